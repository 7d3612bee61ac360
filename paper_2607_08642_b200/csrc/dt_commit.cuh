// dt_commit.cuh -- longest-accepted-path commit over the emitted draft trees:
// PAPER.md:167-169 (Sec. 3.5) "we commit the highest-scoring root-to-leaf path along which every edge is accepted
// (longest-accepted-path)".  One CTA per request, one thread per tree slot: a thread walks its node's root path
// (<= L hops through the parent links staged in shared memory) checking every edge -- greedy verification accepts
// the edge parent u -> node i iff tokens[i] == target_next[u]; otherwise the caller's per-edge
// flags decide -- and the reachable node with the largest (depth, draft score, lower slot) wins a block-wide max
// over one packed 64-bit key.  The winner's path is written root first, padded with -1.
#pragma once
#include "dt_common.cuh"

namespace dt {

struct CommitParams {
    const int32_t *tokens, *parents, *depths, *n_nodes;   // [batch, N] x3, [batch]  (dt_outputs of the build)
    const float *scores;                                   // [batch, N]
    const int32_t *target_next;                            // [batch, N] or nullptr
    const uint8_t *edge_ok;                                // [batch, N] or nullptr
    int32_t *accept_len;                                   // [batch]
    int32_t *path_slots;                                   // [batch, L + 1]
    int32_t *bonus_token;                                  // [batch] or nullptr
    int N, L;
};

__global__ void __launch_bounds__(256) commit_paths_kernel(CommitParams p) {
    __shared__ int sPar[256], sTok[256], sNext[256];
    __shared__ unsigned char sOk[256];
    __shared__ unsigned long long sBest[8];
    const int b = blockIdx.x, tid = threadIdx.x, N = p.N;
    const int n = max(1, min(p.n_nodes[b], N));              // the root always is a node
    const size_t base = (size_t)b * N;
    if (tid < N) {
        sPar[tid] = p.parents[base + tid];
        sTok[tid] = p.tokens[base + tid];
        sNext[tid] = p.target_next ? p.target_next[base + tid] : 0;
        sOk[tid] = p.edge_ok ? p.edge_ok[base + tid] : 0;
    }
    __syncthreads();
    unsigned long long key = 0ull;                         // 0 = not reachable
    if (tid < n) {
        bool ok = true;
        int u = tid;
        for (int hop = 0; hop <= p.L && u != 0; ++hop) {   // every edge of the root path must be accepted
            const int par = sPar[u];
            if (par < 0 || par >= n) { ok = false; break; }
            const bool acc = p.target_next ? (sTok[u] == sNext[par]) : (sOk[u] != 0);
            if (!acc) { ok = false; break; }
            u = par;
        }
        if (ok && u == 0) {
            const unsigned int dep = (unsigned int)p.depths[base + tid];
            key = ((unsigned long long)(dep + 1u) << 48) | ((unsigned long long)ord_key(p.scores[base + tid]) << 16) |
                  (unsigned long long)(0xFFFFu - (unsigned int)tid);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const unsigned long long other = __shfl_xor_sync(0xffffffffu, key, o);
        key = other > key ? other : key;
    }
    if ((tid & 31) == 0) sBest[tid >> 5] = key;
    __syncthreads();
    if (tid == 0) {
        unsigned long long best = sBest[0];
        for (int w = 1; w < 8; ++w) best = sBest[w] > best ? sBest[w] : best;
        const int end = (int)(0xFFFFu - (unsigned int)(best & 0xFFFFull));       // the root always qualifies
        const int len = (int)(best >> 48) - 1;
        p.accept_len[b] = len;
        int32_t *path = p.path_slots + (size_t)b * (p.L + 1);
        for (int i = len + 1; i <= p.L; ++i) path[i] = -1;
        int u = end;
        for (int i = len; i >= 0; --i) { path[i] = u; u = (u == 0) ? 0 : sPar[u]; }
        if (p.bonus_token) p.bonus_token[b] = p.target_next ? sNext[end] : -1;
    }
}

// First-child / next-sibling link arrays for tree-verify kernels that walk the tree instead of reading the mask
// (PAPER.md:169, 187): first_child[i] = smallest slot j > i with parents[j] == i, next_sibling[i] = smallest slot
// j > i with parents[j] == parents[i]; -1 where there is none, for the root's sibling and for dead-leaf padding slots.
// One CTA per request, one thread per slot, the parent links staged in shared memory.
__global__ void __launch_bounds__(256) tree_links_kernel(const int32_t *parents, const int32_t *n_nodes, int N,
                                                         int32_t *first_child, int32_t *next_sibling) {
    __shared__ int sPar[256];
    const int b = blockIdx.x, i = threadIdx.x;
    const int n = max(1, min(n_nodes[b], N));
    const size_t base = (size_t)b * N;
    if (i < N) sPar[i] = parents[base + i];
    __syncthreads();
    if (i >= N) return;
    int fc = -1, ns = -1;
    if (i < n) {
        const int par = sPar[i];
        for (int j = i + 1; j < n; ++j) {
            const int pj = sPar[j];
            if (fc < 0 && pj == i) fc = j;
            if (ns < 0 && i > 0 && pj == par) ns = j;
            if (fc >= 0 && (ns >= 0 || i == 0)) break;
        }
    }
    first_child[base + i] = fc;
    next_sibling[base + i] = ns;
}

}  // namespace dt
