// dt_scorers.cuh -- the factorized scorer arms of the paper's conditioning ladder (
// PAPER.md:553-555): Marg (menus from the base logits alone) and Cond-static (menus corrected once per depth along
// Domino's greedy trajectory, produced by the fused kernel in static mode).  Both share one per-depth menu
// [L][k] of (token, logp) between all nodes of a depth, so the best-first expansion (Alg. 1)
// needs no GRU step: one CTA per request keeps the sorted frontier of dt_fused.cuh and pops B times on its own.
#pragma once
#include "dt_fused.cuh"

namespace dt {

struct ScorerParams {
    ExpandParams e;                 // shapes, candidate tables, outputs
    int32_t *menu_tok;              // [batch, L, k]
    float *menu_lp;                 // [batch, L, k]
};

// Marg menus: per (request, depth) the log-softmax over the top-M slice of base / T_eff (reading A1)
// and its top-k under (logp desc, token asc).  grid = batch * L, block = 256 (M <= 256).
__global__ void __launch_bounds__(256) marg_menu_kernel(ScorerParams p) {
    __shared__ float sZ[256];
    __shared__ int sTok[256];
    __shared__ float sRed[8];
    const ExpandParams &e = p.e;
    const int row = blockIdx.x, tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int M = e.M, k = e.k;
    const float base0 = e.cand_val[(size_t)row * M];
    float z = -INFINITY;
    int tok = 0;
    if (tid < M) {
        z = __fdiv_rn(e.cand_val[(size_t)row * M + tid] - base0, e.T_eff);
        tok = e.cand_id[(size_t)row * M + tid];
        sZ[tid] = z; sTok[tid] = tok;
    }
    float m = warp_max(z);
    if (lane == 0) sRed[warp] = m;
    __syncthreads();
    float zmax = sRed[0];
#pragma unroll
    for (int w = 1; w < 8; ++w) zmax = fmaxf(zmax, sRed[w]);
    __syncthreads();
    float ex = warp_sum((tid < M) ? expf(z - zmax) : 0.f);
    if (lane == 0) sRed[warp] = ex;
    __syncthreads();
    float ssum = 0.f;
#pragma unroll
    for (int w = 0; w < 8; ++w) ssum += sRed[w];
    const float lse = logf(ssum);
    if (tid < M) {
        int rank = 0;
        for (int q = 0; q < M; ++q) {
            const float oz = sZ[q];
            rank += (oz > z) || (oz == z && sTok[q] < tok);
        }
        if (rank < k) {
            p.menu_tok[(size_t)row * k + rank] = tok;
            p.menu_lp[(size_t)row * k + rank] = (z - zmax) - lse;
        }
    }
}

__host__ __device__ inline size_t factorized_smem(int L, int k, int N) {
    auto al = [](size_t x) { return (x + 15) / 16 * 16; };
    return al((size_t)2 * kFusMaxFront * 8) + al((size_t)k * 8) + al((size_t)2 * kFusMaxFront * 4) + al((size_t)k * 4) +
           2 * al((size_t)L * k * 4) + 4 * al((size_t)N * 4) + 64;
}

// Best-first expansion over a per-depth menu + emitter (a9).  grid = batch, block = 256.
__global__ void __launch_bounds__(kFusThreads) factorized_expand_kernel(ScorerParams p) {
    extern __shared__ __align__(16) unsigned char fsm[];
    __shared__ int s_n_valid, s_n_front, s_cur;
    const ExpandParams &e = p.e;
    const int tid = threadIdx.x, b = blockIdx.x;
    const int k = e.k, N = e.N, L = e.L, B = e.B;
    size_t off = 0;
    auto carve = [&](size_t bytes) { unsigned char *q = fsm + off; off += (bytes + 15) / 16 * 16; return q; };
    unsigned long long *fLo = reinterpret_cast<unsigned long long *>(carve((size_t)2 * kFusMaxFront * 8));
    unsigned long long *nLo = reinterpret_cast<unsigned long long *>(carve((size_t)k * 8));
    unsigned int *fHi = reinterpret_cast<unsigned int *>(carve((size_t)2 * kFusMaxFront * 4));
    unsigned int *nHi = reinterpret_cast<unsigned int *>(carve((size_t)k * 4));
    int *mTok = reinterpret_cast<int *>(carve((size_t)L * k * 4));
    float *mLp = reinterpret_cast<float *>(carve((size_t)L * k * 4));
    int *nTok = reinterpret_cast<int *>(carve((size_t)N * 4));
    int *nPar = reinterpret_cast<int *>(carve((size_t)N * 4));
    int *nDep = reinterpret_cast<int *>(carve((size_t)N * 4));
    float *nSco = reinterpret_cast<float *>(carve((size_t)N * 4));

    for (int i = tid; i < L * k; i += kFusThreads) {
        mTok[i] = p.menu_tok[(size_t)b * L * k + i];
        mLp[i] = p.menu_lp[(size_t)b * L * k + i];
    }
    if (tid == 0) {
        nTok[0] = e.root_tokens[b]; nPar[0] = -1; nDep[0] = 0; nSco[0] = 0.f;
        s_n_valid = 1; s_n_front = 0; s_cur = 0;
    }
    __syncthreads();

    for (int t = 0; t < B; ++t) {
        const int n_valid = s_n_valid, n_front = s_n_front, cur = s_cur;
        const bool node_ok = (t < n_valid);
        const int depth = node_ok ? nDep[t] : L;
        const unsigned int *oHi = fHi + cur * kFusMaxFront + 1;            // live frontier = entries 1 .. n_front
        const unsigned long long *oLo = fLo + cur * kFusMaxFront + 1;
        unsigned int *wHi = fHi + (cur ^ 1) * kFusMaxFront;
        unsigned long long *wLo = fLo + (cur ^ 1) * kFusMaxFront;
        int n_new = 0;
        if (node_ok && depth < L) {                                         // children = the shared menu of depth + 1
            if (tid < k) {
                nHi[tid] = ord_key(nSco[t] + mLp[depth * k + tid]);
                nLo[tid] = ((unsigned long long)(0xFFFFFFFFu - (unsigned int)mTok[depth * k + tid]) << 32) |
                           (unsigned long long)(0xFFFFFFFFu - (unsigned int)t);
            }
            n_new = k;
        }
        __syncthreads();
        const int cap = B - t;
        int tot = n_front + n_new;
        if (tot > 0) {
            if (tid < n_front) {
                const unsigned int h = oHi[tid]; const unsigned long long l = oLo[tid];
                int c = 0;
                for (int j = 0; j < n_new; ++j) c += front_gt(nHi[j], nLo[j], h, l);
                const int pos = tid + c;
                if (pos < cap) { wHi[pos] = h; wLo[pos] = l; }
            }
            if (tid >= kFusThreads - n_new) {
                const int j = tid - (kFusThreads - n_new);
                const unsigned int h = nHi[j]; const unsigned long long l = nLo[j];
                int c = 0;
                for (int j2 = 0; j2 < n_new; ++j2) c += front_gt(nHi[j2], nLo[j2], h, l);
                int lo = 0, hi = n_front;
                while (lo < hi) {
                    const int mid = (lo + hi) >> 1;
                    if (front_gt(oHi[mid], oLo[mid], h, l)) lo = mid + 1; else hi = mid;
                }
                const int pos = lo + c;
                if (pos < cap) { wHi[pos] = h; wLo[pos] = l; }
            }
            if (tot > cap) tot = cap;
        }
        __syncthreads();
        if (tid == 0) {
            if (tot > 0) {                                                  // pop entry 0 into slot t + 1
                const unsigned int h = wHi[0]; const unsigned long long l = wLo[0];
                const int par = (int)(0xFFFFFFFFu - (unsigned int)(l & 0xFFFFFFFFull));
                nTok[t + 1] = (int)(0xFFFFFFFFu - (unsigned int)(l >> 32)); nPar[t + 1] = par;
                nDep[t + 1] = nDep[par] + 1; nSco[t + 1] = ord_key_inv(h);
                s_n_valid = t + 2; s_n_front = tot - 1; s_cur = cur ^ 1;
            } else s_n_front = 0;
        }
        __syncthreads();
    }

    // emitter (a9): dead-leaf padding (reading A10), positions, ancestor-or-self mask
    const int n = s_n_valid;
    const int rpos = e.root_positions ? e.root_positions[b] : 0;
    for (int i = tid; i < N; i += kFusThreads) {
        const size_t so = (size_t)b * N + i;
        const bool dead = (i >= n);
        const int dep = dead ? 1 : nDep[i];
        e.tokens[so] = dead ? 0 : nTok[i];
        e.parents[so] = dead ? 0 : nPar[i];
        e.depths[so] = dep;
        e.scores[so] = dead ? -INFINITY : nSco[i];
        e.positions[so] = rpos + dep;
        if (dead) nPar[i] = 0;
    }
    if (tid == 0) e.n_nodes[b] = n;
    uint8_t *mk = e.mask + (size_t)b * N * N;
    for (int i = tid; i < N * N; i += kFusThreads) mk[i] = 0;
    __syncthreads();
    for (int i = tid; i < N; i += kFusThreads) {
        int a = i;
        while (a >= 0) { mk[(size_t)i * N + a] = 1; a = nPar[a]; }
    }
}

}  // namespace dt
