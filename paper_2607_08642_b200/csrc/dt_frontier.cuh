// dt_frontier.cuh -- the depth-synchronous frontier builder, the paper's serving schedule
// (Appendix B 524-528): instead of popping one node at a time, advance a frontier of W lanes per
// request in lockstep across depth; at each depth score the k children of every lane (the same CHILDREN of
// PAPER.md:142-144), write every scored candidate to a ledger [batch, L, W k] with its cumulative log-score and a
// pointer to its parent, keep the top W as the next frontier and advance the GRU state only for those; after L
// depths take the global top-B of the ledger, order parents first, remap the parent pointers, pad with dead leaves
// and emit.  With W = B it selects the same nodes as the heap (scores are monotone along a path, so
// fewer than B candidates at a depth can outscore a top-B node and none is evicted before its children are scored).
//
// This is the alternative SCHEDULE behind the same ABI (dt_set_option "schedule" = 1), fixed-shape and capture-safe
// like the paper's (L + 1 launches, no host synchronisation).  It is a correctness-first implementation: one CTA per
// request walks its lanes with warp-FMA matvecs (weights streamed from L2); at batch 32 x W = 32 its per-depth GEMM
// would have 2048 columns on the tensor cores, which does not beat the heap schedule on B200.
#pragma once
#include "dt_expand.cuh"

namespace dt {

struct FrontierParams {
    ExpandParams e;                 // weights, shapes, candidate tables, outputs (e.B = budget, W = e.B)
    int W;                          // lanes per request
    float *fstate;                  // [2, batch, W, g] ping-pong lane states
    int32_t *led_tok, *led_par;     // [batch, L, W k]  token; ledger index of the parent (-1 = root)
    float *led_g;                   // [batch, L, W k]  cumulative log-score
    int32_t *fr_ref;                // [2, batch, W]    ledger index of each frontier lane (-1 = root)
    int32_t *fr_plane;              // [2, batch, W]    lane of its parent in the previous frontier
    int32_t *n_fr;                  // [2, batch]       lanes in the frontier
    int32_t *led_cnt;               // [batch, L]       entries written at each depth
    int32_t *led_slot;              // [batch, L, W k]  tree slot of a selected entry, -1 otherwise
};

constexpr int kFrLanes = 4;          // frontier lanes advanced together in the GRU phase

// key order of the heap (reading A8): larger pops first
__device__ __forceinline__ bool led_before(float ga, int ta, int pa, float gb, int tb, int pb) {
    return ga > gb || (ga == gb && (ta < tb || (ta == tb && pa < pb)));
}

// One depth for one request: states of the frontier lanes, CHILDREN of every lane into the ledger, next frontier.
// grid = batch, block = 256, dynamic smem = (g + r + 2 M + kFrLanes g) floats + M ints.
template <typename T>
__global__ void __launch_bounds__(kExpThreads) frontier_depth_kernel(FrontierParams p, int d) {
    extern __shared__ float fsm_[];
    __shared__ float s_red[8];
    __shared__ float s_zmax, s_lse;
    const ExpandParams &e = p.e;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, b = blockIdx.x;
    const int g = e.g, r = e.r, M = e.M, k = e.k, L = e.L, W = p.W;
    float *sS = fsm_, *sA = sS + g, *sZ = sA + r, *sLp = sZ + M;
    int *sTok = reinterpret_cast<int *>(sLp + M);
    float *sSp = reinterpret_cast<float *>(sTok + M);           // [kFrLanes][g] parent states of one lane group
    const int cur = d & 1, nxt = cur ^ 1;
    const size_t WK = (size_t)W * k;
    const int nl = (d == 0) ? 1 : p.n_fr[(size_t)cur * e.batch + b];
    const size_t row = (size_t)b * L + d;                       // H_{d+1} pairs with the parent state (A12)
    int32_t *ltok = p.led_tok + ((size_t)b * L + d) * WK, *lpar = p.led_par + ((size_t)b * L + d) * WK;
    float *lg = p.led_g + ((size_t)b * L + d) * WK;
    const T *whh = reinterpret_cast<const T *>(e.w_hh), *w1 = reinterpret_cast<const T *>(e.w1), *w2 = reinterpret_cast<const T *>(e.w2);
    for (int m = tid; m < M; m += kExpThreads) sTok[m] = e.cand_id[row * M + m];
    const float base0 = e.cand_val[row * M];

    // (1) lane states, kFrLanes lanes at a time so that every W_hh row is read once per group, not once per lane:
    //     root S_0 = GRUcell(0, E[root]) (A4), else GRUcell(S_parent-lane, E[token])
    for (int l0 = 0; l0 < nl; l0 += kFrLanes) {
        const int ng = min(kFrLanes, nl - l0);
        __syncthreads();
        for (int i = tid; i < ng * g; i += kExpThreads) {
            const int q = i / g, u = i - q * g;
            float v = 0.f;
            if (d > 0) v = p.fstate[(((size_t)nxt * e.batch + b) * W + p.fr_plane[((size_t)cur * e.batch + b) * W + l0 + q]) * g + u];
            sSp[q * g + u] = v;
        }
        __syncthreads();
        for (int u = warp; u < g; u += kExpThreads / 32) {
            float acc[3][kFrLanes];
#pragma unroll
            for (int gt = 0; gt < 3; ++gt)
#pragma unroll
                for (int q = 0; q < kFrLanes; ++q) acc[gt][q] = 0.f;
            if (d > 0) {
                for (int i = lane; i < g; i += 32) {
#pragma unroll
                    for (int gt = 0; gt < 3; ++gt) {
                        const float wv = ldf(whh, ((size_t)gt * g + u) * g + i);
#pragma unroll
                        for (int q = 0; q < kFrLanes; ++q) acc[gt][q] = fmaf(wv, sSp[q * g + i], acc[gt][q]);
                    }
                }
#pragma unroll
                for (int gt = 0; gt < 3; ++gt)
#pragma unroll
                    for (int q = 0; q < kFrLanes; ++q) acc[gt][q] = warp_sum(acc[gt][q]);
            }
            if (lane < ng) {                                   // lane q finishes unit u of frontier lane l0 + q
                float hr = 0.f, hz = 0.f, hn = 0.f;
#pragma unroll
                for (int q = 0; q < kFrLanes; ++q) if (q == lane) { hr = acc[0][q]; hz = acc[1][q]; hn = acc[2][q]; }
                int tok;
                if (d == 0) tok = min(max(e.root_tokens[b], 0), e.V - 1);
                else tok = p.led_tok[((size_t)b * L + (d - 1)) * WK + p.fr_ref[((size_t)cur * e.batch + b) * W + l0 + lane]];
                const float *pr = e.P + (size_t)tok * 3 * g;
                const float rg = sigmoidf_acc(pr[u] + hr), zg = sigmoidf_acc(pr[g + u] + hz);
                const float ng2 = tanhf(pr[2 * g + u] + rg * hn);
                p.fstate[(((size_t)cur * e.batch + b) * W + l0 + lane) * g + u] = (1.0f - zg) * ng2 + zg * sSp[lane * g + u];
            }
        }
    }
    __threadfence_block();
    __syncthreads();

    for (int l = 0; l < nl; ++l) {
        const int ref = (d == 0) ? -1 : p.fr_ref[((size_t)cur * e.batch + b) * W + l];
        const float gpar = (d == 0) ? 0.f : p.led_g[((size_t)b * L + (d - 1)) * WK + ref];
        const float *Sn = p.fstate + (((size_t)cur * e.batch + b) * W + l) * g;
        __syncthreads();
        for (int u = tid; u < g; u += kExpThreads) sS[u] = Sn[u];
        __syncthreads();
        // (2) a = SiLU(C + W1[:, d:] S)
        for (int j = warp; j < r; j += kExpThreads / 32) {
            const float acc = warp_dot(w1 + (size_t)j * (e.d + g) + e.d, sS, g, lane);
            if (lane == 0) { const float x = e.C[row * r + j] + acc; sA[j] = x * sigmoidf_acc(x); }
        }
        __syncthreads();
        // (3) z, slice log-softmax (A1), top-k into the ledger
        for (int m = warp; m < M; m += kExpThreads / 32) {
            const float acc = warp_dot(w2 + (size_t)sTok[m] * r, sA, r, lane);
            if (lane == 0) sZ[m] = __fdiv_rn((e.cand_val[row * M + m] - base0) + acc, e.T_eff);
        }
        __syncthreads();
        float z = (tid < M) ? sZ[tid] : -INFINITY;
        float wm = warp_max(z);
        if (lane == 0) s_red[warp] = wm;
        __syncthreads();
        if (tid == 0) { float mx = s_red[0]; for (int i = 1; i < 8; ++i) mx = fmaxf(mx, s_red[i]); s_zmax = mx; }
        __syncthreads();
        float ex = warp_sum((tid < M) ? expf(z - s_zmax) : 0.f);
        if (lane == 0) s_red[warp] = ex;
        __syncthreads();
        if (tid == 0) { float sum = 0.f; for (int i = 0; i < 8; ++i) sum += s_red[i]; s_lse = logf(sum); }
        __syncthreads();
        if (tid < M) {
            const float lp = (z - s_zmax) - s_lse;
            sLp[tid] = lp;
        }
        __syncthreads();
        if (tid < M) {
            const float lp = sLp[tid];
            const int mytok = sTok[tid];
            int rank = 0;
            for (int m = 0; m < M; ++m) { const float o = sLp[m]; rank += (o > lp) || (o == lp && sTok[m] < mytok); }
            if (rank < k) {
                ltok[(size_t)l * k + rank] = mytok;
                lpar[(size_t)l * k + rank] = ref;
                lg[(size_t)l * k + rank] = gpar + lp;
                p.led_slot[((size_t)b * L + d) * WK + (size_t)l * k + rank] = -1;
            }
        }
        __syncthreads();
    }
    if (tid == 0) p.led_cnt[(size_t)b * L + d] = nl * k;
    // (4) next frontier: the top W of the nl k entries just written (only needed when another depth follows)
    if (d + 1 < L) {
        __threadfence_block();
        __syncthreads();
        const int ne = nl * k;
        for (int i = tid; i < ne; i += kExpThreads) {
            const float gi = lg[i]; const int ti = ltok[i], pi = lpar[i];
            int rank = 0;
            for (int j = 0; j < ne; ++j) rank += (j != i) && led_before(lg[j], ltok[j], lpar[j], gi, ti, pi);
            if (rank < W) {
                p.fr_ref[((size_t)nxt * e.batch + b) * W + rank] = i;
                p.fr_plane[((size_t)nxt * e.batch + b) * W + rank] = i / k;
            }
        }
        if (tid == 0) p.n_fr[(size_t)nxt * e.batch + b] = min(ne, W);
    }
}

// Selection + emitter: the global top-B of the ledger in heap order (g desc, then depth asc so that a parent always
// precedes a child of equal score, token asc, ledger index asc), B rounds of a block-wide arg-max; parents are
// remapped through led_slot; dead-leaf padding, positions and the ancestor mask as in reading A10.
// grid = batch, block = 256, dynamic smem = 4 N ints.
__global__ void __launch_bounds__(kExpThreads) frontier_finalize_kernel(FrontierParams p) {
    extern __shared__ int fin_sm[];
    __shared__ float s_g[8];
    __shared__ unsigned long long s_k[8];
    __shared__ float s_bg; __shared__ unsigned long long s_bk;
    const ExpandParams &e = p.e;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, b = blockIdx.x;
    const int L = e.L, N = e.N, B = e.B;
    const size_t WK = (size_t)p.W * e.k;
    int *nTok = fin_sm, *nPar = nTok + N, *nDep = nPar + N;
    float *nSco = reinterpret_cast<float *>(nDep + N);
    if (tid == 0) { nTok[0] = e.root_tokens[b]; nPar[0] = -1; nDep[0] = 0; nSco[0] = 0.f; }
    int n = 1;
    for (int s = 1; s <= B; ++s) {
        // arg-max over the entries not taken yet; tie key: smaller is better = depth << 56 | token << 24 | index
        float bg = -INFINITY; unsigned long long bk = ~0ull;
        for (int d = 0; d < L; ++d) {
            const int cnt = p.led_cnt[(size_t)b * L + d];
            const size_t o = ((size_t)b * L + d) * WK;
            for (int i = tid; i < cnt; i += kExpThreads) {
                if (p.led_slot[o + i] >= 0) continue;
                const float gi = p.led_g[o + i];
                const unsigned long long ki = ((unsigned long long)d << 56) | ((unsigned long long)(unsigned int)p.led_tok[o + i] << 24) |
                                              (unsigned long long)(unsigned int)i;
                if (gi > bg || (gi == bg && ki < bk)) { bg = gi; bk = ki; }
            }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const float og = __shfl_xor_sync(0xffffffffu, bg, o);
            const unsigned long long ok = __shfl_xor_sync(0xffffffffu, bk, o);
            if (og > bg || (og == bg && ok < bk)) { bg = og; bk = ok; }
        }
        if (lane == 0) { s_g[warp] = bg; s_k[warp] = bk; }
        __syncthreads();
        if (tid == 0) {
            for (int w = 1; w < 8; ++w) if (s_g[w] > bg || (s_g[w] == bg && s_k[w] < bk)) { bg = s_g[w]; bk = s_k[w]; }
            s_bg = bg; s_bk = bk;
            if (bk != ~0ull) {
                const int d = (int)(bk >> 56), i = (int)(bk & 0xFFFFFFull);
                const size_t o = ((size_t)b * L + d) * WK;
                const int par = p.led_par[o + i];
                nTok[s] = p.led_tok[o + i]; nDep[s] = d + 1; nSco[s] = bg;
                nPar[s] = (par < 0) ? 0 : p.led_slot[((size_t)b * L + (d - 1)) * WK + par];
                p.led_slot[o + i] = s;
            }
        }
        __syncthreads();
        if (s_bk == ~0ull) break;                              // ledger exhausted (short tree)
        n = s + 1;
        __threadfence_block();
    }
    __syncthreads();
    const int rpos = e.root_positions ? e.root_positions[b] : 0;
    for (int i = tid; i < N; i += kExpThreads) {
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
    for (int i = tid; i < N * N; i += kExpThreads) mk[i] = 0;
    __syncthreads();
    for (int i = tid; i < N; i += kExpThreads) {
        int a = i;
        while (a >= 0) { mk[(size_t)i * N + a] = 1; a = nPar[a]; }
    }
}

}  // namespace dt
