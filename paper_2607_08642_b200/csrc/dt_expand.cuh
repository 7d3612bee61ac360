// dt_expand.cuh -- steps (a5)-(a9): the best-first expansion (Alg. 1 steps 3-5).
//
// Lock-step schedule: step t processes, for every request of the batch at once, the node that
// request popped t-th (slot t; slot 0 is the root).  Per step:
//   gru_step_kernel   S[b,t] = GRUcell(S[b,parent], E[token])  (reading A2),
//                     input half read from the P table, hidden half W_hh S computed here;
//                     grid over GRU units so each W_hh row is read once per step for the whole batch.
//   expand_kernel     CHILDREN(S[b,t], depth+1): a = SiLU(C + W1s S),
//                     z_m = (base_m + W2[cand_m,:] a)/T_eff, slice log-softmax (reading A1),
//                     top-k by (logp desc, token asc); push k entries; pop the heap maximum under
//                     (g desc, token asc, parent asc) (reading A8) into slot t+1.
// The child's GRU state is evaluated when the child is popped (a pure function of parent state
// and token, so identical to Alg. 1's eager advance at PAPER.md:144).
#pragma once
#include "dt_common.cuh"

namespace dt {

constexpr int kExpThreads = 256;
constexpr int kGruUnitsPerCta = 8;   // one warp per GRU unit (3 gate rows)

struct ExpandParams {
    // weights
    const void *w_hh;      // [3g, g]
    const void *w1;        // [r, d+g]
    const void *w2;        // [V, r]
    const float *P;        // [V, 3g]
    int V, d, g, r;
    // round state
    int batch, L, M, B, k, N;       // N = B+1
    float inv_unused, T_eff;
    const float *C;        // [batch*L, r]
    const int32_t *cand_id;   // [batch*L, M]
    const float *cand_val;    // [batch*L, M]
    float *states;         // [batch, N, g]
    float *heap_g;         // [batch, heap_cap]
    unsigned long long *heap_tp;   // [batch, heap_cap]  token << 32 | parent
    int32_t *heap_cnt;     // [batch]
    int heap_cap;
    // outputs (also the running tree)
    int32_t *tokens, *parents, *depths, *positions, *n_nodes;
    float *scores;
    uint8_t *mask;
    const int32_t *root_tokens, *root_positions;
};

// dot(w[0..n), s[0..n)) with w of type T (global) and s fp32; whole warp cooperates, result on all lanes.
template <typename T>
__device__ __forceinline__ float warp_dot(const T *__restrict__ w, const float *__restrict__ s, int n, int lane) {
    constexpr int kVec = ElemTraits<T>::kVec;
    float acc = 0.f;
    const bool aligned = ((reinterpret_cast<uintptr_t>(w) & 15u) == 0);
    int n_vec = aligned ? (n / kVec) : 0;
    for (int v = lane; v < n_vec; v += 32) {
        uint4 q = ld_ro_v4(w + (size_t)v * kVec);
        const float *sp = s + (size_t)v * kVec;
        if (sizeof(T) == 2) {
            float f[8];
            unpack8(q, f);
#pragma unroll
            for (int i = 0; i < 8; ++i) acc = fmaf(f[i], sp[i], acc);
        } else {
            acc = fmaf(__uint_as_float(q.x), sp[0], acc);
            acc = fmaf(__uint_as_float(q.y), sp[1], acc);
            acc = fmaf(__uint_as_float(q.z), sp[2], acc);
            acc = fmaf(__uint_as_float(q.w), sp[3], acc);
        }
    }
    for (int i = n_vec * kVec + lane; i < n; i += 32) acc = fmaf(ldf(w, (size_t)i), s[i], acc);
    return warp_sum(acc);
}

// Initialise slot 0 and the heap of every request.  grid = batch.
__global__ void init_round_kernel(ExpandParams p) {
    const int b = blockIdx.x;
    if (threadIdx.x == 0) {
        p.tokens[(size_t)b * p.N] = p.root_tokens[b];
        p.parents[(size_t)b * p.N] = -1;
        p.depths[(size_t)b * p.N] = 0;
        p.scores[(size_t)b * p.N] = 0.f;
        p.n_nodes[b] = 1;
        p.heap_cnt[b] = 0;
    }
}

// Hidden half of the GRU cell for slot t of every request.  grid = ceil(g / 8), block = 256.
template <typename T>
__global__ void __launch_bounds__(kExpThreads) gru_step_kernel(ExpandParams p, int t) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int u = blockIdx.x * kGruUnitsPerCta + warp;
    const int g = p.g;
    if (u >= g) return;
    const T *whh = reinterpret_cast<const T *>(p.w_hh);
    const T *wr = whh + (size_t)u * g, *wz = whh + (size_t)(g + u) * g, *wn = whh + (size_t)(2 * g + u) * g;
    for (int b = 0; b < p.batch; ++b) {
        if (t >= p.n_nodes[b]) continue;                        // request exhausted its candidate tree
        const size_t so = (size_t)b * p.N + t;
        if (p.depths[so] >= p.L) continue;                      // never expanded: state not needed
        const int tok = p.tokens[so], par = p.parents[so];
        const float *Sp = p.states + ((size_t)b * p.N + par) * g;
        float hr = warp_dot(wr, Sp, g, lane);
        float hz = warp_dot(wz, Sp, g, lane);
        float hn = warp_dot(wn, Sp, g, lane);
        if (lane == 0) {
            const float *pr = p.P + (size_t)tok * 3 * g;
            float rg = sigmoidf_acc(pr[u] + hr);
            float zg = sigmoidf_acc(pr[g + u] + hz);
            float ng = tanhf(pr[2 * g + u] + rg * hn);
            p.states[((size_t)b * p.N + t) * g + u] = (1.0f - zg) * ng + zg * Sp[u];
        }
    }
}

struct ExpandSmem {
    float red[8];
    float redk[8];
    unsigned long long redtp[8];
    int redi[8];
    float zmax, lse;
    int pop_idx;
};

// CHILDREN + push + pop for slot t.  grid = batch, block = 256.  Dynamic smem: g + r + 2*M floats + M ints.
template <typename T>
__global__ void __launch_bounds__(kExpThreads) expand_kernel(ExpandParams p, int t) {
    extern __shared__ float dsm[];
    __shared__ ExpandSmem sm;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int b = blockIdx.x;
    const int g = p.g, r = p.r, M = p.M, k = p.k, N = p.N;
    float *sS = dsm;                // [g]
    float *sA = sS + g;             // [r]
    float *sZ = sA + r;             // [M]  z, then logp
    int *sTok = reinterpret_cast<int *>(sZ + M);   // [M]

    const int n_valid = p.n_nodes[b];
    const bool node_ok = (t < n_valid);
    const int depth = node_ok ? p.depths[(size_t)b * N + t] : p.L;
    float *hg = p.heap_g + (size_t)b * p.heap_cap;
    unsigned long long *htp = p.heap_tp + (size_t)b * p.heap_cap;
    int cnt = p.heap_cnt[b];

    if (node_ok && depth < p.L) {               // block-uniform
        const float *S = p.states + ((size_t)b * N + t) * g;
        for (int i = tid; i < g; i += kExpThreads) sS[i] = S[i];
        const size_t row = (size_t)b * p.L + depth;            // H_{depth+1} <-> row index depth (A12)
        for (int m = tid; m < M; m += kExpThreads) sTok[m] = p.cand_id[row * M + m];
        __syncthreads();
        // a = SiLU(C + W1[:, d:d+g] S)
        const T *w1 = reinterpret_cast<const T *>(p.w1);
        for (int j = warp; j < r; j += kExpThreads / 32) {
            float acc = warp_dot(w1 + (size_t)j * (p.d + g) + p.d, sS, g, lane);
            if (lane == 0) {
                float x = p.C[row * r + j] + acc;
                sA[j] = x * sigmoidf_acc(x);
            }
        }
        __syncthreads();
        // z_m = ((base_m - base_0) + W2[cand_m, :] a) / T_eff     PAPER.md:143-144 (shift-invariant)
        const T *w2 = reinterpret_cast<const T *>(p.w2);
        const float base0 = p.cand_val[row * M];
        for (int m = warp; m < M; m += kExpThreads / 32) {
            float acc = warp_dot(w2 + (size_t)sTok[m] * r, sA, r, lane);
            if (lane == 0) sZ[m] = __fdiv_rn((p.cand_val[row * M + m] - base0) + acc, p.T_eff);
        }
        __syncthreads();
        // slice log-softmax (reading A1): one candidate per thread (M <= 256)
        float z = (tid < M) ? sZ[tid] : -INFINITY;
        float wm = warp_max(z);
        if (lane == 0) sm.red[warp] = wm;
        __syncthreads();
        if (tid == 0) { float m = sm.red[0]; for (int i = 1; i < 8; ++i) m = fmaxf(m, sm.red[i]); sm.zmax = m; }
        __syncthreads();
        const float zmax = sm.zmax;
        float e = (tid < M) ? expf(z - zmax) : 0.f;
        float ws = warp_sum(e);
        if (lane == 0) sm.redk[warp] = ws;
        __syncthreads();
        if (tid == 0) { float s = 0.f; for (int i = 0; i < 8; ++i) s += sm.redk[i]; sm.lse = logf(s); }
        __syncthreads();
        const float lp = (z - zmax) - sm.lse;
        if (tid < M) sZ[tid] = lp;
        __syncthreads();
        // top-k by (logp desc, token asc): rank by counting
        if (tid < M) {
            const int mytok = sTok[tid];
            int rank = 0;
            for (int m = 0; m < M; ++m) {
                float o = sZ[m];
                rank += (o > lp) || (o == lp && sTok[m] < mytok);
            }
            if (rank < k) {
                hg[cnt + rank] = p.scores[(size_t)b * N + t] + lp;
                htp[cnt + rank] = ((unsigned long long)(unsigned int)mytok << 32) | (unsigned int)t;
            }
        }
        cnt += k;
        __syncthreads();
    }

    // pop the maximum under (g desc, token asc, parent asc) into slot t+1
    if (cnt == 0 || t + 1 > p.B) {
        if (tid == 0) p.heap_cnt[b] = cnt;
        return;
    }
    float bg = -INFINITY; unsigned long long btp = ~0ull; int bi = -1;
    for (int i = tid; i < cnt; i += kExpThreads) {
        float gi = hg[i]; unsigned long long tp = htp[i];
        if (bi < 0 || gi > bg || (gi == bg && tp < btp)) { bg = gi; btp = tp; bi = i; }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        float og = __shfl_xor_sync(0xffffffffu, bg, o);
        unsigned long long otp = __shfl_xor_sync(0xffffffffu, btp, o);
        int oi = __shfl_xor_sync(0xffffffffu, bi, o);
        if (oi >= 0 && (bi < 0 || og > bg || (og == bg && otp < btp))) { bg = og; btp = otp; bi = oi; }
    }
    if (lane == 0) { sm.redk[warp] = bg; sm.redtp[warp] = btp; sm.redi[warp] = bi; }
    __syncthreads();
    if (tid == 0) {
        for (int w = 0; w < kExpThreads / 32; ++w) {
            float og = sm.redk[w]; unsigned long long otp = sm.redtp[w]; int oi = sm.redi[w];
            if (oi >= 0 && (bi < 0 || og > bg || (og == bg && otp < btp))) { bg = og; btp = otp; bi = oi; }
        }
        const int par = (int)(btp & 0xFFFFFFFFull);
        const size_t so = (size_t)b * N + t + 1;
        p.tokens[so] = (int)(btp >> 32);
        p.parents[so] = par;
        p.depths[so] = p.depths[(size_t)b * N + par] + 1;
        p.scores[so] = bg;
        p.n_nodes[b] = t + 2;
        hg[bi] = hg[cnt - 1];
        htp[bi] = htp[cnt - 1];
        p.heap_cnt[b] = cnt - 1;
    }
}

// Emitter (a9): dead-leaf padding (reading A10), positions, ancestor-or-self mask.
// grid = batch, block = 256 (N <= 256).
__global__ void __launch_bounds__(kExpThreads) emit_kernel(ExpandParams p) {
    const int b = blockIdx.x, tid = threadIdx.x, N = p.N;
    __shared__ int sPar[256];
    const int n = p.n_nodes[b];
    const int rpos = p.root_positions ? p.root_positions[b] : 0;
    if (tid < N) {
        const size_t so = (size_t)b * N + tid;
        if (tid >= n) { p.tokens[so] = 0; p.parents[so] = 0; p.depths[so] = 1; p.scores[so] = -INFINITY; }
        sPar[tid] = p.parents[so];
        p.positions[so] = rpos + p.depths[so];
    }
    uint8_t *mk = p.mask + (size_t)b * N * N;
    for (int i = tid; i < N * N; i += kExpThreads) mk[i] = 0;
    __syncthreads();
    if (tid < N) {
        int a = tid;
        while (a >= 0) { mk[(size_t)tid * N + a] = 1; a = sPar[a]; }
    }
}

}  // namespace dt
