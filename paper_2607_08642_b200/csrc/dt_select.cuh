// dt_select.cuh -- step (a1): exact top-M select per logits row (Alg. 1 step 1).
//
// One streaming pass over the row (every logit is read from HBM exactly once), HBM-bound.
// A CTA owns one chunk of one row.  Per 16-byte vector the fast path is: packed max of the
// vector, packed compare against a threshold tau, fold into the thread's running maxima.  Only
// vectors holding an element >= tau take the slow path, which pushes 64-bit keys
// (ordered value << 32 | ~token) into a shared-memory candidate buffer.
//
// tau is always a PROVEN lower bound on the row's M-th largest value: each thread keeps two
// running maxima over disjoint element subsets (512 per CTA), so the M-th largest of those 512
// maxima has at least M distinct elements at or above it.  It is re-derived at tiles 1,2,4,8,..
// (it tightens like 1/t) by an 8-bit radix select over the 512 maxima, and shared between the
// chunks of one row through an atomicMax word.  Nothing is ever dropped that could be in the
// top M, so the result is exact; ties on the value are resolved by the key (token id asc).
//
// Overflow of the candidate buffer (adversarial rows: ascending, all-equal): a push that finds the
// buffer full stores nothing and is remembered in a per-thread bit mask; the CTA then compacts the
// buffer to the exact top-M so far (bitonic sort, which also yields an exact 64-bit key bound) and
// re-pushes only the remembered elements from registers, one vector per sub-step.
#pragma once
#include "dt_common.cuh"

namespace dt {

constexpr int kSelThreads = 256;
constexpr int kSelU = 4;            // 16-byte vectors per thread per tile
constexpr int kSelCap = 4096;       // candidate buffer capacity (u64 keys), power of two
constexpr int kSelSub = 2 * kSelThreads;   // running maxima per CTA
constexpr int kSelMaxChunks = 32;   // chunks per row; S * M <= kSelCap must hold

struct SelectParams {
    const void *logits;             // [rows, V]
    int rows, V, M, S;              // S = chunks per row
    int row_vecs;                   // ceil(V / kVec)
    int chunk_vecs;                 // ceil(row_vecs / S)
    int32_t *cand_id;               // [rows, M]
    float *cand_val;                // [rows, M]
    unsigned long long *part;       // [rows, S, M] per-chunk sorted keys (S > 1)
    unsigned int *row_counter;      // [rows] arrival tickets, self-resetting
    unsigned int *row_tau;          // [rows] shared lower bound (ordered key), self-resetting
};

template <typename T> struct SelOps;

template <> struct SelOps<__nv_bfloat16> {
    using Run = __nv_bfloat162;
    static __device__ __forceinline__ Run from_bits(uint32_t b) { return *reinterpret_cast<Run *>(&b); }
    static __device__ __forceinline__ uint32_t bits(Run r) { return *reinterpret_cast<uint32_t *>(&r); }
    static __device__ __forceinline__ Run lowest() { return from_bits(0xFF80FF80u); }
    static __device__ __forceinline__ uint4 lowest_vec() { return make_uint4(0xFF80FF80u, 0xFF80FF80u, 0xFF80FF80u, 0xFF80FF80u); }
    static __device__ __forceinline__ Run vmax(const uint4 &v) {
        return __hmax2(__hmax2(from_bits(v.x), from_bits(v.y)), __hmax2(from_bits(v.z), from_bits(v.w)));
    }
    static __device__ __forceinline__ Run rmax(Run a, Run b) { return __hmax2(a, b); }
    static __device__ __forceinline__ bool pass(Run m, Run tau) { return !__hblt2(m, tau); }
    static __device__ __forceinline__ Run make_tau(uint32_t tau_ord) {
        uint32_t b = __float_as_uint(ord_key_inv(tau_ord)) >> 16;
        return from_bits(b | (b << 16));
    }
    static __device__ __forceinline__ void sub_keys(Run r, uint32_t &k0, uint32_t &k1) {
        uint32_t b = bits(r);
        k0 = ord_key(__uint_as_float(b << 16));
        k1 = ord_key(__uint_as_float(b & 0xFFFF0000u));
    }
    static __device__ __forceinline__ void elems(const uint4 &v, float (&f)[8]) { unpack8(v, f); }
    static __device__ __forceinline__ uint4 load_scalar(const __nv_bfloat16 *row, long long e0, int V) {
        uint32_t w[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            uint32_t lo = 0xFF80u, hi = 0xFF80u;
            if (e0 + 2 * i < V) lo = *reinterpret_cast<const unsigned short *>(row + e0 + 2 * i);
            if (e0 + 2 * i + 1 < V) hi = *reinterpret_cast<const unsigned short *>(row + e0 + 2 * i + 1);
            w[i] = lo | (hi << 16);
        }
        return make_uint4(w[0], w[1], w[2], w[3]);
    }
};

template <> struct SelOps<float> {
    struct Run { float a, b; };
    static __device__ __forceinline__ Run lowest() { return Run{-INFINITY, -INFINITY}; }
    static __device__ __forceinline__ uint4 lowest_vec() { return make_uint4(0xFF800000u, 0xFF800000u, 0xFF800000u, 0xFF800000u); }
    static __device__ __forceinline__ Run vmax(const uint4 &v) {
        return Run{fmaxf(__uint_as_float(v.x), __uint_as_float(v.z)), fmaxf(__uint_as_float(v.y), __uint_as_float(v.w))};
    }
    static __device__ __forceinline__ Run rmax(Run x, Run y) { return Run{fmaxf(x.a, y.a), fmaxf(x.b, y.b)}; }
    static __device__ __forceinline__ bool pass(Run m, Run tau) { return !(m.a < tau.a && m.b < tau.a); }
    static __device__ __forceinline__ Run make_tau(uint32_t tau_ord) { float f = ord_key_inv(tau_ord); return Run{f, f}; }
    static __device__ __forceinline__ void sub_keys(Run r, uint32_t &k0, uint32_t &k1) { k0 = ord_key(r.a); k1 = ord_key(r.b); }
    static __device__ __forceinline__ void elems(const uint4 &v, float (&f)[4]) {
        f[0] = __uint_as_float(v.x); f[1] = __uint_as_float(v.y); f[2] = __uint_as_float(v.z); f[3] = __uint_as_float(v.w);
    }
    static __device__ __forceinline__ uint4 load_scalar(const float *row, long long e0, int V) {
        uint32_t w[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) w[i] = (e0 + i < V) ? __float_as_uint(row[e0 + i]) : 0xFF800000u;
        return make_uint4(w[0], w[1], w[2], w[3]);
    }
};

struct SelectSmem {
    unsigned long long cand[kSelCap];
    unsigned int sub[kSelSub];
    unsigned int hist[256];
    unsigned long long tau_key;     // exact 64-bit bound after a compaction (0 = none)
    unsigned int cnt;
    unsigned int cnt2;
    unsigned int sel_bin, sel_rem;
    unsigned int bcast;
    unsigned int is_last;
};

// K-th largest (1-based) of n_keys 32-bit keys in smem; all kSelThreads threads call.  NPASS 8-bit
// radix passes from the top (2 suffice when the low 16 bits of every key are zero).
template <int NPASS>
__device__ __forceinline__ unsigned int block_select_kth(SelectSmem &sm, const unsigned int *keys, int n_keys, unsigned int K) {
    const int tid = threadIdx.x;
    unsigned int prefix = 0, mask = 0, rem = K;
#pragma unroll 1
    for (int p = 0; p < NPASS; ++p) {
        const int shift = 24 - 8 * p;
        sm.hist[tid] = 0;
        __syncthreads();
        for (int i = tid; i < n_keys; i += kSelThreads) {
            unsigned int k = keys[i];
            if ((k & mask) == prefix) atomicAdd(&sm.hist[(k >> shift) & 255u], 1u);
        }
        __syncthreads();
        if (tid < 32) {
            unsigned int c[8], tot = 0;
#pragma unroll
            for (int j = 0; j < 8; ++j) { c[j] = sm.hist[255 - 8 * tid - j]; tot += c[j]; }
            unsigned int incl = tot;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                unsigned int t = __shfl_up_sync(0xffffffffu, incl, o);
                if (tid >= o) incl += t;
            }
            unsigned int excl = incl - tot;
            if (excl < rem && rem <= incl) {
                unsigned int run = excl;
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    if (run < rem && rem <= run + c[j]) { sm.sel_bin = 255 - 8 * tid - j; sm.sel_rem = rem - run; }
                    run += c[j];
                }
            }
        }
        __syncthreads();
        prefix |= sm.sel_bin << shift;
        mask |= 255u << shift;
        rem = sm.sel_rem;
    }
    return prefix;
}

// In-place descending bitonic sort of n (power of two) u64 keys in smem; all threads call.
__device__ __forceinline__ void block_bitonic_desc(unsigned long long *s, int n) {
    const int tid = threadIdx.x;
    for (int k = 2; k <= n; k <<= 1) {
        for (int j = k >> 1; j > 0; j >>= 1) {
            for (int i = tid; i < n; i += kSelThreads) {
                int ixj = i ^ j;
                if (ixj > i) {
                    unsigned long long a = s[i], b = s[ixj];
                    bool desc = ((i & k) == 0);
                    if (desc ? (a < b) : (a > b)) { s[i] = b; s[ixj] = a; }
                }
            }
            __syncthreads();
        }
    }
}

__device__ __forceinline__ int next_pow2(int x) { int p = 1; while (p < x) p <<= 1; return p; }

// Keep the exact top-M of cand[0..cnt): sort, truncate, publish the 64-bit bound.  All threads call.
__device__ __forceinline__ void block_compact(SelectSmem &sm, int M) {
    const int tid = threadIdx.x;
    __syncthreads();
    int cnt = min((int)sm.cnt, kSelCap);
    int n = next_pow2(max(cnt, 2));
    for (int i = cnt + tid; i < n; i += kSelThreads) sm.cand[i] = 0ull;
    __syncthreads();
    block_bitonic_desc(sm.cand, n);
    if (tid == 0) {
        if (cnt >= M) { sm.tau_key = sm.cand[M - 1]; sm.cnt = M; }
        else sm.cnt = cnt;
    }
    __syncthreads();
}

template <typename T, bool ALIGNED>
__global__ void __launch_bounds__(kSelThreads, 4) select_topm_kernel(SelectParams p) {
    using Ops = SelOps<T>;
    using Run = typename Ops::Run;
    constexpr int kVec = ElemTraits<T>::kVec;
    constexpr int kNPass = (sizeof(T) == 2) ? 2 : 4;
    __shared__ SelectSmem sm;

    const int tid = threadIdx.x;
    const int row = blockIdx.y, s = blockIdx.x;
    const int M = p.M, V = p.V;
    const T *rowp = reinterpret_cast<const T *>(p.logits) + (size_t)row * V;
    const int v0 = s * p.chunk_vecs;
    const int v1 = min(p.row_vecs, v0 + p.chunk_vecs);
    const int tile_vecs = kSelThreads * kSelU;
    const int n_tiles = (max(v1 - v0, 0) + tile_vecs - 1) / tile_vecs;

    if (tid == 0) { sm.cnt = 0; sm.cnt2 = 0; sm.tau_key = 0ull; sm.is_last = 0; }
    __syncthreads();

    auto load_tile = [&](int t, uint4 (&buf)[kSelU]) {
#pragma unroll
        for (int u = 0; u < kSelU; ++u) {
            int gv = v0 + t * tile_vecs + u * kSelThreads + tid;
            if (gv < v1) {
                if (ALIGNED) buf[u] = ld_stream_v4(rowp + (size_t)gv * kVec);
                else buf[u] = Ops::load_scalar(rowp, (long long)gv * kVec, V);
            } else buf[u] = Ops::lowest_vec();
        }
    };

    unsigned int tau_ord = 0;
    unsigned long long tau_key = 0ull;
    Run run = Ops::lowest();

    // Re-derive tau from the 512 running maxima (+ the row-shared word when the row is chunked).
    auto update_tau = [&]() {
        unsigned int k0, k1;
        Ops::sub_keys(run, k0, k1);
        sm.sub[2 * tid] = k0; sm.sub[2 * tid + 1] = k1;
        __syncthreads();
        unsigned int t = block_select_kth<kNPass>(sm, sm.sub, kSelSub, (unsigned int)M);
        if (p.S > 1) {
            if (tid == 0) { unsigned int old = atomicMax(&p.row_tau[row], t); sm.bcast = max(old, t); }
            __syncthreads();
            t = sm.bcast;
        }
        tau_ord = max(tau_ord, t);
    };

    // Slow path for one vector: push every element (of those named in `which`) that can still be in
    // the top M.  Returns the bit mask of elements whose push found the buffer full.
    auto push_vec = [&](const uint4 &v, int gv, unsigned int which) -> unsigned int {
        float f[kVec];
        Ops::elems(v, f);
        unsigned int failed = 0;
#pragma unroll
        for (int i = 0; i < kVec; ++i) {
            unsigned int o = ord_key(f[i]);
            unsigned int idx = (unsigned int)gv * kVec + i;
            if (((which >> i) & 1u) && o >= tau_ord && idx < (unsigned int)V) {
                unsigned long long key = ((unsigned long long)o << 32) | (unsigned long long)(0xFFFFFFFFu - idx);
                if (key > tau_key) {
                    unsigned int pos = atomicAdd(&sm.cnt, 1u);
                    if (pos < (unsigned int)kSelCap) sm.cand[pos] = key; else failed |= 1u << i;
                }
            }
        }
        return failed;
    };

    uint4 A[kSelU], Bn[kSelU];
    if (n_tiles > 0) {
        load_tile(0, A);
#pragma unroll
        for (int u = 0; u < kSelU; ++u) run = Ops::rmax(run, Ops::vmax(A[u]));
    }
    update_tau();

    constexpr unsigned int kAllElems = (1u << kVec) - 1u;
    for (int t = 0; t < n_tiles; ++t) {
        if (t + 1 < n_tiles) load_tile(t + 1, Bn);
        const Run tau = Ops::make_tau(tau_ord);
        unsigned int fail = 0;                  // bit u*kVec+i: push of element i of vector u failed
#pragma unroll
        for (int u = 0; u < kSelU; ++u) {
            Run m = Ops::vmax(A[u]);
            run = Ops::rmax(run, m);
            if (Ops::pass(m, tau))
                fail |= push_vec(A[u], v0 + t * tile_vecs + u * kSelThreads + tid, kAllElems) << (u * kVec);
        }
        if (__syncthreads_or(fail != 0)) {      // block-uniform: the candidate buffer overflowed
            // Nothing that failed was stored, so: compact to the exact top-M so far, then re-push
            // only the failed elements, one vector per sub-step (at most kSelThreads*kVec pushes).
            block_compact(sm, M);
            tau_key = sm.tau_key;
            if (tau_key) tau_ord = max(tau_ord, (unsigned int)(tau_key >> 32));
#pragma unroll 1
            for (int u = 0; u < kSelU; ++u) {
                unsigned int c = sm.cnt;
                __syncthreads();
                if (c > (unsigned int)(kSelCap - kSelThreads * kVec)) {
                    block_compact(sm, M);
                    tau_key = sm.tau_key;
                    if (tau_key) tau_ord = max(tau_ord, (unsigned int)(tau_key >> 32));
                }
                uint4 v = A[0];
                if (u == 1) v = A[1]; else if (u == 2) v = A[2]; else if (u == 3) v = A[3];
                unsigned int which = (fail >> (u * kVec)) & kAllElems;
                if (which) push_vec(v, v0 + t * tile_vecs + u * kSelThreads + tid, which);
                __syncthreads();
            }
        }
        if ((((t + 1) & t) == 0) && (t + 1 < n_tiles)) update_tau();
#pragma unroll
        for (int u = 0; u < kSelU; ++u) A[u] = Bn[u];
    }

    // Final: tightest tau, prune, sort, emit.
    update_tau();
    __syncthreads();
    int cnt = min((int)sm.cnt, kSelCap);
    unsigned long long *srt = sm.cand;
    int n_srt;
    if (cnt <= kSelCap / 2) {
        unsigned long long *dst = sm.cand + kSelCap / 2;
        for (int i = tid; i < cnt; i += kSelThreads) {
            unsigned long long key = sm.cand[i];
            if ((unsigned int)(key >> 32) >= tau_ord) { unsigned int q = atomicAdd(&sm.cnt2, 1u); dst[q] = key; }
        }
        __syncthreads();
        int c2 = (int)sm.cnt2;
        n_srt = next_pow2(max(c2, 2));
        for (int i = c2 + tid; i < n_srt; i += kSelThreads) dst[i] = 0ull;
        srt = dst;
    } else {
        n_srt = next_pow2(cnt);
        for (int i = cnt + tid; i < n_srt; i += kSelThreads) sm.cand[i] = 0ull;
    }
    __syncthreads();
    block_bitonic_desc(srt, n_srt);

    auto emit = [&](const unsigned long long *sorted, int n_valid) {
        for (int m = tid; m < M; m += kSelThreads) {
            unsigned long long key = (m < n_valid) ? sorted[m] : 0ull;
            p.cand_id[(size_t)row * M + m] = (int32_t)(0xFFFFFFFFu - (unsigned int)(key & 0xFFFFFFFFull));
            p.cand_val[(size_t)row * M + m] = ord_key_inv((unsigned int)(key >> 32));
        }
    };

    if (p.S == 1) { emit(srt, n_srt); return; }

    // Chunked row: publish this chunk's top-M, the last chunk to arrive merges.
    unsigned long long *part = p.part + ((size_t)row * p.S + s) * M;
    for (int m = tid; m < M; m += kSelThreads) part[m] = (m < n_srt) ? srt[m] : 0ull;
    __threadfence();
    __syncthreads();
    if (tid == 0) {
        unsigned int ticket = atomicAdd(&p.row_counter[row], 1u);
        sm.is_last = (ticket == (unsigned int)(p.S - 1));
    }
    __syncthreads();
    if (!sm.is_last) return;
    __threadfence();
    const int tot = p.S * M;
    const unsigned long long *allp = p.part + (size_t)row * p.S * M;
    for (int i = tid; i < tot; i += kSelThreads) sm.cand[i] = __ldcg(allp + i);
    int n2 = next_pow2(max(tot, 2));
    for (int i = tot + tid; i < n2; i += kSelThreads) sm.cand[i] = 0ull;
    __syncthreads();
    block_bitonic_desc(sm.cand, n2);
    emit(sm.cand, n2);
    if (tid == 0) { p.row_counter[row] = 0u; p.row_tau[row] = 0u; }
}

}  // namespace dt
