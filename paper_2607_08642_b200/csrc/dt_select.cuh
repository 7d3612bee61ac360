// dt_select.cuh -- step (a1): exact top-M select per logits row (Alg. 1 step 1).
//
// One streaming pass over the row (every logit is read from HBM exactly once), HBM-bound by design.
// A CTA owns one chunk of one row; its 8 warps stream independently (no CTA barrier in the main loop):
// per tile a thread loads four 16-byte vectors, folds them into its running maximum with packed max
// instructions and compares the tile maximum against a threshold tau; only when some lane of the warp
// holds an element >= tau does the warp take the slow path, which filters elements with scalar compares
// and appends 64-bit keys (ordered value << 32 | ~token) to the warp's PRIVATE candidate segment in
// shared memory.
//
// tau is always a PROVEN lower bound on the row's M-th largest value.  Each warp publishes a claim
// "at least q = ceil(M/8) of my lanes have seen an element >= c_w" (c_w = q-th largest of its 32 lane
// maxima, found with 16 or 32 ballot steps, no barrier); lanes cover disjoint elements, so
// min_w c_w has at least 8 q >= M elements at or above it.  Claims only grow, so a stale claim is still
// valid and warps refresh tau asynchronously (tiles 0, 1, 3, 7, 15, ...).  A warp that compacts its
// segment publishes the stronger claim "M elements >= the M-th key of my segment".  Chunks of one row
// share tau through an atomicMax word.  Nothing that could be in the top M is ever dropped, so the
// result is exact; ties on the value are resolved by the key (token id asc).
//
// A segment holds 512 keys; before a vector slot that could overflow it (32 lanes x 8 elements) the warp
// sorts its segment, keeps the top M and remembers the exact 64-bit bound, which also turns all-equal and
// ascending rows into cheap rejections.  At the end the CTA prunes all candidates with the final tau,
// ranks the survivors by counting (typically ~100 keys) and emits; chunked rows merge in the last CTA.
#pragma once
#include "dt_common.cuh"

namespace dt {

constexpr int kSelThreads = 256;
constexpr int kSelU = 4;            // 16-byte vectors per thread per tile
constexpr int kSelCap = 4096;       // largest candidate buffer (u64 keys): bounds S * M for chunked rows
constexpr int kSelWarps = kSelThreads / 32;
constexpr int kSelTileBytes = 4096; // bulk-copy tile of one warp: 256 vectors of 16 bytes
constexpr int kSelStages = 2;       // bulk-copy tiles in flight per warp (ring slots)
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
    unsigned long long *span;       // optional measurement aid: [0] min %globaltimer at CTA start, [1] max at CTA end
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
    // bit i set <=> element i >= tau (packed compares, two elements per instruction)
    static __device__ __forceinline__ unsigned int ge_mask(const uint4 &v, Run tau) {
        const unsigned int m0 = __hge2_mask(from_bits(v.x), tau), m1 = __hge2_mask(from_bits(v.y), tau);
        const unsigned int m2 = __hge2_mask(from_bits(v.z), tau), m3 = __hge2_mask(from_bits(v.w), tau);
        return ((m0 & 1u) | ((m0 >> 15) & 2u)) | (((m1 & 1u) | ((m1 >> 15) & 2u)) << 2) |
               (((m2 & 1u) | ((m2 >> 15) & 2u)) << 4) | (((m3 & 1u) | ((m3 >> 15) & 2u)) << 6);
    }
    static __device__ __forceinline__ float elem(const uint4 &v, int i) {
        const unsigned int w = (i < 4) ? ((i < 2) ? v.x : v.y) : ((i < 6) ? v.z : v.w);
        return __uint_as_float((i & 1) ? (w & 0xFFFF0000u) : (w << 16));
    }
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
    static __device__ __forceinline__ unsigned int ge_mask(const uint4 &v, Run tau) {
        return (__uint_as_float(v.x) >= tau.a ? 1u : 0u) | (__uint_as_float(v.y) >= tau.a ? 2u : 0u) |
               (__uint_as_float(v.z) >= tau.a ? 4u : 0u) | (__uint_as_float(v.w) >= tau.a ? 8u : 0u);
    }
    static __device__ __forceinline__ float elem(const uint4 &v, int i) {
        return __uint_as_float((i < 2) ? ((i == 0) ? v.x : v.y) : ((i == 2) ? v.z : v.w));
    }
    static __device__ __forceinline__ uint4 load_scalar(const float *row, long long e0, int V) {
        uint32_t w[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) w[i] = (e0 + i < V) ? __float_as_uint(row[e0 + i]) : 0xFF800000u;
        return make_uint4(w[0], w[1], w[2], w[3]);
    }
};


// Shared-memory state of one CTA.  SEG = keys per warp-private candidate segment (M <= SEG / 2),
// FIN = survivors the epilogue ranks by counting, QCAP = per-warp queue of vectors awaiting the element filter.
template <int SEG, int FIN, int QCAP, int NW>
struct SelectSmemT {
    static constexpr int kSeg = SEG, kCap = SEG * NW, kFin = FIN, kQ = QCAP, kWarps = NW;
    unsigned long long cand[SEG * NW];          // NW warp-private segments; reused for sorting / merging
    unsigned long long fin[FIN];                // survivors of the final prune
    int qi[NW][QCAP];                    // per-warp queue: row index of every vector that held an element >= tau when it
                                                // streamed by; the vectors are read again (from L2) when the queue is filtered,
                                                // normally once, after the chunk, against the FINAL threshold
    unsigned int wcnt[NW];                      // keys in each warp's segment
    unsigned int claim[NW];              // c_w: >= q lanes of warp w have seen an element with ordered key >= c_w
    unsigned int claimM[NW];             // >= M elements of warp w have ordered key >= claimM[w] (after a compaction)
    unsigned int cnt2;
    unsigned int is_last;
};
using SelectSmemBig = SelectSmemT<512, 512, 256, 8>;  // 8 warps, any M <= 256 (44 KB static)
using SelectSmemW4 = SelectSmemT<512, 256, 128, 4>;   // 4 warps, M <= 128 (20 KB static): four CTAs per SM hold all 512 rows of a
                                                      // batch-32 round at once (no second wave)

// In-place descending bitonic sort of n (power of two) u64 keys in smem; all kSelThreads threads call.
__device__ __forceinline__ void block_bitonic_desc(unsigned long long *s, int n) {
    const int tid = threadIdx.x;
    for (int k = 2; k <= n; k <<= 1) {
        for (int j = k >> 1; j > 0; j >>= 1) {
            for (int i = tid; i < n; i += (int)blockDim.x) {
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
// Same for one warp on its own segment (n a power of two); the 32 lanes of the warp call.
__device__ __forceinline__ void warp_bitonic_desc(unsigned long long *s, int n, int lane) {
    for (int k = 2; k <= n; k <<= 1) {
        for (int j = k >> 1; j > 0; j >>= 1) {
            for (int i = lane; i < n; i += 32) {
                int ixj = i ^ j;
                if (ixj > i) {
                    unsigned long long a = s[i], b = s[ixj];
                    bool desc = ((i & k) == 0);
                    if (desc ? (a < b) : (a > b)) { s[i] = b; s[ixj] = a; }
                }
            }
            __syncwarp();
        }
    }
}

__device__ __forceinline__ void sel_span_mark(unsigned long long *span, int which) {
    if (span && threadIdx.x == 0) {
        unsigned long long t;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
        if (which == 0) atomicMin(span, t); else atomicMax(span + 1, t);
    }
}
__device__ __forceinline__ int next_pow2(int x) { int p = 1; while (p < x) p <<= 1; return p; }

// q-th largest (1-based, q <= 32) of the 32 lanes' keys: the largest T with #{key >= T} >= q, built bit by bit
// from the top with one ballot per bit.  NBITS = 16 resolves only the top 16 bits (bf16 keys; the caller completes
// the low half, which is 0xFFFF for negative values and 0 otherwise).
template <int NBITS>
__device__ __forceinline__ unsigned int warp_qth_largest(unsigned int key, int q) {
    unsigned int T = 0;
#pragma unroll
    for (int b = 31; b > 31 - NBITS; --b) {
        const unsigned int cand = T | (1u << b);
        if (__popc(__ballot_sync(0xffffffffu, key >= cand)) >= q) T = cand;
    }
    return T;
}

// Rank `n` distinct keys by counting and hand the top M to `emit(rank, key)`; all threads call.
template <typename F>
__device__ __forceinline__ void block_rank_emit(const unsigned long long *keys, int n, int M, F emit) {
    for (int i = threadIdx.x; i < n; i += (int)blockDim.x) {
        const unsigned long long mk = keys[i];
        int rank = 0;
        int j = 0;
        for (; j + 2 <= n; j += 2) {
            const ulonglong2 o = *reinterpret_cast<const ulonglong2 *>(keys + j);
            rank += (o.x > mk) + (o.y > mk);
        }
        if (j < n) rank += (keys[j] > mk);
        if (rank < M) emit(rank, mk);
    }
}

// Per-warp slow-path state kept in registers by the kernels and handed to the out-of-line helpers by value.
struct SelWarpCtx {
    unsigned int tau_ord;                // ordered-key lower bound on the row's M-th largest value
    unsigned long long wtau_key;         // exact key bound for this warp's own pushes (after a compaction)
    int qcnt;                            // vectors waiting in this warp's queue (warp-uniform)
};

// Keep the top M of this warp's segment (sort), remember the exact bound, publish the strong claim.
template <typename SM>
__device__ __noinline__ SelWarpCtx sel_compact(SM &sm, SelWarpCtx c, int M) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    unsigned long long *seg = sm.cand + warp * SM::kSeg;
    volatile unsigned int *vwcnt = sm.wcnt, *vclaimM = sm.claimM;
    __syncwarp();
    int n = (int)vwcnt[warp];
    const int np2 = next_pow2(max(n, 2));
    for (int i = n + lane; i < np2; i += 32) seg[i] = 0ull;
    __syncwarp();
    warp_bitonic_desc(seg, np2, lane);
    if (n >= M) {
        c.wtau_key = seg[M - 1];
        n = M;
        const unsigned int o = (unsigned int)(c.wtau_key >> 32);
        if (lane == 0) vclaimM[warp] = o;
        c.tau_ord = max(c.tau_ord, o);
    }
    __syncwarp();
    if (lane == 0) vwcnt[warp] = (unsigned int)n;
    __syncwarp();
    return c;
}

// Filter the queued vectors, one vector per lane: append every element that can still be in the top M.
// A batch adds at most SEG / 2 keys; the segment is compacted first when it could overflow.
template <typename T, typename SM>
__device__ __noinline__ SelWarpCtx sel_drain(SM &sm, SelWarpCtx c, int M, int V, const T *rowp, bool aligned) {
    using Ops = SelOps<T>;
    constexpr int kVec = ElemTraits<T>::kVec;
    constexpr int kBatchKeys = SM::kSeg / 2;
    constexpr int kLanes = (kBatchKeys / kVec) < 32 ? (kBatchKeys / kVec) : 32;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    unsigned long long *seg = sm.cand + warp * SM::kSeg;
    volatile unsigned int *vwcnt = sm.wcnt;
    __syncwarp();
    constexpr int kU = 4;                                           // vectors per lane in flight: one L2 round trip per 4 batches (8 spills)
    for (int base0 = 0; base0 < c.qcnt; base0 += kLanes * kU) {
        uint4 vv[kU];
        int gvv[kU];
#pragma unroll
        for (int u = 0; u < kU; ++u) {
            const int qi = base0 + u * kLanes + lane;
            gvv[u] = (lane < kLanes && qi < c.qcnt) ? sm.qi[warp][qi] : -1;
            vv[u] = make_uint4(0u, 0u, 0u, 0u);
            if (gvv[u] >= 0) vv[u] = aligned ? ld_ro_v4(rowp + (size_t)gvv[u] * kVec) : Ops::load_scalar(rowp, (long long)gvv[u] * kVec, V);
        }
#pragma unroll
        for (int u = 0; u < kU; ++u) {
            if (base0 + u * kLanes >= c.qcnt) break;                 // warp-uniform
            if ((int)vwcnt[warp] > SM::kSeg - kBatchKeys) c = sel_compact(sm, c, M);
            if (gvv[u] >= 0) {
                const uint4 v = vv[u];
                const int gv = gvv[u];
                unsigned int mask = Ops::ge_mask(v, Ops::make_tau(c.tau_ord));      // usually one bit
                while (mask) {
                    const int i = __ffs(mask) - 1;
                    mask &= mask - 1;
                    const unsigned int idx = (unsigned int)gv * kVec + i;
                    const unsigned long long key = ((unsigned long long)ord_key(Ops::elem(v, i)) << 32) | (unsigned long long)(0xFFFFFFFFu - idx);
                    if (key > c.wtau_key && idx < (unsigned int)V) {
                        const unsigned int pos = atomicAdd(&sm.wcnt[warp], 1u);
                        seg[pos] = key;
                    }
                }
            }
            __syncwarp();
        }
    }
    c.qcnt = 0;
    return c;
}

// Publish this warp's claim: the q-th largest of its 32 lane maxima.
template <typename T, typename SM>
__device__ __forceinline__ void sel_publish_claim(SM &sm, typename SelOps<T>::Run run, int q) {
    constexpr int kNBits = (sizeof(T) == 2) ? 16 : 32;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    unsigned int k0, k1;
    SelOps<T>::sub_keys(run, k0, k1);
    unsigned int cl = warp_qth_largest<kNBits>(max(k0, k1), q);
    // bf16: only the top 16 bits were resolved; keys of negative values end in 0xFFFF, of non-negative ones in 0
    if (kNBits == 16 && !(cl & 0x80000000u)) cl |= 0xFFFFu;
    if (lane == 0) *reinterpret_cast<volatile unsigned int *>(&sm.claim[warp]) = cl;
}
// tau = max(min_w claim[w], max_w claimM[w], the row-shared word); claims only grow, stale reads stay valid.
template <typename SM>
__device__ __forceinline__ unsigned int sel_read_tau(SM &sm, const SelectParams &p, int row) {
    constexpr unsigned int kFull = 0xffffffffu;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    volatile unsigned int *vclaim = sm.claim, *vclaimM = sm.claimM;
    unsigned int cw = (lane < SM::kWarps) ? vclaim[lane] : 0xFFFFFFFFu;
    unsigned int cm = (lane < SM::kWarps) ? vclaimM[lane] : 0u;
#pragma unroll
    for (int o = 4; o > 0; o >>= 1) {
        cw = min(cw, __shfl_xor_sync(kFull, cw, o));
        cm = max(cm, __shfl_xor_sync(kFull, cm, o));
    }
    unsigned int t = max(__shfl_sync(kFull, cw, 0), __shfl_sync(kFull, cm, 0));
    if (p.S > 1) {
        unsigned int g = 0;
        if (lane == 0) g = (warp == 0) ? atomicMax(&p.row_tau[row], t) : *reinterpret_cast<volatile unsigned int *>(&p.row_tau[row]);
        t = max(t, __shfl_sync(kFull, g, 0));
    }
    return t;
}
// One vector slot of a warp: lanes whose vector holds an element >= tau queue it; a full queue is drained.
template <typename T, typename SM>
__device__ __forceinline__ SelWarpCtx sel_slot(SM &sm, SelWarpCtx c, bool hit, int gv, int M, int V, const T *rowp, bool aligned) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const unsigned int bal = __ballot_sync(0xffffffffu, hit);
    if (bal) {
        if (hit) {
            const int pos = c.qcnt + __popc(bal & ((1u << lane) - 1u));
            sm.qi[warp][pos] = gv;
        }
        c.qcnt += __popc(bal);
        if (c.qcnt > SM::kQ - 32) c = sel_drain<T>(sm, c, M, V, rowp, aligned);
    }
    return c;
}

// Epilogue shared by both kernels: prune every segment with the final tau, rank the survivors, emit; chunked rows
// publish their top M and the last chunk to arrive merges.  All threads call, after a CTA barrier.
template <typename SM>
__device__ __forceinline__ void sel_epilogue(SM &sm, const SelectParams &p, int row, int s, unsigned int tau_ord) {
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int M = p.M;
    unsigned long long *seg = sm.cand + warp * SM::kSeg;
    {
        const int n = (int)sm.wcnt[warp];
        for (int i = lane; i < n; i += 32) {
            const unsigned long long key = seg[i];
            if ((unsigned int)(key >> 32) >= tau_ord) {
                const unsigned int pos = atomicAdd(&sm.cnt2, 1u);
                if (pos < (unsigned int)SM::kFin) sm.fin[pos] = key;
            }
        }
    }
    __syncthreads();
    const int c2 = (int)sm.cnt2;

    unsigned long long *part = p.part + ((size_t)row * p.S + s) * M;
    auto out_single = [&](int rank, unsigned long long key) {
        p.cand_id[(size_t)row * M + rank] = (int32_t)(0xFFFFFFFFu - (unsigned int)(key & 0xFFFFFFFFull));
        p.cand_val[(size_t)row * M + rank] = ord_key_inv((unsigned int)(key >> 32));
    };
    auto out_part = [&](int rank, unsigned long long key) { part[rank] = key; };

    if (c2 <= SM::kFin) {
        if (p.S == 1) { block_rank_emit(sm.fin, c2, M, out_single); return; }
        block_rank_emit(sm.fin, c2, M, out_part);
        for (int i = c2 + tid; i < M; i += (int)blockDim.x) part[i] = 0ull;      // chunk with fewer than M elements
    } else {
        // adversarial rows (more than kFin survivors): sort everything that was kept
        const int n = (int)sm.wcnt[warp];
        for (int i = n + lane; i < SM::kSeg; i += 32) seg[i] = 0ull;
        __syncthreads();
        block_bitonic_desc(sm.cand, SM::kCap);
        for (int i = tid; i < M; i += (int)blockDim.x) { if (p.S == 1) out_single(i, sm.cand[i]); else out_part(i, sm.cand[i]); }
        if (p.S == 1) return;
    }

    // Chunked row: the last chunk to arrive merges the S sorted partial lists.
    __threadfence();
    __syncthreads();
    if (tid == 0) {
        unsigned int ticket = atomicAdd(&p.row_counter[row], 1u);
        sm.is_last = (ticket == (unsigned int)(p.S - 1));
    }
    __syncthreads();
    if (!sm.is_last) return;
    __threadfence();
    // every chunk's final tau went into row_tau: prune the S * M keys with it, then rank
    const unsigned int gtau = *reinterpret_cast<volatile unsigned int *>(&p.row_tau[row]);
    if (tid == 0) sm.cnt2 = 0;
    __syncthreads();
    const int tot = p.S * M;                                   // <= SM::kCap (launcher)
    const unsigned long long *allp = p.part + (size_t)row * p.S * M;
    for (int i = tid; i < tot; i += (int)blockDim.x) {
        const unsigned long long key = __ldcg(allp + i);
        sm.cand[i] = key;
        if ((unsigned int)(key >> 32) >= gtau && key != 0ull) {
            const unsigned int pos = atomicAdd(&sm.cnt2, 1u);
            if (pos < (unsigned int)SM::kFin) sm.fin[pos] = key;
        }
    }
    __syncthreads();
    const int c3 = (int)sm.cnt2;
    if (c3 <= SM::kFin) {
        block_rank_emit(sm.fin, c3, M, out_single);
    } else {
        const int n2 = next_pow2(max(tot, 2));
        for (int i = tot + tid; i < n2; i += (int)blockDim.x) sm.cand[i] = 0ull;
        __syncthreads();
        block_bitonic_desc(sm.cand, n2);
        for (int i = tid; i < M; i += (int)blockDim.x) out_single(i, sm.cand[i]);
    }
    if (tid == 0) { p.row_counter[row] = 0u; p.row_tau[row] = 0u; }
}

// ---------------------------------------------------------------------------------------------------------------
// Register-tile kernel: any alignment, any M <= 256.  Each thread keeps two tiles of four 16-byte vectors in
// registers (ping-pong) and loads them with 128-bit streaming loads (scalar loads when the row is unaligned).
template <typename T, bool ALIGNED>
__global__ void __launch_bounds__(kSelThreads, 4) select_topm_kernel(SelectParams p) {
    using Ops = SelOps<T>;
    using Run = typename Ops::Run;
    using SM = SelectSmemBig;
    constexpr int kVec = ElemTraits<T>::kVec;
    __shared__ __align__(16) SM sm;

    const int tid = threadIdx.x;
    const int row = blockIdx.y, s = blockIdx.x;
    const int M = p.M, V = p.V;
    const int q = (M + kSelWarps - 1) / kSelWarps;             // lanes per warp that must back a claim (<= 32)
    const T *rowp = reinterpret_cast<const T *>(p.logits) + (size_t)row * V;
    const int v0 = s * p.chunk_vecs;
    const int v1 = min(p.row_vecs, v0 + p.chunk_vecs);
    const int tile_vecs = kSelThreads * kSelU;
    const int n_tiles = (max(v1 - v0, 0) + tile_vecs - 1) / tile_vecs;

    if (tid < kSelWarps) { sm.wcnt[tid] = 0; sm.claim[tid] = 0; sm.claimM[tid] = 0; }
    if (tid == 0) { sm.cnt2 = 0; sm.is_last = 0; }
    __syncthreads();

    const int n_full = max(v1 - v0, 0) / tile_vecs;            // tiles that need no bounds checks
    auto load_tile = [&](int t, uint4 (&buf)[kSelU]) {
        if (ALIGNED && t < n_full) {
            const T *qp = rowp + (size_t)(v0 + t * tile_vecs + tid) * kVec;
#pragma unroll
            for (int u = 0; u < kSelU; ++u) buf[u] = ld_stream_v4(qp + (size_t)u * kSelThreads * kVec);
            return;
        }
#pragma unroll
        for (int u = 0; u < kSelU; ++u) {
            int gv = v0 + t * tile_vecs + u * kSelThreads + tid;
            if (gv < v1) {
                if (ALIGNED) buf[u] = ld_stream_v4(rowp + (size_t)gv * kVec);
                else buf[u] = Ops::load_scalar(rowp, (long long)gv * kVec, V);
            } else buf[u] = Ops::lowest_vec();
        }
    };

    SelWarpCtx c;
    c.tau_ord = 0; c.wtau_key = 0ull; c.qcnt = 0;
    Run run = Ops::lowest();                 // this lane's running maximum (two packed halves)

    uint4 A[kSelU], Bn[kSelU];
    if (n_tiles > 0) {
        load_tile(0, A);
#pragma unroll
        for (int u = 0; u < kSelU; ++u) run = Ops::rmax(run, Ops::vmax(A[u]));
    }
    sel_publish_claim<T>(sm, run, q);
    __syncthreads();                          // the only CTA barrier before the epilogue: every warp has a claim
    c.tau_ord = max(c.tau_ord, sel_read_tau(sm, p, row));

    auto process = [&](const uint4 (&X)[kSelU], int t) {
        const Run tau = Ops::make_tau(c.tau_ord);
        const int gv0 = v0 + t * tile_vecs + tid;
#pragma unroll
        for (int u = 0; u < kSelU; ++u) {
            const Run m = Ops::vmax(X[u]);
            run = Ops::rmax(run, m);
            c = sel_slot<T>(sm, c, Ops::pass(m, tau), gv0 + u * kSelThreads, M, V, rowp, ALIGNED);
        }
        if (t > 0 && (((t + 1) & t) == 0) && (t + 1 < n_tiles)) {
            sel_publish_claim<T>(sm, run, q);
            __syncwarp();
            c.tau_ord = max(c.tau_ord, sel_read_tau(sm, p, row));
        }
    };
    for (int t = 0; t < n_tiles; t += 2) {      // ping-pong between the two register tiles
        if (t + 1 < n_tiles) load_tile(t + 1, Bn);
        process(A, t);
        if (t + 1 < n_tiles) {
            if (t + 2 < n_tiles) load_tile(t + 2, A);
            process(Bn, t + 1);
        }
    }
    // the queue is filtered against the chunk's final threshold
    sel_publish_claim<T>(sm, run, q);
    __syncthreads();
    c.tau_ord = max(c.tau_ord, sel_read_tau(sm, p, row));
    c = sel_drain<T>(sm, c, M, V, rowp, ALIGNED);
    __syncthreads();
    sel_epilogue(sm, p, row, s, c.tau_ord);
}

// ---------------------------------------------------------------------------------------------------------------
// Bulk-copy kernel (16-byte aligned rows, M <= 128): every warp streams its own 2 KB tiles from HBM into a private
// ring in shared memory with cp.async.bulk (one elected lane issues; completion on an mbarrier), kSelStages tiles
// in flight per warp, and reads them back with conflict-free 128-bit shared loads.  No load instruction or
// register is spent per vector on the global side, so more bytes are in flight per SM (3 CTAs x 8 warps x 2 tiles).
__device__ __forceinline__ void sel_mbar_init(unsigned int bar, unsigned int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void sel_mbar_wait(unsigned int bar, unsigned int parity) {
    asm volatile(
        "{\n\t.reg .pred p;\n"
        "DT_SEL_WAIT:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DT_SEL_DONE;\n\t"
        "bra DT_SEL_WAIT;\n"
        "DT_SEL_DONE:\n\t}\n" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void sel_bulk_load(unsigned int dst, const void *src, unsigned int bytes, unsigned int bar) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}

constexpr int kSelTileVecs = kSelTileBytes / 16;
constexpr int kBulkU = kSelTileVecs / 32;        // vectors per lane per tile
template <typename SM> constexpr size_t sel_bulk_dyn_smem() { return (size_t)SM::kWarps * kSelStages * kSelTileBytes + (size_t)SM::kWarps * kSelStages * 8; }

template <typename T, typename SM>
__global__ void __launch_bounds__(SM::kWarps * 32, SM::kWarps == 4 ? 4 : 2) select_topm_bulk_kernel(SelectParams p) {
    using Ops = SelOps<T>;
    using Run = typename Ops::Run;
    constexpr int kNW = SM::kWarps;
    constexpr int kVec = ElemTraits<T>::kVec;
    __shared__ __align__(16) SM sm;
    extern __shared__ __align__(128) unsigned char sel_dyn[];

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    sel_span_mark(p.span, 0);
    const int row = blockIdx.y, s = blockIdx.x;
    const int M = p.M, V = p.V;
    const int q = (M + kNW - 1) / kNW;
    const T *rowp = reinterpret_cast<const T *>(p.logits) + (size_t)row * V;
    const int v0 = s * p.chunk_vecs;
    const int v1 = min(p.row_vecs, v0 + p.chunk_vecs);
    const int n_ctiles = (max(v1 - v0, 0) + kSelTileVecs - 1) / kSelTileVecs;       // 2 KB tiles of the chunk
    const int n_w = (n_ctiles > warp) ? (n_ctiles - warp + kNW - 1) / kNW : 0;   // tiles of this warp

    unsigned char *ring = sel_dyn + (size_t)warp * kSelStages * kSelTileBytes;
    const unsigned int ring_a = (unsigned int)__cvta_generic_to_shared(ring);
    const unsigned int bar_a = (unsigned int)__cvta_generic_to_shared(sel_dyn + (size_t)kNW * kSelStages * kSelTileBytes) +
                               (unsigned int)warp * kSelStages * 8;

    if (tid < kNW) { sm.wcnt[tid] = 0; sm.claim[tid] = 0; sm.claimM[tid] = 0; }
    if (tid == 0) { sm.cnt2 = 0; sm.is_last = 0; }
    if (lane == 0) {
        for (int i = 0; i < kSelStages; ++i) sel_mbar_init(bar_a + 8 * i, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    // tile i of this warp = chunk tile warp + 8 i: vectors [tv0, tv0 + nv)
    auto issue = [&](int i) {
        const int tv0 = v0 + (warp + kNW * i) * kSelTileVecs;
        const int nv = min(kSelTileVecs, v1 - tv0);
        const int slot = i % kSelStages;
        sel_bulk_load(ring_a + slot * kSelTileBytes, rowp + (size_t)tv0 * kVec, (unsigned int)nv * 16u, bar_a + 8 * slot);
    };
    if (lane == 0) for (int i = 0; i < kSelStages && i < n_w; ++i) issue(i);

    SelWarpCtx c;
    c.tau_ord = 0; c.wtau_key = 0ull; c.qcnt = 0;
    Run run = Ops::lowest();
    auto load_slot = [&](int i, uint4 (&X)[kBulkU]) {            // lane's vectors u * 32 + lane of tile i
        const int nv = min(kSelTileVecs, v1 - (v0 + (warp + kNW * i) * kSelTileVecs));
        const uint4 *src = reinterpret_cast<const uint4 *>(ring + (size_t)(i % kSelStages) * kSelTileBytes);
#pragma unroll
        for (int u = 0; u < kBulkU; ++u) X[u] = (u * 32 + lane < nv) ? src[u * 32 + lane] : Ops::lowest_vec();
    };

    // first tile: fold into the running maxima so that every warp can back a claim before any push
    uint4 X[kBulkU];
    if (n_w > 0) {
        sel_mbar_wait(bar_a, 0);
        load_slot(0, X);
#pragma unroll
        for (int u = 0; u < kBulkU; ++u) run = Ops::rmax(run, Ops::vmax(X[u]));
    }
    sel_publish_claim<T>(sm, run, q);
    __syncthreads();
    c.tau_ord = max(c.tau_ord, sel_read_tau(sm, p, row));

    for (int i = 0; i < n_w; ++i) {
        if (i > 0) { sel_mbar_wait(bar_a + 8 * (i % kSelStages), (unsigned int)((i / kSelStages) & 1)); load_slot(i, X); }
        __syncwarp();                                           // every lane has read the slot: refill it
        if (lane == 0 && i + kSelStages < n_w) {
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");      // generic reads above, async write below
            issue(i + kSelStages);
        }
        const Run tau = Ops::make_tau(c.tau_ord);
        const int gv0 = v0 + (warp + kNW * i) * kSelTileVecs + lane;
#pragma unroll
        for (int u = 0; u < kBulkU; ++u) {
            const Run m = Ops::vmax(X[u]);
            run = Ops::rmax(run, m);
            c = sel_slot<T>(sm, c, Ops::pass(m, tau), gv0 + u * 32, M, V, rowp, true);
        }
        if (i > 0 && (((i + 1) & i) == 0) && (i + 1 < n_w)) {
            sel_publish_claim<T>(sm, run, q);
            __syncwarp();
            c.tau_ord = max(c.tau_ord, sel_read_tau(sm, p, row));
        }
    }
    sel_publish_claim<T>(sm, run, q);
    __syncthreads();
    c.tau_ord = max(c.tau_ord, sel_read_tau(sm, p, row));
    c = sel_drain<T>(sm, c, M, V, rowp, true);
    __syncthreads();
    sel_epilogue(sm, p, row, s, c.tau_ord);
    sel_span_mark(p.span, 1);
}

}  // namespace dt
