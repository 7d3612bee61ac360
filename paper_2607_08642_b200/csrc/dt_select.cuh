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
constexpr int kSelCap = 4096;       // candidate buffer capacity (u64 keys), power of two
constexpr int kSelWarps = kSelThreads / 32;
constexpr int kSelSeg = kSelCap / kSelWarps;       // candidate segment per warp (512 keys)
constexpr int kSelFin = 1024;       // survivors ranked by counting; more than that falls back to a bitonic sort
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

