// dt_wave.cuh -- steps (a4)-(a9) as ONE persistent kernel with an exact WAVEFRONT schedule (bf16 weights).
//
// Algorithm 1 pops one node per step, so a round is a chain of B dependent
// GRU -> correction -> pop steps.  By the equivalence lemma of Appendix B (scores are
// monotone along a path, so best-first returns exactly the B best nodes of the candidate tree, an
// ancestor-closed set) the ORDER in which CHILDREN(.) is evaluated does not matter, only that every
// node the heap would expand has been expanded before the heap run is replayed.  This kernel therefore
// lets every request expand up to W nodes per step:
//
//   repeat   replay the best-first heap on what is known (children lists of the nodes expanded so far);
//            the first popped node whose children are unknown is exactly the node Algorithm 1 would
//            expand next (NEEDED); the next W-1 unexpanded nodes the replay pops are SPECULATIVE picks
//            (each lies in the top-B of the known scores, a necessary condition for being in the tree);
//            expand all of them in one batched GRU step;
//   until    a replay pops B nodes (or runs dry) without meeting an unexpanded node among its first B-1
//            pops: that replay IS Algorithm 1's run, pop for pop, ties included (reading A8).
//
// W = 1 is the plain heap schedule (B steps); a bushy tree of depth D finishes in about D + 1 steps.
// Speculative expansions that turn out useless cost GRU columns, never correctness.
//
// Two CTA roles, co-resident (cooperative launch), hand-over through self-describing words in L2 as in
// dt_fused.cuh:
//  * GRU CTAs (g / 16 of them, weight-stationary: 48 rows of W_hh + 16 columns of W1[:, d:] in shared
//    memory).  Step s: gather the items {request, parent state slot, token} every request published,
//    and for passes of up to 64 items run D1[node, row] = S_parent[node, :] . W_hh[row, :]^T on
//    tcgen05 with the NODES as the M dimension (M = 128 rows = 64 nodes x {bf16 hi, bf16 lo}, N = 48,
//    accumulators in TMEM; states stream from L2 through a cp.async ring in the 128-byte-swizzled
//    K-major layout), gates with the input half gathered from P = E W_ih^T, new
//    state to L2, and D2[node, j] = S_new[node, my 16 units] . W1[j, d + my units]^T, this CTA's
//    split-K share of W1[:, d:] S_new, one M = 128, N = r MMA.
//  * Request CTAs (one per request) keep the children lists, replay the heap, nominate, and for every
//    expanded node compute a = SiLU(C + sum of partials), z = (base + W2[cand] a) / T_eff over the M
//    candidate rows of the node's depth (rows staged per depth in shared memory "slices"), slice
//    log-softmax (reading A1) and top-k; at the end they emit (a9).
#pragma once
#include "dt_fused.cuh"

namespace dt {

constexpr int kWvThreads = 256;
constexpr int kWvNP = 64;                       // items per GRU pass (M = 128 operand rows: hi | lo)
constexpr int kWvKC = 128;                      // k per ring slot (two 64-wide swizzle blocks)
constexpr int kWvRingBytes = 96 * 1024;         // state ring: three 128-row chunks, or more slots of fewer rows
constexpr int kWvCS = 4;                        // GRU CTAs per thread-block cluster
constexpr int kWvLdH = 68;                      // floats per row of the pre-activation buffer (64 nodes + pad)
constexpr int kWvDescWords = 16;                // u64 words per request descriptor: header + 15 items, one 128-byte line
constexpr int kWvMaxW = kWvDescWords - 1;
constexpr int kWvMaxBatch = 128;                // requests per launch (headers are polled by four warps)
constexpr int kWvTmemCols = 512;                // 4 or 8 independent D1 accumulators of N <= 128 / 64 columns; D2 reuses column 0 ..
constexpr int kWvMaxSlices = 8;
constexpr unsigned int kWvAct = 0x100u;         // replay word: cursor (8) | active (1) | pop slot (16, from bit 16)

struct WaveParams {
    ExpandParams e;
    int n_gru;                     // GRU CTAs = g / 16
    int slot_stride;               // state slots per request (slot 0 = zeros, expansion x lives in slot x + 1)
    int W;                         // items a request may publish per step (1 .. kWvMaxW)
    int n_slices;                  // W2 slices in a request CTA's shared memory
    int e_max;                     // expansions per request = slot_stride - 1
    int P;                         // partial vectors per item = n_gru / kWvCS (one per cluster of GRU CTAs)
    int rpc;                       // rows of W1 each CTA of a cluster reduces: 16 ceil(r / (16 kWvCS))
    __nv_bfloat16 *s_hi, *s_lo;    // [batch, slot_stride, g]
    float *s32;                    // [batch, slot_stride, g]
    float *partial;                // [batch, kWvMaxW, P, r]
    unsigned long long *desc;      // [batch, kWvDescWords]
    unsigned int *flags;           // [n_gru] one 128-byte line each
    unsigned int *round_ctr;       // rounds this handle has run (tags every hand-over word)
    unsigned int *err;             // set to 1 when a hand-over wait timed out (protocol slip: fail, do not hang)
    unsigned int *stats;           // [4] optional counters of request 0: steps, expansions (measurement aid)
};

// ---- hand-over words ---------------------------------------------------------------------------------
// header: round (24) | epoch (12) | first new state slot (12) | done (1) | count (15)
// item:   token (32) | parent state slot (10) | epoch (10) | round (12)
// Every word is self-validating (relaxed stores need no ordering between them); epoch = step + 1, so
// zero-initialised memory never matches.
__device__ __forceinline__ unsigned long long wave_hdr_pack(unsigned int rnd, int epoch, int first, int done, int count) {
    return ((unsigned long long)(rnd & 0xFFFFFFu) << 40) | ((unsigned long long)(epoch & 0xFFF) << 28) |
           ((unsigned long long)(first & 0xFFF) << 16) | ((unsigned long long)(done & 1) << 15) | (unsigned long long)(count & 0x7FFF);
}
__device__ __forceinline__ bool wave_hdr_ok(unsigned long long h, unsigned int rnd, int epoch) {
    if ((unsigned int)(h >> 40) != (rnd & 0xFFFFFFu)) return false;
    return ((h >> 15) & 1ull) || (int)((h >> 28) & 0xFFFu) == (epoch & 0xFFF);
}
__device__ __forceinline__ unsigned long long wave_item_pack(unsigned int rnd, int epoch, int pslot, int tok) {
    return ((unsigned long long)(unsigned int)tok << 32) | ((unsigned long long)(pslot & 0x3FF) << 22) |
           ((unsigned long long)(epoch & 0x3FF) << 12) | (unsigned long long)(rnd & 0xFFFu);
}
__device__ __forceinline__ bool wave_item_ok(unsigned long long w, unsigned int rnd, int epoch) {
    return (unsigned int)(w & 0x3FFFFFull) == ((((unsigned int)epoch & 0x3FFu) << 12) | (rnd & 0xFFFu));
}

__device__ __forceinline__ unsigned long long wave_timer() {
    unsigned long long t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); return t;
}
// In-kernel timeline (measurement builds only: `python -m paper_2607_08642_b200.build --trace` compiles the separate
// libdominotree_trace.so with -DDT_TRACE, read by `bench.py --trace`): thread 0 of GRU CTA 0 (role 0) and of request
// CTA 0 (role 1) stamp %globaltimer at fixed points of the first kWvTraceSteps steps.
constexpr int kWvTraceSteps = 64, kWvTraceStamps = 16;
#ifdef DT_TRACE
__device__ unsigned long long g_wv_trace[2][kWvTraceSteps][kWvTraceStamps];
__device__ unsigned long long g_wv_trace_sink[kWvThreads];
// branch-free on purpose: a thread-0-only branch would leave its warp diverged and slow every warp collective after it
#define WV_TR(role, cond, step, i) do { \
        const bool wv_on__ = (threadIdx.x == 0) && (cond) && (step) < kWvTraceSteps; \
        unsigned long long *wv_dst__ = wv_on__ ? &g_wv_trace[role][wv_on__ ? (step) : 0][i] : &g_wv_trace_sink[threadIdx.x]; \
        *wv_dst__ = wave_timer(); } while (0)
#else
#define WV_TR(role, cond, step, i) do { } while (0)
#endif
constexpr unsigned long long kWvTimeoutNs = 4000000000ull;     // 4 s: far beyond any round; a slip fails instead of hanging

// TMEM -> registers: 8 consecutive fp32 columns of this thread's lane
__device__ __forceinline__ void wave_tmem_ld8(uint32_t taddr, float (&v)[8]) {
    uint32_t r[8];
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
                 : "r"(taddr) : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
    for (int i = 0; i < 8; ++i) v[i] = __uint_as_float(r[i]);
}

// shared-memory footprints (bytes)
__host__ __device__ inline size_t wave_gru_smem(int g, int r) {
    const size_t r16 = (size_t)((r + 15) & ~15);
    (void)r16;
    const size_t rpc = (size_t)16 * ((r + 16 * kWvCS - 1) / (16 * kWvCS));
    return (size_t)48 * g * 2 + (size_t)kWvRingBytes + (size_t)kWvCS * 4096 + (size_t)kWvCS * rpc * 32 +
           (size_t)(5 * kWvNP + 3 * kWvMaxBatch + 8) * 4 + 20 * 8 + 64 + 1024;
}
__host__ __device__ inline size_t wave_slice_bytes(int r, int M) {
    return (size_t)((M + 7) / 8) * (size_t)((r + 63) / 64) * 1024;
}
__host__ __device__ inline size_t wave_req_smem(int r, int M, int N, int k, int W, int e_max, int n_slices) {
    auto al = [](size_t x) { return (x + 15) / 16 * 16; };
    size_t s = (size_t)n_slices * wave_slice_bytes(r, M) + 2 * al((size_t)n_slices * M * 4);
    s += al((size_t)e_max * k * 8) + al((size_t)e_max * k * 2) + 4 * al((size_t)e_max * 4) + 2 * al((size_t)e_max * 4) + al((size_t)e_max * 8);
    s += 4 * al((size_t)N * 4);
    s += al((size_t)W * r * 4) + al((size_t)W * M * 4) + al((size_t)W * M * 8) + al((size_t)W * M);
    s += al((size_t)4 * kWvMaxW * 4) + al(256);
    return s + 1024;
}

// bounded spin on a hand-over word; returns false on timeout (and raises *err)
template <typename F>
__device__ __forceinline__ bool wave_spin(F ready, unsigned int *err) {
    if (ready()) return true;
    const unsigned long long t0 = wave_timer();
    unsigned int n = 0;
    while (!ready()) {
        if (((++n) & 1023u) == 0u) {
            if (ld_relaxed_u32(err) != 0u) return false;
            if (wave_timer() - t0 > kWvTimeoutNs) { atomicExch(err, 1u); return false; }
        }
    }
    return true;
}

// ------------------------------------------------------------------------------------------ GRU role
// thread-block cluster helpers (the GRU CTAs run in clusters of kWvCS: the W1 partial is reduced over the cluster's
// 16 kWvCS units inside the tensor core after an all-gather of the new states through distributed shared memory)
__device__ __forceinline__ uint32_t wave_cluster_rank() { uint32_t r; asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ uint32_t wave_mapa(uint32_t saddr, uint32_t rank) {
    uint32_t r; asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(saddr), "r"(rank)); return r;
}
__device__ __forceinline__ void wave_st_cluster_v2(uint32_t addr, uint2 v) {
    asm volatile("st.shared::cluster.v2.b32 [%0], {%1, %2};" ::"r"(addr), "r"(v.x), "r"(v.y) : "memory");
}
__device__ __forceinline__ void wave_cluster_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
__device__ __forceinline__ void wave_cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }

__device__ __forceinline__ void wave_tmem_ld16(uint32_t taddr, float (&v)[16]) {
    uint32_t r[16];
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
                   "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
                 : "r"(taddr) : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
    for (int i = 0; i < 16; ++i) v[i] = __uint_as_float(r[i]);
}
// make the mbarrier count this thread's earlier cp.async copies: it arrives once they have landed (the barrier's expected
// count includes these arrivals)
__device__ __forceinline__ void wave_cp_async_arrive(uint32_t mbar_addr) {
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(mbar_addr) : "memory");
}
__device__ __forceinline__ void wave_tmem_ld16x2(uint32_t ta, uint32_t tb, float (&va)[16], float (&vb)[16]) {
    uint32_t r[32];
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
                   "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
                 : "r"(ta) : "memory");
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
                 : "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]),
                   "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
                 : "r"(tb) : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
    for (int i = 0; i < 16; ++i) { va[i] = __uint_as_float(r[i]); vb[i] = __uint_as_float(r[16 + i]); }
}
template <int N> __device__ __forceinline__ void wave_cp_wait_n(int n) {
    if (n >= N) cp_async_wait<N>();
    else if constexpr (N > 0) wave_cp_wait_n<N - 1>(n);
}

__device__ __forceinline__ void wave_gru_role(const WaveParams &p, unsigned char *smem_raw) {
    const ExpandParams &e = p.e;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int g = e.g, r = e.r, batch = e.batch;
    const int cta = blockIdx.x, u0 = cta * 16;
    const int crank = (int)wave_cluster_rank(), cbase = cta - crank;   // rank in the cluster, first CTA of the cluster
    const size_t stride = (size_t)p.slot_stride;
    const int n_kc = g / kWvKC;
    const int rpc = p.rpc;                                             // rows of W1 this CTA reduces (multiple of 16)

    // carve (smem_raw is 1024-byte aligned by the kernel)
    unsigned char *sW = smem_raw;                                     // W_hh slice, K-major sw128: [6 row groups][g/64 atoms][1 KB]
    const uint32_t sboW = (uint32_t)g * 16;                           // bytes between 8-row groups
    unsigned char *sRing = sW + (size_t)48 * g * 2;                   // [slot][2 k-blocks][N / 8 row groups][1 KB]
    float *sH = reinterpret_cast<float *>(sRing);                    // [48][kWvLdH] hidden-half pre-activations (aliases the ring after D1)
    unsigned char *sS2 = sRing + kWvRingBytes;                        // [kWvCS][16 groups][2 k-halves][8 rows][16 B]: new states of
                                                                      // the cluster's 16 kWvCS units (block c written by rank c)
    unsigned char *sW1 = sS2 + (size_t)kWvCS * 4096;                  // [kWvCS][rpc/8 groups][2 k-halves][8 rows][16 B]
    int *sRow = reinterpret_cast<int *>(sW1 + (size_t)kWvCS * rpc * 32);   // [64] request * stride + parent slot  (state row)
    int *sNew = sRow + kWvNP;                                         // [64] request * stride + new slot
    int *sTok = sNew + kWvNP;                                         // [64]
    int *sIt = sTok + kWvNP;                                          // [64] request * kWvMaxW + item index (partial row)
    int *sPz = sIt + kWvNP;                                           // [64] parent slot is the zero slot
    int *sCnt = sPz + kWvNP;                                          // [128] items per request this step
    int *sOff = sCnt + kWvMaxBatch;                                   // [129] exclusive prefix
    int *sFirst = sOff + kWvMaxBatch + 4;                             // [128] first new state slot per request
    unsigned long long *mbar = reinterpret_cast<unsigned long long *>(sFirst + kWvMaxBatch);   // [0..7] slot full, [8] D1, [9] D2, [10..17] slot empty
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(mbar + 20);
    int *sCtl = reinterpret_cast<int *>(tmem_slot + 2);               // [0] items this step, [1] requests not done, [2] abort, [4..7] live masks

    {   // resident weights
        const __nv_bfloat16 *whh = reinterpret_cast<const __nv_bfloat16 *>(e.w_hh);
        const int vpr = g / 8;
        for (int i = tid; i < 48 * vpr; i += kWvThreads) {
            const int m = i / vpr, c = i - m * vpr;                // local row m = gate * 16 + unit, 16-byte piece c
            const int gate = m >> 4, ul = m & 15;
            const uint4 q = ld_ro_v4(whh + ((size_t)gate * g + u0 + ul) * g + (size_t)c * 8);
            *reinterpret_cast<uint4 *>(sW + (size_t)(m >> 3) * sboW + (size_t)(c >> 3) * 1024 + (m & 7) * 128 + (((c & 7) ^ (m & 7)) << 4)) = q;
        }
        // W1 rows [crank * rpc, crank * rpc + rpc) x the 16 units of every CTA of the cluster (one K = 16 step each)
        const __nv_bfloat16 *w1 = reinterpret_cast<const __nv_bfloat16 *>(e.w1);
        for (int i = tid; i < kWvCS * rpc * 16; i += kWvThreads) {
            const int c = i / (rpc * 16), rem = i - c * rpc * 16;
            const int jl = rem >> 4, ul = rem & 15, j = crank * rpc + jl;
            const __nv_bfloat16 v = (j < r) ? w1[(size_t)j * (e.d + g) + e.d + (cbase + c) * 16 + ul] : __float2bfloat16_rn(0.f);
            *reinterpret_cast<__nv_bfloat16 *>(sW1 + (size_t)c * rpc * 32 + (size_t)(jl >> 3) * 256 + (ul >> 3) * 128 + (jl & 7) * 16 + (ul & 7) * 2) = v;
        }
        for (int i = tid; i < kWvCS * 1024; i += kWvThreads) reinterpret_cast<uint32_t *>(sS2)[i] = 0u;
        if (tid == 0) {
            for (int i = 0; i < 8; ++i) { tc::mbar_init(tc::smem_u32(mbar + i), kWvThreads - 128); tc::mbar_init(tc::smem_u32(mbar + 10 + i), 4); }
            tc::mbar_init(tc::smem_u32(mbar + 8), 4);
            tc::mbar_init(tc::smem_u32(mbar + 9), 1);
            tc::mbar_init_fence();
            sCtl[2] = 0;
        }
        if (warp == 0) tc::tmem_alloc<kWvTmemCols>(tmem_slot);
    }
    tc::fence_proxy_async();
    tc::fence_before_sync();
    __syncthreads();
    tc::fence_after_sync();
    wave_cluster_arrive();                                            // peers' sS2 is zeroed before anyone stores into it
    wave_cluster_wait();
    const uint32_t tmem = *tmem_slot;
    const uint32_t idesc2 = tc::make_idesc_bf16(128, rpc);
    const uint32_t mb0 = tc::smem_u32(mbar);
    const uint64_t descW0 = tc::make_desc_sw128(tc::smem_u32(sW), sboW), descR0 = tc::make_desc_sw128(tc::smem_u32(sRing), 1024);
    const uint64_t descS2 = tc::make_desc(tc::smem_u32(sS2), 128, 256), descW1 = tc::make_desc(tc::smem_u32(sW1), 128, 256);
    uint32_t ph_full = 0, ph_empty = 0, ph_d1 = 0, ph_d2 = 0;      // mbarrier phases (each role keeps the bits of the barriers it waits on)
    bool pend2 = false;                                             // a cluster arrive (sS2 consumed) awaits its wait

    // epilogue geometry: TMEM lane quadrant q4, unit half hsel; lanes 0..15 hold the hi rows of nodes 16 q4 + lane,
    // lanes 16..31 the lo rows of the same nodes; after the hi + lo exchange lane < 16 finishes units 8 hsel + 0..3,
    // lane >= 16 units 8 hsel + 4..7
    const int q4 = warp & 3, hsel = warp >> 2, il = lane & 15, uh = lane >> 4;
    const int my_node = 16 * q4 + il;
    const int my_u = 8 * hsel + 4 * uh;                              // first of this thread's 4 local units
    const uint32_t tlane = (uint32_t)(32 * q4) << 16;
    // where this thread's new states go in every cluster CTA's sS2 (block crank): rows 32 q4 + il (hi) and + 16 (lo)
    uint32_t s2_hi[kWvCS], s2_lo[kWvCS];
    {
        const int rh = 32 * q4 + il, rl = rh + 16;
        const uint32_t oh = (uint32_t)(crank * 4096 + (rh >> 3) * 256 + hsel * 128 + (rh & 7) * 16 + uh * 8);
        const uint32_t ol = (uint32_t)(crank * 4096 + (rl >> 3) * 256 + hsel * 128 + (rl & 7) * 16 + uh * 8);
#pragma unroll
        for (int c = 0; c < kWvCS; ++c) {
            s2_hi[c] = wave_mapa(tc::smem_u32(sS2) + oh, (uint32_t)c);
            s2_lo[c] = wave_mapa(tc::smem_u32(sS2) + ol, (uint32_t)c);
        }
    }

    // every GRU CTA walks the K chunks of a pass in its own rotation: 64 CTAs asking L2 for the same lines at the same
    // moment is a hot spot; the order depends on the CTA only, never on the batch, so results stay batch-invariant
    const int kshift = cta % n_kc;
    const unsigned int rnd = ld_relaxed_u32(p.round_ctr), fbase = rnd << 10;
    for (int s = 0;; ++s) {
        // ---- headers of step s: one lane per request
        if (warp < 4) {
            const int b = warp * 32 + lane;
            int cnt = 0, first = 0, live = 0;
            if (b < batch) {
                unsigned long long hdr = 0ull;
                const unsigned long long *hp = p.desc + (size_t)b * kWvDescWords;
                const bool ok = wave_spin([&] { hdr = ld_relaxed_u64(hp); return wave_hdr_ok(hdr, rnd, s + 1); }, p.err);
                if (!ok) sCtl[2] = 1;
                else if (!((hdr >> 15) & 1ull)) { cnt = (int)(hdr & 0x7FFFull); first = (int)((hdr >> 16) & 0xFFFull); live = 1; }
            }
            sCnt[b] = cnt; sFirst[b] = first;
            const unsigned int lv = __ballot_sync(0xffffffffu, live != 0);
            if (lane == 0) sCtl[4 + warp] = (int)lv;
        }
        __syncthreads();
        if (warp == 0) {                                            // exclusive prefix of the counts (4 per lane)
            int c[4], sum = 0;
#pragma unroll
            for (int i = 0; i < 4; ++i) { c[i] = sCnt[lane * 4 + i]; sum += c[i]; }
            int inc = sum;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { const int v = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += v; }
            int run = inc - sum;
#pragma unroll
            for (int i = 0; i < 4; ++i) { sOff[lane * 4 + i] = run; run += c[i]; }
            if (lane == 31) { sOff[kWvMaxBatch] = inc; sCtl[0] = inc; }
            if (lane == 0) sCtl[1] = (sCtl[4] | sCtl[5] | sCtl[6] | sCtl[7]) != 0;
        }
        __syncthreads();
        const int total = sCtl[0];
        if (sCtl[2] || !sCtl[1]) break;                              // abort, or every request is done
        WV_TR(0, cta == 0, s, 0);

        for (int p0 = 0; p0 < total; p0 += kWvNP) {
            const int n = min(kWvNP, total - p0);
            // ---- items of this pass: thread i < n fetches item p0 + i
            if (tid < kWvNP) {
                int row = 0, nw = 0, tok = 0, it = 0, pz = 1;
                if (tid < n) {
                    const int qi = p0 + tid;
                    int lo = 0, hi = kWvMaxBatch - 1;                // last b with sOff[b] <= qi: its list is not empty
                    while (lo < hi) { const int mid = (lo + hi + 1) >> 1; if (sOff[mid] <= qi) lo = mid; else hi = mid - 1; }
                    const int b = lo, j = qi - sOff[b];
                    unsigned long long w = 0ull;
                    const unsigned long long *ip = p.desc + (size_t)b * kWvDescWords + 1 + j;
                    const bool ok = wave_spin([&] { w = ld_relaxed_u64(ip); return wave_item_ok(w, rnd, s + 1); }, p.err);
                    if (!ok) sCtl[2] = 1;
                    const int ps = (int)((w >> 22) & 0x3FFull);
                    tok = (int)(w >> 32);
                    tok = min(max(tok, 0), e.V - 1);
                    row = b * (int)stride + ps; nw = b * (int)stride + sFirst[b] + j; it = b * kWvMaxW + j; pz = (ps == 0);
                }
                sRow[tid] = row; sNew[tid] = nw; sTok[tid] = tok; sIt[tid] = it; sPz[tid] = pz;
            }
            __syncthreads();
            WV_TR(0, cta == 0 && p0 == 0, s, 1);

            // ---- this pass: the parents' states are operand B of D1[64 x N] = W_hh slice . [S_hi | S_lo]^T with N = 2 nh columns
            // (hi halves of the nh = 4 ceil(n / 4) nodes, then their lo halves); ring slots of N / 8 row groups per k-block
            const int nh = 4 * ((n + 3) >> 2), N = 2 * nh;
            const int kb_bytes = (N >> 3) * 1024, slot_bytes = 2 * kb_bytes;
            const int nslot = min(min(n_kc, 8), kWvRingBytes / slot_bytes);
            const uint32_t idesc1 = tc::make_idesc_bf16(64, N);
            // independent D1 accumulators, npad columns apart; the same four whatever N is, so that the association of the
            // K sum (and with it every bit of the result) does not depend on how many nodes share the pass
            constexpr int NA = 4, npad = kWvTmemCols / NA;
            // ---- epilogue operands (input half from P, previous state): issued now, consumed after the MMAs
            float4 pr = make_float4(0.f, 0.f, 0.f, 0.f), pz4 = pr, pn = pr, hp = pr;
            const bool mine = (my_node < n);
            if (mine) {
                const float *prow = e.P + (size_t)sTok[my_node] * 3 * g + u0 + my_u;
                pr = __ldg(reinterpret_cast<const float4 *>(prow));
                pz4 = __ldg(reinterpret_cast<const float4 *>(prow + g));
                pn = __ldg(reinterpret_cast<const float4 *>(prow + 2 * g));
                if (!sPz[my_node]) hp = __ldcg(reinterpret_cast<const float4 *>(p.s32 + (size_t)sRow[my_node] * g + u0 + my_u));
            }
            WV_TR(0, cta == 0 && p0 == 0, s, 2);

            // ---- D1[64 x N] = W_hh slice . [S_hi | S_lo]^T, K streamed through the ring by a warp-specialised pipeline with no
            // CTA barrier inside: warps 2..7 produce (cp.async into the slot, completion tracked by the slot's `full`
            // mbarrier), lane 0 of warps 0 and 1 consume (tcgen05.mma, tcgen05.commit on the slot's `empty` mbarrier).
            if (warp >= 4) {
                // producer: 16-byte piece ptid & 15 of operand rows rho = (ptid >> 4) + 8 i
                const int ptid = tid - 128, piece = ptid & 15, kb = piece >> 3, pc = piece & 7;
                const __nv_bfloat16 *src[16];
#pragma unroll
                for (int i = 0; i < 16; ++i) {
                    const int rho = (ptid >> 4) + 8 * i;
                    const int hl = (rho >= nh), node = rho - (hl ? nh : 0);
                    src[i] = nullptr;
                    if (rho < N && node < n) src[i] = (hl ? p.s_lo : p.s_hi) + (size_t)sRow[node] * g + (size_t)piece * 8;
                }
                const int r7 = (ptid >> 4) & 7;                      // rho & 7 is the same for all 16 rows of a thread
                const uint32_t doff = (uint32_t)(kb * kb_bytes + r7 * 128 + ((pc ^ r7) << 4));
#pragma unroll 1
                for (int kc = 0; kc < n_kc; ++kc) {
                    const int sl = kc % nslot;
                    if (kc >= nslot) {                           // the MMAs of the slot's previous chunk have read it
                        tc::mbar_wait(mb0 + 80 + 8 * sl, (ph_empty >> sl) & 1u);
                        ph_empty ^= 1u << sl;
                    }
                    unsigned char *dst = sRing + (size_t)sl * slot_bytes + doff;
                    const size_t k0 = (size_t)((kc + kshift) % n_kc) * kWvKC;
#pragma unroll
                    for (int i = 0; i < 16; ++i)
                        if (src[i]) cp_async16(dst + i * 1024, src[i] + k0);   // rho >> 3 = i
                    wave_cp_async_arrive(mb0 + 8 * sl);
                }
            } else if (lane == 0) {
                // consumer: warp w issues K = 16 steps 2 w, 2 w + 1 of every chunk into its own accumulator D1[w] (a thread needs
                // ~120 cycles to issue one tcgen05.mma and ~200 for a commit, so four threads share the work)
                const int kbw = warp >> 1, s40 = (warp & 1) * 2;
#pragma unroll 1
                for (int kc = 0; kc < n_kc; ++kc) {
                    const int sl = kc % nslot;
                    tc::mbar_wait(mb0 + 8 * sl, (ph_full >> sl) & 1u);
                    ph_full ^= 1u << sl;
                    tc::fence_proxy_async();
                    tc::fence_after_sync();
                    const uint64_t da = descW0 + (uint64_t)((((kc + kshift) % n_kc) * 2 + kbw) * 64 + s40 * 2);
                    const uint64_t db = descR0 + (uint64_t)((sl * slot_bytes + kbw * kb_bytes) / 16 + s40 * 2);
                    tc::mma_bf16(tmem + warp * npad, da, db, idesc1, kc ? 1u : 0u);
                    tc::mma_bf16(tmem + warp * npad, da + 2, db + 2, idesc1, 1u);
                    if (kc + nslot < n_kc) tc::commit(mb0 + 80 + 8 * sl);        // this slot will be refilled
                    if (kc == n_kc - 1) tc::commit(mb0 + 64);
                }
            }
            __syncwarp();
            tc::mbar_wait(mb0 + 64, ph_d1); ph_d1 ^= 1u;
            tc::fence_after_sync();
            __syncwarp();
            WV_TR(0, cta == 0 && p0 == 0, s, 3);

            // ---- TMEM -> shared: an M = 64 accumulator keeps row 16 q + i in lane 32 q + i (i < 16), so quadrant q holds gate q
            // (r, z, n) of the 16 units; the two accumulators and the hi / lo column blocks are added here (fixed order)
            if (q4 < 3 && 16 * hsel < nh) {
#pragma unroll 1
                for (int c16 = hsel; 16 * c16 < nh; c16 += 2) {
                    float v0[16], v1[16], v2[16];
#pragma unroll
                    for (int c = 0; c < 16; ++c) v0[c] = 0.f;
#pragma unroll 1
                    for (int a = 0; a < NA; ++a) {                   // accumulators in index order, hi then lo column block
                        wave_tmem_ld16x2(tmem + tlane + a * npad + 16 * c16, tmem + tlane + a * npad + nh + 16 * c16, v1, v2);
#pragma unroll
                        for (int c = 0; c < 16; ++c) v0[c] += v1[c] + v2[c];
                    }
                    if (lane < 16) {
                        float4 *dst = reinterpret_cast<float4 *>(sH + (size_t)(16 * q4 + lane) * kWvLdH + 16 * c16);
#pragma unroll
                        for (int c = 0; c < 4; ++c) dst[c] = make_float4(v0[4 * c], v0[4 * c + 1], v0[4 * c + 2], v0[4 * c + 3]);
                    }
                }
            }
            tc::fence_before_sync();
            __syncthreads();
            // ---- gates (reading A2): thread = (node 16 q4 + il, units 8 hsel + 4 uh ..)
            float acc[12];
#pragma unroll
            for (int gate = 0; gate < 3; ++gate)
#pragma unroll
                for (int c = 0; c < 4; ++c) acc[gate * 4 + c] = sH[(size_t)(16 * gate + my_u + c) * kWvLdH + my_node];
            {
                const float prv[4] = {pr.x, pr.y, pr.z, pr.w}, pzv[4] = {pz4.x, pz4.y, pz4.z, pz4.w};
                const float pnv[4] = {pn.x, pn.y, pn.z, pn.w}, hpv[4] = {hp.x, hp.y, hp.z, hp.w};
                float hn[4];
                __nv_bfloat16 bh[4], bl[4];
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    const float rg = sigmoidf_fast(prv[c] + acc[c]);
                    const float zg = sigmoidf_fast(pzv[c] + acc[4 + c]);
                    const float ng = tanhf_fast(pnv[c] + rg * acc[8 + c]);
                    hn[c] = mine ? ((1.0f - zg) * ng + zg * hpv[c]) : 0.f;
                    bh[c] = __float2bfloat16_rn(hn[c]);
                    bl[c] = __float2bfloat16_rn(hn[c] - __bfloat162float(bh[c]));
                }
                uint2 ph, pl;
                ph.x = (uint32_t)__bfloat16_as_ushort(bh[0]) | ((uint32_t)__bfloat16_as_ushort(bh[1]) << 16);
                ph.y = (uint32_t)__bfloat16_as_ushort(bh[2]) | ((uint32_t)__bfloat16_as_ushort(bh[3]) << 16);
                pl.x = (uint32_t)__bfloat16_as_ushort(bl[0]) | ((uint32_t)__bfloat16_as_ushort(bl[1]) << 16);
                pl.y = (uint32_t)__bfloat16_as_ushort(bl[2]) | ((uint32_t)__bfloat16_as_ushort(bl[3]) << 16);
                if (mine) {                                          // publish S_new: fp32 and the bf16 hi/lo split
                    const size_t o = (size_t)sNew[my_node] * g + u0 + my_u;
                    __stcg(reinterpret_cast<float4 *>(p.s32 + o), make_float4(hn[0], hn[1], hn[2], hn[3]));
                    __stcg(reinterpret_cast<uint2 *>(p.s_hi + o), ph);
                    __stcg(reinterpret_cast<uint2 *>(p.s_lo + o), pl);
                }
                // all-gather over the cluster: block `crank` of every cluster CTA's sS2 (operand A of the W1 GEMM)
                if (pend2) { wave_cluster_wait(); pend2 = false; }   // every peer's previous W1 GEMM has read its sS2
#pragma unroll
                for (int c = 0; c < kWvCS; ++c) { wave_st_cluster_v2(s2_hi[c], ph); wave_st_cluster_v2(s2_lo[c], pl); }
            }
            wave_cluster_arrive();
            wave_cluster_wait();
            tc::fence_proxy_async();
            tc::fence_before_sync();
            __syncthreads();
            WV_TR(0, cta == 0 && p0 == 0, s, 4);
            // ---- D2[128 x rpc] = S_new[rows, the cluster's 16 kWvCS units] . W1[my rpc rows, d + those units]^T:
            // one K = 16 step per cluster CTA, accumulated in rank order
            if (tid == 0) {
                tc::fence_after_sync();
#pragma unroll
                for (int c = 0; c < kWvCS; ++c)
                    tc::mma_bf16(tmem, descS2 + (uint64_t)(c * 256), descW1 + (uint64_t)(c * rpc * 2), idesc2, c ? 1u : 0u);   // D1's columns are dead
                tc::commit(mb0 + 72);
            }
            tc::mbar_wait(mb0 + 72, ph_d2); ph_d2 ^= 1u;
            tc::fence_after_sync();
            __syncwarp();
            wave_cluster_arrive(); pend2 = true;                     // my sS2 may be overwritten by the next pass
            WV_TR(0, cta == 0 && p0 == 0, s, 5);
            {
                // partial[item][cluster][crank * rpc + col]: lanes < 16 store columns 0..7 of a 16-column block, lanes >= 16 8..15
                float *prow = p.partial + ((size_t)(mine ? sIt[my_node] : 0) * p.P + (cta / kWvCS)) * r + crank * rpc;
#pragma unroll 1
                for (int blk = hsel; blk < rpc / 16; blk += 2) {
                    float v[16];
                    wave_tmem_ld16(tmem + tlane + 16 * blk, v);
#pragma unroll
                    for (int c = 0; c < 16; ++c) v[c] += __shfl_xor_sync(0xffffffffu, v[c], 16);
                    if (mine) {
                        const int col = 16 * blk + 8 * uh;
                        const float4 o0 = uh ? make_float4(v[8], v[9], v[10], v[11]) : make_float4(v[0], v[1], v[2], v[3]);
                        const float4 o1 = uh ? make_float4(v[12], v[13], v[14], v[15]) : make_float4(v[4], v[5], v[6], v[7]);
                        if (crank * rpc + col + 3 < r) __stcg(reinterpret_cast<float4 *>(prow + col), o0);
                        if (crank * rpc + col + 7 < r) __stcg(reinterpret_cast<float4 *>(prow + col + 4), o1);
                    }
                }
            }
            tc::fence_before_sync();
            __syncthreads();
            WV_TR(0, cta == 0 && p0 == 0, s, 6);
        }
        if (sCtl[2]) break;
        if (tid == 0) { fence_release_gpu(); st_relaxed_u32(p.flags + (size_t)cta * kFusFlagStride, fbase + (unsigned int)(s + 1)); }
        WV_TR(0, cta == 0, s, 7);
    }
    __syncthreads();
    if (pend2) wave_cluster_wait();
    if (warp == 0) tc::tmem_free<kWvTmemCols>(tmem);
    // every CTA of the grid has read the counter: a request is done only after all GRU CTAs finished step 0
    if (cta == 0 && tid == 0) st_relaxed_u32(p.round_ctr, rnd + 1u);
}

// -------------------------------------------------------------------------------------- request role
struct WaveCtl {
    int n_exp;          // expansions allocated so far (expansion 0 = the root)
    int c;              // committed pops: slots 1 .. c are final
    int n_items;        // items published for the coming step
    int done, n_valid, n_stage, abort_, pad;
    int slDepth[kWvMaxSlices];      // depth whose candidate rows a slice holds (-1 = empty)
    int slUsed[kWvMaxSlices];       // last step that needs the slice
    int stage[kWvMaxSlices];        // slices to fill before the coming step
    signed char d2s[DT_MAX_L];      // depth -> slice (-1 = not resident)
};

__device__ __forceinline__ void wave_req_role(const WaveParams &p, unsigned char *smem_raw) {
    const ExpandParams &e = p.e;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int b = blockIdx.x - p.n_gru;
    const int r = e.r, M = e.M, k = e.k, N = e.N, L = e.L, B = e.B;
    const int W = p.W, nsl = p.n_slices, e_max = p.e_max, P = p.P;
    const unsigned int rnd = ld_relaxed_u32(p.round_ctr), fbase = rnd << 10;
    const size_t slice_bytes = wave_slice_bytes(r, M);
    const int Ka = (r + 63) / 64, nvec = r / 8;

    size_t off = 0;
    auto carve = [&](size_t bytes) { unsigned char *q = smem_raw + off; off += (bytes + 15) / 16 * 16; return q; };
    unsigned char *sW2 = carve((size_t)nsl * slice_bytes);
    int *slTok = reinterpret_cast<int *>(carve((size_t)nsl * M * 4));
    float *slBase = reinterpret_cast<float *>(carve((size_t)nsl * M * 4));
    unsigned long long *cKey = reinterpret_cast<unsigned long long *>(carve((size_t)e_max * k * 8));   // children of expansion x, best first
    short *cExp = reinterpret_cast<short *>(carve((size_t)e_max * k * 2));                             // expansion of that child, -1 = none
    int *eTok = reinterpret_cast<int *>(carve((size_t)e_max * 4));
    int *ePar = reinterpret_cast<int *>(carve((size_t)e_max * 4));
    int *eDep = reinterpret_cast<int *>(carve((size_t)e_max * 4));
    float *eSco = reinterpret_cast<float *>(carve((size_t)e_max * 4));
    unsigned int *simC = reinterpret_cast<unsigned int *>(carve((size_t)e_max * 4));   // replay state at the commit point
    unsigned int *simT = reinterpret_cast<unsigned int *>(carve((size_t)e_max * 4));   // ... of the running replay
    unsigned long long *hT = reinterpret_cast<unsigned long long *>(carve((size_t)e_max * 8));   // head key of every active list (0 = none)
    int *nTok = reinterpret_cast<int *>(carve((size_t)N * 4));
    int *nPar = reinterpret_cast<int *>(carve((size_t)N * 4));
    int *nDep = reinterpret_cast<int *>(carve((size_t)N * 4));
    float *nSco = reinterpret_cast<float *>(carve((size_t)N * 4));
    float *sA = reinterpret_cast<float *>(carve((size_t)W * r * 4));
    float *sZ = reinterpret_cast<float *>(carve((size_t)W * M * 4));
    unsigned long long *sKey = reinterpret_cast<unsigned long long *>(carve((size_t)W * M * 8));   // (z, ~token) of every candidate
    unsigned char *sRank = carve((size_t)W * M);
    int *itE = reinterpret_cast<int *>(carve((size_t)4 * kWvMaxW * 4));
    int *itTok = itE + kWvMaxW, *itPs = itTok + kWvMaxW;
    WaveCtl &ctl = *reinterpret_cast<WaveCtl *>(carve(256));

    const __nv_bfloat16 *w2 = reinterpret_cast<const __nv_bfloat16 *>(e.w2);
    unsigned long long *my_desc = p.desc + (size_t)b * kWvDescWords;

    // fill the slices listed in ctl.stage with the candidate table of their depth: ids, base logits, the M rows of W2
    // (compact code on purpose: the step loop has to stay inside the instruction cache)
    auto stage_slices = [&]() {
        const int ns = ctl.n_stage;
#pragma unroll 1
        for (int q = 0; q < ns; ++q) {
            const int si = ctl.stage[q];
            const size_t row = (size_t)b * L + ctl.slDepth[si];
#pragma unroll 1
            for (int m = tid; m < M; m += kWvThreads) {
                slTok[si * M + m] = e.cand_id[row * M + m];
                slBase[si * M + m] = e.cand_val[row * M + m];
            }
        }
        __syncthreads();
        const int v = tid % nvec, m0 = tid / nvec, dm = kWvThreads / nvec;   // a thread keeps its 16-byte piece, rows m0, m0 + dm, ..
        if (m0 < dm) {
#pragma unroll 1
            for (int q = 0; q < ns; ++q) {
                const int si = ctl.stage[q];
                unsigned char *dst = sW2 + (size_t)si * slice_bytes + (size_t)(v >> 3) * 1024;
                const int *tk = slTok + si * M;
#pragma unroll 2
                for (int m = m0; m < M; m += dm)
                    cp_async16(dst + (size_t)(m >> 3) * Ka * 1024 + (m & 7) * 128 + (((v & 7) ^ (m & 7)) << 4),
                               w2 + (size_t)tk[m] * r + (size_t)v * 8);
            }
        }
        cp_async_commit();
    };

    if (tid == 0) {
        const int root = e.root_tokens[b];
        ctl.n_exp = 1; ctl.c = 0; ctl.n_items = 1; ctl.done = 0; ctl.n_valid = 1; ctl.abort_ = 0;
        for (int i = 0; i < kWvMaxSlices; ++i) { ctl.slDepth[i] = -1; ctl.slUsed[i] = -1; }
        for (int i = 0; i < DT_MAX_L; ++i) ctl.d2s[i] = -1;
        ctl.slDepth[0] = 0; ctl.slUsed[0] = 0; ctl.d2s[0] = 0; ctl.stage[0] = 0; ctl.n_stage = 1;
        eTok[0] = root; ePar[0] = -1; eDep[0] = 0; eSco[0] = 0.f; simC[0] = 0u; simT[0] = 0u;
        nTok[0] = root; nPar[0] = -1; nDep[0] = 0; nSco[0] = 0.f;
        itE[0] = 0;
        // step 0: the root, whose parent state is the zero slot (reading A4)
        st_relaxed_u64(my_desc + 1, wave_item_pack(rnd, 1, 0, min(max(root, 0), e.V - 1)));
        st_relaxed_u64(my_desc, wave_hdr_pack(rnd, 1, 1, 0, 1));
    }
    __syncthreads();
    stage_slices();
    if (tid == 0) ctl.n_stage = 0;                               // every thread read the list before the barrier inside

    for (int s = 0;; ++s) {
        const int n_it = ctl.n_items;
        // C = H W1h^T of the item's depth does not depend on the GRU CTAs: fetch it while waiting for them (A12: row = depth)
        float4 cpre = make_float4(0.f, 0.f, 0.f, 0.f);
        if (tid < n_it * (r >> 2)) {
            const int j = tid / (r >> 2), jq = tid - j * (r >> 2);
            cpre = __ldg(reinterpret_cast<const float4 *>(e.C + ((size_t)b * L + eDep[itE[j]]) * r) + jq);
        }
        if (warp == 0) {
            bool ok = true;
            for (int q = lane; q < p.n_gru; q += 32) {
                const unsigned int *fp = p.flags + (size_t)q * kFusFlagStride;
                ok = wave_spin([&] { return (int)(ld_relaxed_u32(fp) - (fbase + (unsigned int)(s + 1))) >= 0; }, p.err) && ok;
            }
            if (!ok) ctl.abort_ = 1;
        }
        __syncthreads();
        if (ctl.abort_) break;
        WV_TR(1, b == 0, s, 0);

        // ---- a_j = SiLU(C + W1[:, d:] S_j): the P cluster partials are summed in a fixed order (batch-invariant);
        // one thread per (item, four columns), all loads of a thread in flight at once
        {
            const int r4 = r >> 2;
#pragma unroll 1
            for (int pair = tid; pair < n_it * r4; pair += kWvThreads) {
                const int j = pair / r4, jq = pair - j * r4;
                const float4 cv = (pair == tid) ? cpre : __ldg(reinterpret_cast<const float4 *>(e.C + ((size_t)b * L + eDep[itE[j]]) * r) + jq);
                const float4 *pp = reinterpret_cast<const float4 *>(p.partial + ((size_t)(b * kWvMaxW + j) * P) * r) + jq;
                float4 s0 = make_float4(0.f, 0.f, 0.f, 0.f), s1 = s0;
                int q = 0;
                for (; q + 16 <= P; q += 16) {
                    float4 v[16];
#pragma unroll
                    for (int i = 0; i < 16; ++i) v[i] = __ldcg(pp + (size_t)(q + i) * r4);
#pragma unroll
                    for (int i = 0; i < 16; i += 2) {
                        s0.x += v[i].x; s0.y += v[i].y; s0.z += v[i].z; s0.w += v[i].w;
                        s1.x += v[i + 1].x; s1.y += v[i + 1].y; s1.z += v[i + 1].z; s1.w += v[i + 1].w;
                    }
                }
#pragma unroll 1
                for (; q < P; ++q) {
                    const float4 v = __ldcg(pp + (size_t)q * r4);
                    s0.x += v.x; s0.y += v.y; s0.z += v.z; s0.w += v.w;
                }
                float4 o;
                o.x = cv.x + (s0.x + s1.x); o.y = cv.y + (s0.y + s1.y); o.z = cv.z + (s0.z + s1.z); o.w = cv.w + (s0.w + s1.w);
                o.x *= sigmoidf_acc(o.x); o.y *= sigmoidf_acc(o.y); o.z *= sigmoidf_acc(o.z); o.w *= sigmoidf_acc(o.w);
                *reinterpret_cast<float4 *>(sA + (size_t)j * r + 4 * jq) = o;
            }
        }
        cp_async_wait<0>();
        __syncthreads();
        WV_TR(1, b == 0, s, 1);

        // ---- z_m = ((base_m - base_0) + W2[cand_m, :] a) / T_eff   PAPER.md:143-144 (shift-invariant)
        // a warp takes 8 candidate rows (one swizzle row group), four lanes per row
#pragma unroll 1
        for (int j = 0; j < n_it; ++j) {
            const int si = ctl.d2s[eDep[itE[j]]];
            const unsigned char *sl = sW2 + (size_t)si * slice_bytes;
            const float *bs = slBase + si * M;
            const float base0 = bs[0];
            const float *aj = sA + (size_t)j * r;
            const int rw = lane & 7, qq = lane >> 3;
#pragma unroll 1
            for (int rg = warp; rg < (M + 7) / 8; rg += kWvThreads / 32) {
                const unsigned char *rowp = sl + (size_t)rg * Ka * 1024 + rw * 128;
                float acc = 0.f;
#pragma unroll 2
                for (int v = qq; v < nvec; v += 4) {
                    const uint4 q = *reinterpret_cast<const uint4 *>(rowp + (size_t)(v >> 3) * 1024 + (((v & 7) ^ rw) << 4));
                    const float4 a0 = *reinterpret_cast<const float4 *>(aj + (size_t)v * 8);
                    const float4 a1 = *reinterpret_cast<const float4 *>(aj + (size_t)v * 8 + 4);
                    float f[8];
                    unpack8(q, f);
                    acc = fmaf(f[0], a0.x, acc); acc = fmaf(f[1], a0.y, acc); acc = fmaf(f[2], a0.z, acc); acc = fmaf(f[3], a0.w, acc);
                    acc = fmaf(f[4], a1.x, acc); acc = fmaf(f[5], a1.y, acc); acc = fmaf(f[6], a1.z, acc); acc = fmaf(f[7], a1.w, acc);
                }
                acc += __shfl_xor_sync(0xffffffffu, acc, 8);
                acc += __shfl_xor_sync(0xffffffffu, acc, 16);
                const int m = 8 * rg + rw;
                if (qq == 0 && m < M) {
                    const float z = __fdiv_rn((bs[m] - base0) + acc, e.T_eff);
                    sZ[(size_t)j * M + m] = z;
                    sKey[(size_t)j * M + m] = ((unsigned long long)ord_key(z) << 32) | (unsigned long long)(0xFFFFFFFFu - (unsigned int)slTok[si * M + m]);
                }
            }
        }
        __syncthreads();
        WV_TR(1, b == 0, s, 2);

        // ---- top-k by (z desc, token asc): rank by counting over the sortable keys, `tpc` neighbouring lanes per candidate
        {
            const int tot = n_it * M;
            int tpc = 1;
            while (tpc < 8 && tot * tpc * 2 <= kWvThreads) tpc <<= 1;
            const int per = (M + tpc - 1) / tpc;
#pragma unroll 1
            for (int base = 0; base < tot * tpc; base += kWvThreads) {      // block-uniform trip count
                const int idx = base + tid, pair = idx / tpc, part = idx - pair * tpc;
                const bool act = pair < tot;
                const int j = act ? pair / M : 0, m = act ? pair - j * M : 0;
                const unsigned long long *kj = sKey + (size_t)j * M;
                const unsigned long long mk = kj[m];
                int rank = 0;
                if (act) {
                    const int m0 = part * per, m1 = min(M, m0 + per);
                    int q = m0;
                    if (!(m0 & 1))
#pragma unroll 4
                        for (; q + 2 <= m1; q += 2) {
                            const ulonglong2 o = *reinterpret_cast<const ulonglong2 *>(kj + q);
                            rank += (o.x > mk) + (o.y > mk);
                        }
#pragma unroll 1
                    for (; q < m1; ++q) rank += (kj[q] > mk);
                }
                for (int o = 1; o < tpc; o <<= 1) rank += __shfl_xor_sync(0xffffffffu, rank, o);
                if (act && part == 0) sRank[(size_t)j * M + m] = (unsigned char)min(rank, 255);
            }
        }
        __syncthreads();
        // ---- slice log-softmax (reading A1) and the children list: one warp per node
#pragma unroll 1
        for (int j = warp; j < n_it; j += kWvThreads / 32) {
            const int x = itE[j];
            const float *zj = sZ + (size_t)j * M;
            float zmax = -INFINITY;
#pragma unroll 1
            for (int m = lane; m < M; m += 32) zmax = fmaxf(zmax, zj[m]);
            zmax = warp_max(zmax);
            float ssum = 0.f;
#pragma unroll 1
            for (int m = lane; m < M; m += 32) ssum += expf(zj[m] - zmax);
            ssum = warp_sum(ssum);
            const float lse = logf(ssum);
            const float gpar = eSco[x];
            unsigned long long *ck = cKey + (size_t)x * k;
#pragma unroll 1
            for (int m = lane; m < M; m += 32) {
                const int rank = sRank[(size_t)j * M + m];
                if (rank < k) {
                    const float lpm = (zj[m] - zmax) - lse;
                    ck[rank] = ((unsigned long long)ord_key(gpar + lpm) << 32) | (sKey[(size_t)j * M + m] & 0xFFFFFFFFull);
                }
            }
            __syncwarp();
            // the list is kept sorted by the pop comparator itself (fp32 rounding of g + logp may merge two scores)
            unsigned long long mk = 0ull;
            int rk2 = 0;
            if (lane < k) {
                mk = ck[lane];
#pragma unroll 1
                for (int q = 0; q < k; ++q) rk2 += (ck[q] > mk);
            }
            __syncwarp();
            if (lane < k) { ck[rk2] = mk; cExp[(size_t)x * k + lane] = -1; }
        }
        __syncthreads();
        WV_TR(1, b == 0, s, 3);

        // ---- replay the heap from the commit point, nominate, publish (warp 0)
        if (warp == 0) {
            WV_TR(1, b == 0, s, 6);
            const int n_exp = ctl.n_exp;
            int t = ctl.c;
            int n_pops = 0;
            if (s == 0 && lane == 0) { simC[0] = kWvAct; }          // the root is slot 0; its children are known now
            __syncwarp();
#pragma unroll 1
            for (int x = lane; x < n_exp; x += 32) {
                const unsigned int w = simC[x];
                simT[x] = w;
                hT[x] = ((w & kWvAct) && (int)(w & 0xFFu) < k) ? cKey[(size_t)x * k + (w & 0xFFu)] : 0ull;
            }
            __syncwarp();
            WV_TR(1, b == 0, s, 7);
            bool committing = true, finished = false;
            int found = 0, c_new = t;
            const int step_next = s + 1;
            while (true) {
                if (t >= B) { finished = committing; break; }
                // every lane scans the lists it owns and keeps the best head with what the pop needs to know about it
                unsigned long long bk = 0ull;
                unsigned int bw = 0u;
                int be = -1;
#pragma unroll 1
                for (int x = lane; x < n_exp; x += 32) {
                    const unsigned long long key = hT[x];
                    if (key == 0ull) continue;
                    const unsigned int w = simT[x];
                    if (be < 0 || key > bk || (key == bk && (w >> 16) < (bw >> 16))) { bk = key; bw = w; be = x; }
                }
#ifdef DT_TRACE
                const unsigned int wv_am = __activemask();
                const bool wv_pr = (b == 0 && s < kWvTraceSteps && n_pops == 1 && lane == 0);
                *(wv_pr ? &g_wv_trace[1][wv_pr ? s : 0][11] : &g_wv_trace_sink[threadIdx.x]) = wv_am;
                const long long ck0 = clock64();
#endif
                if (__ballot_sync(0xffffffffu, be >= 0) == 0u) { finished = committing; break; }   // the candidate tree ran dry
                // pop comparator of reading A8: score desc, token asc, parent slot asc
                const unsigned int hi = (be >= 0) ? (unsigned int)(bk >> 32) : 0u;
                const unsigned int mh = __reduce_max_sync(0xffffffffu, hi);
                bool el = (be >= 0) && hi == mh;
                const unsigned int ml = __reduce_max_sync(0xffffffffu, el ? (unsigned int)(bk & 0xFFFFFFFFull) : 0u);
                el = el && (unsigned int)(bk & 0xFFFFFFFFull) == ml;
                unsigned int bal = __ballot_sync(0xffffffffu, el);
                if (__popc(bal) > 1) {                              // the same token at the same score under two parents
                    const unsigned int mp = __reduce_min_sync(0xffffffffu, el ? (bw >> 16) : 0xFFFFFFFFu);
                    bal = __ballot_sync(0xffffffffu, el && (bw >> 16) == mp);
                }
                const int wl = __ffs(bal) - 1;
#ifdef DT_TRACE
                *(wv_pr ? &g_wv_trace[1][wv_pr ? s : 0][12] : &g_wv_trace_sink[threadIdx.x]) = (unsigned long long)(clock64() - ck0);
#endif
                // the winning lane looks up its node; the rest of the warp gets the few words it needs by shuffle
                int jc = 0, dep = 0, x = -1;
                if (lane == wl) {
                    jc = (int)(bw & 0xFFu);
                    dep = eDep[be] + 1;
                    x = cExp[(size_t)be * k + jc];
                }
                const int es = __shfl_sync(0xffffffffu, be, wl);
                const unsigned int wv = __shfl_sync(0xffffffffu, bw, wl);
                jc = __shfl_sync(0xffffffffu, jc, wl);
                dep = __shfl_sync(0xffffffffu, dep, wl);
                x = __shfl_sync(0xffffffffu, x, wl);
                const int tok = (int)(0xFFFFFFFFu - ml);
                const bool needs = (x < 0) && dep < L && (t + 1 < B);
                if (committing && needs) {                          // everything before this pop is final
#pragma unroll 1
                    for (int y = lane; y < n_exp; y += 32) simC[y] = simT[y];
                    c_new = t;
                    committing = false;
                    __syncwarp();
                }
                t += 1;
                if (lane == wl) {
                    simT[es] = wv + 1u;
                    hT[es] = (jc + 1 < k) ? cKey[(size_t)es * k + jc + 1] : 0ull;
                    nTok[t] = tok; nPar[t] = (int)(wv >> 16); nDep[t] = dep; nSco[t] = ord_key_inv(mh);
                    if (x >= 0) { simT[x] = kWvAct | ((unsigned int)t << 16); hT[x] = cKey[(size_t)x * k]; }
                }
                bool stop = false;
                if (needs) {                                        // warp-uniform; lane 0 decides, the verdict is broadcast
                    // resources: a state slot (speculative picks leave room for the expansions Algorithm 1 still needs)
                    // and a W2 slice for the node's depth
                    int add = 0;
                    if (lane == 0) {
                        const int xn = n_exp + found;
                        bool can = (xn < e_max) && (found == 0 || xn + 1 + (B - c_new) <= e_max);
                        int si = -1;
                        if (can) {
                            si = ctl.d2s[dep];
                            if (si < 0) {
                                int best = -1, bu = 0x7FFFFFFF;
#pragma unroll 1
                                for (int q = 0; q < nsl; ++q)
                                    if (ctl.slUsed[q] != step_next && ctl.slUsed[q] < bu) { bu = ctl.slUsed[q]; best = q; }
                                si = best;
                                if (si >= 0) {
                                    if (ctl.slDepth[si] >= 0) ctl.d2s[ctl.slDepth[si]] = -1;
                                    ctl.slDepth[si] = dep; ctl.d2s[dep] = (signed char)si;
                                    ctl.stage[ctl.n_stage] = si; ctl.n_stage += 1;
                                }
                            }
                            can = (si >= 0);
                        }
                        if (can) {
                            ctl.slUsed[si] = step_next;
                            cExp[(size_t)es * k + jc] = (short)xn;
                            eTok[xn] = tok; ePar[xn] = es; eDep[xn] = dep; eSco[xn] = ord_key_inv(mh);
                            simC[xn] = 0u; simT[xn] = 0u; hT[xn] = 0ull;
                            itE[found] = xn; itTok[found] = tok; itPs[found] = es + 1;
                            add = 1;
                        }
                    }
                    add = __shfl_sync(0xffffffffu, add, 0);
                    found += add;
                    stop = (add == 0) || found >= W;                // out of slots / slices, or the step is full
                }
                __syncwarp();
#ifdef DT_TRACE
                *(wv_pr ? &g_wv_trace[1][wv_pr ? s : 0][13] : &g_wv_trace_sink[threadIdx.x]) = (unsigned long long)(clock64() - ck0);
#endif
                n_pops += 1;
                if (stop) break;
            }
            WV_TR(1, b == 0, s, 8);
#ifdef DT_TRACE
            { const bool on = (threadIdx.x == 0 && b == 0 && s < kWvTraceSteps); *(on ? &g_wv_trace[1][on ? s : 0][10] : &g_wv_trace_sink[threadIdx.x]) = (unsigned long long)n_pops; }
#endif
            if (finished) {
                if (lane == 0) {
                    ctl.done = 1; ctl.n_valid = t + 1; ctl.n_items = 0; ctl.c = t;
                    st_relaxed_u64(my_desc, wave_hdr_pack(rnd, s + 2, 0, 1, 0));
                    if (p.stats && b == 0) { p.stats[0] = (unsigned int)(s + 1); p.stats[1] = (unsigned int)n_exp; }
                }
            } else {
                if (lane < found) st_relaxed_u64(my_desc + 1 + lane, wave_item_pack(rnd, s + 2, itPs[lane], min(max(itTok[lane], 0), e.V - 1)));
                if (lane == 0) {
                    st_relaxed_u64(my_desc, wave_hdr_pack(rnd, s + 2, n_exp + 1, 0, found));
                    ctl.n_items = found; ctl.n_exp = n_exp + found; ctl.c = c_new;
                }
            }
            WV_TR(1, b == 0, s, 9);
        }
        __syncthreads();
        WV_TR(1, b == 0, s, 4);
        if (ctl.done) break;
        stage_slices();
        WV_TR(1, b == 0, s, 5);
        if (tid == 0) ctl.n_stage = 0;
    }
    __syncthreads();

    // emitter (a9): dead-leaf padding (reading A10), positions, ancestor-or-self mask
    const int n = ctl.abort_ ? 1 : ctl.n_valid;
    const int rpos = e.root_positions ? e.root_positions[b] : 0;
    for (int i = tid; i < N; i += kWvThreads) {
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
    for (int i = tid; i < N * N; i += kWvThreads) mk[i] = 0;
    __syncthreads();
    for (int i = tid; i < N; i += kWvThreads) {
        int a = i;
        while (a >= 0) { mk[(size_t)i * N + a] = 1; a = nPar[a]; }
    }
}

__global__ void __launch_bounds__(kWvThreads, 1) wave_expand_kernel(WaveParams p) {
    extern __shared__ __align__(1024) unsigned char wave_smem[];
    if ((int)blockIdx.x < p.n_gru) wave_gru_role(p, wave_smem);
    else if ((int)blockIdx.x - p.n_gru < p.e.batch) wave_req_role(p, wave_smem);   // CTAs padding the last cluster leave
}

}  // namespace dt
