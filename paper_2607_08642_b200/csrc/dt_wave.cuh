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
// Speculative expansions that turn out useless cost GRU rows, never correctness.
//
// Two CTA roles, co-resident (cooperative launch), hand-over through self-describing words in L2:
//  * GRU CTAs (g / 16 of them, in clusters of 4, weight-stationary: 48 rows of W_hh and the W1[:, d:] block of the
//    cluster's 64 units in shared memory).  Step s: poll every request's item line (one 128-byte line of up to 15
//    self-validating words {token, parent state slot, count, epoch, round}), compact the items, and for passes of up
//    to 64 items run D1[row, gate unit] = S_parent[row, :] . W_hh[gate unit, :]^T on tcgen05 with the NODES as the
//    M dimension (M = 128 rows = 64 nodes x {bf16 hi, bf16 lo}, N = 48, four accumulators in TMEM, one per issuing
//    thread; the states stream from L2 through a cp.async ring in the 128-byte-swizzled K-major layout, completion
//    tracked by mbarriers, no CTA barrier inside), gates in registers with the input half gathered from
//    P = E W_ih^T, new state to L2 and, over distributed shared memory, to every CTA of the
//    cluster, then D2[row, j] = S_new[row, the cluster's 64 units] . W1[j, d + those units]^T: the cluster's
//    split-K share of W1[:, d:] S_new, 16 partial vectors per node.
//  * Request CTAs (one per request) keep the children lists, replay the heap, nominate, and for every
//    expanded node compute a = SiLU(C + sum of partials), z = (base + W2[cand] a) / T_eff over the M
//    candidate rows of the node's depth (rows staged per depth in shared memory "slices"), slice
//    log-softmax (reading A1) and top-k; at the end they emit (a9).
#pragma once
#include "dt_fused.cuh"

namespace dt {

constexpr int kWvThreads = 256;
constexpr int kWvNP = 64;                       // items per GRU pass (N = 128 operand columns: hi and lo of 64 nodes)
constexpr int kWvKC = 128;                      // k per ring slot (two 64-wide swizzle blocks)
constexpr int kWvSlots = 3;
constexpr int kWvSlotBytes = 32 * 1024;         // 128 rows x 128 k x 2 B
constexpr int kWvRingBytes = kWvSlots * kWvSlotBytes;
constexpr int kWvCS = 4;                        // GRU CTAs per thread-block cluster
constexpr int kWvDescWords = 16;                // u64 words per request line: 15 items + one spare, one 128-byte line
constexpr int kWvMaxW = kWvDescWords - 1;
constexpr int kWvMaxBatch = 64;                 // requests per launch (larger batches run as consecutive launches)
constexpr int kWvMaxItems = 512;                // items per step over all requests of a launch (W is clamped to this)
constexpr int kWvTmemCols = 512;                // D1: 4 accumulators of N <= 128 columns; D2 reuses column 0 ..
constexpr int kWvLdH = 68;                      // floats per row of the pre-activation buffer (64 nodes + pad)
constexpr int kWvMaxSlices = 8;
constexpr unsigned int kWvAct = 0x100u;         // replay word: cursor (8) | active (1) | pop slot (16, from bit 16)

struct WaveParams {
    ExpandParams e;
    int n_gru;                     // GRU CTAs = g / 16
    int slot_stride;               // state slots per request (slot 0 = zeros, expansion x lives in slot x + 1)
    int W;                         // items a request may publish per step (1 .. kWvMaxW)
    int n_groups;                  // 1 .. 4: the requests of a launch form groups the GRU CTAs serve in turn (ping-pong)
    int n_slices;                  // W2 slices in a request CTA's shared memory
    int e_max;                     // expansions per request = slot_stride - 1
    int P;                         // partial vectors per item = n_gru / kWvCS (one per cluster of GRU CTAs)
    int rpc;                       // rows of W1 each CTA of a cluster reduces: 16 ceil(r / (16 kWvCS))
    __nv_bfloat16 *s_hi, *s_lo;    // [batch, slot_stride, g]
    float *s32;                    // [batch, slot_stride, g]
    float *partial;                // [batch, kWvMaxW, P, r]
    unsigned long long *desc;      // [batch, kWvDescWords]
    unsigned int *flags;           // [n_gru] one 128-byte line each: steps completed (released: states and partials visible)
    unsigned int *round_ctr;       // rounds this handle has run (tags every hand-over word)
    unsigned int *err;             // set to 1 when a hand-over wait timed out (protocol slip: fail, do not hang)
    unsigned int *stats;           // [4] optional counters of request 0: steps, expansions (measurement aid)
    // adaptive schedule (null selector: always run, width W): the round is `flat` when *sched_sel < sched_thr; on a peaked round
    // the kernel runs only if run_peaked, with the narrower width W_peaked (speculative nodes rarely pay on chains)
    const unsigned int *sched_sel; unsigned int sched_thr; int run_peaked, W_peaked;
};

// ---- hand-over words ---------------------------------------------------------------------------------
// item word j of a request's line:  token (20) | parent state slot (10) | done (1) | count (4) | epoch (10) | round (19)
// Every word is self-validating (relaxed stores need no ordering between them) and carries the request's item count
// of the step, so one poll of the line tells a GRU CTA everything; epoch = step + 1, so zero-initialised memory never
// matches.  Word 0 is written every step (count 0 .. 15, or `done`, which stays valid for the rest of the round).
__device__ __forceinline__ unsigned long long wave_item_pack(unsigned int rnd, int epoch, int count, int done, int pslot, int tok) {
    return ((unsigned long long)((unsigned int)tok & 0xFFFFFu) << 44) | ((unsigned long long)(pslot & 0x3FF) << 34) |
           ((unsigned long long)(done & 1) << 33) | ((unsigned long long)(count & 0xF) << 29) |
           ((unsigned long long)(epoch & 0x3FF) << 19) | (unsigned long long)(rnd & 0x7FFFFu);
}
__device__ __forceinline__ bool wave_item_ok(unsigned long long w, unsigned int rnd, int epoch) {
    return (unsigned int)(w & 0x1FFFFFFFull) == ((((unsigned int)epoch & 0x3FFu) << 19) | (rnd & 0x7FFFFu));
}
__device__ __forceinline__ bool wave_item0_ok(unsigned long long w, unsigned int rnd, int epoch) {
    if ((unsigned int)(w & 0x7FFFFull) != (rnd & 0x7FFFFu)) return false;
    return ((w >> 33) & 1ull) || (int)((w >> 19) & 0x3FFu) == (epoch & 0x3FF);
}
// compacted item in a GRU CTA's shared memory: token (20) | parent slot (10) | new slot (10) | request (7) | item index (4)
__device__ __forceinline__ unsigned long long wave_citem_pack(int tok, int ps, int ns, int b, int j) {
    return (unsigned long long)(unsigned int)tok | ((unsigned long long)ps << 20) | ((unsigned long long)ns << 30) |
           ((unsigned long long)b << 40) | ((unsigned long long)j << 47);
}

constexpr unsigned long long kWvTimeoutNs = 4000000000ull;     // 4 s: far beyond any round; a slip fails instead of hanging

// shared-memory footprints (bytes)
__host__ __device__ inline size_t wave_gru_smem(int g, int r) {
    const size_t rpc = (size_t)16 * ((r + 16 * kWvCS - 1) / (16 * kWvCS));
    return (size_t)48 * g * 2 + (size_t)kWvRingBytes + (size_t)kWvCS * 4096 + (size_t)kWvCS * rpc * 32 +
           (size_t)kWvMaxItems * 12 + (size_t)(2 * kWvMaxBatch + 8) * 4 + 24 * 8 + 64 + 1024;
}
__host__ __device__ inline size_t wave_slice_bytes(int r, int M) {
    return (size_t)((M + 7) / 8) * (size_t)((r + 63) / 64) * 1024;
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
__device__ __forceinline__ void wave_st_cluster_v4(uint32_t addr, uint4 v) {
    asm volatile("st.shared::cluster.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
__device__ __forceinline__ void wave_cluster_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
__device__ __forceinline__ void wave_cluster_arrive_relaxed() { asm volatile("barrier.cluster.arrive.relaxed.aligned;" ::: "memory"); }
__device__ __forceinline__ void wave_cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }

__device__ __forceinline__ unsigned int wave_ld_acquire_u32(const unsigned int *p) {
    unsigned int v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
// TMEM -> registers without the wait: 8 / 16 consecutive fp32 columns of this thread's lane
__device__ __forceinline__ void wave_tmem_ld8_nw(uint32_t taddr, uint32_t (&r)[8]) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
                 : "r"(taddr) : "memory");
}
__device__ __forceinline__ void wave_tmem_ld16_nw(uint32_t taddr, uint32_t (&r)[16]) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
                   "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
                 : "r"(taddr) : "memory");
}
__device__ __forceinline__ void wave_tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
// make the mbarrier count this thread's earlier cp.async copies: it arrives once they have landed (the barrier's expected
// count includes these arrivals)
__device__ __forceinline__ void wave_mbar_arrive(uint32_t mbar_addr) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(mbar_addr) : "memory");
}
__device__ __forceinline__ void wave_cp_async16_s(uint32_t saddr, const void *gmem) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(saddr), "l"(gmem));
}
__device__ __forceinline__ void wave_cp_async_arrive(uint32_t mbar_addr) {
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(mbar_addr) : "memory");
}

__device__ __forceinline__ void wave_gru_role(const WaveParams &p, unsigned char *smem_raw) {
    const ExpandParams &e = p.e;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int g = e.g, r = e.r, batch = e.batch;
    const int cta = blockIdx.x, u0 = cta * 16;
    const int crank = (int)wave_cluster_rank(), cbase = cta - crank;   // rank in the cluster, first CTA of the cluster
    const int stride = p.slot_stride;
    const int n_kc = g / kWvKC;
    const int rpc = p.rpc;                                             // rows of W1 this CTA reduces (multiple of 16)

    // carve (smem_raw is 1024-byte aligned by the kernel)
    unsigned char *sW = smem_raw;                                     // W_hh slice, K-major sw128: [6 row groups][g/64 atoms][1 KB]
    const uint32_t sboW = (uint32_t)g * 16;                           // bytes between 8-row groups
    unsigned char *sRing = sW + (size_t)48 * g * 2;                   // [slot][2 k-blocks][16 row groups][1 KB]
    unsigned long long *sRaw = reinterpret_cast<unsigned long long *>(sRing);   // [batch][16] polled lines (between steps the ring is idle)
    float *sH = reinterpret_cast<float *>(sRing);                    // [48][kWvLdH] hidden-half pre-activations (aliases the ring after D1)
    unsigned char *sS2 = sRing + kWvRingBytes;                        // [kWvCS][16 groups][2 k-halves][8 rows][16 B]: new states of
                                                                      // the cluster's 16 kWvCS units (block c written by rank c)
    unsigned char *sW1 = sS2 + (size_t)kWvCS * 4096;                  // [kWvCS][rpc/8 groups][2 k-halves][8 rows][16 B]
    unsigned long long *sItems = reinterpret_cast<unsigned long long *>(sW1 + (size_t)kWvCS * rpc * 32);   // [kWvMaxItems] compacted items of the step
    int *sCnt = reinterpret_cast<int *>(sItems + kWvMaxItems);        // [64] items per request this step (-1 = done)
    int *sCum = sCnt + kWvMaxBatch;                                   // [64] items per request so far = expansions allocated
    unsigned long long *mbar = reinterpret_cast<unsigned long long *>(sCum + kWvMaxBatch + 8);   // [0..7] slot full, [8..15] slot empty, [16] D1, [17] D2, [18] first group of chunks full
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(mbar + 24);
    int *sCtl = reinterpret_cast<int *>(tmem_slot + 2);               // [2] abort
    uint32_t *sOff = reinterpret_cast<uint32_t *>(sCtl + 8);          // [kWvMaxItems] parent state row of an item, in 16-byte pieces

    {   // resident weights
        const __nv_bfloat16 *whh = reinterpret_cast<const __nv_bfloat16 *>(e.w_hh);
        const int vpr = g / 8;
        // as asynchronous copies, all in flight at once: the weights come from HBM every round (the select has streamed
        // 150 MB through L2 since the last one) and a load -> store loop pays that latency once per iteration
        for (int i = tid; i < 48 * vpr; i += kWvThreads) {
            const int m = i / vpr, c = i - m * vpr;                // local row m = gate * 16 + unit, 16-byte piece c
            const int gate = m >> 4, ul = m & 15;
            cp_async16(sW + (size_t)(m >> 3) * sboW + (size_t)(c >> 3) * 1024 + (m & 7) * 128 + (((c & 7) ^ (m & 7)) << 4),
                       whh + ((size_t)gate * g + u0 + ul) * g + (size_t)c * 8);
        }
        // W1 rows [crank * rpc, crank * rpc + rpc) x the 16 units of every CTA of the cluster (one K = 16 step each)
        const __nv_bfloat16 *w1 = reinterpret_cast<const __nv_bfloat16 *>(e.w1);
        if ((e.d & 7) == 0 && (reinterpret_cast<uintptr_t>(w1) & 15) == 0) {                                      // 8 units = one aligned 16-byte piece of a W1 row (g % 128 == 0)
            for (int i = tid; i < kWvCS * rpc * 2; i += kWvThreads) {
                const int c = i / (rpc * 2), rem = i - c * rpc * 2;
                const int jl = rem >> 1, uh = rem & 1, j = crank * rpc + jl;
                unsigned char *dst = sW1 + (size_t)c * rpc * 32 + (size_t)(jl >> 3) * 256 + uh * 128 + (jl & 7) * 16;
                if (j < r) cp_async16(dst, w1 + (size_t)j * (e.d + g) + e.d + (cbase + c) * 16 + 8 * uh);
                else *reinterpret_cast<uint4 *>(dst) = make_uint4(0u, 0u, 0u, 0u);
            }
        } else {
            for (int i = tid; i < kWvCS * rpc * 16; i += kWvThreads) {
                const int c = i / (rpc * 16), rem = i - c * rpc * 16;
                const int jl = rem >> 4, ul = rem & 15, j = crank * rpc + jl;
                const __nv_bfloat16 v = (j < r) ? w1[(size_t)j * (e.d + g) + e.d + (cbase + c) * 16 + ul] : __float2bfloat16_rn(0.f);
                *reinterpret_cast<__nv_bfloat16 *>(sW1 + (size_t)c * rpc * 32 + (size_t)(jl >> 3) * 256 + (ul >> 3) * 128 + (jl & 7) * 16 + (ul & 7) * 2) = v;
            }
        }
        cp_async_commit();
        cp_async_wait<0>();
        for (int i = tid; i < kWvCS * 1024; i += kWvThreads) reinterpret_cast<uint32_t *>(sS2)[i] = 0u;
        for (int i = tid; i < kWvMaxBatch; i += kWvThreads) sCum[i] = 0;
        if (tid == 0) {
            for (int i = 0; i < 8; ++i) { tc::mbar_init(tc::smem_u32(mbar + i), kWvThreads - 128); tc::mbar_init(tc::smem_u32(mbar + 8 + i), 4); }
            tc::mbar_init(tc::smem_u32(mbar + 16), 4);
            tc::mbar_init(tc::smem_u32(mbar + 17), 1);
            tc::mbar_init(tc::smem_u32(mbar + 18), kWvThreads - 128);
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
    const uint32_t mbFull = mb0, mbEmpty = mb0 + 64, mbD1 = mb0 + 128, mbD2 = mb0 + 136, mbGrp = mb0 + 144;
    const uint64_t descW0 = tc::make_desc_sw128(tc::smem_u32(sW), sboW), descR0 = tc::make_desc_sw128(tc::smem_u32(sRing), 1024);
    const uint64_t descS2 = tc::make_desc(tc::smem_u32(sS2), 128, 256), descW1 = tc::make_desc(tc::smem_u32(sW1), 128, 256);
    uint32_t ph_full = 0, ph_empty = 0, ph_d1 = 0, ph_d2 = 0, ph_grp = 0;      // mbarrier phases (each role keeps the bits of the barriers it waits on)
    bool pend2 = false;                                             // a cluster arrive (sS2 consumed) awaits its wait

    // epilogue geometry: TMEM lane quadrant q4, unit half hsel; lanes 0..15 hold the hi rows of nodes 16 q4 + lane,
    // lanes 16..31 the lo rows of the same nodes (operand row rho = 32 q4 + lane); after the hi + lo exchange lane < 16
    // finishes units 8 hsel + 0..3, lane >= 16 units 8 hsel + 4..7
    const int q4 = warp & 3, hsel = warp >> 2, il = lane & 15, uh = lane >> 4;
    const int my_node = 16 * q4 + il;
    const int my_u = 8 * hsel + 4 * uh;                              // first of this thread's 4 local units
    const uint32_t tlane = (uint32_t)(32 * q4) << 16;
    // where this thread's 16-byte piece of the new states (8 units, hi for lanes < 16, lo for the others) goes in every
    // cluster CTA's sS2 (block crank): row rho, k-half hsel
    uint32_t s2_dst[kWvCS];
    {
        const int rho = 32 * q4 + lane;
        const uint32_t o = (uint32_t)(crank * 4096 + (rho >> 3) * 256 + hsel * 128 + (rho & 7) * 16);
#pragma unroll
        for (int c = 0; c < kWvCS; ++c) s2_dst[c] = wave_mapa(tc::smem_u32(sS2) + o, (uint32_t)c);
    }

    // every GRU CTA walks the K chunks of a pass in its own rotation: 64 CTAs asking L2 for the same lines at the same
    // moment is a hot spot; the order depends on the CTA only, never on the batch, so results stay batch-invariant
    const int kshift = cta % n_kc;
    const unsigned int rnd = ld_relaxed_u32(p.round_ctr), fbase = rnd << 10;
    // Ping-pong: the requests form up to four groups served in turn, so that while the request CTAs of one group score their
    // nodes the GRU CTAs already run the other group's pass (a group's step still costs pass + hand-over + request role,
    // but two groups share that time).  Each group has its own step counter and its own flag word.
    const int G = p.n_groups, gsplit = (batch + G - 1) / G;
    WV_TR(0, cta == 0, kWvTraceSteps - 1, 1);
    int sg[4] = {0, 0, 0, 0};
    bool glive[4] = {true, G > 1, G > 2, G > 3};
    for (int grp = 0; glive[0] || glive[1] || glive[2] || glive[3]; grp = (grp + 1 == G) ? 0 : grp + 1) {
        if (!glive[grp]) continue;
        const int s = sg[grp];
        const int b_lo = grp * gsplit, b_hi = min(batch, b_lo + gsplit);
        // ---- item lines of step s: a half-warp per request, a lane per word of its 128-byte line
        for (int b0 = b_lo + 2 * warp; b0 < b_hi; b0 += 2 * (kWvThreads / 32)) {
            const int b = b0 + (lane >> 4), j = lane & 15;
            const bool have = b < b_hi;
            const unsigned long long *wp = p.desc + (size_t)(have ? b : 0) * kWvDescWords + j;
            unsigned long long w = 0ull, t0 = 0ull;
            bool v = false, ok = !have;
            int cnt = 0, dn = 0;
            unsigned int n = 0;
            while (true) {
                if (have && !v) {
                    w = ld_relaxed_u64(wp);
                    v = (j == 0) ? wave_item0_ok(w, rnd, s + 1) : wave_item_ok(w, rnd, s + 1);
                }
                const unsigned long long w0 = __shfl_sync(0xffffffffu, w, lane & 16);
                const int v0 = __shfl_sync(0xffffffffu, (int)v, lane & 16);
                if (v0) { cnt = (int)((w0 >> 29) & 0xFull); dn = (int)((w0 >> 33) & 1ull); }
                ok = !have || (v0 && (dn || j >= cnt || v));
                if (__all_sync(0xffffffffu, ok)) break;
                bool to = false;
                if (((++n) & 1023u) == 0u) {
                    if (n == 1024u) t0 = wave_timer();
                    to = (ld_relaxed_u32(p.err) != 0u) || (wave_timer() - t0 > kWvTimeoutNs);
                }
                if (__any_sync(0xffffffffu, to)) { if (lane == 0) { atomicExch(p.err, 1u); sCtl[2] = 1; } break; }
            }
            if (have) {
                if (j == 0) sCnt[b] = dn ? -1 : cnt;
                if (!dn && j < cnt) sRaw[b * kWvDescWords + j] = w;
            }
        }
        if (s > 0 && warp >= 6) {
            // the parents' states were written by other GRU CTAs in earlier steps: acquire their `states visible` words (they
            // were set long ago: a request only nominates after it has seen the partials of that step)
            const unsigned int want = fbase + (unsigned int)s;
            const bool ok = wave_spin([&] {
                bool all = true;
                for (int q = tid - 192; q < p.n_gru; q += 64)        // one flag per lane (acquire loads complete in order)
                    all = all && ((int)(wave_ld_acquire_u32(p.flags + (size_t)q * kFusFlagStride + grp) - want) >= 0);
                return all; }, p.err);
            if (!ok) sCtl[2] = 1;
        }
        __syncthreads();
        // ---- compaction: every warp scans the counts (two requests per lane), warp w packs requests w, w + 8, ..
        int total;
        {
            const int r0 = (lane >= b_lo && lane < b_hi) ? sCnt[lane] : -1, r1 = (lane + 32 >= b_lo && lane + 32 < b_hi) ? sCnt[lane + 32] : -1;
            const int c0 = max(r0, 0), c1 = max(r1, 0);
            int i0 = c0, i1 = c1;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int a0 = __shfl_up_sync(0xffffffffu, i0, o), a1 = __shfl_up_sync(0xffffffffu, i1, o);
                if (lane >= o) { i0 += a0; i1 += a1; }
            }
            const int tot0 = __shfl_sync(0xffffffffu, i0, 31);
            total = tot0 + __shfl_sync(0xffffffffu, i1, 31);
            const int ex0 = i0 - c0, ex1 = tot0 + i1 - c1;
            const bool live = __any_sync(0xffffffffu, r0 >= 0 || r1 >= 0);
            if (sCtl[2]) break;                                      // abort (block-uniform)
            if (!live) { glive[grp] = false; __syncthreads(); continue; }   // every request of the group is done
            for (int b = b_lo + warp; b < b_hi; b += kWvThreads / 32) {
                const int off = __shfl_sync(0xffffffffu, (b < 32) ? ex0 : ex1, b & 31);
                const int cb = __shfl_sync(0xffffffffu, (b < 32) ? c0 : c1, b & 31);
                const int first = 1 + sCum[b];
                if (lane < cb) {
                    const unsigned long long w = sRaw[b * kWvDescWords + lane];
                    const int tok = min((int)(w >> 44), e.V - 1), ps = (int)((w >> 34) & 0x3FFull);
                    sItems[off + lane] = wave_citem_pack(tok, ps, first + lane, b, lane);
                    sOff[off + lane] = (uint32_t)(b * stride + ps) * (uint32_t)(g >> 3);
                }
                __syncwarp();
                if (lane == 0) sCum[b] = first - 1 + cb;
            }
        }
        __syncthreads();
        WV_TR(0, cta == 0, s, 0);

        for (int p0 = 0; p0 < total; p0 += kWvNP) {
            const int n = min(kWvNP, total - p0);
            // this pass: the parents' states are operand B of D1[64 x N] = W_hh slice . [S_hi | S_lo]^T with N = 2 nh columns (hi halves
            // of the nh = 4 ceil(n / 4) nodes, then their lo halves): the tensor core fetches (64 + N) x 32 bytes of operands per
            // K = 16 step at ~64 B/clk, so a pass of few nodes is short.  A ring slot holds two k-blocks of N rows, so such a pass
            // also keeps every K chunk in flight at once and a full pass streams through 3 slots
            const int nh = 4 * ((n + 3) >> 2), N = 2 * nh;
            const int kb_bytes = (N >> 3) * 1024, slot_bytes = 2 * kb_bytes;
            const int nslot = min(min(n_kc, 8), kWvRingBytes / slot_bytes);
            const uint32_t idesc1 = tc::make_idesc_bf16(64, N);
            // independent D1 accumulators, npad columns apart; the same four whatever N is, so that the association of the
            // K sum (and with it every bit of the result) does not depend on how many nodes share the pass
            constexpr int NA = 4, npad = kWvTmemCols / NA;
            WV_TR(0, cta == 0 && p0 == 0, s, 1);
            // ---- epilogue operands (input half from P, previous state): issued now, consumed after the MMAs
            float4 pr = make_float4(0.f, 0.f, 0.f, 0.f), pz4 = pr, pn = pr, hp = pr;
            const bool mine = (my_node < n);
            int my_new = 0, my_it = 0;
            // (the producer warps issue theirs after the operand copies: the copies head the pass's critical path and the
            // load / store unit serves both in order)
            auto load_mine = [&]() {
                if (!mine) return;
                const unsigned long long it = sItems[p0 + my_node];
                const int tok = (int)(it & 0xFFFFFull), ps = (int)((it >> 20) & 0x3FFull), bq = (int)((it >> 40) & 0x7Full);
                my_new = bq * stride + (int)((it >> 30) & 0x3FFull);
                my_it = bq * kWvMaxW + (int)((it >> 47) & 0xFull);
                const float *prow = e.P + (size_t)tok * 3 * g + u0 + my_u;
                pr = __ldg(reinterpret_cast<const float4 *>(prow));
                pz4 = __ldg(reinterpret_cast<const float4 *>(prow + g));
                pn = __ldg(reinterpret_cast<const float4 *>(prow + 2 * g));
                if (ps) hp = __ldcg(reinterpret_cast<const float4 *>(p.s32 + ((size_t)bq * stride + ps) * g + u0 + my_u));
            };
            if (warp < 4) load_mine();
            WV_TR(0, cta == 0 && p0 == 0, s, 2);

            // ---- D1[64 x N] = W_hh slice . [S_hi | S_lo]^T, K streamed through the ring by a warp-specialised pipeline
            // with no CTA barrier inside: warps 4..7 produce (cp.async into the slot, completion tracked by the slot's `full`
            // mbarrier), lane 0 of warps 0..3 consume (tcgen05.mma, tcgen05.commit on the slot's `empty` mbarrier).
            if (warp >= 4) {
                // producer: 16-byte piece ptid & 15 of operand rows rho = (ptid >> 4) + 8 i (row rho < nh: hi half of node rho)
                const int ptid = tid - 128, piece = ptid & 15, kb = piece >> 3, pc = piece & 7;
                const int r7 = ptid >> 4;                            // rho & 7, the same for all rows of a thread
                const uint32_t doff = tc::smem_u32(sRing) + (uint32_t)(kb * kb_bytes + r7 * 128 + ((pc ^ r7) << 4));
                const int nfirst = min(nslot, n_kc), ngrp = N >> 3;
                // source of this thread's piece of row group i, in 16-byte pieces from s_hi (kNoRow: the row is not in use).
                // Branch-free (clamped index), so that the shared-memory loads of all row groups are in flight together
                constexpr uint32_t kNoRow = 0xFFFFFFFFu;
                const uint32_t lo_delta = (uint32_t)((p.s_lo - p.s_hi) >> 3);
                auto off_of = [&](int i) -> uint32_t {
                    const int rho = r7 + 8 * i;
                    const int hl = (rho >= nh), node = rho - (hl ? nh : 0);
                    const uint32_t o = sOff[p0 + min(node, n - 1)] + (uint32_t)piece + (hl ? lo_delta : 0u);
                    return (node < n) ? o : kNoRow;
                };
                // A copy instruction occupies the LSU for ~14 cycles even with every lane predicated off, divisions and address
                // conversions cost hundreds of cycles with one warp per scheduler: real (uniform) branches around unused row
                // groups, no division, shared-space addresses.  The chunks that fit the ring at once go row group by row group
                // and share ONE arrive-on-completion (it sits in the copy queue: later copies would wait behind it).
                if (nfirst == n_kc) {
                    uint32_t o_next = off_of(0);
#pragma unroll 2
                    for (int i = 0; i < ngrp; ++i) {
                        const uint32_t o = o_next;
                        if (i + 1 < ngrp) o_next = off_of(i + 1);
                        if (__ballot_sync(0xffffffffu, o != kNoRow) == 0u) continue;     // nobody in the warp has this row group
                        if (o != kNoRow) {
                            const __nv_bfloat16 *sp = p.s_hi + ((size_t)o << 3);
                            int kcs = kshift;
#pragma unroll 4
                            for (int kc = 0; kc < nfirst; ++kc) {
                                wave_cp_async16_s(doff + (uint32_t)(kc * slot_bytes + i * 1024), sp + (size_t)kcs * kWvKC);
                                if (++kcs == n_kc) kcs = 0;
                            }
                        }
                    }
                    wave_cp_async_arrive(mbGrp);
                } else {
                    // a large pass streams through the ring: chunk by chunk, a slot refilled once the MMAs of its previous chunk
                    // have read it (at least 7 of the 16 row groups are in use, so the sources live in registers)
                    uint32_t so[16];
#pragma unroll
                    for (int i = 0; i < 16; ++i) so[i] = (i < ngrp) ? off_of(i) : kNoRow;
                    WV_TRT(128, 0, cta == 0 && p0 == 0, s, 14);
                    int sl = 0, kcs = kshift;
#pragma unroll 1
                    for (int kc = 0; kc < n_kc; ++kc) {
                        if (kc >= nslot) {
                            tc::mbar_wait(mbEmpty + 8 * sl, (ph_empty >> sl) & 1u);
                            ph_empty ^= 1u << sl;
                        }
                        const uint32_t dst = doff + (uint32_t)(sl * slot_bytes);
                        const __nv_bfloat16 *base = p.s_hi + (size_t)kcs * kWvKC;
#pragma unroll
                        for (int i = 0; i < 16; ++i)
                            if (so[i] != kNoRow) wave_cp_async16_s(dst + i * 1024, base + ((size_t)so[i] << 3));
                        if (kc == nfirst - 1) { wave_cp_async_arrive(mbGrp); WV_TRT(128, 0, cta == 0 && p0 == 0, s, 15); }
                        else if (kc >= nfirst) wave_cp_async_arrive(mbFull + 8 * sl);
                        if (++sl == nslot) sl = 0;
                        if (++kcs == n_kc) kcs = 0;
                    }
                }
                load_mine();
            } else if (lane == 0) {
                // consumer: warp w issues K = 16 steps 2 w, 2 w + 1 of every chunk into its own accumulator D1[w].  MMAs are issued
                // in bursts: every wait -> proxy fence -> issue round costs a few hundred ns, the MMAs themselves tens, so the
                // first burst takes every chunk the ring holds (all of K when the pass is small), the rest follow chunk by chunk
                const int kbw = warp >> 1, s40 = (warp & 1) * 2;
                tc::fence_after_sync();
                int kc = 0, sl = 0, kcs = kshift;
                const uint64_t daw = descW0 + (uint64_t)(kbw * 64 + s40 * 2);
                const uint64_t dbw = descR0 + (uint64_t)((kbw * kb_bytes) / 16 + s40 * 2);
#pragma unroll 1
                while (kc < n_kc) {
                    const int k1 = (kc == 0) ? min(nslot, n_kc) : kc + 1;
                    if (kc == 0) { tc::mbar_wait(mbGrp, ph_grp); ph_grp ^= 1u; }
                    else { tc::mbar_wait(mbFull + 8 * sl, (ph_full >> sl) & 1u); ph_full ^= 1u << sl; }
                    WV_TR(0, cta == 0 && p0 == 0 && kc == 0, s, 8);
                    tc::fence_proxy_async();
#pragma unroll 1
                    for (int q = kc; q < k1; ++q) {
                        const uint64_t da = daw + (uint64_t)(kcs * 128);
                        const uint64_t db = dbw + (uint64_t)((sl * slot_bytes) >> 4);
                        tc::mma_bf16(tmem + warp * npad, da, db, idesc1, q ? 1u : 0u);
                        tc::mma_bf16(tmem + warp * npad, da + 2, db + 2, idesc1, 1u);
                        if (q + nslot < n_kc) tc::commit(mbEmpty + 8 * sl);      // this slot will be refilled
                        if (++sl == nslot) sl = 0;
                        if (++kcs == n_kc) kcs = 0;
                    }
                    kc = k1;
                }
                tc::commit(mbD1);
                WV_TR(0, cta == 0 && p0 == 0, s, 9);
            }
            __syncwarp();
            tc::mbar_wait(mbD1, ph_d1); ph_d1 ^= 1u;
            tc::fence_after_sync();
            __syncwarp();
            WV_TR(0, cta == 0 && p0 == 0, s, 3);

            // ---- TMEM -> shared: an M = 64 accumulator keeps row 16 q + i in lane 32 q + i (i < 16), so quadrant q holds gate q
            // (r, z, n) of the 16 units; the four accumulators and the hi / lo column blocks are added here (fixed order)
            if (q4 < 3 && 16 * hsel < nh) {
#pragma unroll 1
                for (int c16 = hsel; 16 * c16 < nh; c16 += 2) {
                    float v0[16];
#pragma unroll
                    for (int c = 0; c < 16; ++c) v0[c] = 0.f;
#pragma unroll
                    for (int a2 = 0; a2 < NA; a2 += 2) {             // accumulators in index order, hi then lo column block
                        uint32_t u[4][16];
                        wave_tmem_ld16_nw(tmem + tlane + a2 * npad + 16 * c16, u[0]);
                        wave_tmem_ld16_nw(tmem + tlane + a2 * npad + nh + 16 * c16, u[1]);
                        wave_tmem_ld16_nw(tmem + tlane + (a2 + 1) * npad + 16 * c16, u[2]);
                        wave_tmem_ld16_nw(tmem + tlane + (a2 + 1) * npad + nh + 16 * c16, u[3]);
                        wave_tmem_wait_ld();
#pragma unroll
                        for (int c = 0; c < 16; ++c) {
                            v0[c] += __uint_as_float(u[0][c]) + __uint_as_float(u[1][c]);
                            v0[c] += __uint_as_float(u[2][c]) + __uint_as_float(u[3][c]);
                        }
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
            float acc[24];
#pragma unroll
            for (int gate = 0; gate < 3; ++gate)
#pragma unroll
                for (int c = 0; c < 4; ++c) acc[gate * 8 + c] = sH[(size_t)(16 * gate + my_u + c) * kWvLdH + my_node];
            {
                const float prv[4] = {pr.x, pr.y, pr.z, pr.w}, pzv[4] = {pz4.x, pz4.y, pz4.z, pz4.w};
                const float pnv[4] = {pn.x, pn.y, pn.z, pn.w}, hpv[4] = {hp.x, hp.y, hp.z, hp.w};
                float hn[4];
                __nv_bfloat16 bh[4], bl[4];
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    const float rg = sigmoidf_fast(prv[c] + acc[c]);
                    const float zg = sigmoidf_fast(pzv[c] + acc[8 + c]);
                    const float ng = tanhf_fast(pnv[c] + rg * acc[16 + c]);
                    hn[c] = mine ? ((1.0f - zg) * ng + zg * hpv[c]) : 0.f;
                    bh[c] = __float2bfloat16_rn(hn[c]);
                    bl[c] = __float2bfloat16_rn(hn[c] - __bfloat162float(bh[c]));
                }
                uint2 ph, pl;
                ph.x = (uint32_t)__bfloat16_as_ushort(bh[0]) | ((uint32_t)__bfloat16_as_ushort(bh[1]) << 16);
                ph.y = (uint32_t)__bfloat16_as_ushort(bh[2]) | ((uint32_t)__bfloat16_as_ushort(bh[3]) << 16);
                pl.x = (uint32_t)__bfloat16_as_ushort(bl[0]) | ((uint32_t)__bfloat16_as_ushort(bl[1]) << 16);
                pl.y = (uint32_t)__bfloat16_as_ushort(bl[2]) | ((uint32_t)__bfloat16_as_ushort(bl[3]) << 16);
                // lane < 16 (hi row) collects the hi halves of units 8 hsel .. + 8, its partner (lo row) the lo halves
                const uint2 snd = uh ? ph : pl;
                uint2 rcv;
                rcv.x = __shfl_xor_sync(0xffffffffu, snd.x, 16);
                rcv.y = __shfl_xor_sync(0xffffffffu, snd.y, 16);
                const uint4 piece = uh ? make_uint4(rcv.x, rcv.y, pl.x, pl.y) : make_uint4(ph.x, ph.y, rcv.x, rcv.y);
                WV_TR(0, cta == 0 && p0 == 0, s, 10);
                // all-gather over the cluster: block `crank` of every cluster CTA's sS2 (operand A of the W1 GEMM)
                if (pend2) { wave_cluster_wait(); pend2 = false; }   // every peer's previous W1 GEMM has read its sS2
                if (mine) {
#pragma unroll
                    for (int c = 0; c < kWvCS; ++c) wave_st_cluster_v4(s2_dst[c], piece);
                }
                // the release of the arrive covers what was stored BEFORE it: the global stores come after, so the cluster
                // does not wait for their round trip to L2 (the gpu fence in front of the flag does)
                wave_cluster_arrive();
                WV_TR(0, cta == 0 && p0 == 0, s, 11);
                if (mine) {                                          // publish S_new: fp32 and the bf16 hi / lo split
                    __stcg(reinterpret_cast<float4 *>(p.s32 + (size_t)my_new * g + u0 + my_u), make_float4(hn[0], hn[1], hn[2], hn[3]));
                    __stcg(reinterpret_cast<uint4 *>((uh ? p.s_lo : p.s_hi) + (size_t)my_new * g + u0 + 8 * hsel), piece);
                }
            }
            wave_cluster_wait();
            WV_TR(0, cta == 0 && p0 == 0, s, 12);
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
                tc::commit(mbD2);
            }
            WV_TR(0, cta == 0 && p0 == 0, s, 13);
            tc::mbar_wait(mbD2, ph_d2); ph_d2 ^= 1u;
            tc::fence_after_sync();
            __syncwarp();
            WV_TR(0, cta == 0 && p0 == 0, s, 5);
            wave_cluster_arrive_relaxed(); pend2 = true;             // my sS2 may be overwritten by the next pass (no data to release)
            {
                // partial[item][cluster][crank * rpc + col]: lanes < 16 store columns 0..7 of a 16-column block, lanes >= 16 8..15
                float *prow = p.partial + ((size_t)my_it * p.P + (cta / kWvCS)) * r + crank * rpc;
#pragma unroll 1
                for (int blk = hsel; blk < rpc / 16; blk += 2) {
                    uint32_t u[16];
                    wave_tmem_ld16_nw(tmem + tlane + 16 * blk, u);
                    wave_tmem_wait_ld();
                    float v[16];
#pragma unroll
                    for (int c = 0; c < 16; ++c) { v[c] = __uint_as_float(u[c]); v[c] += __shfl_xor_sync(0xffffffffu, v[c], 16); }
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
        if (tid == 0) {
            fence_release_gpu();                                     // states and partials of this step are visible before the flag
            st_relaxed_u32(p.flags + (size_t)cta * kFusFlagStride + grp, fbase + (unsigned int)(s + 1));
        }
        WV_TR(0, cta == 0, s, 7);
        sg[grp] = s + 1;
    }
    __syncthreads();
    WV_TR(0, cta == 0, kWvTraceSteps - 1, 2);
    if (pend2) wave_cluster_wait();
    if (warp == 0) tc::tmem_free<kWvTmemCols>(tmem);
    // every CTA of the grid has read the counter: a request is done only after all GRU CTAs finished step 0
    if (cta == 0 && tid == 0) st_relaxed_u32(p.round_ctr, rnd + 1u);
}

// -------------------------------------------------------------------------------------- request role
// The frontier is kept as a SORTED list G of the best known nodes (children of the nodes expanded so far), cut at B
// entries: the known set only grows, so a node ranked beyond B can never enter the tree.  Sort key (larger = earlier):
//     score desc, depth asc, token asc        [then parent position asc, then arrival order: never equal]
// `depth asc` keeps a parent in front of a child whose fp32 score rounds to the parent's (g + logp == g happens for
// saturated slices); everything else is the pop comparator of reading A8.  The first B - 1 entries are exactly the
// nodes Algorithm 1 expands, so a step nominates the first W of them that are not expanded yet
// (the first one is the node Algorithm 1 needs next, the others are speculative) and the round ends when there is none.
struct WaveCtl {
    int n_exp;          // expansions allocated so far (expansion 0 = the root)
    int n_items;        // items published for the coming step
    int nG;             // entries of the sorted frontier
    int cur;            // which of the two frontier buffers is current
    int done, n_stage, abort_, pad;
    int slDepth[kWvMaxSlices];      // depth whose candidate rows a slice holds (-1 = empty)
    int slUsed[kWvMaxSlices];       // last step that needs the slice
    int stage[kWvMaxSlices];        // slices to fill before the coming step
    signed char d2s[DT_MAX_L];      // depth -> slice (-1 = not resident)
};
// frontier entry: key = ord(score) (32) | 63 - depth (6, from bit 20) | 0xFFFFF - token (20);
//                 meta = depth (6) | own expansion + 1 (10, from bit 6; 0 = not expanded) | parent expansion (10, from bit 16)
__device__ __forceinline__ unsigned long long wave_gkey(float score, int depth, int tok) {
    return ((unsigned long long)ord_key(score) << 32) | ((unsigned long long)(63 - min(depth, 63)) << 20) |
           (unsigned long long)(0xFFFFFu - ((unsigned int)tok & 0xFFFFFu));
}
constexpr int kWvDropped = 0x3FFFFFFF;

__host__ __device__ inline size_t wave_req_smem2(int r, int M, int B, int k, int W, int e_max, int n_slices) {
    auto al = [](size_t x) { return (x + 15) / 16 * 16; };
    size_t s = (size_t)n_slices * wave_slice_bytes(r, M) + 2 * al((size_t)n_slices * M * 4);
    s += 2 * al((size_t)B * 8) + 2 * al((size_t)B * 4);                     // frontier, two buffers
    s += al((size_t)W * k * 8) + al((size_t)W * k * 4);                     // new children
    s += 3 * al((size_t)e_max * 4);                                         // eDep, eSco, ePos
    s += al((size_t)W * r * 4) + al((size_t)W * M * 8);
    s += al((size_t)4 * kWvMaxW * 4) + al(256) + al((size_t)kWvThreads * 8) + al((size_t)kWvMaxW * 8);
    return s + 1024;
}

// Rank of frontier entry i (old entry i < n_old, or new candidate i - n_old) in the merged order; strict total order: key
// desc, then parent position asc, then index asc (old entries before new ones).  Out of line on purpose: the request
// role's step loop has to stay inside the instruction cache (it runs once per step, on one latency chain).
__device__ __noinline__ int wave_merge_rank(const unsigned long long *oK, const unsigned int *oM, int n_old,
                                            const unsigned long long *nKey, const unsigned int *nMeta, int n_new,
                                            const int *ePos, int i, unsigned long long mkh, unsigned int mmh) {
    auto prec = [&](unsigned long long ka, unsigned int ma, int ia, unsigned long long kb, unsigned int mb, int ib) {
        if (ka != kb) return ka > kb;
        const int pa = ePos[(ma >> 16) & 0x3FFu], pb = ePos[(mb >> 16) & 0x3FFu];
        if (pa != pb) return pa < pb;
        return ia < ib;
    };
    const bool is_old = i < n_old;
    int rank = 0;
    if (is_old) rank = i;
    else {                                               // old entries in front of it: the list is sorted
        int lo = 0, hi = n_old;
        while (lo < hi) {
            const int mid = (lo + hi) >> 1;
            const unsigned long long km = oK[mid];
            if (km > mkh || (km == mkh && prec(km, oM[mid], mid, mkh, mmh, i))) lo = mid + 1; else hi = mid;
        }
        rank = lo;
    }
    // new entries in front of it: keys only, two per load; equal keys (the same score, depth and token under two
    // parents: rare) go through the full comparator
    int n_eq = 0, q = 0;
#pragma unroll 2
    for (; q + 2 <= n_new; q += 2) {
        const ulonglong2 o = *reinterpret_cast<const ulonglong2 *>(nKey + q);
        rank += (o.x > mkh) + (o.y > mkh);
        n_eq += (o.x == mkh) + (o.y == mkh);
    }
    if (q < n_new) { rank += (nKey[q] > mkh); n_eq += (nKey[q] == mkh); }
    if (n_eq > (is_old ? 0 : 1)) {
#pragma unroll 1
        for (int q2 = 0; q2 < n_new; ++q2)
            if (nKey[q2] == mkh && n_old + q2 != i) rank += prec(nKey[q2], nMeta[q2], n_old + q2, mkh, mmh, i) ? 1 : 0;
    }
    return rank;
}

__device__ __forceinline__ void wave_req_role(const WaveParams &p, unsigned char *smem_raw) {
    const ExpandParams &e = p.e;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int b = blockIdx.x - p.n_gru;
    const int r = e.r, M = e.M, k = e.k, N = e.N, L = e.L, B = e.B;
    const int W = p.W, nsl = p.n_slices, e_max = p.e_max, P = p.P;
    const unsigned int rnd = ld_relaxed_u32(p.round_ctr), fbase = rnd << 10;
    const int my_grp = b / ((e.batch + p.n_groups - 1) / p.n_groups);
    const size_t slice_bytes = wave_slice_bytes(r, M);
    const int Ka = (r + 63) / 64, nvec = r / 8;

    size_t off = 0;
    auto carve = [&](size_t bytes) { unsigned char *q = smem_raw + off; off += (bytes + 15) / 16 * 16; return q; };
    unsigned char *sW2 = carve((size_t)nsl * slice_bytes);
    int *slTok = reinterpret_cast<int *>(carve((size_t)nsl * M * 4));
    float *slBase = reinterpret_cast<float *>(carve((size_t)nsl * M * 4));
    unsigned long long *gKey[2];
    unsigned int *gMeta[2];
    gKey[0] = reinterpret_cast<unsigned long long *>(carve((size_t)B * 8));
    gKey[1] = reinterpret_cast<unsigned long long *>(carve((size_t)B * 8));
    gMeta[0] = reinterpret_cast<unsigned int *>(carve((size_t)B * 4));
    gMeta[1] = reinterpret_cast<unsigned int *>(carve((size_t)B * 4));
    unsigned long long *nKey = reinterpret_cast<unsigned long long *>(carve((size_t)W * k * 8));   // children of this step's items
    unsigned int *nMeta = reinterpret_cast<unsigned int *>(carve((size_t)W * k * 4));
    int *eDep = reinterpret_cast<int *>(carve((size_t)e_max * 4));                 // depth of expansion x's node
    float *eSco = reinterpret_cast<float *>(carve((size_t)e_max * 4));             // its score
    int *ePos = reinterpret_cast<int *>(carve((size_t)e_max * 4));                 // its position in the frontier (-1 root)
    float *sA = reinterpret_cast<float *>(carve((size_t)W * r * 4));
    unsigned long long *sKey = reinterpret_cast<unsigned long long *>(carve((size_t)W * M * 8));   // (z, ~token) of every candidate
    int *itE = reinterpret_cast<int *>(carve((size_t)4 * kWvMaxW * 4));
    unsigned long long *sSvK = reinterpret_cast<unsigned long long *>(carve((size_t)kWvThreads * 8));   // per warp: keys at or above the top-k threshold
    float2 *sStat = reinterpret_cast<float2 *>(carve((size_t)kWvMaxW * 8));        // per node: slice maximum, log-sum-exp
    int *itTok = itE + kWvMaxW, *itPs = itTok + kWvMaxW;
    WaveCtl &ctl = *reinterpret_cast<WaveCtl *>(carve(256));

    const __nv_bfloat16 *w2 = reinterpret_cast<const __nv_bfloat16 *>(e.w2);
    unsigned long long *my_desc = p.desc + (size_t)b * kWvDescWords;

    // fill the slices listed in ctl.stage with the candidate table of their depth: ids, base logits, the M rows of W2
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
        ctl.n_exp = 1; ctl.n_items = 1; ctl.nG = 0; ctl.cur = 0; ctl.done = 0; ctl.abort_ = 0;
        for (int i = 0; i < kWvMaxSlices; ++i) { ctl.slDepth[i] = -1; ctl.slUsed[i] = -1; }
        for (int i = 0; i < DT_MAX_L; ++i) ctl.d2s[i] = -1;
        ctl.slDepth[0] = 0; ctl.slUsed[0] = 0; ctl.d2s[0] = 0; ctl.stage[0] = 0; ctl.n_stage = 1;
        eDep[0] = 0; eSco[0] = 0.f; ePos[0] = -1;
        itE[0] = 0;
        // step 0: the root, whose parent state is the zero slot (reading A4)
        st_relaxed_u64(my_desc, wave_item_pack(rnd, 1, 1, 0, 0, min(max(root, 0), e.V - 1)));
    }
    __syncthreads();
    stage_slices();
    if (tid == 0) ctl.n_stage = 0;                               // every thread read the list before the barrier inside

    WV_TR(1, b == 0, kWvTraceSteps - 1, 1);
    for (int s = 0;; ++s) {
        const int n_it = ctl.n_items;
        // the first round of the partial sums: who am I, where are my partials, and C = H W1h^T of the node's depth (A12: row =
        // depth), which does not depend on the GRU CTAs: all of it while they work
        const int r4 = r >> 2;
        const int pair0 = tid >> 1, j0 = pair0 / r4, jq0 = pair0 - j0 * r4;
        const bool act0 = pair0 < n_it * r4;
        float4 cv0 = make_float4(0.f, 0.f, 0.f, 0.f);
        if (act0 && !(tid & 1)) cv0 = __ldg(reinterpret_cast<const float4 *>(e.C + ((size_t)b * L + eDep[itE[j0]]) * r) + jq0);
        if (warp < 2) {
            // two warps, so that with up to 64 GRU CTAs a lane has ONE flag: acquire loads of one thread complete in order,
            // a second flag per lane would cost a second round trip to L2
            const unsigned int want = fbase + (unsigned int)(s + 1);
            const bool ok = wave_spin([&] {
                bool all = true;
                for (int q = tid; q < p.n_gru; q += 64)
                    all = all && ((int)(wave_ld_acquire_u32(p.flags + (size_t)q * kFusFlagStride + my_grp) - want) >= 0);
                return all; }, p.err);
            if (!ok) ctl.abort_ = 1;
        }
        __syncthreads();
        if (ctl.abort_) break;
        WV_TR(1, b == 0, s, 0);

        // ---- a_j = SiLU(C + W1[:, d:] S_j): the P cluster partials are summed in a fixed order (batch-invariant): two
        // neighbouring lanes per (node, four columns) take the even / the odd clusters, all loads of a lane in flight at once
        {
            const int n_task = 2 * n_it * r4;
#pragma unroll 1
            for (int base = 0; base < n_task; base += 2 * kWvThreads) {             // block-uniform trip count; two tasks per thread,
                bool act[2];                                                        // the loads of both in flight together
                int jj[2], jq[2], hh[2];
                float4 cv[2], v[2][8];
                const float4 *pp[2];
#pragma unroll
                for (int t = 0; t < 2; ++t) {
                    const int idx = base + t * kWvThreads + tid, pair = idx >> 1;
                    hh[t] = idx & 1;
                    const bool first = (base == 0 && t == 0);
                    act[t] = first ? act0 : (pair < n_it * r4);
                    jj[t] = first ? j0 : (act[t] ? pair / r4 : 0);
                    jq[t] = first ? jq0 : (act[t] ? pair - jj[t] * r4 : 0);
                    cv[t] = first ? cv0 : make_float4(0.f, 0.f, 0.f, 0.f);
                    pp[t] = reinterpret_cast<const float4 *>(p.partial + ((size_t)(b * kWvMaxW + jj[t]) * P) * r) + jq[t];
                    if (act[t]) {
                        if (!first && hh[t] == 0) cv[t] = __ldg(reinterpret_cast<const float4 *>(e.C + ((size_t)b * L + eDep[itE[jj[t]]]) * r) + jq[t]);
#pragma unroll
                        for (int i = 0; i < 8; ++i)
                            v[t][i] = (hh[t] + 2 * i < P) ? __ldcg(pp[t] + (size_t)(hh[t] + 2 * i) * r4) : make_float4(0.f, 0.f, 0.f, 0.f);
                    }
                }
#pragma unroll
                for (int t = 0; t < 2; ++t) {
                    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
                    if (act[t]) {
#pragma unroll
                        for (int i = 0; i < 8; ++i) { acc.x += v[t][i].x; acc.y += v[t][i].y; acc.z += v[t][i].z; acc.w += v[t][i].w; }
#pragma unroll 1
                        for (int q0 = hh[t] + 16; q0 < P; q0 += 16) {               // more than 16 clusters (g > 1024)
                            float4 w8[8];
#pragma unroll
                            for (int i = 0; i < 8; ++i) w8[i] = (q0 + 2 * i < P) ? __ldcg(pp[t] + (size_t)(q0 + 2 * i) * r4) : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
                            for (int i = 0; i < 8; ++i) { acc.x += w8[i].x; acc.y += w8[i].y; acc.z += w8[i].z; acc.w += w8[i].w; }
                        }
                    }
                    // even clusters + odd clusters, then C
                    acc.x += __shfl_xor_sync(0xffffffffu, acc.x, 1); acc.y += __shfl_xor_sync(0xffffffffu, acc.y, 1);
                    acc.z += __shfl_xor_sync(0xffffffffu, acc.z, 1); acc.w += __shfl_xor_sync(0xffffffffu, acc.w, 1);
                    if (act[t] && hh[t] == 0) {
                        float4 o;
                        o.x = cv[t].x + acc.x; o.y = cv[t].y + acc.y; o.z = cv[t].z + acc.z; o.w = cv[t].w + acc.w;
                        o.x *= sigmoidf_acc(o.x); o.y *= sigmoidf_acc(o.y); o.z *= sigmoidf_acc(o.z); o.w *= sigmoidf_acc(o.w);
                        *reinterpret_cast<float4 *>(sA + (size_t)jj[t] * r + 4 * jq[t]) = o;
                    }
                }
            }
        }
        cp_async_wait<0>();
        __syncthreads();
        WV_TR(1, b == 0, s, 1);

        // ---- z_m = ((base_m - base_0) + W2[cand_m, :] a) / T_eff   PAPER.md:143-144 (shift-invariant)
        // a warp takes 8 candidate rows (one swizzle row group), four lanes per row; two accumulation chains per lane
        const int rb_n = (M + 31) >> 5;                              // 32-row blocks per node
        if (n_it * rb_n >= kWvThreads / 32) {
            // enough (node, row block) tasks for every warp: a lane owns one candidate row and walks all of it -- no cross-lane
            // reduction, 8 accumulation chains -- with EXACTLY the association of the four-lanes-per-row form below (class
            // c = piece index mod 4 is what lane group qq sums there; (q0 + q1) + (q2 + q3) is what its two shuffles add), so a
            // node's scores do not depend on how many nodes share the step (batch invariance)
#pragma unroll 1
            for (int task = warp; task < n_it * rb_n; task += kWvThreads / 32) {
                int j = 0, rb = task;
                while (rb >= rb_n) { rb -= rb_n; ++j; }
                const int si = ctl.d2s[eDep[itE[j]]];
                const unsigned char *sl = sW2 + (size_t)si * slice_bytes;
                const float *bs = slBase + si * M;
                const float *aj = sA + (size_t)j * r;
                const int m = 32 * rb + lane, mc = min(m, M - 1), rw = mc & 7;
                const unsigned char *rowp = sl + (size_t)(mc >> 3) * Ka * 1024 + rw * 128;
                float A0[4] = {0.f, 0.f, 0.f, 0.f}, A1[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll 2
                for (int v0 = 0; v0 < nvec; v0 += 4) {
#pragma unroll
                    for (int c = 0; c < 4; ++c) {
                        const int v = v0 + c;
                        if (v < nvec) {
                            const uint4 q = *reinterpret_cast<const uint4 *>(rowp + (size_t)(v >> 3) * 1024 + (((v & 7) ^ rw) << 4));
                            const float4 a0 = *reinterpret_cast<const float4 *>(aj + (size_t)v * 8);
                            const float4 a1 = *reinterpret_cast<const float4 *>(aj + (size_t)v * 8 + 4);
                            float f[8];
                            unpack8(q, f);
                            A0[c] = fmaf(f[0], a0.x, A0[c]); A1[c] = fmaf(f[1], a0.y, A1[c]); A0[c] = fmaf(f[2], a0.z, A0[c]); A1[c] = fmaf(f[3], a0.w, A1[c]);
                            A0[c] = fmaf(f[4], a1.x, A0[c]); A1[c] = fmaf(f[5], a1.y, A1[c]); A0[c] = fmaf(f[6], a1.z, A0[c]); A1[c] = fmaf(f[7], a1.w, A1[c]);
                        }
                    }
                }
                const float acc = ((A0[0] + A1[0]) + (A0[1] + A1[1])) + ((A0[2] + A1[2]) + (A0[3] + A1[3]));
                if (m < M) {
                    const float z = __fdiv_rn((bs[m] - bs[0]) + acc, e.T_eff);
                    sKey[(size_t)j * M + m] = ((unsigned long long)ord_key(z) << 32) | (unsigned long long)(0xFFFFFFFFu - (unsigned int)slTok[si * M + m]);
                }
            }
        } else
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
                float acc0 = 0.f, acc1 = 0.f;
#pragma unroll 4
                for (int v = qq; v < nvec; v += 4) {
                    const uint4 q = *reinterpret_cast<const uint4 *>(rowp + (size_t)(v >> 3) * 1024 + (((v & 7) ^ rw) << 4));
                    const float4 a0 = *reinterpret_cast<const float4 *>(aj + (size_t)v * 8);
                    const float4 a1 = *reinterpret_cast<const float4 *>(aj + (size_t)v * 8 + 4);
                    float f[8];
                    unpack8(q, f);
                    acc0 = fmaf(f[0], a0.x, acc0); acc1 = fmaf(f[1], a0.y, acc1); acc0 = fmaf(f[2], a0.z, acc0); acc1 = fmaf(f[3], a0.w, acc1);
                    acc0 = fmaf(f[4], a1.x, acc0); acc1 = fmaf(f[5], a1.y, acc1); acc0 = fmaf(f[6], a1.z, acc0); acc1 = fmaf(f[7], a1.w, acc1);
                }
                float acc = acc0 + acc1;
                acc += __shfl_xor_sync(0xffffffffu, acc, 8);
                acc += __shfl_xor_sync(0xffffffffu, acc, 16);
                const int m = 8 * rg + rw;
                if (qq == 0 && m < M) {
                    const float z = __fdiv_rn((bs[m] - base0) + acc, e.T_eff);
                    sKey[(size_t)j * M + m] = ((unsigned long long)ord_key(z) << 32) | (unsigned long long)(0xFFFFFFFFu - (unsigned int)slTok[si * M + m]);
                }
            }
        }
        __syncthreads();
        WV_TR(1, b == 0, s, 2);

        // ---- slice log-softmax (reading A1) and top-k by (z desc, token asc).  A warp per node finds the k best without
        // anything that scales with M * M: (1) every lane takes the best of its own M / 32 keys and k rounds of a warp
        // max reduction give L, the k-th best of the 32 lane maxima: at least k keys lie at or above L, so the true top k
        // do; (2) the keys at or above L (k plus a few) are handed one to a lane and ranked among themselves by counting
        // over the full 64-bit keys through shuffles.  The result is the exact top k in the exact order.  With at most
        // four nodes a second warp per node computes the slice maximum and log-sum-exp meanwhile (named barrier 1 + j);
        // otherwise the node's warp does both.  The k best become frontier candidates with score g_parent + logp
        {
            const int MI = (M + 31) >> 5;
            const bool split = 2 * n_it <= kWvThreads / 32;
            const bool stat_only = split && (warp & 1);
            const int jstep = split ? kWvThreads / 64 : kWvThreads / 32;
            unsigned long long *svK = sSvK + warp * 32;
#pragma unroll 1
            for (int j = split ? (warp >> 1) : warp; j < n_it; j += jstep) {
                const int x = itE[j];
                const unsigned long long *kj = sKey + (size_t)j * M;
                float zmax = 0.f, lse = 0.f;
                if (!split || stat_only) {
                    float zr[8];
                    zmax = -INFINITY;
#pragma unroll
                    for (int i = 0; i < 8; ++i) {
                        const int m = lane + 32 * i;
                        zr[i] = -INFINITY;
                        if (i < MI && m < M) {
                            zr[i] = ord_key_inv((unsigned int)(kj[m] >> 32));
                            zmax = fmaxf(zmax, zr[i]);
                        }
                    }
                    zmax = ord_key_inv(__reduce_max_sync(0xffffffffu, ord_key(zmax)));
                    float ssum = 0.f;
#pragma unroll
                    for (int i = 0; i < 8; ++i)
                        if (i < MI && lane + 32 * i < M) ssum += __expf(zr[i] - zmax);
                    ssum = warp_sum(ssum);
                    lse = __logf(ssum);
                    if (stat_only) {
                        if (lane == 0) sStat[j] = make_float2(zmax, lse);
                        __threadfence_block();
                        asm volatile("bar.arrive %0, 64;" ::"r"(1 + j) : "memory");
                        continue;
                    }
                }
                unsigned long long kk[8];
                unsigned int hmax = 0u;
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    const int m = lane + 32 * i;
                    kk[i] = (i < MI && m < M) ? kj[m] : 0ull;
                    hmax = max(hmax, (unsigned int)(kk[i] >> 32));
                }
                unsigned int cur = (hmax & ~31u) | (unsigned int)(31 - lane), L = 0u;   // lane in the low bits: all distinct
#pragma unroll 1
                for (int rr = 0; rr < k; ++rr) {
                    L = __reduce_max_sync(0xffffffffu, cur);
                    if (cur == L) cur = 0u;
                }
                L &= ~31u;
                WV_TR(1, b == 0, s, 10);
                int ns = 0;
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    if (i >= MI) break;
                    const bool in = (unsigned int)(kk[i] >> 32) >= L && kk[i] != 0ull;
                    const unsigned int bal = __ballot_sync(0xffffffffu, in);
                    const int at = ns + __popc(bal & ((1u << lane) - 1u));
                    if (in && at < 32) svK[at] = kk[i];
                    ns += __popc(bal);
                }
                __syncwarp();
                if (split) {
                    asm volatile("bar.sync %0, 64;" ::"r"(1 + j) : "memory");
                    const float2 st = sStat[j];
                    zmax = st.x;
                    lse = st.y;
                }
                const float gpar = eSco[x];
                const int cdep = eDep[x] + 1;
                if (ns <= 32) {
                    const unsigned long long mk = lane < ns ? svK[lane] : 0ull;
                    int rank = 0;
#pragma unroll 4
                    for (int q = 0; q < ns; ++q) rank += (__shfl_sync(0xffffffffu, mk, q) > mk);
                    if (lane < ns && rank < k) {
                        const float lpm = (ord_key_inv((unsigned int)(mk >> 32)) - zmax) - lse;
                        const int tok = (int)(0xFFFFFFFFu - (unsigned int)(mk & 0xFFFFFFFFull));
                        nKey[j * k + rank] = wave_gkey(gpar + lpm, cdep, tok);
                        nMeta[j * k + rank] = (unsigned int)cdep | ((unsigned int)x << 16);
                    }
                } else {                                             // many equal keys at the threshold: count over the slice
#pragma unroll 1
                    for (int m = lane; m < M; m += 32) {
                        const unsigned long long mk = kj[m];
                        if ((unsigned int)(mk >> 32) < L) continue;
                        int rank = 0;
#pragma unroll 1
                        for (int q = 0; q < M; ++q) rank += (kj[q] > mk);
                        if (rank < k) {
                            const float lpm = (ord_key_inv((unsigned int)(mk >> 32)) - zmax) - lse;
                            const int tok = (int)(0xFFFFFFFFu - (unsigned int)(mk & 0xFFFFFFFFull));
                            nKey[j * k + rank] = wave_gkey(gpar + lpm, cdep, tok);
                            nMeta[j * k + rank] = (unsigned int)cdep | ((unsigned int)x << 16);
                        }
                    }
                }
                __syncwarp();
                WV_TR(1, b == 0, s, 11);
            }
        }
        __syncthreads();
        WV_TR(1, b == 0, s, 3);

        // ---- merge the n_it k new candidates into the sorted frontier (rank by counting, cut at B)
        {
            const int cur = ctl.cur, n_old = ctl.nG, n_new = n_it * k, tot = n_old + n_new;
            const unsigned long long *oK = gKey[cur];
            const unsigned int *oM = gMeta[cur];
            unsigned long long *dK = gKey[cur ^ 1];
            unsigned int *dM = gMeta[cur ^ 1];
            int rk[2] = {0, 0};
            unsigned long long mk[2] = {0ull, 0ull};
            unsigned int mm[2] = {0u, 0u};
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int i = tid + h * kWvThreads;
                if (i >= tot) continue;
                const bool is_old = i < n_old;
                mk[h] = is_old ? oK[i] : nKey[i - n_old];
                mm[h] = is_old ? oM[i] : nMeta[i - n_old];
                const int rank = wave_merge_rank(oK, oM, n_old, nKey, nMeta, n_new, ePos, i, mk[h], mm[h]);
                rk[h] = rank;
            }
            __syncthreads();                                         // every rank is computed from the old positions
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int i = tid + h * kWvThreads;
                if (i >= tot) continue;
                const int own = (int)((mm[h] >> 6) & 0x3FFu);
                if (rk[h] < B) { dK[rk[h]] = mk[h]; dM[rk[h]] = mm[h]; if (own) ePos[own - 1] = rk[h]; }
                else if (own) ePos[own - 1] = kWvDropped;
            }
            if (tid == 0) { ctl.cur = cur ^ 1; ctl.nG = min(tot, B); }
        }
        __syncthreads();
        WV_TR(1, b == 0, s, 6);

        // ---- nominate (warp 0): the first W frontier entries among the first B - 1 that have depth < L and no expansion yet
        if (warp == 0) {
            const int cur = ctl.cur, nG = ctl.nG, n_exp = ctl.n_exp;
            unsigned long long *cK = gKey[cur];
            unsigned int *cM = gMeta[cur];
            const int lim = min(nG, B - 1), step_next = s + 1;
            int found = 0, c_first = -1;
            bool stop = false;
#pragma unroll 1
            for (int i0 = 0; i0 < lim && !stop; i0 += 32) {
                const int i = i0 + lane;
                unsigned int m = 0u;
                bool want = false;
                if (i < lim) { m = cM[i]; want = ((m >> 6) & 0x3FFu) == 0u && (int)(m & 0x3Fu) < L; }
                unsigned int bal = __ballot_sync(0xffffffffu, want);
                while (bal && !stop) {
                    const int ln = __ffs(bal) - 1;
                    bal &= bal - 1;
                    const int idx = i0 + ln;
                    if (c_first < 0) c_first = idx;
                    int add = 0;
                    if (lane == 0) {
                        const unsigned int mt = cM[idx];
                        const unsigned long long ky = cK[idx];
                        const int dep = (int)(mt & 0x3Fu), par = (int)((mt >> 16) & 0x3FFu);
                        const int xn = n_exp + found;
                        // resources: a state slot (speculative picks leave room for the expansions Algorithm 1 still needs)
                        // and a W2 slice for the node's depth
                        bool can = (xn < e_max) && (found == 0 || xn + 1 + (B - c_first) <= e_max);
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
                            cM[idx] = mt | ((unsigned int)(xn + 1) << 6);
                            eDep[xn] = dep; eSco[xn] = ord_key_inv((unsigned int)(ky >> 32)); ePos[xn] = idx;
                            itE[found] = xn; itTok[found] = (int)(0xFFFFFu - (unsigned int)(ky & 0xFFFFFull)); itPs[found] = par + 1;
                            add = 1;
                        }
                    }
                    add = __shfl_sync(0xffffffffu, add, 0);
                    found += add;
                    stop = (add == 0) || found >= W;                // out of slots / slices, or the step is full
                }
            }
            __syncwarp();
            if (c_first < 0) {                                       // nothing left to expand: the frontier is Algorithm 1's tree
                if (lane == 0) {
                    ctl.done = 1; ctl.n_items = 0;
                    st_relaxed_u64(my_desc, wave_item_pack(rnd, s + 2, 0, 1, 0, 0));
                    if (p.stats && b == 0) { p.stats[0] = (unsigned int)(s + 1); p.stats[1] = (unsigned int)n_exp; }
                }
            } else {
                // every word carries the count; word 0 is written even when nothing could be nominated
                if (lane < max(found, 1))
                    st_relaxed_u64(my_desc + lane, wave_item_pack(rnd, s + 2, found, 0, lane < found ? itPs[lane] : 0,
                                                                  lane < found ? itTok[lane] : 0));
                if (lane == 0) { ctl.n_items = found; ctl.n_exp = n_exp + found; }
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

    WV_TR(1, b == 0, kWvTraceSteps - 1, 2);
    // emitter (a9): slots in frontier order, dead-leaf padding (reading A10), positions, ancestor-or-self mask
    const int n = ctl.abort_ ? 1 : ctl.nG + 1;
    const unsigned long long *fK = gKey[ctl.cur];
    const unsigned int *fM = gMeta[ctl.cur];
    int *nPar = reinterpret_cast<int *>(gKey[ctl.cur ^ 1]);         // parent slot of every output slot (the spare frontier buffer: 8 B >= 4 (B + 1))
    const int rpos = e.root_positions ? e.root_positions[b] : 0;
    for (int i = tid; i < N; i += kWvThreads) {
        const size_t so = (size_t)b * N + i;
        int tok = 0, par = 0, dep = 1;
        float sc = -INFINITY;
        if (i == 0) { tok = e.root_tokens[b]; par = -1; dep = 0; sc = 0.f; }
        else if (i < n) {
            const unsigned long long ky = fK[i - 1];
            const unsigned int mt = fM[i - 1];
            tok = (int)(0xFFFFFu - (unsigned int)(ky & 0xFFFFFull));
            par = ePos[(mt >> 16) & 0x3FFu] + 1;
            dep = (int)(mt & 0x3Fu);
            sc = ord_key_inv((unsigned int)(ky >> 32));
        }
        e.tokens[so] = tok; e.parents[so] = par; e.depths[so] = dep; e.scores[so] = sc; e.positions[so] = rpos + dep;
        nPar[i] = (i < n) ? par : 0;
    }
    if (tid == 0) e.n_nodes[b] = n;
    uint8_t *mk = e.mask + (size_t)b * N * N;
    for (int i = tid; i < N * N; i += kWvThreads) mk[i] = 0;
    __syncthreads();
    for (int i = tid; i < N; i += kWvThreads) {
        int a = i;
        while (a >= 0) { mk[(size_t)i * N + a] = 1; a = nPar[a]; }
    }
    WV_TR(1, b == 0, kWvTraceSteps - 1, 3);
}

// Which schedule pays is a property of the round's candidate tables: bushy trees (flat slices) finish in a few wide
// wavefront steps, chains (peaked slices) need one dependent step per node whatever the width, and there the lock-step
// kernel's shorter step wins.  The decision is taken for the whole batch from the a1 output: the mean top-1 probability
// of the base slices, p1 = 1 / sum_m exp((v_m - v_0) / T_eff) (reading A1 without the correction), against a threshold.
// A warp per row adds its p1 in 16-bit fixed point to one device word (integer adds: the sum does not depend on their order);
// the word is cleared by a memset node at the start of the round and compared with `sched_thr` by the expansion kernels.
__global__ void __launch_bounds__(256) wave_regime_kernel(const float *cand_val, int rows, int M, float inv_T, unsigned int *acc) {
    const int row = blockIdx.x * 8 + (threadIdx.x >> 5);
    if (row >= rows) return;
    const float *v = cand_val + (size_t)row * M;
    const float v0 = v[0];
    float ssum = 0.f;
    for (int m = threadIdx.x & 31; m < M; m += 32) ssum += __expf((v[m] - v0) * inv_T);
    ssum = warp_sum(ssum);
    if ((threadIdx.x & 31) == 0) atomicAdd(acc, (unsigned int)(65536.0f / ssum + 0.5f));
}

__global__ void __launch_bounds__(kWvThreads, 1) wave_expand_kernel(WaveParams p) {
    extern __shared__ __align__(1024) unsigned char wave_smem[];
    if (p.sched_sel && !(*p.sched_sel < p.sched_thr)) {            // a peaked round (grid-uniform)
        if (!p.run_peaked) return;                                  // the lock-step kernel takes it
        p.W = p.W_peaked;
    }
    WV_TR(0, blockIdx.x == 0, kWvTraceSteps - 1, 0);
    WV_TR(1, (int)blockIdx.x == p.n_gru, kWvTraceSteps - 1, 0);
    if ((int)blockIdx.x < p.n_gru) wave_gru_role(p, wave_smem);
    else if ((int)blockIdx.x - p.n_gru < p.e.batch) wave_req_role(p, wave_smem);   // CTAs padding the last cluster leave
}

}  // namespace dt
