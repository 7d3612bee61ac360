// dt_fused.cuh -- steps (a5)-(a9) as ONE persistent kernel (bf16 weights): the whole best-first
// expansion of Algorithm 1 for every request of the batch, without a launch or a
// host round trip per popped node (the paper's builder pays one of each per pop).
//
// Two CTA roles, co-resident on the chip (cooperative launch), in lock-step over t = 0 .. B-1:
//
//  * GRU CTAs (n_gru = g / 16 of them) are weight-stationary: CTA j keeps the 48 rows of W_hh that
//    produce GRU units [16 j, 16 j + 16) and the matching columns of W1[:, d:] in shared memory for
//    the whole round.  Step t: for the node every request popped t-th, hidden half W_hh S_parent on
//    the 5th-generation tensor cores (fused_gru_role_tc: tcgen05.mma M = 64, N = hi|lo columns of up
//    to 32 requests, accumulators in TMEM; the parents' states, split bf16 hi + lo so that every
//    bf16 x bf16 product is exact and the state is carried to ~2^-17 relative, stream from L2 through
//    a cp.async ring in the 128-byte-swizzled operand layout), gates with the input half gathered
//    from the table P = E W_ih^T, new state S_t, and this CTA's split-K share of
//    W1[:, d:] S_t, a second small tcgen05 GEMM, written as a partial [batch, r].
//    fused_gru_role<UPC> is the same role on legacy mma.sync for shapes tcgen05 path rejects
//    (g not a multiple of 256, r > 256): ~256 MAC/clk/SM on B200, kept as the fallback.
//  * Request CTAs (one per request) own that request's heap in shared memory.  Step t: sum the
//    partials in a fixed order (deterministic, batch-invariant), a = SiLU(C + .),
//    z_m = (base_m + W2[cand_m, :] a) / T_eff over the M candidate rows of the node's depth
//    (rows staged into shared memory by cp.async while the GRU CTAs work),
//    slice log-softmax (reading A1), top-k, publish the next node's descriptor, merge the children
//    into the sorted frontier, pop entry 0 (reading A8) into slot t+1.
//    After the last pop the same CTA emits positions, padding and the ancestor mask (a9).
//
// The two roles hand over through self-describing words in global memory, one per producer and one
// 128-byte line each, so nothing is contended: request b publishes {step, round tag, parent state
// slot, token} in its descriptor word and GRU CTA c publishes round * 256 + its completed step count
// in its flag word; consumers poll with L1-bypassing loads (one lane per producer) and release the
// CTA through one barrier.  The round counter lives on the device, so no kernel has to reset anything.
// The request CTA keeps its frontier as a SORTED array (one entry per thread, truncated to the pops
// that remain), so a pop is "take entry 0" and a push is a rank-and-scatter merge of the k children.
// Static mode (Cond-static arm) walks only the greedy chain and records per-depth menus.
#pragma once
#include "dt_expand.cuh"
#include "dt_gemm_mma.cuh"
#include "dt_tcgen05.cuh"

namespace dt {

constexpr int kFusThreads = 256;
constexpr int kFusWarps = 8;
constexpr int kFusWPad = 32;      // bf16 elements of padding per W_hh row in smem (64 B: conflict-free LDS.128)
constexpr int kFusRedLd = 40;     // floats per row of the split-K reduction buffer
constexpr int kFusChunk = 32;     // requests per MMA pass (4 n8 tiles)
constexpr int kFusKB = 32;        // k per MMA block (two k16 steps)
constexpr int kFusRing = 3;       // state blocks in flight per warp (cp.async ring)
constexpr int kFusW2Pad = 32;     // bf16 elements of padding per staged W2 row (row stride = 16 banks mod 32)
constexpr int kFusMaxFront = 256; // frontier entries kept (>= DT_MAX_B)
constexpr int kFusDescStride = 16; // u64 words between two requests' descriptors (one 128-byte line each: concurrent
constexpr int kFusFlagStride = 32; // u32 words between two GRU CTAs' flags         partial writes to one line serialise in L2)

struct FusedParams {
    ExpandParams e;
    int n_gru, upc, m_tiles;       // GRU CTAs, units per CTA, ceil(3*upc/16)
    int gsz;                       // requests per GRU pass (<= kFusChunk): the batch is served in groups of gsz, each with its own
                                   // flag word, so the request CTAs of one group work while the GRU CTAs run the next group's pass
    int slot_stride;               // state slots per request = max_B + 2 (slot 0 = zeros, node t at t+1)
    int w2_smem;                   // request CTAs stage the M W2 rows in shared memory
    int w2_bufs;                   // ... in two buffers (the next depth is prefetched) or, if they do not fit, one
    __nv_bfloat16 *s_hi, *s_lo;    // [batch, slot_stride, g]
    float *s32;                    // [batch, slot_stride, g]
    float *partial;                // [n_gru, batch, r]
    unsigned long long *desc;      // [batch]  hand-over word request -> GRU: epoch(16) | state slot + 1 (16) | token (32)
    unsigned int *flags;           // [n_gru]  hand-over word GRU -> request: round base + steps completed by that GRU CTA
    unsigned int *round_ctr;       // rounds this handle has run: tags every hand-over word, so nothing needs zeroing
    // Cond-static arm: walk only the greedy chain (the frontier is dropped after every pop) for
    // B = L steps and record each depth's corrected top-k menu; the tree is then built by dt_scorers.cuh
    int static_mode;
    // adaptive schedule (dt_api.cu): the kernel runs only when (*sched_sel < sched_thr) == sched_want (null: always)
    const unsigned int *sched_sel; unsigned int sched_want, sched_thr;
    unsigned int *err;             // device error word: a hand-over wait that times out raises it and gives up (no hang)
    // speculation (tcgen05 GRU role only): while the request CTAs score node t the GRU CTAs already run the pass of the
    // node a chain would pop next (parent = node t, token = the marginal top-1 of the next depth) into the other of two
    // partial buffers; a request whose pop is that node continues on the `speculative pass done` flag
    int spec;
    size_t partial_buf;            // floats between the two partial buffers
    unsigned int *stats;           // optional (measurement aid): [0] GRU passes request 0 needed, [1] the most any request needed
    int32_t *menu_tok;             // [batch, L, k]
    float *menu_lp;                // [batch, L, k]
};

// ---- hand-over words -------------------------------------------------------------------------------
// Both directions use one self-describing word per producer (no shared counter, so no serialised
// atomics).  GRU -> request: the GRU CTA's threads store states / partials, a CTA barrier, then thread 0
// fences at gpu scope (the data is in L2 before the flag can be seen) and stores the flag.  Consumers
// poll with relaxed gpu-scope loads and read ALL hand-over data with L1-bypassing loads (ld.global.cg,
// cp.async.cg), i.e. from L2, the single point of coherence, after the control dependency on the polled
// word; they need no fence of their own.  Request -> GRU: the descriptor word is the whole payload.
// Release fence at gpu scope (MEMBAR.ALL.GPU): lighter than __threadfence(), which is sequentially consistent
// (MEMBAR.SC.GPU) and also invalidates L1.
__device__ __forceinline__ void fence_release_gpu() { asm volatile("fence.acq_rel.gpu;" ::: "memory"); }
__device__ __forceinline__ unsigned int ld_relaxed_u32(const unsigned int *p) {
    unsigned int v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ unsigned long long ld_relaxed_u64(const unsigned long long *p) {
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
// Bounded hand-over wait: spin on `ready`, look at the clock every 1024 polls, after 4 s (or when another CTA
// has given up) raise the device error word and return false: a protocol slip fails the call instead of hanging the GPU.
template <typename F>
__device__ __forceinline__ bool fused_spin(F ready, unsigned int *err) {
    unsigned long long t0 = 0ull;
    unsigned int n = 0;
    while (!ready()) {
        if (((++n) & 1023u) == 0u && err) {
            unsigned long long t;
            asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
            if (n == 1024u) t0 = t;
            if (*reinterpret_cast<volatile unsigned int *>(err) != 0u) return false;
            if (t - t0 > 4000000000ull) { atomicExch(err, 1u); return false; }
        }
    }
    return true;
}
__device__ __forceinline__ void st_relaxed_u32(unsigned int *p, unsigned int v) {
    asm volatile("st.relaxed.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ void st_relaxed_u64(unsigned long long *p, unsigned long long v) {
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
// descriptor word: step epoch (12 bits) | round tag (8) | parent state slot + 1 (12) | token (32)
__device__ __forceinline__ unsigned long long fused_desc_pack(int epoch, unsigned int tag, int sidx, int tok) {
    return ((unsigned long long)(unsigned int)epoch << 52) | ((unsigned long long)(tag & 0xFFu) << 44) |
           ((unsigned long long)(unsigned int)(sidx + 1) << 32) | (unsigned long long)(unsigned int)tok;
}
__device__ __forceinline__ bool fused_desc_is(unsigned long long d, int epoch, unsigned int tag) {
    return (unsigned int)(d >> 44) == (((unsigned int)epoch << 8) | (tag & 0xFFu));
}
__device__ __forceinline__ int fused_desc_sidx(unsigned long long d) { return (int)((d >> 32) & 0xFFFu) - 1; }
constexpr int kFusMaxGroups = 8;   // request groups the speculation keeps predictions for

// No initialisation kernel: the hand-over words carry the handle's round counter (flags: round * 256 + steps done,
// compared as a signed difference; descriptors: an 8-bit round tag), each request CTA publishes its own root
// descriptor (parent state = the zero slot, reading A4), and GRU CTA 0 bumps the counter when it leaves.
// shared-memory footprints (bytes) of the two roles
__host__ __device__ inline size_t fused_gru_smem(int g, int r, int upc, int m_tiles) {
    size_t w = (size_t)3 * upc * (g + kFusWPad) * 2;
    size_t ring = (size_t)kFusWarps * kFusRing * (2 * kFusChunk * kFusKB * 2);          // hi + lo blocks
    size_t red = (size_t)kFusWarps * m_tiles * 16 * kFusRedLd * 4;                      // aliases the ring
    size_t w1 = (size_t)r * 16 * 2;
    size_t snew = (size_t)2 * kFusChunk * 16 * 2;
    (void)upc;
    return w + (ring > red ? ring : red) + w1 + snew + 3 * kFusChunk * 4 + 64;
}
__host__ __device__ inline size_t fused_req_smem(int r, int M, int N, int k, int w2_smem, int w2_bufs = 2) {
    auto al = [](size_t x) { return (x + 15) / 16 * 16; };
    size_t s = al((size_t)2 * kFusMaxFront * 8) + al((size_t)k * 8) + al((size_t)M * 8) + al((size_t)2 * kFusMaxFront * 4) +
               al((size_t)k * 4) + 9 * al((size_t)r * 4) + al((size_t)M * 4) + 2 * al((size_t)2 * M * 4) + 4 * al((size_t)N * 4);
    if (w2_smem) s += al((size_t)w2_bufs * M * (r + kFusW2Pad) * 2);   // staging buffers: current depth (+ prefetched depth)
    return s + 16 + 64;
}

__device__ __forceinline__ void cp_async16(void *smem, const void *gmem) {
    unsigned int s = (unsigned int)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gmem));
}

// ------------------------------------------------------------------------------------------ GRU role
template <int UPC>
__device__ __forceinline__ void fused_gru_role(const FusedParams &p, unsigned char *smem_raw) {
    constexpr int MT = (3 * UPC + 15) / 16;
    constexpr int ROWS = 3 * UPC;
    constexpr int PP = UPC * kFusChunk / kFusThreads;          // epilogue (unit, request) pairs per thread
    constexpr int kBlkBytes = 2 * kFusChunk * kFusKB * 2;      // one k-block of states: [hi|lo][32 cols][32 k] bf16
    const ExpandParams &e = p.e;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, gq = lane >> 2, c4 = lane & 3;
    const int g = e.g, r = e.r, batch = e.batch;
    const int cta = blockIdx.x, u0 = cta * UPC;
    const int ldw = g + kFusWPad;
    const size_t stride = (size_t)p.slot_stride;

    __nv_bfloat16 *sW = reinterpret_cast<__nv_bfloat16 *>(smem_raw);
    unsigned char *sRingAll = reinterpret_cast<unsigned char *>(sW + (size_t)ROWS * ldw);
    const size_t ring_bytes = (size_t)kFusWarps * kFusRing * kBlkBytes;
    const size_t red_bytes = (size_t)kFusWarps * MT * 16 * kFusRedLd * 4;
    float *sRed = reinterpret_cast<float *>(sRingAll);                                  // aliases the ring
    unsigned int *sW1b = reinterpret_cast<unsigned int *>(sRingAll + (ring_bytes > red_bytes ? ring_bytes : red_bytes));  // [r][16] bf16
    __nv_bfloat16 *sNewH = reinterpret_cast<__nv_bfloat16 *>(sW1b + (size_t)r * 8);     // [32 requests][16 units]
    __nv_bfloat16 *sNewL = sNewH + kFusChunk * 16;
    int *sIdx = reinterpret_cast<int *>(sNewL + kFusChunk * 16);
    int *sTok = sIdx + kFusChunk;
    unsigned char *myRing = sRingAll + (size_t)warp * kFusRing * kBlkBytes;

    // resident weights: rows (gate, u0 + ul) of W_hh, columns d + u0 + ul of W1
    {
        const __nv_bfloat16 *whh = reinterpret_cast<const __nv_bfloat16 *>(e.w_hh);
        const int vpr = g / 8;
        for (int i = tid; i < ROWS * vpr; i += kFusThreads) {
            const int lr = i / vpr, v = i - lr * vpr;
            const int gate = lr / UPC, ul = lr - gate * UPC;
            uint4 q = ld_ro_v4(whh + ((size_t)gate * g + u0 + ul) * g + (size_t)v * 8);
            *reinterpret_cast<uint4 *>(sW + (size_t)lr * ldw + v * 8) = q;
        }
        const __nv_bfloat16 *w1 = reinterpret_cast<const __nv_bfloat16 *>(e.w1);
        __nv_bfloat16 *sW1h = reinterpret_cast<__nv_bfloat16 *>(sW1b);
        for (int i = tid; i < r * 16; i += kFusThreads) {       // K padded to 16 with zeros when UPC == 8
            const int j = i >> 4, ul = i & 15;
            sW1h[i] = (ul < UPC) ? w1[(size_t)j * (e.d + g) + e.d + u0 + ul] : __float2bfloat16_rn(0.f);
        }
        for (int i = tid; i < 2 * kFusChunk * 16; i += kFusThreads) sNewH[i] = __float2bfloat16_rn(0.f);   // H and L are adjacent
    }
    __syncthreads();

    // split-K over the warps: warp w owns k-blocks [blk0, blk1) of 32 k each
    const int nblk = g / kFusKB;
    const int blk0 = warp * nblk / kFusWarps, blk1 = (warp + 1) * nblk / kFusWarps;

    const unsigned int rnd = ld_relaxed_u32(p.round_ctr), fbase = rnd << 10;  // this round's tag / flag base
    for (int t = 0; t < e.B; ++t) {
        for (int c0 = 0; c0 < batch; c0 += p.gsz) {
            const int nb = min(p.gsz, batch - c0);
            const int ntiles = (nb + 7) >> 3;
            // wait for the descriptors of step t (lane = request), then broadcast through shared memory
            if (warp == 0) {
                int sidx = -1, tok = 0;
                if (lane < nb) {
                    unsigned long long dsc;
                    fused_spin([&] { dsc = ld_relaxed_u64(p.desc + (size_t)(c0 + lane) * kFusDescStride + (t & 1)); return fused_desc_is(dsc, t + 1, rnd); }, p.err);
                    sidx = fused_desc_sidx(dsc);
                    tok = (int)(dsc & 0xFFFFFFFFull);
                }
                sIdx[lane] = sidx; sTok[lane] = tok;
            }
            __syncthreads();

            // stream this warp's k-blocks of the parents' states (bf16 hi | lo) into its ring
            auto issue_block = [&](int blk) {
                unsigned char *dst = myRing + (size_t)((blk - blk0) % kFusRing) * kBlkBytes;
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    const int idx = i * 32 + lane;                   // 256 16-byte pieces: [hl][col][piece]
                    const int hl = idx >> 7, col = (idx >> 2) & 31, pc = idx & 3;
                    const int sidx = sIdx[col];
                    const size_t off = (sidx > 0) ? ((size_t)(c0 + col) * stride + sidx) * g : 0;   // 0 = zero slot
                    const __nv_bfloat16 *src = (hl ? p.s_lo : p.s_hi) + off + (size_t)blk * kFusKB + pc * 8;
                    cp_async16(dst + (size_t)idx * 16, src);
                }
                cp_async_commit();
            };
#pragma unroll
            for (int i = 0; i < kFusRing; ++i) {
                if (blk0 + i < blk1) issue_block(blk0 + i); else cp_async_commit();
            }

            // epilogue operands (input half from P, previous state): issued now, consumed after the MMAs
            float pr[PP], pz[PP], pn[PP], hp[PP];
#pragma unroll
            for (int i = 0; i < PP; ++i) {
                const int idx = tid + i * kFusThreads, ul = idx >> 5, bl = idx & 31;
                const int sidx = sIdx[bl];
                pr[i] = pz[i] = pn[i] = hp[i] = 0.f;
                if (sidx >= 0) {
                    const float *prow = e.P + (size_t)sTok[bl] * 3 * g + u0 + ul;
                    pr[i] = __ldg(prow); pz[i] = __ldg(prow + g); pn[i] = __ldg(prow + 2 * g);
                    if (sidx > 0) hp[i] = __ldcg(p.s32 + ((size_t)(c0 + bl) * stride + sidx) * g + u0 + ul);
                }
            }

            // hidden half W_hh S_parent on the tensor cores; A (weights) and B (states) use the same
            // k permutation inside a block, so 16-byte loads feed both operands directly
            float acc[MT][4][4];
#pragma unroll
            for (int mt = 0; mt < MT; ++mt)
#pragma unroll
                for (int nt = 0; nt < 4; ++nt)
#pragma unroll
                    for (int q = 0; q < 4; ++q) acc[mt][nt][q] = 0.f;
            for (int blk = blk0; blk < blk1; ++blk) {
                cp_async_wait<kFusRing - 1>();
                __syncwarp();
                const unsigned char *src = myRing + (size_t)((blk - blk0) % kFusRing) * kBlkBytes;
                uint4 bh[4], bl4[4];
#pragma unroll
                for (int nt = 0; nt < 4; ++nt) {
                    bh[nt] = *reinterpret_cast<const uint4 *>(src + (size_t)((nt * 8 + gq) * 4 + c4) * 16);
                    bl4[nt] = *reinterpret_cast<const uint4 *>(src + (size_t)(128 + (nt * 8 + gq) * 4 + c4) * 16);
                }
                __syncwarp();
                if (blk + kFusRing < blk1) issue_block(blk + kFusRing); else cp_async_commit();
                const int k0 = blk * kFusKB + 8 * c4;
                unsigned int aA[MT][4], aB[MT][4];
#pragma unroll
                for (int mt = 0; mt < MT; ++mt) {
                    const int r0 = mt * 16 + gq, r1 = r0 + 8;
                    uint4 A0 = make_uint4(0, 0, 0, 0), A1 = make_uint4(0, 0, 0, 0);
                    if (r0 < ROWS) A0 = *reinterpret_cast<const uint4 *>(sW + (size_t)r0 * ldw + k0);
                    if (r1 < ROWS) A1 = *reinterpret_cast<const uint4 *>(sW + (size_t)r1 * ldw + k0);
                    aA[mt][0] = A0.x; aA[mt][1] = A1.x; aA[mt][2] = A0.y; aA[mt][3] = A1.y;
                    aB[mt][0] = A0.z; aB[mt][1] = A1.z; aB[mt][2] = A0.w; aB[mt][3] = A1.w;
                }
                // four passes over the MT x 4 independent accumulators: consecutive MMAs never chain
#pragma unroll
                for (int nt = 0; nt < 4; ++nt)
#pragma unroll
                    for (int mt = 0; mt < MT; ++mt)
                        if (nt < ntiles) mma_bf16_16816(acc[mt][nt], aA[mt], bh[nt].x, bh[nt].y);
#pragma unroll
                for (int nt = 0; nt < 4; ++nt)
#pragma unroll
                    for (int mt = 0; mt < MT; ++mt)
                        if (nt < ntiles) mma_bf16_16816(acc[mt][nt], aB[mt], bh[nt].z, bh[nt].w);
#pragma unroll
                for (int nt = 0; nt < 4; ++nt)
#pragma unroll
                    for (int mt = 0; mt < MT; ++mt)
                        if (nt < ntiles) mma_bf16_16816(acc[mt][nt], aA[mt], bl4[nt].x, bl4[nt].y);
#pragma unroll
                for (int nt = 0; nt < 4; ++nt)
#pragma unroll
                    for (int mt = 0; mt < MT; ++mt)
                        if (nt < ntiles) mma_bf16_16816(acc[mt][nt], aB[mt], bl4[nt].z, bl4[nt].w);
            }
            cp_async_wait<0>();
            __syncthreads();                                    // every warp is done with its ring: reuse it as sRed
            {
                float *red = sRed + (size_t)warp * MT * 16 * kFusRedLd;
#pragma unroll
                for (int mt = 0; mt < MT; ++mt)
#pragma unroll
                    for (int nt = 0; nt < 4; ++nt) {
                        float *q0 = red + (size_t)(mt * 16 + gq) * kFusRedLd + nt * 8 + 2 * c4;
                        *reinterpret_cast<float2 *>(q0) = make_float2(acc[mt][nt][0], acc[mt][nt][1]);
                        *reinterpret_cast<float2 *>(q0 + 8 * kFusRedLd) = make_float2(acc[mt][nt][2], acc[mt][nt][3]);
                    }
            }
            __syncthreads();
            // gates (reading A2): r, z, n rows of unit ul are local rows ul, UPC + ul, 2 UPC + ul
#pragma unroll
            for (int i = 0; i < PP; ++i) {
                const int idx = tid + i * kFusThreads, ul = idx >> 5, bl = idx & 31;
                float hr = 0.f, hz = 0.f, hn = 0.f;
#pragma unroll
                for (int w = 0; w < kFusWarps; ++w) {
                    const float *red = sRed + (size_t)w * MT * 16 * kFusRedLd + bl;
                    hr += red[(size_t)ul * kFusRedLd];
                    hz += red[(size_t)(UPC + ul) * kFusRedLd];
                    hn += red[(size_t)(2 * UPC + ul) * kFusRedLd];
                }
                float hnew = 0.f;
                if (sIdx[bl] >= 0) {
                    const float rg = sigmoidf_fast(pr[i] + hr);
                    const float zg = sigmoidf_fast(pz[i] + hz);
                    const float ng = tanhf_fast(pn[i] + rg * hn);
                    hnew = (1.0f - zg) * ng + zg * hp[i];
                }
                const __nv_bfloat16 hi = __float2bfloat16_rn(hnew);
                const __nv_bfloat16 lo = __float2bfloat16_rn(hnew - __bfloat162float(hi));
                if (sIdx[bl] >= 0) {                             // publish S_t (slot t+1): fp32 and the bf16 hi/lo split
                    const size_t o = ((size_t)(c0 + bl) * stride + (t + 1)) * g + u0 + ul;
                    __stcg(p.s32 + o, hnew);
                    p.s_hi[o] = hi;
                    p.s_lo[o] = lo;
                }
                sNewH[bl * 16 + ul] = hi;
                sNewL[bl * 16 + ul] = lo;
            }
            __syncthreads();
            // this CTA's split-K share of W1[:, d:] S_t on the tensor cores:
            // [r x 16] (bf16 weights, exact) x [16 x 32] (new states, bf16 hi + lo)
            for (int mt = warp; mt < (r + 15) / 16; mt += kFusWarps) {
                const int j0 = mt * 16 + gq, j1 = j0 + 8;
                unsigned int a[4] = {0u, 0u, 0u, 0u};
                if (j0 < r) { a[0] = sW1b[j0 * 8 + c4]; a[2] = sW1b[j0 * 8 + 4 + c4]; }
                if (j1 < r) { a[1] = sW1b[j1 * 8 + c4]; a[3] = sW1b[j1 * 8 + 4 + c4]; }
                float c[4][4];
#pragma unroll
                for (int nt = 0; nt < 4; ++nt) {
                    c[nt][0] = c[nt][1] = c[nt][2] = c[nt][3] = 0.f;
                    const unsigned int *bh32 = reinterpret_cast<const unsigned int *>(sNewH) + (nt * 8 + gq) * 8;
                    const unsigned int *bl32 = reinterpret_cast<const unsigned int *>(sNewL) + (nt * 8 + gq) * 8;
                    mma_bf16_16816(c[nt], a, bh32[c4], bh32[4 + c4]);
                    mma_bf16_16816(c[nt], a, bl32[c4], bl32[4 + c4]);
                }
#pragma unroll
                for (int nt = 0; nt < 4; ++nt) {
                    const int col = nt * 8 + 2 * c4;
                    float *o0 = p.partial + ((size_t)cta * batch + c0 + col) * r;
                    if (col < nb) { if (j0 < r) __stcg(o0 + j0, c[nt][0]); if (j1 < r) __stcg(o0 + j1, c[nt][2]); }
                    if (col + 1 < nb) { if (j0 < r) __stcg(o0 + r + j0, c[nt][1]); if (j1 < r) __stcg(o0 + r + j1, c[nt][3]); }
                }
            }
            __syncthreads();
            if (tid == 0) { fence_release_gpu(); st_relaxed_u32(p.flags + (size_t)cta * kFusFlagStride + c0 / p.gsz, fbase + (unsigned int)(t + 1)); }
        }
    }
    if (cta == 0 && tid == 0) st_relaxed_u32(p.round_ctr, rnd + 1u);      // every CTA read it long ago
}

// ------------------------------------------------------------------------- GRU role, tcgen05 + TMEM
// Same work as fused_gru_role<16>, on the 5th-generation tensor cores: legacy mma.sync runs at about
// 256 MAC/clk/SM on B200 (measured, profiles/), which made the 3072 x 1024 x 64 hidden half 6 us per
// step; tcgen05.mma does it in ~1 us.  One CTA owns 16 GRU units = 48 rows of W_hh (M = 64 tile, rows
// 48..63 are phantom and ignored), N = 64 columns per pass (32 requests x {bf16 hi, bf16 lo} of the
// parent state), K = g streamed in 128-wide chunks through a 6-slot cp.async ring.  The accumulator
// lives in TMEM; a second, tiny tcgen05 GEMM [r x 16] x [16 x 64] gives this CTA's split-K share of
// W1[:, d:] S_t.  Operand layout of the big GEMM: K-major, 128-byte swizzle (a warp-wide cp.async moves four whole
// 128-byte state rows and lands conflict-free); the tiny one uses unswizzled core matrices (dt_tcgen05.cuh).
constexpr int kTcUPC = 16;
constexpr int kTcKC = 256;            // k per ring slot = four 64-wide swizzle blocks, one per issuing warp
constexpr int kTcSlots = 3;
constexpr int kTcSlotBytes = 64 * kTcKC * 2;          // 64 columns x 256 k bf16 = 32 KB
constexpr int kTcIssuers = 4;         // warps 0..3 each issue the MMAs of one k-block into their own accumulator
constexpr int kTcCols = 512;          // TMEM columns: D1[w] at 64 w (w < 4), D2 tiles at 256 and 320

__host__ __device__ inline size_t fused_tc_smem(int g, int r) {
    const size_t a = (size_t)48 * g * 2;                              // W_hh slice as core matrices
    const size_t ring = (size_t)kTcSlots * kTcSlotBytes;              // must cover the phantom rows: >= 16 * g * 2
    const size_t a2 = (size_t)((r + 127) / 128) * 128 * 32;           // W1[:, d + u0 ..] slice [r_pad x 16] bf16
    const size_t b2 = 64 * 32;                                        // new states [64 cols x 16] bf16
    const size_t sh = 48 * 34 * 4;                                    // hidden-half pre-activations
    return a + ring + a2 + b2 + sh + 3 * kFusChunk * 4 + 8 * 8 + 64 + (size_t)(4 * kFusMaxGroups * kFusChunk + 32) * 4 + 1024;
}

__device__ __forceinline__ void fused_gru_role_tc(const FusedParams &p, unsigned char *smem_raw) {
    constexpr int UPC = kTcUPC;
    constexpr int PP = UPC * kFusChunk / kFusThreads;          // (unit, request) pairs per thread = 2
    const ExpandParams &e = p.e;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int g = e.g, r = e.r, batch = e.batch;
    const int cta = blockIdx.x, u0 = cta * UPC;
    const size_t stride = (size_t)p.slot_stride;
    const int n_kc = g / kTcKC;                                // ring chunks per pass
    const int m2_tiles = (r + 127) / 128;

    // carve (smem_raw is 1024-byte aligned by the kernel)
    unsigned char *sA = smem_raw;                                             // 6 row groups x (g/64 swizzle atoms of 1 KB)
    const uint32_t sboA = (uint32_t)g * 16;                                   // bytes between 8-row groups
    unsigned char *sRing = sA + (size_t)48 * g * 2;
    unsigned char *sA2 = sRing + (size_t)kTcSlots * kTcSlotBytes;             // [r_pad/8 groups][2 chunks][8 rows][16 B]
    unsigned char *sB2 = sA2 + (size_t)m2_tiles * 128 * 32;                   // [8 groups][2 chunks][8 cols][16 B]
    float *sH = reinterpret_cast<float *>(sB2 + 64 * 32);                     // [48][34]
    int *sIdx = reinterpret_cast<int *>(sH + 48 * 34);
    int *sTok = sIdx + kFusChunk;
    unsigned long long *mbar = reinterpret_cast<unsigned long long *>(sTok + 2 * kFusChunk);   // [0],[1] slot free, [2] D1, [3] D2
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(mbar + 8);
    // per request (speculation, see the pass loop): predicted parent slot (-1 none, -2 nothing speculated) and token of node rE,
    // the node whose descriptor is expected next, and the state (0 = A: a speculation for rE may exist, its descriptor
    // decides; 1 = B: the real node rE ran in the previous pass; 2 = finished)
    int *sPredIdx = reinterpret_cast<int *>(tmem_slot + 16);                  // [groups][32]
    int *sPredTok = sPredIdx + kFusMaxGroups * kFusChunk;
    int *rE = sPredTok + kFusMaxGroups * kFusChunk;
    int *rSt = rE + kFusMaxGroups * kFusChunk;
    int *sCtl = rSt + kFusMaxGroups * kFusChunk;                              // [0] this pass has columns, [1] the group is finished
    int *sNode = sTok + kFusChunk;                                            // [32] node of this pass's column
    for (int i = tid; i < kFusMaxGroups * kFusChunk; i += kFusThreads) { sPredIdx[i] = -2; sPredTok[i] = 0; rE[i] = 0; rSt[i] = 0; }

    // resident weights in core-matrix layout
    {
        const __nv_bfloat16 *whh = reinterpret_cast<const __nv_bfloat16 *>(e.w_hh);
        const int vpr = g / 8;
        // as asynchronous copies, all in flight at once: the weights come from HBM every round (the select has streamed
        // 150 MB through L2 since the last one) and a load -> store loop pays that latency once per iteration
        for (int i = tid; i < 48 * vpr; i += kFusThreads) {
            const int m = i / vpr, c = i - m * vpr;                // local row m = gate * 16 + ul, k-chunk c
            const int gate = m >> 4, ul = m & 15;
            cp_async16(sA + (size_t)(m >> 3) * sboA + (size_t)(c >> 3) * 1024 + (m & 7) * 128 + (((c & 7) ^ (m & 7)) << 4),
                       whh + ((size_t)gate * g + u0 + ul) * g + (size_t)c * 8);
        }
        const __nv_bfloat16 *w1 = reinterpret_cast<const __nv_bfloat16 *>(e.w1);
        if (((e.d | g) & 7) == 0 && (reinterpret_cast<uintptr_t>(w1) & 15) == 0) {                                // 8 units = one aligned 16-byte piece of a W1 row
            for (int i = tid; i < m2_tiles * 128 * 2; i += kFusThreads) {
                const int j = i >> 1, uh = i & 1;
                unsigned char *dst = sA2 + (size_t)(j >> 3) * 256 + uh * 128 + (j & 7) * 16;
                if (j < r) cp_async16(dst, w1 + (size_t)j * (e.d + g) + e.d + u0 + 8 * uh);
                else *reinterpret_cast<uint4 *>(dst) = make_uint4(0u, 0u, 0u, 0u);
            }
        } else {
            for (int i = tid; i < m2_tiles * 128 * 16; i += kFusThreads) {
                const int j = i >> 4, ul = i & 15;
                const __nv_bfloat16 v = (j < r) ? w1[(size_t)j * (e.d + g) + e.d + u0 + ul] : __float2bfloat16_rn(0.f);
                *reinterpret_cast<__nv_bfloat16 *>(sA2 + (size_t)(j >> 3) * 256 + (ul >> 3) * 128 + (j & 7) * 16 + (ul & 7) * 2) = v;
            }
        }
        cp_async_commit();
        cp_async_wait<0>();
        if (tid == 0) {
            tc::mbar_init(tc::smem_u32(mbar + 0), kTcIssuers);      // slot free
            tc::mbar_init(tc::smem_u32(mbar + 1), kTcIssuers);
            tc::mbar_init(tc::smem_u32(mbar + 2), kTcIssuers);      // D1 complete (one commit per issuing warp)
            tc::mbar_init(tc::smem_u32(mbar + 3), 1);               // D2 complete
            tc::mbar_init_fence();
        }
        if (warp == 0) tc::tmem_alloc<kTcCols>(tmem_slot);
    }
    tc::fence_proxy_async();
    tc::fence_before_sync();
    __syncthreads();
    tc::fence_after_sync();
    const uint32_t tmem = *tmem_slot;
    const uint32_t idesc2 = tc::make_idesc_bf16(128, 64);
    const uint32_t aA = tc::smem_u32(sA), aRing = tc::smem_u32(sRing), aA2 = tc::smem_u32(sA2), aB2 = tc::smem_u32(sB2);
    const uint32_t mb0 = tc::smem_u32(mbar);
    const uint64_t descA0 = tc::make_desc_sw128(aA, sboA), descB0 = tc::make_desc_sw128(aRing, 1024);
    uint32_t ph_free = 0, ph_d1 = 0, ph_d2 = 0;                 // mbarrier phases (uniform across the CTA)

    // this thread's share of one ring slot: the 16-byte piece `my_c` of the 128-byte rows of request `my_rq`
    // (hi and lo, both 64-wide k-blocks of the slot); a warp instruction moves 4 whole 128-byte rows
    const int my_c = tid & 7, my_rq = tid >> 3;

    const unsigned int rnd = ld_relaxed_u32(p.round_ctr), fbase = rnd << 10;  // this round's tag / flag base
    WV_TR(0, cta == 0, kWvTraceSteps - 1, 1);
    // Passes, not steps.  Pass k serves every request of a group with ONE column: the node its descriptor asks for, or --
    // speculation -- the node a chain would pop next (parent = the node just confirmed, token = the marginal top-1 of the
    // next depth), computed while the request CTA still scores that parent.  Per request, identically in every GRU CTA
    // (the decisions depend on descriptor CONTENTS only, never on their timing) and mirrored by the request CTA:
    //   state A (a speculation for node e may exist): wait for descriptor e; if it is the speculated node (or a leaf, which
    //            needs no state) e is final: speculate e + 1 in this pass and stay in A; else run the real node e -> B;
    //   state B (the real node e ran in the previous pass): speculate e + 1 in this pass -> A.
    // A hit costs a request one pass per node (and the pass overlaps its scoring), a miss two.  Without p.spec every
    // pass runs the real node k of every request (the plain lock-step schedule).  Flag of pass k: round base + k + 1.
    const int n_grp = (batch + p.gsz - 1) / p.gsz;
    unsigned int done_mask = 0u;
    __syncthreads();
    for (int t = 0; done_mask != (1u << n_grp) - 1u; ++t) {     // t = pass index
        for (int c0 = 0; c0 < batch; c0 += p.gsz) {
            const int nb = min(p.gsz, batch - c0);
            const int gi = c0 / p.gsz;
            if ((done_mask >> gi) & 1u) continue;
            // Columns of the hidden-half GEMM: requests' hi halves in rows [0, lo_off), lo halves in [lo_off, 2 lo_off);
            // N shrinks with the batch (8 columns serve up to 4 requests), and so do the ring traffic and the MMA time.
            const int ncol = (nb <= 4) ? 8 : (nb <= 8) ? 16 : (nb <= 16) ? 32 : 64;
            const int lo_off = ncol >> 1;
            const uint32_t idesc1 = tc::make_idesc_bf16(64, ncol);
            const int n_lo = lo_off + my_rq;
            const uint32_t my_dst_hi = (uint32_t)((my_rq >> 3) * 1024 + (my_rq & 7) * 128 + ((my_c ^ (my_rq & 7)) << 4));
            const uint32_t my_dst_lo = (uint32_t)((n_lo >> 3) * 1024 + (n_lo & 7) * 128 + ((my_c ^ (n_lo & 7)) << 4));
            unsigned int *my_flag = p.flags + (size_t)cta * kFusFlagStride + gi;
            if (warp == 0) {
                int c_sidx = -1, c_tok = 0, c_node = 0;          // this pass's column of request c0 + lane (none: -1)
                int st = 2, en = 0;
                if (lane < nb) {
                    const int ri = gi * kFusChunk + lane;
                    st = rSt[ri]; en = rE[ri];
                    int pi = sPredIdx[ri], pt = sPredTok[ri];
                    bool advance = false;                        // node en is final: go on to en + 1 with a speculation
                    if (st == 0) {
                        unsigned long long dsc, hnt = 0ull;     // descriptor and (speculation) the request's hint, both self-validating
                        const unsigned long long *dw = p.desc + (size_t)(c0 + lane) * kFusDescStride + (en & 1);
                        fused_spin([&] {
                            dsc = ld_relaxed_u64(dw);
                            if (!p.spec) return fused_desc_is(dsc, en + 1, rnd);
                            hnt = ld_relaxed_u64(dw + 2);
                            return fused_desc_is(dsc, en + 1, rnd) && fused_desc_is(hnt, en + 1, rnd); }, p.err);
                        const int sidx = fused_desc_sidx(dsc);
                        int tok = (int)(dsc & 0xFFFFFFFFull);
                        if (p.spec) tok &= 0xFFFFFF;
                        const bool hit = p.spec ? (sidx < 0 || (sidx == pi && tok == pt)) : (sidx < 0);
                        if (!hit) { c_sidx = sidx; c_tok = tok; c_node = en; st = 1; }
                        advance = hit || !p.spec;                // (without speculation there is no state B: next node, next pass)
                        // the node to speculate on after en: the request CTA's hint (en's marginal top-1 child -- a chain -- or the
                        // best entry left in its frontier)
                        pi = -1; pt = 0;
                        if (p.spec && fused_desc_sidx(hnt) >= 0) { pi = fused_desc_sidx(hnt); pt = (int)(hnt & 0xFFFFFFull); }
                    } else if (st == 1) advance = true;
                    if (advance) {
                        en += 1;
                        if (!p.spec) st = (en >= e.B) ? 2 : 0;
                        else if (en >= e.B) st = 2;
                        else {
                            st = 0;
                            if (pi >= 0) { c_sidx = pi; c_tok = pt; c_node = en; }
                            else pi = -2;                            // nothing speculated for en: only a leaf descriptor is a hit
                        }
                    }
                    rSt[ri] = st; rE[ri] = en; sPredIdx[ri] = pi; sPredTok[ri] = pt;
                }
                sIdx[lane] = c_sidx; sTok[lane] = c_tok; sNode[lane] = c_node;
                const unsigned int anyc = __ballot_sync(0xffffffffu, c_sidx >= 0);
                const unsigned int live = __ballot_sync(0xffffffffu, lane < nb && st != 2);
                if (lane == 0) { sCtl[0] = anyc != 0u; sCtl[1] = live == 0u; }
            } else if (warp == 1 && p.spec && t > 0) {
                // meanwhile: the parents' states were written by the other GRU CTAs, at the latest in the previous pass (every
                // CTA flags every pass, so this never waits for long; without speculation a descriptor is only published once
                // its request has seen every flag of that pass)
                const unsigned int want = fbase + (unsigned int)t;
                fused_spin([&] {
                    bool ok = true;
                    for (int q = lane; q < p.n_gru; q += 32) ok = ok & ((int)(ld_relaxed_u32(p.flags + (size_t)q * kFusFlagStride + gi) - want) >= 0);
                    return ok; }, p.err);
            }
            __syncthreads();
            {
                const bool anyc = sCtl[0] != 0, fin = sCtl[1] != 0;
                if (fin) done_mask |= 1u << gi;
                if (!anyc) {                                     // nothing to compute: the pass still counts
                    if (tid == 0) st_relaxed_u32(my_flag, fbase + (unsigned int)(t + 1));
                    __syncthreads();                             // sCtl is rewritten by the next poll
                    continue;
                }
            }
            WV_TR(0, cta == 0 && c0 == 0, t, 0);

            // source rows of this thread's ring pieces (column n < 32: hi of request n, else lo of request n - 32)
            const int my_sidx = sIdx[my_rq];
            const size_t my_off = (my_sidx > 0) ? ((size_t)(c0 + my_rq) * stride + my_sidx) * g : 0;   // 0 = zero slot
            const __nv_bfloat16 *src_hi = p.s_hi + my_off + (size_t)my_c * 8, *src_lo = p.s_lo + my_off + (size_t)my_c * 8;
            auto issue_chunk = [&](int kc) {
                if (my_rq >= lo_off) return;                        // columns beyond N: nothing to stream
                unsigned char *dst = sRing + (size_t)(kc % kTcSlots) * kTcSlotBytes;
                const size_t k0 = (size_t)kc * kTcKC;
#pragma unroll
                for (int kb = 0; kb < kTcKC / 64; ++kb) {           // per 64-wide k-block (8 KB apart in the slot)
                    cp_async16(dst + kb * 8192 + my_dst_hi, src_hi + k0 + kb * 64);
                    cp_async16(dst + kb * 8192 + my_dst_lo, src_lo + k0 + kb * 64);
                }
            };
            // A group of at most 16 requests needs N <= 32 columns: with the k-blocks packed N rows apart (not 64) all of K fits
            // the ring, so every chunk is in flight at once and the MMAs go out in ONE burst behind one wait and one barrier
            // instead of a wait / barrier / issue / refill round per chunk (same accumulators, same order: same bits)
            const int kb_bytes = (ncol >> 3) * 1024, slot_b = (kTcKC / 64) * kb_bytes;
            const bool burst = (size_t)n_kc * slot_b <= (size_t)kTcSlots * kTcSlotBytes && ncol < 64;
            if (burst) {
                if (my_rq < lo_off) {
#pragma unroll 1
                    for (int kc = 0; kc < n_kc; ++kc) {
                        unsigned char *dst = sRing + (size_t)kc * slot_b;
                        const size_t k0 = (size_t)kc * kTcKC;
#pragma unroll
                        for (int kb = 0; kb < kTcKC / 64; ++kb) {
                            cp_async16(dst + kb * kb_bytes + my_dst_hi, src_hi + k0 + kb * 64);
                            cp_async16(dst + kb * kb_bytes + my_dst_lo, src_lo + k0 + kb * 64);
                        }
                    }
                }
                cp_async_commit();
            } else {
#pragma unroll 1
                for (int kc = 0; kc < kTcSlots; ++kc) { if (kc < n_kc) issue_chunk(kc); cp_async_commit(); }
            }

            // epilogue operands (input half from P, previous state): issued now, consumed after the MMAs
            float pr[PP], pz[PP], pn[PP], hp[PP];
#pragma unroll
            for (int i = 0; i < PP; ++i) {
                const int idx = tid + i * kFusThreads, ul = idx & 15, bl = idx >> 4;   // lanes along the units: 64 B per row
                const int sidx = sIdx[bl];
                pr[i] = pz[i] = pn[i] = hp[i] = 0.f;
                if (sidx >= 0) {
                    const float *prow = e.P + (size_t)sTok[bl] * 3 * g + u0 + ul;
                    pr[i] = __ldg(prow); pz[i] = __ldg(prow + g); pn[i] = __ldg(prow + 2 * g);
                    if (sidx > 0) hp[i] = __ldcg(p.s32 + ((size_t)(c0 + bl) * stride + sidx) * g + u0 + ul);
                }
            }

            WV_TR(0, cta == 0 && c0 == 0, t, 1);
            // hidden half: D1[64 x 64] = W_hh slice [64 x g] . [S_hi | S_lo]^T, K streamed through the ring
            if (burst) {
                cp_async_wait<0>();
                tc::fence_proxy_async();
                __syncthreads();
                if (warp < kTcIssuers && lane == 0) {
                    tc::fence_after_sync();
#pragma unroll 1
                    for (int kc = 0; kc < n_kc; ++kc) {
                        const uint64_t da = descA0 + (uint64_t)((kc * (kTcKC / 64) + warp) * 64);
                        const uint64_t db = descB0 + (uint64_t)((kc * slot_b + warp * kb_bytes) >> 4);
#pragma unroll
                        for (int s4 = 0; s4 < 4; ++s4)
                            tc::mma_bf16(tmem + 64 * warp, da + (uint64_t)(s4 * 2), db + (uint64_t)(s4 * 2), idesc1, (kc | s4) ? 1u : 0u);
                    }
                    tc::commit(mb0 + 16);
                }
            } else
#pragma unroll 1
            for (int kc = 0; kc < n_kc; ++kc) {
                cp_async_wait<kTcSlots - 1>();
                tc::fence_proxy_async();
                __syncthreads();
                if (warp < kTcIssuers && lane == 0) {
                    // warp w issues k-block w of the slot (A: +1 KB per block, B: +8 KB) as four K = 16 steps (+32 B)
                    // into its own accumulator D1[w]; the epilogue adds the four
                    tc::fence_after_sync();
                    const uint64_t da = descA0 + (uint64_t)((kc * (kTcKC / 64) + warp) * 64);
                    const uint64_t db = descB0 + (uint64_t)((kc % kTcSlots) * (kTcSlotBytes / 16) + warp * 512);
#pragma unroll
                    for (int s4 = 0; s4 < 4; ++s4)
                        tc::mma_bf16(tmem + 64 * warp, da + (uint64_t)(s4 * 2), db + (uint64_t)(s4 * 2), idesc1, (kc | s4) ? 1u : 0u);
                    if (kc + kTcSlots < n_kc) tc::commit(mb0 + 8 * (kc & 1));       // this slot is refilled below
                    if (kc == n_kc - 1) tc::commit(mb0 + 16);
                }
                if (kc + kTcSlots < n_kc) {                  // refill the slot once its MMAs have read it
                    tc::mbar_wait(mb0 + 8 * (kc & 1), (ph_free >> (kc & 1)) & 1u);
                    ph_free ^= 1u << (kc & 1);
                    issue_chunk(kc + kTcSlots);
                }
                cp_async_commit();
            }
            cp_async_wait<0>();
            tc::mbar_wait(mb0 + 16, ph_d1); ph_d1 ^= 1u;
            tc::fence_after_sync();
            WV_TR(0, cta == 0 && c0 == 0, t, 3);
            // TMEM -> shared: row m = 16 w + i sits in lane 32 w + i (i < 16) for an M = 64 accumulator
            __syncwarp();
            if (warp < 3) {
                float acc[32], v[32];
#pragma unroll
                for (int c = 0; c < 32; ++c) acc[c] = 0.f;
                // the same association for every N, (hi + lo) per accumulator, so results do not depend on the batch
                if (ncol == 64) {
                    float vl[32];
#pragma unroll
                    for (int q = 0; q < kTcIssuers; ++q) {       // four accumulators x {hi, lo} column halves
                        tc::tmem_ld32(tmem + ((uint32_t)(32 * warp) << 16) + 64 * q, v);
                        tc::tmem_ld32(tmem + ((uint32_t)(32 * warp) << 16) + 64 * q + 32, vl);
#pragma unroll
                        for (int c = 0; c < 32; ++c) acc[c] += v[c] + vl[c];
                    }
                } else {
#pragma unroll
                    for (int q = 0; q < kTcIssuers; ++q) {       // hi and lo halves both sit in the first N <= 32 columns
                        tc::tmem_ld32(tmem + ((uint32_t)(32 * warp) << 16) + 64 * q, v);
                        if (ncol == 32) {
#pragma unroll
                            for (int c = 0; c < 16; ++c) acc[c] += v[c] + v[16 + c];
                        } else if (ncol == 16) {
#pragma unroll
                            for (int c = 0; c < 8; ++c) acc[c] += v[c] + v[8 + c];
                        } else {
#pragma unroll
                            for (int c = 0; c < 4; ++c) acc[c] += v[c] + v[4 + c];
                        }
                    }
                }
                if (lane < 16) {
#pragma unroll
                    for (int c = 0; c < 32; ++c) sH[(16 * warp + lane) * 34 + c] = acc[c];
                }
            }
            tc::fence_before_sync();
            __syncthreads();
            WV_TR(0, cta == 0 && c0 == 0, t, 10);
            // gates (reading A2): rows ul, 16 + ul, 32 + ul are the r, z, n pre-activations of unit ul
#pragma unroll
            for (int i = 0; i < PP; ++i) {
                const int idx = tid + i * kFusThreads, ul = idx & 15, bl = idx >> 4;
                float hnew = 0.f;
                if (sIdx[bl] >= 0) {
                    const float rg = sigmoidf_fast(pr[i] + sH[ul * 34 + bl]);
                    const float zg = sigmoidf_fast(pz[i] + sH[(16 + ul) * 34 + bl]);
                    const float ng = tanhf_fast(pn[i] + rg * sH[(32 + ul) * 34 + bl]);
                    hnew = (1.0f - zg) * ng + zg * hp[i];
                }
                const __nv_bfloat16 hi = __float2bfloat16_rn(hnew);
                const __nv_bfloat16 lo = __float2bfloat16_rn(hnew - __bfloat162float(hi));
                if (sIdx[bl] >= 0) {                             // publish S_t (slot t+1): fp32 and the bf16 hi/lo split
                    const size_t o = ((size_t)(c0 + bl) * stride + (sNode[bl] + 1)) * g + u0 + ul;
                    __stcg(p.s32 + o, hnew);
                    p.s_hi[o] = hi;
                    p.s_lo[o] = lo;
                }
                // operand B of the W1 GEMM: column bl (hi) and 32 + bl (lo), k = ul
                unsigned char *q = sB2 + (size_t)(bl >> 3) * 256 + (ul >> 3) * 128 + (bl & 7) * 16 + (ul & 7) * 2;
                *reinterpret_cast<__nv_bfloat16 *>(q) = hi;
                *reinterpret_cast<__nv_bfloat16 *>(q + 4 * 256) = lo;
            }
            tc::fence_proxy_async();
            __syncthreads();
            WV_TR(0, cta == 0 && c0 == 0, t, 11);
            // this CTA's split-K share of W1[:, d:] S_t: D2[r x 64] = W1 slice [r x 16] . [S_hi | S_lo]^T
            if (tid == 0) {
                tc::fence_after_sync();
                const uint64_t db = tc::make_desc(aB2, 128, 256);
                for (int mt = 0; mt < m2_tiles; ++mt)
                    tc::mma_bf16(tmem + 256 + 64 * mt, tc::make_desc(aA2 + (uint32_t)mt * 4096, 128, 256), db, idesc2, 0u);
                tc::commit(mb0 + 24);
            }
            tc::mbar_wait(mb0 + 24, ph_d2); ph_d2 ^= 1u;
            tc::fence_after_sync();
            __syncwarp();
            WV_TR(0, cta == 0 && c0 == 0, t, 5);
            const unsigned int live = __ballot_sync(0xffffffffu, lane < nb && sIdx[lane] >= 0);   // requests of this pass
            const unsigned int odd = __ballot_sync(0xffffffffu, p.spec && (sNode[lane] & 1));       // their partial buffer (node parity)
            for (int mt = warp >> 2; mt < m2_tiles; mt += 2) {
                float vh[32], vl[32];
                const uint32_t ta = tmem + ((uint32_t)(32 * (warp & 3)) << 16) + 256 + 64 * mt;
                tc::tmem_ld32(ta, vh);
                tc::tmem_ld32(ta + 32, vl);
                const int j = mt * 128 + 32 * (warp & 3) + lane;
                if (j < r) {
                    float *o = p.partial + ((size_t)cta * batch + c0) * r + j;
#pragma unroll
                    for (int c = 0; c < 32; ++c)
                        if ((live >> c) & 1u) __stcg(o + (size_t)c * r + (((odd >> c) & 1u) ? p.partial_buf : 0), vh[c] + vl[c]);
                }
            }
            tc::fence_before_sync();
            __syncthreads();
            WV_TR(0, cta == 0 && c0 == 0, t, 6);
            if (tid == 0) { fence_release_gpu(); st_relaxed_u32(my_flag, fbase + (unsigned int)(t + 1)); }
            WV_TR(0, cta == 0 && c0 == 0, t, 7);
        }
    }
    __syncthreads();
    WV_TR(0, cta == 0, kWvTraceSteps - 1, 2);
    if (warp == 0) tc::tmem_free<kTcCols>(tmem);
    if (cta == 0 && tid == 0) st_relaxed_u32(p.round_ctr, rnd + 1u);      // every CTA read it long ago
}

// -------------------------------------------------------------------------------------- request role
// Frontier entries are ordered by the pop comparator of reading A8, (g desc, token asc, parent asc),
// packed so that a larger (hi, lo) pair pops first: hi = ord_key(g), lo = ~token << 32 | ~parent.
__device__ __forceinline__ bool front_gt(unsigned int ah, unsigned long long al, unsigned int bh, unsigned long long bl) {
    return ah > bh || (ah == bh && al > bl);
}

struct FusedReqSmem {
    int kwait;          // GRU pass that produces the current node's partials (its flag is waited for)
    int kspec;          // GRU pass that speculates on the next node (see fused_gru_role_tc)
    int pred_sidx, pred_tok;   // the frontier entry hinted for the next node (parent slot, token); -1: none, the chain child
    int n_valid;        // tree slots filled so far (root included)
    int n_front;        // live frontier entries
    int cur;            // which of the two frontier buffers is live
};

__device__ __forceinline__ void fused_req_role(const FusedParams &p, unsigned char *smem_raw) {
    __shared__ FusedReqSmem sm;
    __shared__ float sLp1[DT_MAX_L];                            // marginal log-probability of every depth's top-1 candidate (hints)
    __shared__ int sTop1[DT_MAX_L];                             // and its token
    const ExpandParams &e = p.e;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int b = blockIdx.x - p.n_gru;
    const int r = e.r, M = e.M, k = e.k, N = e.N, L = e.L, batch = e.batch, B = e.B;
    const int ldw2 = r + kFusW2Pad;
    const unsigned int rnd = ld_relaxed_u32(p.round_ctr), fbase = rnd << 10;  // this round's tag / flag base

    // carve, every array 16-byte aligned: [W2 rows bf16] [frontier lo u64 x2] [new lo] [frontier hi u32 x2]
    // [new hi] [a] [z] [base] [cand tok] [tree tok / par / dep / score]
    size_t off = 0;
    auto carve = [&](size_t bytes) { unsigned char *q = smem_raw + off; off += (bytes + 15) / 16 * 16; return q; };
    __nv_bfloat16 *sW2_ = reinterpret_cast<__nv_bfloat16 *>(carve(p.w2_smem ? (size_t)p.w2_bufs * M * ldw2 * 2 : 0));   // [buffers][M rows]
    unsigned long long *fLo = reinterpret_cast<unsigned long long *>(carve((size_t)2 * kFusMaxFront * 8));
    unsigned long long *nLo = reinterpret_cast<unsigned long long *>(carve((size_t)k * 8));
    unsigned int *fHi = reinterpret_cast<unsigned int *>(carve((size_t)2 * kFusMaxFront * 4));
    unsigned int *nHi = reinterpret_cast<unsigned int *>(carve((size_t)k * 4));
    float *sA = reinterpret_cast<float *>(carve((size_t)r * 4));
    float *sP = reinterpret_cast<float *>(carve((size_t)8 * r * 4));        // group sums of the split-K partials
    float *sWst = reinterpret_cast<float *>(carve((size_t)2 * kFusWarps * 4)); // per-warp softmax (max, sum)
    float *sZ = reinterpret_cast<float *>(carve((size_t)M * 4));
    float *sBase_ = reinterpret_cast<float *>(carve((size_t)2 * M * 4));      // [2 buffers][M]
    int *sTok_ = reinterpret_cast<int *>(carve((size_t)2 * M * 4));
    int *nTok = reinterpret_cast<int *>(carve((size_t)N * 4));
    int *nPar = reinterpret_cast<int *>(carve((size_t)N * 4));
    int *nDep = reinterpret_cast<int *>(carve((size_t)N * 4));
    float *nSco = reinterpret_cast<float *>(carve((size_t)N * 4));

    const __nv_bfloat16 *w2 = reinterpret_cast<const __nv_bfloat16 *>(e.w2);

    // stage the candidate table of depth `dep` (row b*L + dep): ids, base logits, the M rows of W2
    // wait for the GRU CTAs' flags of pass `kpass` (warp 0; a lane's flags are polled together: one L2 round trip, not one each)
    auto wait_flags = [&](int kpass) {
        const unsigned int want = fbase + (unsigned int)(kpass + 1);
        const unsigned int *fl = p.flags + b / p.gsz;
        fused_spin([&] {
            bool ok = true;
            for (int q = lane; q < p.n_gru; q += 32) ok = ok & ((int)(ld_relaxed_u32(fl + (size_t)q * kFusFlagStride) - want) >= 0);
            return ok; }, p.err);
    };
    // `kpass` >= 0: warp 0 also looks ONCE at the next step's flags here, under the latency of the candidate loads (with
    // speculation they are usually set already, but even a successful poll is a round trip to L2); returns whether they
    // were all there (warp 0; else the loop top waits for them, after the staging has been issued)
    auto stage_depth = [&](int dep, int kpass) -> bool {
        const size_t row = (size_t)b * L + dep;
        int ctok[(DT_MAX_M + kFusThreads - 1) / kFusThreads];
        float cval[(DT_MAX_M + kFusThreads - 1) / kFusThreads];
#pragma unroll
        for (int i = 0; i < (DT_MAX_M + kFusThreads - 1) / kFusThreads; ++i) {
            const int m = tid + i * kFusThreads;
            if (m < M) { ctok[i] = e.cand_id[row * M + m]; cval[i] = e.cand_val[row * M + m]; }
        }
        bool seen = false;
        if (warp == 0 && kpass >= 0) {
            const unsigned int want = fbase + (unsigned int)(kpass + 1);
            bool ok = true;
            for (int q = lane; q < p.n_gru; q += 32) ok = ok & ((int)(ld_relaxed_u32(p.flags + b / p.gsz + (size_t)q * kFusFlagStride) - want) >= 0);
            seen = __all_sync(0xffffffffu, ok);
        }
#pragma unroll
        for (int i = 0; i < (DT_MAX_M + kFusThreads - 1) / kFusThreads; ++i) {
            const int m = tid + i * kFusThreads;
            if (m < M) { sTok_[m] = ctok[i]; sBase_[m] = cval[i]; }
        }
        __syncthreads();
        if (p.w2_smem) {
            const int vpr = r / 8;
            for (int i = tid; i < M * vpr; i += kFusThreads) {
                const int m = i / vpr, v = i - m * vpr;
                cp_async16(sW2_ + (size_t)m * ldw2 + v * 8, w2 + (size_t)sTok_[m] * r + (size_t)v * 8);
            }
        }
        cp_async_commit();
        return seen;
    };

    // warps 1..7 (224 threads, named barrier 1) stage depth `dep` into staging buffer `buf` while warp 0 does something else
    auto stage_side = [&](int dep, int buf) {
        constexpr int nw = kFusThreads - 32;
        const int wt = tid - 32;
        const size_t row = (size_t)b * L + dep;
        int *dTok = sTok_ + buf * M;
        float *dBase = sBase_ + buf * M;
        __nv_bfloat16 *dW2 = sW2_ + (size_t)buf * M * ldw2;
        for (int m = wt; m < M; m += nw) { dTok[m] = e.cand_id[row * M + m]; dBase[m] = e.cand_val[row * M + m]; }
        asm volatile("bar.sync 1, %0;" ::"n"(nw) : "memory");
        if (p.w2_smem) {
            const int vpr = r / 8;
            for (int i = wt; i < M * vpr; i += nw) {
                const int m = i / vpr, v = i - m * vpr;
                cp_async16(dW2 + (size_t)m * ldw2 + v * 8, w2 + (size_t)dTok[m] * r + (size_t)v * 8);
            }
        }
        cp_async_commit();
    };
    int cb = 0;                                                 // staging buffer of the current node's depth
    const bool two_bufs = !p.w2_smem || p.w2_bufs == 2;         // (without staged rows only ids / base logits are buffered)
    int buf_dep0 = 0, buf_dep1 = -1;                            // depth whose rows each staging buffer holds (or is being filled with)

    if (p.spec) {                                               // slice log-softmax of the base logits at position 0 (sorted: v_0 is the max)
        for (int row = warp; row < L; row += kFusWarps) {
            const float *v = e.cand_val + ((size_t)b * L + row) * M;
            const float v0 = v[0];
            float ssum = 0.f;
            for (int m = lane; m < M; m += 32) ssum += __expf((v[m] - v0) / e.T_eff);
            ssum = warp_sum(ssum);
            if (lane == 0) { sLp1[row] = -__logf(ssum); sTop1[row] = e.cand_id[((size_t)b * L + row) * M]; }
        }
        __syncthreads();
    }
    if (tid == 0) {
        nTok[0] = e.root_tokens[b]; nPar[0] = -1; nDep[0] = 0; nSco[0] = 0.f;
        // step-0 descriptor: the root, whose parent state is the zero slot (reading A4)
        // (the hint words are written in every round, speculating or not, like the descriptors: a word then never outlives
        // the round that wrote it, and the 8-bit round tag cannot alias)
        st_relaxed_u64(p.desc + (size_t)b * kFusDescStride + 2,                               // hint for node 1: the root's top-1 child
                       fused_desc_pack(1, rnd, (p.spec && 1 < L && 1 < B) ? 1 : -1, p.spec ? sTop1[0] : 0));
        st_relaxed_u64(p.desc + (size_t)b * kFusDescStride, fused_desc_pack(1, rnd, 0, min(max(e.root_tokens[b], 0), e.V - 1)));
        sm.n_valid = 1; sm.n_front = 0; sm.cur = 0; sm.kwait = 0; sm.kspec = 1; sm.pred_sidx = (p.spec && 1 < L && 1 < B) ? 1 : -1; sm.pred_tok = p.spec ? sTop1[0] : 0;
        if (p.stats && b == 0) p.stats[1] = 0u;
    }
    __syncthreads();
    stage_depth(0, -1);
    bool polled = false;                                        // the flags of the coming step were seen while staging

    WV_TR(1, b == 0, kWvTraceSteps - 1, 1);
    for (int t = 0; t < B; ++t) {
        const int n_valid = sm.n_valid;
        const int n_front = sm.n_front, cur = sm.cur;
        const bool node_ok = (t < n_valid);
        const int depth = node_ok ? nDep[t] : L;
        const bool expand = node_ok && depth < L;               // block-uniform
        __nv_bfloat16 *const sW2 = sW2_ + (size_t)cb * M * ldw2;
        float *const sBase = sBase_ + cb * M;
        int *const sTok = sTok_ + cb * M;
        // Every request CTA waits for the GRU CTAs' step t, expanded or not: nobody runs ahead, so the
        // descriptor word and the partial buffer are never overwritten while still in use.
        // C = H W1h^T of the node's depth does not depend on the GRU CTAs: fetch it while waiting for them
        float cpre = 0.f;
        if (expand && tid < r) cpre = e.C[((size_t)b * L + depth) * r + tid];
        if (warp == 0 && !polled) wait_flags(p.spec ? sm.kwait : t);
        __syncthreads();
        WV_TR(1, b == 0, t, 0);
        // the live frontier is entries 1 .. n_front of buffer `cur` (entry 0 was popped by the previous step)
        const unsigned int *oHi = fHi + cur * kFusMaxFront + 1;
        const unsigned long long *oLo = fLo + cur * kFusMaxFront + 1;
        unsigned int *wHi = fHi + (cur ^ 1) * kFusMaxFront;
        unsigned long long *wLo = fLo + (cur ^ 1) * kFusMaxFront;
        int n_new = 0;
        if (expand) {
            const size_t row = (size_t)b * L + depth;           // H_{depth+1} <-> row index depth (A12)
            // a = SiLU(C + W1[:, d:] S_t): the n_gru split-K partials are summed in a fixed order (batch-invariant):
            // G thread groups each sum a contiguous range of GRU CTAs with 16-byte loads, then the groups are added
            {
                const int r4 = r >> 2;
                const int G = min(8, kFusThreads / r4);
                const int per = (p.n_gru + G - 1) / G;
                const int jq = tid % r4, qg = tid / r4;
                if (qg < G) {
                    const size_t ps4 = ((size_t)batch * r) >> 2;
                    const float4 *pp = reinterpret_cast<const float4 *>(p.partial + (size_t)(p.spec ? (t & 1) : 0) * p.partial_buf + (size_t)b * r) + jq;
                    const int q0 = qg * per, q1 = min(p.n_gru, q0 + per);
                    float4 s0 = make_float4(0.f, 0.f, 0.f, 0.f), s1 = s0;
                    int q = q0;
                    for (; q + 16 <= q1; q += 16) {
                        float4 v[16];
#pragma unroll
                        for (int i = 0; i < 16; ++i) v[i] = __ldcg(pp + (size_t)(q + i) * ps4);
#pragma unroll
                        for (int i = 0; i < 16; i += 2) {
                            s0.x += v[i].x; s0.y += v[i].y; s0.z += v[i].z; s0.w += v[i].w;
                            s1.x += v[i + 1].x; s1.y += v[i + 1].y; s1.z += v[i + 1].z; s1.w += v[i + 1].w;
                        }
                    }
                    for (; q < q1; ++q) {
                        const float4 v = __ldcg(pp + (size_t)q * ps4);
                        s0.x += v.x; s0.y += v.y; s0.z += v.z; s0.w += v.w;
                    }
                    *reinterpret_cast<float4 *>(sP + (size_t)qg * r + 4 * jq) = make_float4(s0.x + s1.x, s0.y + s1.y, s0.z + s1.z, s0.w + s1.w);
                }
                __syncthreads();
                for (int j = tid; j < r; j += kFusThreads) {
                    float acc = sP[j];
                    for (int gq = 1; gq < G; ++gq) acc += sP[(size_t)gq * r + j];
                    const float x = ((j == tid) ? cpre : e.C[row * r + j]) + acc;
                    sA[j] = x * sigmoidf_acc(x);
                }
            }
            cp_async_wait<0>();
            __syncthreads();
            WV_TR(1, b == 0, t, 1);
            // z_m = ((base_m - base_0) + W2[cand_m, :] a) / T_eff     PAPER.md:143-144 (shift-invariant)
            // four lanes per candidate row, interleaved 16-byte pieces
            const float base0 = sBase[0];
            {
                const int q4 = tid & 3, nvec = r / 8;
                float wmx = -INFINITY, wsm = 0.f;                     // this warp's running (max, sum exp(z - max))
                for (int mb = 0; mb < M; mb += kFusThreads / 4) {     // warp-uniform trip count (shuffles below)
                    const int m = mb + (tid >> 2);
                    float acc = 0.f;
                    if (m >= M) {
                    } else if (p.w2_smem) {
                        const __nv_bfloat16 *wr = sW2 + (size_t)m * ldw2;
                        for (int v = q4; v < nvec; v += 4) {
                            const uint4 q = *reinterpret_cast<const uint4 *>(wr + (size_t)v * 8);
                            const float4 a0 = *reinterpret_cast<const float4 *>(sA + (size_t)v * 8);
                            const float4 a1 = *reinterpret_cast<const float4 *>(sA + (size_t)v * 8 + 4);
                            float f[8];
                            unpack8(q, f);
                            acc = fmaf(f[0], a0.x, acc); acc = fmaf(f[1], a0.y, acc); acc = fmaf(f[2], a0.z, acc); acc = fmaf(f[3], a0.w, acc);
                            acc = fmaf(f[4], a1.x, acc); acc = fmaf(f[5], a1.y, acc); acc = fmaf(f[6], a1.z, acc); acc = fmaf(f[7], a1.w, acc);
                        }
                    } else {
                        const __nv_bfloat16 *wr = w2 + (size_t)sTok[m] * r;
                        for (int v = q4; v < nvec; v += 4) {
                            const uint4 q = ld_ro_v4(wr + (size_t)v * 8);
                            const float *sp = sA + (size_t)v * 8;
                            float f[8];
                            unpack8(q, f);
#pragma unroll
                            for (int i = 0; i < 8; ++i) acc = fmaf(f[i], sp[i], acc);
                        }
                    }
                    acc += __shfl_xor_sync(0xffffffffu, acc, 1);
                    acc += __shfl_xor_sync(0xffffffffu, acc, 2);
                    float z = -INFINITY;
                    if (m < M) { z = __fdiv_rn((sBase[m] - base0) + acc, e.T_eff); if (q4 == 0) sZ[m] = z; }
                    // slice log-softmax statistics (reading A1), online: the 8 candidates of this warp pass ...
                    float zm = fmaxf(z, __shfl_xor_sync(0xffffffffu, z, 4));
                    zm = fmaxf(zm, __shfl_xor_sync(0xffffffffu, zm, 8));
                    zm = fmaxf(zm, __shfl_xor_sync(0xffffffffu, zm, 16));
                    const float nmx = fmaxf(wmx, zm);
                    float ex = (q4 == 0 && m < M) ? expf(z - nmx) : 0.f;
                    ex += __shfl_xor_sync(0xffffffffu, ex, 4);
                    ex += __shfl_xor_sync(0xffffffffu, ex, 8);
                    ex += __shfl_xor_sync(0xffffffffu, ex, 16);
                    if (nmx > -INFINITY) { wsm = wsm * expf(wmx - nmx) + ex; wmx = nmx; }
                }
                if (lane == 0) { sWst[2 * warp] = wmx; sWst[2 * warp + 1] = wsm; }
            }
            __syncthreads();
            WV_TR(1, b == 0, t, 2);
            // While warp 0 picks the top-k and the pop, the other warps prefetch the candidate rows of the NEXT depth into the
            // other staging buffer: a chain (and most pops of a bushy tree's subtree) goes one level down, and the fetch of
            // M W2 rows takes longer than what is left between two steps.  A different depth is staged after the pop.
            if (two_bufs && depth + 1 < L && t + 1 < B && (cb ? buf_dep0 : buf_dep1) != depth + 1) {
                if (warp != 0) stage_side(depth + 1, cb ^ 1);       // (what that buffer held was waited for before the dots)
                if (cb) buf_dep0 = depth + 1; else buf_dep1 = depth + 1;
            }
            // ... then warp 0 merges the 8 warps' (max, sum) pairs in warp order and picks the top-k by (logp desc, token asc)
            // = (z desc, token asc) without anything that scales with M * M: every lane takes the best of its own M / 32
            // sortable keys (ord(z), ~token) and k rounds of a warp max reduction give L, the k-th best of the 32 lane maxima
            // (lane in the low bits, so the 32 values are distinct): at least k keys lie at or above L, so the true top k do;
            // the keys at or above L (k plus a few) go one to a lane and are ranked among themselves by counting over the
            // full keys through shuffles.  The exact top k in the exact order; the k winners become the new entries
            if (warp == 0) {
                float zmax = -INFINITY;
#pragma unroll
                for (int w = 0; w < kFusWarps; ++w) zmax = fmaxf(zmax, sWst[2 * w]);
                float ssum = 0.f;
#pragma unroll
                for (int w = 0; w < kFusWarps; ++w) { const float mw = sWst[2 * w]; if (mw > -INFINITY) ssum += sWst[2 * w + 1] * expf(mw - zmax); }
                const float lse = logf(ssum);
                const float gpar = nSco[t];
                unsigned long long *svK = reinterpret_cast<unsigned long long *>(sP);   // the group sums are dead
                const int MI = (M + 31) >> 5;
                unsigned long long kk[8];
                unsigned int hmax = 0u;
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    const int m = lane + 32 * i;
                    kk[i] = 0ull;
                    if (i < MI && m < M)
                        kk[i] = ((unsigned long long)ord_key(sZ[m]) << 32) | (unsigned long long)(0xFFFFFFFFu - (unsigned int)sTok[m]);
                    hmax = max(hmax, (unsigned int)(kk[i] >> 32));
                }
                unsigned int cur_l = (hmax & ~31u) | (unsigned int)(31 - lane), Lh = 0u;
#pragma unroll 1
                for (int rr = 0; rr < k; ++rr) {
                    Lh = __reduce_max_sync(0xffffffffu, cur_l);
                    if (cur_l == Lh) cur_l = 0u;
                }
                Lh &= ~31u;
                int ns = 0;
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    if (i >= MI) break;
                    const bool in = (unsigned int)(kk[i] >> 32) >= Lh && kk[i] != 0ull;
                    const unsigned int bal = __ballot_sync(0xffffffffu, in);
                    const int at = ns + __popc(bal & ((1u << lane) - 1u));
                    if (in && at < 32) svK[at] = kk[i];
                    ns += __popc(bal);
                }
                __syncwarp();
                auto emit = [&](unsigned long long mk, int rank) {
                    const float mz = ord_key_inv((unsigned int)(mk >> 32));
                    const int mtok = (int)(0xFFFFFFFFu - (unsigned int)(mk & 0xFFFFFFFFull));
                    const float lpm = (mz - zmax) - lse;
                    nHi[rank] = ord_key(gpar + lpm);
                    nLo[rank] = ((unsigned long long)(0xFFFFFFFFu - (unsigned int)mtok) << 32) |
                                (unsigned long long)(0xFFFFFFFFu - (unsigned int)t);
                    if (p.static_mode) {                        // the depth's shared menu (row index = depth of node t)
                        p.menu_tok[((size_t)b * L + depth) * k + rank] = mtok;
                        p.menu_lp[((size_t)b * L + depth) * k + rank] = lpm;
                    }
                };
                if (ns <= 32) {
                    const unsigned long long mk = lane < ns ? svK[lane] : 0ull;
                    int rank = 0;
#pragma unroll 4
                    for (int q = 0; q < ns; ++q) rank += (__shfl_sync(0xffffffffu, mk, q) > mk);
                    if (lane < ns && rank < k) emit(mk, rank);
                } else {                                        // many equal keys at the threshold: count over the slice
#pragma unroll 1
                    for (int m = lane; m < M; m += 32) {
                        const unsigned long long mk = ((unsigned long long)ord_key(sZ[m]) << 32) | (unsigned long long)(0xFFFFFFFFu - (unsigned int)sTok[m]);
                        if ((unsigned int)(mk >> 32) < Lh) continue;
                        int rank = 0;
#pragma unroll 1
                        for (int q = 0; q < M; ++q)
                            rank += ((((unsigned long long)ord_key(sZ[q]) << 32) | (unsigned long long)(0xFFFFFFFFu - (unsigned int)sTok[q])) > mk);
                        if (rank < k) emit(mk, rank);
                    }
                }
                __syncwarp();
            }
            n_new = k;
            WV_TR(1, b == 0, t, 3);
        }
        // The node popped now is the better of the old frontier head and the best new entry: warp 0 publishes its descriptor
        // BEFORE the merge (and before the CTA barrier that hands the new entries to the other warps), so the GRU CTAs start
        // step t+1 while this CTA is still merging.
        const int cap = B - t;                                  // pops still to do, this one included
        int tot = n_front + n_new;
        if (warp == 0) {
            if (tot > 0) {
                // best new entry: max of (hi, lo) over the k new entries (lo's low word, ~parent, is the same for all)
                unsigned int h = 0u; unsigned long long l = 0ull; bool have = false;
                if (n_new > 0) {
                    const unsigned int mh = (lane < n_new) ? nHi[lane] : 0u;
                    const unsigned long long ml = (lane < n_new) ? nLo[lane] : 0ull;
                    h = __reduce_max_sync(0xffffffffu, mh);
                    const unsigned int l_hi = __reduce_max_sync(0xffffffffu, (lane < n_new && mh == h) ? (unsigned int)(ml >> 32) : 0u);
                    l = ((unsigned long long)l_hi << 32) | (unsigned long long)(0xFFFFFFFFu - (unsigned int)t);
                    have = true;
                }
                if (lane == 0) {
                    const unsigned int hn = h; const unsigned long long ln = l;      // best new entry
                    const bool pop_old = n_front > 0 && (!have || !front_gt(h, l, oHi[0], oLo[0]));
                    if (pop_old) { h = oHi[0]; l = oLo[0]; }
                    const int tok = (int)(0xFFFFFFFFu - (unsigned int)(l >> 32));
                    const int par = (int)(0xFFFFFFFFu - (unsigned int)(l & 0xFFFFFFFFull));
                    const int dep = nDep[par] + 1;
                    // Hint for the GRU CTAs' speculation on the node AFTER this one.  Default: this node's marginal top-1 child (a
                    // chain).  But if the best entry left in the frontier beats the score that child can be expected to have
                    // (this node's score + the marginal log-probability of the next depth's top-1), or this node is a leaf, the
                    // frontier entry is the better guess.  Only a guess: a hit is decided by comparing with the real pop.
                    int h_sidx = -1, h_tok = 0;
                    if (p.spec && t + 2 < B && dep + 1 < L) { h_sidx = t + 2; h_tok = sTop1[dep]; }     // the chain: slot of node t + 1
                    if (p.spec && !p.static_mode && t + 2 < B) {
                        unsigned int h2 = 0u; unsigned long long l2 = 0ull; bool have2 = false;
                        if (pop_old) {
                            if (n_front > 1) { h2 = oHi[1]; l2 = oLo[1]; have2 = true; }
                            if (have && (!have2 || front_gt(hn, ln, h2, l2))) { h2 = hn; l2 = ln; have2 = true; }
                        } else {
                            if (n_front > 0) { h2 = oHi[0]; l2 = oLo[0]; have2 = true; }
                            if (n_new > 1 && (!have2 || front_gt(nHi[1], nLo[1], h2, l2))) { h2 = nHi[1]; l2 = nLo[1]; have2 = true; }   // (ranked)
                        }
                        if (have2) {
                            const int par2 = (int)(0xFFFFFFFFu - (unsigned int)(l2 & 0xFFFFFFFFull));
                            const int dep2 = nDep[par2] + 1;
                            if (dep2 < L && (dep >= L || ord_key_inv(h2) > ord_key_inv(h) + sLp1[dep])) {
                                h_sidx = par2 + 1; h_tok = (int)(0xFFFFFFFFu - (unsigned int)(l2 >> 32));
                            }
                        }
                    }
                    // (the descriptor of step s lives in word s & 1 of the request's line: with speculation this CTA may publish
                    // step t + 1 before every GRU CTA has read step t; the depth rides in the token's top byte)
                    if (t + 1 < B) {
                        st_relaxed_u64(p.desc + (size_t)b * kFusDescStride + 2 + ((t + 1) & 1), fused_desc_pack(t + 2, rnd, h_sidx, h_tok));
                        st_relaxed_u64(p.desc + (size_t)b * kFusDescStride + ((t + 1) & 1),
                                       fused_desc_pack(t + 2, rnd, dep < L ? par + 1 : -1, p.spec ? (tok | (min(dep, 255) << 24)) : tok));
                    }
                    // What the GRU CTAs speculated for THIS node (told a step ago): the hinted frontier entry, else the marginal
                    // top-1 child of the node expanded now.  A hit (or a leaf, which needs no state) is served by the
                    // speculating pass, a miss by the pass after it
                    const bool hit = dep >= L || (sm.pred_sidx >= 0 && par + 1 == sm.pred_sidx && tok == sm.pred_tok);
                    sm.kwait = sm.kspec + (hit ? 0 : 1); sm.kspec = sm.kwait + 1;
                    sm.pred_sidx = h_sidx; sm.pred_tok = h_tok;
                    nTok[t + 1] = tok; nPar[t + 1] = par; nDep[t + 1] = dep; nSco[t + 1] = ord_key_inv(h);
                    sm.n_valid = t + 2; sm.n_front = p.static_mode ? 0 : min(tot, cap) - 1; sm.cur = cur ^ 1;
                }
            } else if (lane == 0) {
                sm.n_front = 0; sm.kwait = sm.kspec; sm.kspec = sm.kwait + 1; sm.pred_sidx = -1;
                if (t + 1 < B) {
                    st_relaxed_u64(p.desc + (size_t)b * kFusDescStride + 2 + ((t + 1) & 1), fused_desc_pack(t + 2, rnd, -1, 0));
                    st_relaxed_u64(p.desc + (size_t)b * kFusDescStride + ((t + 1) & 1), fused_desc_pack(t + 2, rnd, -1, 0));
                }
            }
        }
        WV_TR(1, b == 0, t, 9);
        __syncthreads();                                        // the new entries (and the pop) are visible to every warp
        // Between two steps: warp 0 waits for the flags of the pass the NEXT node needs (with speculation they are usually there,
        // but even a successful poll is a round trip to L2) while warps 1..7 merge the new entries into the sorted frontier
        // (other buffer, truncated to the pops that remain) and stage the next depth's candidate rows; they meet at the
        // barrier on top of the loop.
        int next_dep = L;                                       // depth of the node popped now (L = none / leaf)
        if (tot > 0) next_dep = nDep[t + 1];
        polled = false;
        if (warp == 0) {
            if (t + 1 < B) { wait_flags(p.spec ? sm.kwait : t + 1); polled = true; }
            WV_TR(1, b == 0, t, 4);
        } else {
            constexpr int nw = kFusThreads - 32;
            const int wt = tid - 32;
            if (tot > 0) {
                for (int i = wt; i < n_front; i += nw) {
                    const unsigned int h = oHi[i]; const unsigned long long l = oLo[i];
                    int c = 0;
                    for (int j = 0; j < n_new; ++j) c += front_gt(nHi[j], nLo[j], h, l);
                    const int pos = i + c;
                    if (pos < cap) { wHi[pos] = h; wLo[pos] = l; }
                }
                if (wt >= nw - n_new) {                         // the last n_new threads place the new entries
                    const int j = wt - (nw - n_new);
                    const unsigned int h = nHi[j]; const unsigned long long l = nLo[j];
                    int c = 0;
                    for (int j2 = 0; j2 < n_new; ++j2) c += front_gt(nHi[j2], nLo[j2], h, l);
                    int lo = 0, hi = n_front;                    // first old entry that does not beat (h, l)
                    while (lo < hi) {
                        const int mid = (lo + hi) >> 1;
                        if (front_gt(oHi[mid], oLo[mid], h, l)) lo = mid + 1; else hi = mid;
                    }
                    const int pos = lo + c;
                    if (pos < cap) { wHi[pos] = h; wLo[pos] = l; }
                }
            }
            // neither the prefetched depth nor the current one (a sibling): stage it now (overlaps the GRU CTAs' next pass), once
            // whatever is still landing in that buffer has landed
            if (t + 1 < B && next_dep < L && next_dep != buf_dep0 && next_dep != buf_dep1) {
                cp_async_wait<0>();
                asm volatile("bar.sync 1, %0;" ::"n"(nw) : "memory");
                stage_side(next_dep, two_bufs ? cb ^ 1 : 0);
            }
        }
        if (t + 1 < B && next_dep < L) {                        // (block-uniform) which buffer holds the next node's rows
            if (next_dep != buf_dep0 && next_dep != buf_dep1) { if (cb || !two_bufs) buf_dep0 = next_dep; else buf_dep1 = next_dep; }
            cb = (next_dep == buf_dep0) ? 0 : 1;
        }
    }
    cp_async_wait<0>();                                         // (a prefetch nobody used)
    __syncthreads();

    if (p.stats && tid == 0) {
        const unsigned int np = (unsigned int)((p.spec ? sm.kwait : B - 1) + 1);
        if (b == 0) p.stats[0] = np;
        atomicMax(p.stats + 1, np);
    }
    if (p.static_mode) return;                                  // menus are out; dt_scorers.cuh builds and emits the tree
    WV_TR(1, b == 0, kWvTraceSteps - 1, 2);
    // emitter (a9): dead-leaf padding (reading A10), positions, ancestor-or-self mask
    const int n = sm.n_valid;
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
    WV_TR(1, b == 0, kWvTraceSteps - 1, 3);
}

template <int UPC>
__global__ void __launch_bounds__(kFusThreads, 1) fused_expand_kernel(FusedParams p) {
    extern __shared__ __align__(1024) unsigned char fused_smem[];
    if (p.sched_sel && (unsigned int)(*p.sched_sel < p.sched_thr) != p.sched_want) return;   // the other schedule was chosen (grid-uniform)
    WV_TR(0, blockIdx.x == 0, kWvTraceSteps - 1, 0);
    WV_TR(1, (int)blockIdx.x == p.n_gru, kWvTraceSteps - 1, 0);
    if ((int)blockIdx.x < p.n_gru) {
        if constexpr (UPC == 0) fused_gru_role_tc(p, fused_smem);
        else fused_gru_role<UPC>(p, fused_smem);
    } else fused_req_role(p, fused_smem);
}

}  // namespace dt
