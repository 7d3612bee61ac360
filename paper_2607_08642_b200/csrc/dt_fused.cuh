// dt_fused.cuh -- steps (a5)-(a9) as ONE persistent kernel (bf16 weights): the whole best-first
// expansion of Algorithm 1 for every request of the batch, without a launch or a
// host round trip per popped node (the paper's builder pays one of each per pop).
//
// Two CTA roles, co-resident on the chip (cooperative launch), in lock-step over t = 0 .. B-1:
//
//  * GRU CTAs (n_gru of them) are weight-stationary: CTA j keeps the 3*upc rows of W_hh that
//    produce GRU units [j*upc, (j+1)*upc) and the matching columns of W1[:, d:] in shared memory for
//    the whole round.  Step t: for the node every request popped t-th, hidden half W_hh S_parent on
//    the tensor cores (mma.sync m16n8k16, states split bf16 hi + lo so the bf16 x bf16 products are
//    exact and the state is carried to ~2^-17 relative), gates with the input half gathered from the
//    table P = E W_ih^T, new state S_t, and this CTA's split-K share of
//    W1[:, d:] S_t written as a partial [batch, r].
//  * Request CTAs (one per request) own that request's heap in shared memory.  Step t: sum the
//    partials in CTA order (fixed order => deterministic, batch-invariant), a = SiLU(C + .),
//    z_m = (base_m + W2[cand_m, :] a) / T_eff over the M candidate rows of the node's depth
//    (rows staged into shared memory by cp.async while the GRU CTAs work),
//    slice log-softmax (reading A1), top-k, push, pop the maximum (reading A8) into slot t+1.
//    After the last pop the same CTA emits positions, padding and the ancestor mask (a9).
//
// The two roles hand over through two monotone counters in global memory (release: fence + atomic
// add; acquire: ld.acquire spin by one thread + bar.sync) and a double-buffered node descriptor.
#pragma once
#include "dt_expand.cuh"
#include "dt_gemm_mma.cuh"

namespace dt {

constexpr int kFusThreads = 256;
constexpr int kFusWarps = 8;
constexpr int kFusWPad = 32;      // bf16 elements of padding per W_hh row in smem (64 B: conflict-free LDS.128)
constexpr int kFusRedLd = 40;     // floats per row of the split-K reduction buffer
constexpr int kFusChunk = 32;     // requests per MMA pass (4 n8 tiles)

struct FusedParams {
    ExpandParams e;
    int n_gru, upc, m_tiles;       // GRU CTAs, units per CTA, ceil(3*upc/16)
    int slot_stride;               // state slots per request = max_B + 2 (slot 0 = zeros, node t at t+1)
    int w2_smem;                   // request CTAs stage the M W2 rows in shared memory
    __nv_bfloat16 *s_hi, *s_lo;    // [batch, slot_stride, g]
    float *s32;                    // [batch, slot_stride, g]
    float *partial;                // [n_gru, batch, r]
    int2 *desc;                    // [2, batch]  {state slot of the parent or -1 = skip, token}
    unsigned int *sync;            // [0] ready (request -> GRU), [32] done (GRU -> request)
};

__device__ __forceinline__ unsigned int ld_acquire_u32(const unsigned int *p) {
    unsigned int v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
// All threads of the CTA call: waits until *ctr >= target.
__device__ __forceinline__ void cta_wait_counter(const unsigned int *ctr, unsigned int target) {
    if (threadIdx.x == 0) {
        while (ld_acquire_u32(ctr) < target) { }
    }
    __syncthreads();
}
// All threads call after their global writes: publishes them and bumps *ctr by one.
__device__ __forceinline__ void cta_signal_counter(unsigned int *ctr) {
    __syncthreads();
    if (threadIdx.x == 0) { __threadfence(); atomicAdd(ctr, 1u); }
}

// Zero the hand-over words and write the step-0 descriptor (the root: parent state = zeros, reading A4).
__global__ void fused_init_kernel(FusedParams p) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i == 0) { p.sync[0] = 0u; p.sync[32] = 0u; }
    if (i < p.e.batch) {
        int tok = p.e.root_tokens[i];
        tok = min(max(tok, 0), p.e.V - 1);
        p.desc[i] = make_int2(0, tok);
    }
}

// shared-memory footprints (bytes) of the two roles
__host__ __device__ inline size_t fused_gru_smem(int g, int r, int upc, int m_tiles) {
    size_t w = (size_t)3 * upc * (g + kFusWPad) * 2;
    size_t red = (size_t)kFusWarps * m_tiles * 16 * kFusRedLd * 4;
    size_t w1 = (size_t)r * upc * 4;
    size_t snew = (size_t)upc * (kFusChunk + 1) * 4;
    return w + red + w1 + snew + 3 * kFusChunk * 4;
}
__host__ __device__ inline size_t fused_req_smem(int r, int M, int N, int heap_cap, int w2_smem) {
    size_t s = (size_t)r * 4 + (size_t)M * 12 + (size_t)N * 16 + (size_t)heap_cap * 12 + 64;
    if (w2_smem) s += (size_t)M * (r + 8) * 2;
    return (s + 15) / 16 * 16 + 16;
}

// ------------------------------------------------------------------------------------------ GRU role
template <int UPC>
__device__ __forceinline__ void fused_gru_role(const FusedParams &p, unsigned char *smem_raw) {
    constexpr int MT = (3 * UPC + 15) / 16;
    constexpr int ROWS = 3 * UPC;
    constexpr int PP = UPC * kFusChunk / kFusThreads;          // epilogue (unit, request) pairs per thread
    constexpr int kNewLd = kFusChunk + 1;
    const ExpandParams &e = p.e;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, gq = lane >> 2, c4 = lane & 3;
    const int g = e.g, r = e.r, batch = e.batch;
    const int cta = blockIdx.x, u0 = cta * UPC;
    const int ldw = g + kFusWPad;
    const size_t stride = (size_t)p.slot_stride;

    __nv_bfloat16 *sW = reinterpret_cast<__nv_bfloat16 *>(smem_raw);
    float *sRed = reinterpret_cast<float *>(sW + (size_t)ROWS * ldw);
    float *sW1 = sRed + (size_t)kFusWarps * MT * 16 * kFusRedLd;
    float *sNew = sW1 + (size_t)r * UPC;
    int *sIdx = reinterpret_cast<int *>(sNew + UPC * kNewLd);
    int *sTok = sIdx + kFusChunk;

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
        for (int i = tid; i < r * UPC; i += kFusThreads) {
            const int j = i / UPC, ul = i - j * UPC;
            sW1[i] = __bfloat162float(w1[(size_t)j * (e.d + g) + e.d + u0 + ul]);
        }
    }
    __syncthreads();

    const int nblk = g / 32;
    const int blk0 = warp * nblk / kFusWarps, blk1 = (warp + 1) * nblk / kFusWarps;

    for (int t = 0; t < e.B; ++t) {
        if (t > 0) cta_wait_counter(&p.sync[0], (unsigned int)batch * (unsigned int)t);
        const int2 *desc = p.desc + (size_t)(t & 1) * batch;
        for (int c0 = 0; c0 < batch; c0 += kFusChunk) {
            const int nb = min(kFusChunk, batch - c0);
            const int ntiles = (nb + 7) >> 3;
            if (tid < kFusChunk) {
                int2 dsc = (tid < nb) ? __ldcg(desc + c0 + tid) : make_int2(-1, 0);
                sIdx[tid] = dsc.x; sTok[tid] = dsc.y;
            }
            __syncthreads();

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

            // hidden half W_hh S_parent: split-K over the warps, 32 k per block (two k16 MMA steps)
            float acc[MT][4][4];
#pragma unroll
            for (int mt = 0; mt < MT; ++mt)
#pragma unroll
                for (int nt = 0; nt < 4; ++nt)
#pragma unroll
                    for (int q = 0; q < 4; ++q) acc[mt][nt][q] = 0.f;
            size_t boff[4];
#pragma unroll
            for (int nt = 0; nt < 4; ++nt) {
                const int n = nt * 8 + gq;
                const int sidx = sIdx[n];
                boff[nt] = (sidx > 0) ? ((size_t)(c0 + n) * stride + sidx) * g : 0;     // 0 = zero slot of request 0
            }
            for (int blk = blk0; blk < blk1; ++blk) {
                const int k0 = blk * 32 + 8 * c4;
                uint4 bh[4], bl4[4];
#pragma unroll
                for (int nt = 0; nt < 4; ++nt) {
                    if (nt < ntiles) {
                        bh[nt] = __ldcg(reinterpret_cast<const uint4 *>(p.s_hi + boff[nt] + k0));
                        bl4[nt] = __ldcg(reinterpret_cast<const uint4 *>(p.s_lo + boff[nt] + k0));
                    } else { bh[nt] = make_uint4(0, 0, 0, 0); bl4[nt] = make_uint4(0, 0, 0, 0); }
                }
#pragma unroll
                for (int mt = 0; mt < MT; ++mt) {
                    const int r0 = mt * 16 + gq, r1 = r0 + 8;
                    uint4 A0 = make_uint4(0, 0, 0, 0), A1 = make_uint4(0, 0, 0, 0);
                    if (r0 < ROWS) A0 = *reinterpret_cast<const uint4 *>(sW + (size_t)r0 * ldw + k0);
                    if (r1 < ROWS) A1 = *reinterpret_cast<const uint4 *>(sW + (size_t)r1 * ldw + k0);
                    const unsigned int aA[4] = {A0.x, A1.x, A0.y, A1.y};
                    const unsigned int aB[4] = {A0.z, A1.z, A0.w, A1.w};
#pragma unroll
                    for (int nt = 0; nt < 4; ++nt) {
                        if (nt < ntiles) {
                            mma_bf16_16816(acc[mt][nt], aA, bh[nt].x, bh[nt].y);
                            mma_bf16_16816(acc[mt][nt], aB, bh[nt].z, bh[nt].w);
                            mma_bf16_16816(acc[mt][nt], aA, bl4[nt].x, bl4[nt].y);
                            mma_bf16_16816(acc[mt][nt], aB, bl4[nt].z, bl4[nt].w);
                        }
                    }
                }
            }
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
                    const float rg = sigmoidf_acc(pr[i] + hr);
                    const float zg = sigmoidf_acc(pz[i] + hz);
                    const float ng = tanhf(pn[i] + rg * hn);
                    hnew = (1.0f - zg) * ng + zg * hp[i];
                }
                sNew[ul * kNewLd + bl] = hnew;
            }
            __syncthreads();
            // publish S_t (slot t+1): fp32 and the bf16 hi/lo split, UPC consecutive units per request row
            for (int idx = tid; idx < UPC * nb; idx += kFusThreads) {
                const int bl = idx / UPC, ul = idx - bl * UPC;
                if (sIdx[bl] >= 0) {
                    const float h = sNew[ul * kNewLd + bl];
                    const size_t o = ((size_t)(c0 + bl) * stride + (t + 1)) * g + u0 + ul;
                    const __nv_bfloat16 hi = __float2bfloat16_rn(h);
                    __stcg(p.s32 + o, h);
                    p.s_hi[o] = hi;
                    p.s_lo[o] = __float2bfloat16_rn(h - __bfloat162float(hi));
                }
            }
            // this CTA's split-K share of W1[:, d:] S_t
            for (int j = tid; j < r; j += kFusThreads) {
                float w1r[UPC];
#pragma unroll
                for (int ul = 0; ul < UPC; ++ul) w1r[ul] = sW1[j * UPC + ul];
                for (int bl = 0; bl < nb; ++bl) {
                    float s = 0.f;
#pragma unroll
                    for (int ul = 0; ul < UPC; ++ul) s = fmaf(w1r[ul], sNew[ul * kNewLd + bl], s);
                    __stcg(p.partial + ((size_t)cta * batch + c0 + bl) * r + j, s);
                }
            }
            __syncthreads();
        }
        cta_signal_counter(&p.sync[32]);
    }
}

// -------------------------------------------------------------------------------------- request role
__device__ __forceinline__ void cp_async16(void *smem, const void *gmem) {
    unsigned int s = (unsigned int)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gmem));
}

// dot(w[0..n) bf16 in SHARED memory (16 B aligned, n % 8 == 0), s[0..n) fp32 in shared memory).
__device__ __forceinline__ float warp_dot_smem_bf16(const __nv_bfloat16 *w, const float *s, int n, int lane) {
    float acc = 0.f;
    for (int v = lane; v < n / 8; v += 32) {
        const uint4 q = *reinterpret_cast<const uint4 *>(w + (size_t)v * 8);
        const float *sp = s + (size_t)v * 8;
        float f[8];
        unpack8(q, f);
#pragma unroll
        for (int i = 0; i < 8; ++i) acc = fmaf(f[i], sp[i], acc);
    }
    return warp_sum(acc);
}

struct FusedReqSmem {
    float red[8];
    float redk[8];
    unsigned long long redtp[8];
    int redi[8];
    float zmax, lse;
    int n_valid, cnt;
};

__device__ __forceinline__ void fused_req_role(const FusedParams &p, unsigned char *smem_raw) {
    __shared__ FusedReqSmem sm;
    const ExpandParams &e = p.e;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int b = blockIdx.x - p.n_gru;
    const int g = e.g, r = e.r, M = e.M, k = e.k, N = e.N, L = e.L, batch = e.batch;
    (void)g;
    const int ldw2 = r + 8;

    // carve: [W2 rows (bf16, 16 B aligned)] [heap tp u64] [fp32 / int arrays]
    __nv_bfloat16 *sW2 = reinterpret_cast<__nv_bfloat16 *>(smem_raw);
    size_t off = p.w2_smem ? ((size_t)M * ldw2 * 2 + 15) / 16 * 16 : 0;
    unsigned long long *htp = reinterpret_cast<unsigned long long *>(smem_raw + off);
    off += (size_t)e.heap_cap * 8;
    float *hg = reinterpret_cast<float *>(smem_raw + off);
    float *sA = hg + e.heap_cap;
    float *sZ = sA + r;
    float *sBase = sZ + M;
    int *sTok = reinterpret_cast<int *>(sBase + M);
    int *nTok = sTok + M;
    int *nPar = nTok + N;
    int *nDep = nPar + N;
    float *nSco = reinterpret_cast<float *>(nDep + N);

    const __nv_bfloat16 *w2 = reinterpret_cast<const __nv_bfloat16 *>(e.w2);

    // stage the candidate table of depth `dep` (row b*L + dep): ids, base logits, the M rows of W2
    auto stage_depth = [&](int dep) {
        const size_t row = (size_t)b * L + dep;
        for (int m = tid; m < M; m += kFusThreads) {
            sTok[m] = e.cand_id[row * M + m];
            sBase[m] = e.cand_val[row * M + m];
        }
        __syncthreads();
        if (p.w2_smem) {
            const int vpr = r / 8;
            for (int i = tid; i < M * vpr; i += kFusThreads) {
                const int m = i / vpr, v = i - m * vpr;
                cp_async16(sW2 + (size_t)m * ldw2 + v * 8, w2 + (size_t)sTok[m] * r + (size_t)v * 8);
            }
        }
        cp_async_commit();
    };

    if (tid == 0) {
        nTok[0] = e.root_tokens[b]; nPar[0] = -1; nDep[0] = 0; nSco[0] = 0.f;
        sm.n_valid = 1; sm.cnt = 0;
    }
    __syncthreads();
    stage_depth(0);

    for (int t = 0; t < e.B; ++t) {
        const int n_valid = sm.n_valid;
        int cnt = sm.cnt;
        const bool node_ok = (t < n_valid);
        const int depth = node_ok ? nDep[t] : L;
        // Every request CTA waits for the GRU CTAs' step t, expanded or not: nobody runs ahead, so the
        // double-buffered descriptor and the partial buffer are never overwritten while still in use.
        cta_wait_counter(&p.sync[32], (unsigned int)p.n_gru * (unsigned int)(t + 1));
        if (node_ok && depth < L) {                 // block-uniform
            const size_t row = (size_t)b * L + depth;           // H_{depth+1} <-> row index depth (A12)
            // a = SiLU(C + W1[:, d:] S_t): split-K partials summed in CTA order
            for (int j = tid; j < r; j += kFusThreads) {
                const float *pp = p.partial + (size_t)b * r + j;
                const size_t ps = (size_t)batch * r;
                float s0 = 0.f, s1 = 0.f, s2 = 0.f, s3 = 0.f;
                int q = 0;
                for (; q + 4 <= p.n_gru; q += 4) {
                    s0 += __ldcg(pp + (size_t)q * ps);
                    s1 += __ldcg(pp + (size_t)(q + 1) * ps);
                    s2 += __ldcg(pp + (size_t)(q + 2) * ps);
                    s3 += __ldcg(pp + (size_t)(q + 3) * ps);
                }
                for (; q < p.n_gru; ++q) s0 += __ldcg(pp + (size_t)q * ps);
                const float x = e.C[row * r + j] + ((s0 + s1) + (s2 + s3));
                sA[j] = x * sigmoidf_acc(x);
            }
            cp_async_wait<0>();
            __syncthreads();
            // z_m = ((base_m - base_0) + W2[cand_m, :] a) / T_eff     PAPER.md:143-144 (shift-invariant)
            const float base0 = sBase[0];
            for (int m = warp; m < M; m += kFusWarps) {
                float acc = p.w2_smem ? warp_dot_smem_bf16(sW2 + (size_t)m * ldw2, sA, r, lane)
                                      : warp_dot(w2 + (size_t)sTok[m] * r, sA, r, lane);
                if (lane == 0) sZ[m] = __fdiv_rn((sBase[m] - base0) + acc, e.T_eff);
            }
            __syncthreads();
            // slice log-softmax (reading A1): one candidate per thread (M <= 256)
            const float z = (tid < M) ? sZ[tid] : -INFINITY;
            const float wm = warp_max(z);
            if (lane == 0) sm.red[warp] = wm;
            __syncthreads();
            if (tid == 0) { float m = sm.red[0]; for (int i = 1; i < 8; ++i) m = fmaxf(m, sm.red[i]); sm.zmax = m; }
            __syncthreads();
            const float zmax = sm.zmax;
            const float ex = (tid < M) ? expf(z - zmax) : 0.f;
            const float ws = warp_sum(ex);
            if (lane == 0) sm.redk[warp] = ws;
            __syncthreads();
            if (tid == 0) { float s = 0.f; for (int i = 0; i < 8; ++i) s += sm.redk[i]; sm.lse = logf(s); }
            __syncthreads();
            const float lp = (z - zmax) - sm.lse;
            if (tid < M) sZ[tid] = lp;
            __syncthreads();
            // top-k by (logp desc, token asc): rank by counting; push
            if (tid < M) {
                const int mytok = sTok[tid];
                int rank = 0;
                for (int m = 0; m < M; ++m) {
                    const float o = sZ[m];
                    rank += (o > lp) || (o == lp && sTok[m] < mytok);
                }
                if (rank < k) {
                    hg[cnt + rank] = nSco[t] + lp;
                    htp[cnt + rank] = ((unsigned long long)(unsigned int)mytok << 32) | (unsigned int)t;
                }
            }
            cnt += k;
            __syncthreads();
        }

        // pop the maximum under (g desc, token asc, parent asc) into slot t+1
        int next_dep = L;                           // depth of the node popped now (L = none / leaf)
        if (cnt > 0) {
            float bg = -INFINITY; unsigned long long btp = ~0ull; int bi = -1;
            for (int i = tid; i < cnt; i += kFusThreads) {
                const float gi = hg[i]; const unsigned long long tp = htp[i];
                if (bi < 0 || gi > bg || (gi == bg && tp < btp)) { bg = gi; btp = tp; bi = i; }
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                const float og = __shfl_xor_sync(0xffffffffu, bg, o);
                const unsigned long long otp = __shfl_xor_sync(0xffffffffu, btp, o);
                const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
                if (oi >= 0 && (bi < 0 || og > bg || (og == bg && otp < btp))) { bg = og; btp = otp; bi = oi; }
            }
            if (lane == 0) { sm.redk[warp] = bg; sm.redtp[warp] = btp; sm.redi[warp] = bi; }
            __syncthreads();
            if (tid == 0) {
                for (int w = 0; w < kFusWarps; ++w) {
                    const float og = sm.redk[w]; const unsigned long long otp = sm.redtp[w]; const int oi = sm.redi[w];
                    if (oi >= 0 && (bi < 0 || og > bg || (og == bg && otp < btp))) { bg = og; btp = otp; bi = oi; }
                }
                const int par = (int)(btp & 0xFFFFFFFFull), tok = (int)(btp >> 32);
                const int dep = nDep[par] + 1;
                nTok[t + 1] = tok; nPar[t + 1] = par; nDep[t + 1] = dep; nSco[t + 1] = bg;
                hg[bi] = hg[cnt - 1];
                htp[bi] = htp[cnt - 1];
                sm.n_valid = t + 2; sm.cnt = cnt - 1;
                if (t + 1 < e.B)
                    p.desc[(size_t)((t + 1) & 1) * batch + b] = make_int2(dep < L ? par + 1 : -1, tok);
            }
            __syncthreads();
            next_dep = nDep[t + 1];
        } else {
            if (tid == 0) {
                sm.cnt = 0;
                if (t + 1 < e.B) p.desc[(size_t)((t + 1) & 1) * batch + b] = make_int2(-1, 0);
            }
        }
        if (t + 1 < e.B) {
            cta_signal_counter(&p.sync[0]);
            if (next_dep < L) stage_depth(next_dep);   // overlaps the GRU CTAs' step t+1
            else __syncthreads();
        }
    }
    __syncthreads();

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
}

template <int UPC>
__global__ void __launch_bounds__(kFusThreads, 1) fused_expand_kernel(FusedParams p) {
    extern __shared__ __align__(16) unsigned char fused_smem[];
    if ((int)blockIdx.x < p.n_gru) fused_gru_role<UPC>(p, fused_smem);
    else fused_req_role(p, fused_smem);
}

}  // namespace dt
