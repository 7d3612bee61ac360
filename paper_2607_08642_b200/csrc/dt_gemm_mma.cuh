// dt_gemm_mma.cuh -- bf16 x bf16 -> fp32 "NT" contraction on the tensor cores for the two
// path-independent GEMMs of the builder:
//   * P = E W_ih^T            [V, 3g]        once per handle
//   * C = H W1[:, 0:d]^T      [batch*L, r]   once per round   (Fact B PAPER.md:83-89)
// out[m, n] = sum_k A[m, k] * Bm[n, k], both operands K-contiguous.  Products of bf16 values are
// exact in fp32 and the accumulation is fp32, so the result differs from the float64 oracle only
// by fp32 summation rounding.
//
// Why warp-level mma.sync and not tcgen05 here: the per-round GEMM is 512 x 256 x 4096 (1 GFLOP,
// batch 32) or 16 x 256 x 4096 (batch 1) -- a few microseconds of tensor time on a latency chain;
// it is split-K'd over the whole chip for latency, every CTA owning a 64x64x(K/S) slab whose
// accumulators fit registers.  The UMMA/TMEM path pays for itself on tiles >= 128 x 128 x long-K,
// which this problem does not have on the per-round path.  (DESIGN.md "Kernels".)
//
// Tiling: CTA 64x64x32, 4 warps (2x2, warp tile 32x32 = 2 m16 x 4 n8 mma tiles), 3-stage cp.async
// pipeline, ldmatrix from padded (conflict-free) shared tiles.  Split-K: blockIdx.z owns a K range;
// partials go to a workspace and the LAST CTA of a tile (arrival ticket) sums them in split order,
// so the result does not depend on arrival order (deterministic, batch-invariant).
#pragma once
#include "dt_common.cuh"

namespace dt {

constexpr int kMmaBM = 64, kMmaBN = 64, kMmaBK = 32, kMmaStages = 4, kMmaThreads = 128;
constexpr int kMmaLd = kMmaBK + 8;      // padded row (80 B): ldmatrix rows land in distinct banks

struct GemmMmaParams {
    const __nv_bfloat16 *A; long long lda;      // [M, K]
    const __nv_bfloat16 *Bm; long long ldb;     // [N, K]
    float *out; long long ldo;                  // [M, N]
    int M, N, K;
    int splits;                                 // gridDim.z
    int k_per_split;                            // multiple of kMmaBK
    float *partial;                             // [splits, M, N] (splits > 1)
    unsigned int *tile_counter;                 // [tiles] self-resetting tickets (splits > 1)
};

__device__ __forceinline__ void cp_async16_zfill(void *smem, const void *gmem, bool valid) {
    unsigned int s = (unsigned int)__cvta_generic_to_shared(smem);
    int sz = valid ? 16 : 0;
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(s), "l"(gmem), "r"(sz));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N)); }

__device__ __forceinline__ void ldmatrix_x4(unsigned int (&r)[4], const void *smem) {
    unsigned int s = (unsigned int)__cvta_generic_to_shared(smem);
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0, %1, %2, %3}, [%4];\n"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(s));
}
__device__ __forceinline__ void mma_bf16_16816(float (&d)[4], const unsigned int (&a)[4], unsigned int b0, unsigned int b1) {
    asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0, %1, %2, %3}, {%4, %5, %6, %7}, {%8, %9}, {%0, %1, %2, %3};\n"
                 : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}

__global__ void __launch_bounds__(kMmaThreads) gemm_nt_bf16_mma_kernel(GemmMmaParams p) {
    __shared__ __align__(16) __nv_bfloat16 sA[kMmaStages][kMmaBM][kMmaLd];
    __shared__ __align__(16) __nv_bfloat16 sB[kMmaStages][kMmaBN][kMmaLd];
    __shared__ unsigned int s_last;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int wm = warp >> 1, wn = warp & 1;
    const long long m0 = (long long)blockIdx.y * kMmaBM, n0 = (long long)blockIdx.x * kMmaBN;
    const int kb = blockIdx.z * p.k_per_split;
    const int ke = min(p.K, kb + p.k_per_split);
    const int n_kt = (ke > kb) ? (ke - kb + kMmaBK - 1) / kMmaBK : 0;

    // loader: a 64 x 32 tile = 256 chunks of 16 B, two per thread (rows r and r + 32)
    const int lrow = tid >> 2, lk = (tid & 3) * 8;
    auto load_stage = [&](int stage, int kt) {
        const int k = kb + kt * kMmaBK + lk;
        const bool kin = (k < ke);                       // K % 8 == 0 is required by the launcher
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int r = lrow + 32 * h;
            const long long am = m0 + r, bn = n0 + r;
            const bool va = kin && am < p.M, vb = kin && bn < p.N;
            cp_async16_zfill(&sA[stage][r][lk], p.A + (va ? am * p.lda + k : 0), va);
            cp_async16_zfill(&sB[stage][r][lk], p.Bm + (vb ? bn * p.ldb + k : 0), vb);
        }
    };

    float acc[2][4][4];
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j)
#pragma unroll
            for (int q = 0; q < 4; ++q) acc[i][j][q] = 0.f;

#pragma unroll
    for (int s = 0; s < kMmaStages - 1; ++s) {
        if (s < n_kt) load_stage(s, s);
        cp_async_commit();
    }
    for (int kt = 0; kt < n_kt; ++kt) {
        cp_async_wait<kMmaStages - 2>();
        __syncthreads();
        const int nxt = kt + kMmaStages - 1;
        if (nxt < n_kt) load_stage(nxt % kMmaStages, nxt);
        cp_async_commit();
        const int st = kt % kMmaStages;
#pragma unroll
        for (int ks = 0; ks < kMmaBK; ks += 16) {
            unsigned int a[2][4], b[2][4];
#pragma unroll
            for (int i = 0; i < 2; ++i) {
                const int row = wm * 32 + i * 16 + (lane & 7) + 8 * ((lane >> 3) & 1);
                ldmatrix_x4(a[i], &sA[st][row][ks + 8 * (lane >> 4)]);
            }
#pragma unroll
            for (int j = 0; j < 2; ++j) {                // each x4 covers two n8 tiles
                const int nrow = wn * 32 + j * 16 + (lane & 7) + 8 * (lane >> 4);
                ldmatrix_x4(b[j], &sB[st][nrow][ks + 8 * ((lane >> 3) & 1)]);
            }
#pragma unroll
            for (int i = 0; i < 2; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) mma_bf16_16816(acc[i][j], a[i], b[j >> 1][2 * (j & 1)], b[j >> 1][2 * (j & 1) + 1]);
        }
    }
    cp_async_wait<0>();

    // epilogue: accumulator (i, j, q) -> row m0 + wm*32 + i*16 + lane/4 + 8*(q/2), col n0 + wn*32 + j*8 + 2*(lane%4) + (q&1)
    const bool split = p.splits > 1;
    float *dst = split ? p.partial + (size_t)blockIdx.z * p.M * p.N : p.out;
    const long long ldd = split ? p.N : p.ldo;
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j)
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const long long m = m0 + wm * 32 + i * 16 + (lane >> 2) + 8 * (q >> 1);
                const long long n = n0 + wn * 32 + j * 8 + 2 * (lane & 3) + (q & 1);
                if (m < p.M && n < p.N) {
                    if (split) __stcg(dst + m * ldd + n, acc[i][j][q]);
                    else dst[m * ldd + n] = acc[i][j][q];
                }
            }
    if (!split) return;
    // the last CTA of this output tile sums the partials in split order (fixed => deterministic)
    __threadfence();
    __syncthreads();
    const unsigned int tile = blockIdx.y * gridDim.x + blockIdx.x;
    if (tid == 0) {
        unsigned int ticket = atomicAdd(&p.tile_counter[tile], 1u);
        s_last = (ticket == (unsigned int)(p.splits - 1));
        if (s_last) p.tile_counter[tile] = 0u;
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    for (int e = tid; e < kMmaBM * kMmaBN; e += kMmaThreads) {
        const long long m = m0 + e / kMmaBN, n = n0 + e % kMmaBN;
        if (m < p.M && n < p.N) {
            float s = 0.f;
            for (int z = 0; z < p.splits; ++z) s += __ldcg(p.partial + ((size_t)z * p.M + m) * p.N + n);
            p.out[m * p.ldo + n] = s;
        }
    }
}

}  // namespace dt
