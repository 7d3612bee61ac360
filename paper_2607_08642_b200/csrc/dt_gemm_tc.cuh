// dt_gemm_tc.cuh -- the per-round precompute C = H W1[:, 0:d]^T (Fact B PAPER.md:83-89) on the
// 5th-generation tensor cores: out[m, n] = sum_k A[m, k] Bm[n, k], bf16 x bf16 -> fp32, both operands K-major.
//
// One CTA owns a 128-row tile of A and one of kTcgSplits K-slices (the split depends on K only, never on the batch,
// so every output is summed in the same order whatever the batch size).  Per 64-wide K block all threads copy the A
// tile (128 x 128 B) and the whole B slice (N x 128 B) into a 4-deep cp.async ring in the 128-byte-swizzled layout
// (dt_tcgen05.cuh); one thread issues four tcgen05.mma (M = 128, N <= 256, K = 16) per block into one TMEM
// accumulator; the epilogue moves it to a [split, row, col] fp32 partial and a second tiny kernel adds the splits
// in split order.  Legacy mma.sync (dt_gemm_mma.cuh) runs this 512 x 256 x 4096 problem in 30 us on B200
// (~256 MAC/clk/SM); this kernel is measured in profiles/.
#pragma once
#include "dt_gemm_mma.cuh"
#include "dt_tcgen05.cuh"

namespace dt {

constexpr int kTcgSplits = 8;
constexpr int kTcgStages = 4;
constexpr int kTcgThreads = 256;
constexpr int kTcgStageBytes = 128 * 128 + 256 * 128;       // A tile + B slice of one 64-wide K block

struct GemmTcParams {
    const __nv_bfloat16 *A; long long lda;      // [Mr, K]
    const __nv_bfloat16 *Bm; long long ldb;     // [Nc, K]
    float *partial;                             // [kTcgSplits, Mr_pad, Nc]  (Mr_pad = row tiles * 128)
    float *out; long long ldo;                  // [Mr, Nc]
    int Mr, Nc, K, Mr_pad;
};

__host__ __device__ inline size_t gemm_tc_smem() { return (size_t)kTcgStages * kTcgStageBytes + 64 + 1024; }

__global__ void __launch_bounds__(kTcgThreads, 1) gemm_c_tc_kernel(GemmTcParams p) {
    extern __shared__ __align__(1024) unsigned char gsm[];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int m0 = blockIdx.x * 128, ks = blockIdx.y;
    const int Kc = p.K / kTcgSplits, kb0 = ks * Kc, n_blk = Kc / 64;
    unsigned char *ring = gsm;
    unsigned long long *mbar = reinterpret_cast<unsigned long long *>(gsm + (size_t)kTcgStages * kTcgStageBytes);  // [0..3] free, [4] done
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(mbar + 6);

    if (tid == 0) {
        for (int i = 0; i < 5; ++i) tc::mbar_init(tc::smem_u32(mbar + i), 1);
        tc::mbar_init_fence();
    }
    if (warp == 0) tc::tmem_alloc<256>(tmem_slot);
    tc::fence_before_sync();
    __syncthreads();
    tc::fence_after_sync();
    const uint32_t tmem = *tmem_slot;
    const uint32_t idesc = tc::make_idesc_bf16(128, p.Nc);
    const uint32_t ring_a = tc::smem_u32(ring), mb0 = tc::smem_u32(mbar);

    // this thread's 16-byte pieces of a stage: piece c of rows r0 + 32 i
    const int c = tid & 7, r0 = tid >> 3;
    auto issue = [&](int blk) {
        unsigned char *st = ring + (size_t)(blk % kTcgStages) * kTcgStageBytes;
        const long long k = kb0 + (long long)blk * 64 + c * 8;
#pragma unroll
        for (int i = 0; i < 4; ++i) {                       // A tile: 128 rows
            const int r = r0 + 32 * i;
            const bool v = (m0 + r) < p.Mr;
            cp_async16_zfill(st + (r >> 3) * 1024 + (r & 7) * 128 + ((c ^ (r & 7)) << 4), p.A + (v ? (long long)(m0 + r) * p.lda + k : 0), v);
        }
        unsigned char *sb = st + 128 * 128;
        for (int r = r0; r < p.Nc; r += 32)                 // B slice: Nc rows
            cp_async16(sb + (r >> 3) * 1024 + (r & 7) * 128 + ((c ^ (r & 7)) << 4), p.Bm + (long long)r * p.ldb + k);
    };
    for (int i = 0; i < kTcgStages; ++i) { if (i < n_blk) issue(i); cp_async_commit(); }

    uint32_t ph_free = 0;
    for (int blk = 0; blk < n_blk; ++blk) {
        cp_async_wait<kTcgStages - 1>();
        tc::fence_proxy_async();
        __syncthreads();
        const int stg = blk % kTcgStages;
        if (tid == 0) {
            tc::fence_after_sync();
            const uint64_t da = tc::make_desc_sw128(ring_a + (uint32_t)stg * kTcgStageBytes, 1024);
            const uint64_t db = tc::make_desc_sw128(ring_a + (uint32_t)stg * kTcgStageBytes + 128 * 128, 1024);
#pragma unroll
            for (int s4 = 0; s4 < 4; ++s4) tc::mma_bf16(tmem, da + (uint64_t)(s4 * 2), db + (uint64_t)(s4 * 2), idesc, (blk | s4) ? 1u : 0u);
            if (blk + kTcgStages < n_blk) tc::commit(mb0 + 8 * stg);
            if (blk == n_blk - 1) tc::commit(mb0 + 32);
        }
        if (blk + kTcgStages < n_blk) {                     // refill the stage once its MMAs have read it
            tc::mbar_wait(mb0 + 8 * stg, (ph_free >> stg) & 1u);
            ph_free ^= 1u << stg;
            issue(blk + kTcgStages);
        }
        cp_async_commit();
    }
    cp_async_wait<0>();
    tc::mbar_wait(mb0 + 32, 0);
    tc::fence_after_sync();
    __syncwarp();
    // epilogue: row m0 + 32 (warp % 4) + lane, columns [128 (warp / 4), +128)
    {
        const int row = m0 + 32 * (warp & 3) + lane;
        float *dst = p.partial + ((size_t)ks * p.Mr_pad + row) * p.Nc;
#pragma unroll 1
        for (int q = 0; q < 4; ++q) {
            const int col0 = 128 * (warp >> 2) + 32 * q;
            if (col0 < p.Nc) {                               // warp-uniform
                float v[32];
                tc::tmem_ld32(tmem + ((uint32_t)(32 * (warp & 3)) << 16) + col0, v);
#pragma unroll
                for (int j = 0; j < 32; j += 4)
                    if (col0 + j < p.Nc) __stcg(reinterpret_cast<float4 *>(dst + col0 + j), make_float4(v[j], v[j + 1], v[j + 2], v[j + 3]));
            }
        }
    }
    tc::fence_before_sync();
    __syncthreads();
    if (warp == 0) tc::tmem_free<256>(tmem);
}

// out[m, n] = sum over the splits, in split order.  One float4 per thread.
__global__ void gemm_c_reduce_kernel(GemmTcParams p) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int n4 = p.Nc / 4;
    if (i >= (long long)p.Mr * n4) return;
    const int m = (int)(i / n4), n = (int)(i % n4) * 4;
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
    for (int s = 0; s < kTcgSplits; ++s) {
        const float4 v = __ldcg(reinterpret_cast<const float4 *>(p.partial + ((size_t)s * p.Mr_pad + m) * p.Nc + n));
        acc.x += v.x; acc.y += v.y; acc.z += v.z; acc.w += v.w;
    }
    float *o = p.out + (long long)m * p.ldo + n;
    o[0] = acc.x; o[1] = acc.y; o[2] = acc.z; o[3] = acc.w;
}

}  // namespace dt
