// dt_precompute.cuh -- path-independent contractions:
//   * P = E W_ih^T  [V, 3g]  (once per handle): the input half W_ih E[v] of every GRU step
//      becomes a row gather of P.
//   * C[b,i,:] = W1[:, 0:d] H[b,i,:]  [batch*L, r]  (once per round): by Fact B
//     H_i is path independent, so this half of W1 [H_i; S] is shared by all nodes.
//   * S_0 = GRUcell(0, E[root]) (reading A4): with h = 0 the hidden half
//     vanishes, so S_0 = (1 - sigmoid(P_z)) * tanh(P_n) elementwise from row P[root].
#pragma once
#include "dt_common.cuh"

namespace dt {

// out[m, n] = sum_k A[m, k] * Bm[n, k]   (A: [Mr, K] lda, Bm: [Nc, K] ldb, out fp32 [Mr, Nc] ldo)
// 64x64 output tile per CTA, 256 threads, 4x4 micro-tile, K-tile 16, fp32 accumulate.
constexpr int kGemmBM = 64, kGemmBN = 64, kGemmBK = 16;

template <typename T>
__global__ void __launch_bounds__(256) gemm_nt_kernel(const T *__restrict__ A, long long lda,
                                                      const T *__restrict__ Bm, long long ldb,
                                                      float *__restrict__ out, long long ldo,
                                                      int Mr, int Nc, int K) {
    __shared__ float As[kGemmBK][kGemmBM + 4];
    __shared__ float Bs[kGemmBK][kGemmBN + 4];
    const int tid = threadIdx.x;
    const int tx = tid & 15, ty = tid >> 4;
    const long long m0 = (long long)blockIdx.y * kGemmBM, n0 = (long long)blockIdx.x * kGemmBN;
    float acc[4][4];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = 0.f;

    // loader mapping: 64 rows x 16 k = 1024 elements, 4 per thread: row = tid/4, k = (tid%4)*4 .. +3
    const int lr = tid >> 2, lk = (tid & 3) * 4;
    for (int k0 = 0; k0 < K; k0 += kGemmBK) {
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            int kk = k0 + lk + q;
            long long am = m0 + lr, bn = n0 + lr;
            As[lk + q][lr] = (am < Mr && kk < K) ? ldf(A, (size_t)(am * lda + kk)) : 0.f;
            Bs[lk + q][lr] = (bn < Nc && kk < K) ? ldf(Bm, (size_t)(bn * ldb + kk)) : 0.f;
        }
        __syncthreads();
#pragma unroll
        for (int kk = 0; kk < kGemmBK; ++kk) {
            float a[4], b[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) a[i] = As[kk][ty * 4 + i];
#pragma unroll
            for (int j = 0; j < 4; ++j) b[j] = Bs[kk][tx * 4 + j];
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(a[i], b[j], acc[i][j]);
        }
        __syncthreads();
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        long long m = m0 + ty * 4 + i;
        if (m >= Mr) continue;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            long long n = n0 + tx * 4 + j;
            if (n < Nc) out[m * ldo + n] = acc[i][j];
        }
    }
}

// S_0[b, j] = (1 - sigmoid(P[root_b, g + j])) * tanh(P[root_b, 2g + j]);  also writes slot 0 of the
// per-request tree arrays.  grid = batch, any block size.
__global__ void root_state_kernel(const float *__restrict__ P, const int32_t *__restrict__ root_tokens,
                                  int g, int V, float *__restrict__ states, long long state_stride_b) {
    const int b = blockIdx.x;
    int tok = root_tokens[b];
    tok = min(max(tok, 0), V - 1);
    const float *pr = P + (size_t)tok * 3 * g;
    float *S0 = states + (size_t)b * state_stride_b;
    for (int j = threadIdx.x; j < g; j += blockDim.x) {
        float zg = sigmoidf_acc(pr[g + j]);
        float ng = tanhf(pr[2 * g + j]);
        S0[j] = (1.0f - zg) * ng;
    }
}

}  // namespace dt
