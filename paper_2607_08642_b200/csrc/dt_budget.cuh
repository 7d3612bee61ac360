// dt_budget.cuh -- cost-aware adaptive budget: CaDDTree's stopping rule applied to the
// conditional heap's pop order: theta(n) = (1 + Phi(n)) / (C_d + C_v(n)),
// Phi(n) = sum_{s <= n} exp(score of the s-th popped node); keep growing while theta improves.  The trees are
// already built to the cap B, so the rule is a scan over at most 255 scores per request: one thread per request,
// sequential, in double precision (the decision is a comparison of two nearly equal ratios).
#pragma once
#include "dt_common.cuh"

namespace dt {

__global__ void adaptive_budget_kernel(const float *__restrict__ scores, const int32_t *__restrict__ n_nodes, int N, int batch,
                                       double C_d, const float *__restrict__ cv, int32_t *__restrict__ n_star,
                                       float *__restrict__ phi_out) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= batch) return;
    const float *s = scores + (size_t)b * N;
    const int nn = min(n_nodes[b], N);
    int n = 0;
    double phi = 0.0;
    double theta = (1.0 + phi) / (C_d + (double)cv[0]);
    while (n + 1 < nn) {
        const double phi_next = phi + exp((double)s[n + 1]);
        const double theta_next = (1.0 + phi_next) / (C_d + (double)cv[n + 1]);
        if (theta_next <= theta) break;
        ++n; phi = phi_next; theta = theta_next;
    }
    n_star[b] = n;
    if (phi_out) phi_out[b] = (float)phi;
}

}  // namespace dt
