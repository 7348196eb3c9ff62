// fk_chi2.cuh -- the step after the convolution in a fit iteration (reading R22):
//     d[n][r] = sigma[n][r] - data[n]
//     g[n][r] = 2 sum_m Cinv[n][m] d[m][r]          (the upstream gradient the VJP then takes; Cinv symmetric)
//     chi2[r] = sum_n d[n][r] * (g[n][r] / 2)
// fk_chi2_grad_kernel: CTA = one row n of Cinv (read once, coalesced), block (32, 8): lanes stride over m with 4
// interleaved chains, warps stride over r; fixed xor butterfly.  fk_chi2_sum_kernel: one warp per replica.
// No atomics: bitwise repeatable.
#pragma once

#include "fk_common.cuh"

namespace fk {

__global__ void __launch_bounds__(256) fk_chi2_grad_kernel(const double* __restrict__ sigma, const double* __restrict__ data,
                                                            const double* __restrict__ cinv, double* __restrict__ g, int N, int R) {
    const int n = blockIdx.x, lane = threadIdx.x, w = threadIdx.y;
    const double* __restrict__ row = cinv + (long long)n * N;
    for (int r = w; r < R; r += blockDim.y) {
        double acc[4] = {0.0, 0.0, 0.0, 0.0};
        int q = 0;
        for (int m = lane; m < N; m += 32, ++q) acc[q & 3] = fma(row[m], sigma[(long long)m * R + r] - data[m], acc[q & 3]);
        const double s = warp_sum((acc[0] + acc[1]) + (acc[2] + acc[3]));
        if (lane == 0) g[(long long)n * R + r] = 2.0 * s;
    }
}

__global__ void __launch_bounds__(256) fk_chi2_sum_kernel(const double* __restrict__ sigma, const double* __restrict__ data,
                                                           const double* __restrict__ g, double* __restrict__ chi2, int N, int R) {
    const int lane = threadIdx.x & 31;
    const int r = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    if (r >= R) return;
    double acc[4] = {0.0, 0.0, 0.0, 0.0};
    int q = 0;
    for (int n = lane; n < N; n += 32, ++q)
        acc[q & 3] = fma(sigma[(long long)n * R + r] - data[n], 0.5 * g[(long long)n * R + r], acc[q & 3]);
    const double s = warp_sum((acc[0] + acc[1]) + (acc[2] + acc[3]));
    if (lane == 0) chi2[r] = s;
}

}  // namespace fk
