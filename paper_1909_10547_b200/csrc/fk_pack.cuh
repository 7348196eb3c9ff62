// fk_pack.cuh -- one-time, untimed table pack: logical channel-innermost fp64 table
// -> device layout: channel-major, x innermost, rows padded with zeros to a 16-byte multiple,
// optionally demoted to fp32 with round-to-nearest (reading R18).  Tables are loaded once and kept
// resident for the whole fit, so this runs off the timed path.
#pragma once

#include "fk_common.cuh"

namespace fk {

// out[n][kp] = (T) in[n][klog(kp)],  kp in packed order (hadronic: channel blocks of cstride elements,
// x-rows jp apart, the tail of each x-row and of each block zero); pad columns [K, row_stride) = 0
template <typename T>
__global__ void __launch_bounds__(256)
fk_pack_kernel(const double* __restrict__ in, T* __restrict__ out, int N, int nx, int C, int kind,
               int K, int cstride, int jp, long long row_stride) {
    const long long total = (long long)N * row_stride;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total;
         t += (long long)gridDim.x * blockDim.x) {
        const long long n = t / row_stride;
        const int kp = (int)(t - n * row_stride);
        T v = T(0);
        if (kp < K) {
            int klog = -1;
            long long klen;  // logical row length
            if (kind == KIND_HADRONIC) {
                const int c = kp / cstride, rem = kp - c * cstride;
                const int i = rem / jp, j = rem - i * jp;
                if (i < nx && j < nx) klog = (i * nx + j) * C + c;
                klen = (long long)C * nx * nx;
            } else {
                const int c = kp / nx, i = kp - c * nx;
                klog = i * C + c;
                klen = (long long)C * nx;
            }
            if (klog >= 0) v = (T)in[n * klen + klog];  // fp64 -> fp32: cvt.rn
        }
        out[t] = v;
    }
}

// Two-PDF (p pbar) form of Eq. (1) (PAPER.md:43 with distinct f, fbar): the second hadron's PDFs become
// nfl extra flavours of ONE stacked grid F[r][2 nfl][nx] = (f1[r] ; f2[r]), and the pair (a, b) becomes (a, nfl + b):
// the single-PDF kernels then compute sum f1[a][i] f2[b][j] FK, and their VJP returns dF = (df1 ; df2).
template <typename T>
__global__ void __launch_bounds__(256) fk_stack2_kernel(const T* __restrict__ f1, const T* __restrict__ f2, T* __restrict__ F,
                                                         int R, int slots) {
    const long long total = 2LL * R * slots;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const long long r = t / (2 * slots);
        const int s = (int)(t - r * 2 * slots);
        F[t] = s < slots ? f1[r * slots + s] : f2[r * slots + s - slots];
    }
}
template <typename T>
__global__ void __launch_bounds__(256) fk_unstack2_kernel(const T* __restrict__ dF, T* __restrict__ df1, T* __restrict__ df2,
                                                           int R, int slots) {
    const long long total = 2LL * R * slots;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const long long r = t / (2 * slots);
        const int s = (int)(t - r * 2 * slots);
        if (s < slots) df1[r * slots + s] = dF[t];
        else df2[r * slots + s - slots] = dF[t];
    }
}

}  // namespace fk
