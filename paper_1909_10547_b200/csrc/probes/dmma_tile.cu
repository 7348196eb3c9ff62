// dmma_tile.cu -- design probe, not part of libfkconv.so: ceiling of the DMMA consumer loop of the R >> 1 kernels
// (fragments loaded from a static shared-memory tile, 1 CTA per SM, no global traffic) for several warp tilings,
// with and without a CTA barrier per K-tile, with double-buffered fragments, and with the B fragment formed as
// shared * register (the forward kernel's luminosity-on-the-fly).
// Build + run:  python -m paper_1909_10547_b200.build --probes && paper_1909_10547_b200/probes/dmma_tile
// Results: profiles/r01_dense_kernels.md
#include <cstdio>
#include <cuda_runtime.h>
__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}
constexpr int SA = 36, SB = 132, KT = 32, STAGES = 3;
// MODE 0: plain; 1: __syncthreads per K-tile; 2: fragments double-buffered; 3: B fragment = smem * reg (DMUL)
template <int WARPS, int MI, int NJ, int MODE>
__global__ void __launch_bounds__(WARPS * 32, 1) tile_kernel(double* out, int ktiles) {
    extern __shared__ double sm[];
    double* As = sm;                         // [STAGES][128][SA]
    double* Bs = sm + STAGES * 128 * SA;     // [STAGES][KT][SB]
    for (int i = threadIdx.x; i < STAGES * 128 * SA + STAGES * KT * SB; i += blockDim.x) sm[i] = 1e-3 * (i % 7);
    __syncthreads();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int wm = warp % (16 / MI), wn = warp / (16 / MI);
    double acc[MI][NJ][2];
#pragma unroll
    for (int i = 0; i < MI; ++i)
#pragma unroll
        for (int j = 0; j < NJ; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
    double fa[NJ];
#pragma unroll
    for (int j = 0; j < NJ; ++j) fa[j] = 1.0 + 1e-9 * j;
    for (int t = 0; t < ktiles; ++t) {
        const int st = t % STAGES;
        const double* At = As + (st * 128 + wm * MI * 8 + (lane >> 2)) * SA + (lane & 3);
        const double* Bt = Bs + (st * KT + (lane & 3)) * SB + (wn * NJ * 8) % 128 + (lane >> 2);
        if (MODE == 2) {
            double a[2][MI], b[2][NJ];
#pragma unroll
            for (int i = 0; i < MI; ++i) a[0][i] = At[i * 8 * SA];
#pragma unroll
            for (int j = 0; j < NJ; ++j) b[0][j] = Bt[j * 8];
#pragma unroll
            for (int s = 0; s < KT / 4; ++s) {
                if (s + 1 < KT / 4) {
#pragma unroll
                    for (int i = 0; i < MI; ++i) a[(s + 1) & 1][i] = At[i * 8 * SA + (s + 1) * 4];
#pragma unroll
                    for (int j = 0; j < NJ; ++j) b[(s + 1) & 1][j] = Bt[(s + 1) * 4 * SB + j * 8];
                }
#pragma unroll
                for (int j = 0; j < NJ; ++j)
#pragma unroll
                    for (int i = 0; i < MI; ++i) dmma884(acc[i][j][0], acc[i][j][1], a[s & 1][i], b[s & 1][j]);
            }
        } else {
#pragma unroll
            for (int s = 0; s < KT / 4; ++s) {
                double a[MI], b[NJ];
#pragma unroll
                for (int i = 0; i < MI; ++i) a[i] = At[i * 8 * SA + s * 4];
#pragma unroll
                for (int j = 0; j < NJ; ++j) b[j] = MODE == 3 ? Bt[s * 4 * SB + j * 8] * fa[j] : Bt[s * 4 * SB + j * 8];
#pragma unroll
                for (int j = 0; j < NJ; ++j)
#pragma unroll
                    for (int i = 0; i < MI; ++i) dmma884(acc[i][j][0], acc[i][j][1], a[i], b[j]);
            }
        }
        if (MODE == 1) __syncthreads();
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < MI; ++i)
#pragma unroll
        for (int j = 0; j < NJ; ++j) s += acc[i][j][0] + acc[i][j][1];
    if (s == 12345.678) out[threadIdx.x] = s;
}
template <int WARPS, int MI, int NJ, int MODE>
void run(const char* name, double* out) {
    const int ktiles = 4096;
    const size_t smem = (STAGES * 128 * SA + STAGES * KT * SB) * 8;  // force 1 CTA/SM
    cudaFuncSetAttribute(tile_kernel<WARPS, MI, NJ, MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    tile_kernel<WARPS, MI, NJ, MODE><<<148, WARPS * 32, smem>>>(out, ktiles);
    cudaDeviceSynchronize();
    cudaEventRecord(e0);
    for (int r = 0; r < 3; ++r) tile_kernel<WARPS, MI, NJ, MODE><<<148, WARPS * 32, smem>>>(out, ktiles);
    cudaEventRecord(e1); cudaEventSynchronize(e1);
    float ms; cudaEventElapsedTime(&ms, e0, e1); ms /= 3;
    double fl = 148.0 * WARPS * MI * NJ * 512.0 * (KT / 4) * ktiles;
    printf("%-44s %.3f ms  %.2f TFLOP/s (%s)\n", name, ms, fl / ms / 1e9, cudaGetErrorString(cudaGetLastError()));
}
int main() {
    double* out; cudaMalloc(&out, 4096 * 8);
    run<8, 4, 8, 0>("W8 32x64 plain", out);
    run<8, 4, 8, 1>("W8 32x64 syncthreads/Ktile", out);
    run<8, 4, 8, 2>("W8 32x64 double-buffered frags", out);
    run<8, 4, 8, 3>("W8 32x64 B=smem*reg", out);
    run<16, 4, 4, 0>("W16 32x32 plain", out);
    run<16, 4, 4, 1>("W16 32x32 syncthreads/Ktile", out);
    run<16, 4, 4, 2>("W16 32x32 double-buffered frags", out);
    run<16, 4, 4, 3>("W16 32x32 B=smem*reg", out);
    run<8, 8, 4, 0>("W8 64x32 plain", out);
    run<8, 8, 4, 2>("W8 64x32 double-buffered", out);
    run<16, 2, 8, 0>("W16 16x64 plain", out);
    run<16, 2, 8, 2>("W16 16x64 double-buffered", out);
    run<4, 4, 8, 0>("W4 32x64 plain (1 warp/sched)", out);
    run<4, 4, 8, 2>("W4 32x64 double-buffered (1 warp/sched)", out);
    return 0;
}
