// fp64_peak.cu -- design probe, not part of libfkconv.so: FP64 throughput of DFMA chains and of the
// mma.sync f64 shapes (DMMA) on sm_100a, the roofline denominator of the R >> 1 contraction.
// Build + run:  python -m paper_1909_10547_b200.build --probes && paper_1909_10547_b200/probes/fp64_peak
// Results: profiles/r01_fp64_peak.md
#include <cstdio>
#include <cuda_runtime.h>

#define ITERS 2048

template <int ILP>
__global__ void dfma_kernel(double* out, double x, double y) {
    double a[ILP];
#pragma unroll
    for (int i = 0; i < ILP; ++i) a[i] = threadIdx.x + i;
    for (int it = 0; it < ITERS; ++it) {
#pragma unroll
        for (int i = 0; i < ILP; ++i) a[i] = fma(a[i], x, y);
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < ILP; ++i) s += a[i];
    if (s == 12345.678) out[threadIdx.x] = s;
}

template <int ILP>
__global__ void dmma884_kernel(double* out, double x, double y) {
    double c[ILP][2];
#pragma unroll
    for (int i = 0; i < ILP; ++i) { c[i][0] = threadIdx.x + i; c[i][1] = i; }
    double a = x, b = y;
    for (int it = 0; it < ITERS; ++it) {
#pragma unroll
        for (int i = 0; i < ILP; ++i)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                         : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(a), "d"(b));
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < ILP; ++i) s += c[i][0] + c[i][1];
    if (s == 12345.678) out[threadIdx.x] = s;
}

template <int ILP>
__global__ void dmma1688_kernel(double* out, double x, double y) {
    double c[ILP][4];
#pragma unroll
    for (int i = 0; i < ILP; ++i) { c[i][0] = threadIdx.x + i; c[i][1] = i; c[i][2] = 1; c[i][3] = 2; }
    double a0 = x, a1 = x + 1, a2 = x + 2, a3 = x + 3, b0 = y, b1 = y + 1;
    for (int it = 0; it < ITERS; ++it) {
#pragma unroll
        for (int i = 0; i < ILP; ++i)
            asm volatile("mma.sync.aligned.m16n8k8.row.col.f64.f64.f64.f64 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                         : "+d"(c[i][0]), "+d"(c[i][1]), "+d"(c[i][2]), "+d"(c[i][3])
                         : "d"(a0), "d"(a1), "d"(a2), "d"(a3), "d"(b0), "d"(b1));
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < ILP; ++i) s += c[i][0] + c[i][1] + c[i][2] + c[i][3];
    if (s == 12345.678) out[threadIdx.x] = s;
}

template <int ILP>
__global__ void dmma16816_kernel(double* out, double x, double y) {
    double c[ILP][4];
#pragma unroll
    for (int i = 0; i < ILP; ++i) { c[i][0] = threadIdx.x + i; c[i][1] = i; c[i][2] = 1; c[i][3] = 2; }
    double a[8], b[4];
#pragma unroll
    for (int i = 0; i < 8; ++i) a[i] = x + i;
#pragma unroll
    for (int i = 0; i < 4; ++i) b[i] = y + i;
    for (int it = 0; it < ITERS; ++it) {
#pragma unroll
        for (int i = 0; i < ILP; ++i)
            asm volatile("mma.sync.aligned.m16n8k16.row.col.f64.f64.f64.f64 {%0,%1,%2,%3}, {%4,%5,%6,%7,%8,%9,%10,%11}, {%12,%13,%14,%15}, {%0,%1,%2,%3};"
                         : "+d"(c[i][0]), "+d"(c[i][1]), "+d"(c[i][2]), "+d"(c[i][3])
                         : "d"(a[0]), "d"(a[1]), "d"(a[2]), "d"(a[3]), "d"(a[4]), "d"(a[5]), "d"(a[6]), "d"(a[7]),
                           "d"(b[0]), "d"(b[1]), "d"(b[2]), "d"(b[3]));
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < ILP; ++i) s += c[i][0] + c[i][1] + c[i][2] + c[i][3];
    if (s == 12345.678) out[threadIdx.x] = s;
}

template <typename F>
void run(const char* name, F launch, double flops_per_thread_iter, int blocks, int threads) {
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    launch(); launch();
    cudaDeviceSynchronize();
    cudaEventRecord(e0);
    for (int r = 0; r < 5; ++r) launch();
    cudaEventRecord(e1);
    cudaEventSynchronize(e1);
    float ms; cudaEventElapsedTime(&ms, e0, e1); ms /= 5;
    double fl = flops_per_thread_iter * ITERS * (double)blocks * threads;
    printf("%-28s blocks=%5d thr=%4d  %.3f ms  %.2f TFLOP/s  (%s)\n", name, blocks, threads, ms, fl / ms / 1e9,
           cudaGetErrorString(cudaGetLastError()));
}

int main() {
    double* out; cudaMalloc(&out, 4096 * 8);
    int sms = 148;
    for (int wps : {4, 8, 16, 32}) {   // warps per SM
        int threads = 256, blocks = sms * wps * 32 / threads * 4;
        if (wps * 32 < 256) { threads = wps * 32; blocks = sms * 4; }
        printf("--- %d warps/SM resident (approx)\n", wps);
        // limit residency by launching exactly blocks that fit: use blocks = sms * (wps*32/threads) waves x4
        run("dfma ilp8", [&] { dfma_kernel<8><<<blocks, threads>>>(out, 1.0000001, 1e-9); }, 2.0 * 8, blocks, threads);
        run("dfma ilp16", [&] { dfma_kernel<16><<<blocks, threads>>>(out, 1.0000001, 1e-9); }, 2.0 * 16, blocks, threads);
        run("dmma m8n8k4 ilp8", [&] { dmma884_kernel<8><<<blocks, threads>>>(out, 1.0000001, 1e-9); }, 2.0 * 256 / 32 * 8, blocks, threads);
        run("dmma m8n8k4 ilp16", [&] { dmma884_kernel<16><<<blocks, threads>>>(out, 1.0000001, 1e-9); }, 2.0 * 256 / 32 * 16, blocks, threads);
        run("dmma m16n8k8 ilp8", [&] { dmma1688_kernel<8><<<blocks, threads>>>(out, 1.0000001, 1e-9); }, 2.0 * 1024 / 32 * 8, blocks, threads);
        run("dmma m16n8k16 ilp8", [&] { dmma16816_kernel<8><<<blocks, threads>>>(out, 1.0000001, 1e-9); }, 2.0 * 2048 / 32 * 8, blocks, threads);
    }
    return 0;
}
