// read_patterns.cu -- design probe, not part of libfkconv.so: HBM read bandwidth of a config-2-shaped table
// ([512 rows][250000 doubles], 1.024 GB) under the access patterns considered for the forward kernel:
// linear grid-stride, "column" CTAs (4 KB of U rows in flight), warp-private row pieces (register
// staged), and per-warp cp.async.bulk + mbarrier rings.  Every kernel only sums what it reads.
// Build + run:  python -m paper_1909_10547_b200.build --probes && paper_1909_10547_b200/probes/read_patterns
// Results: profiles/r01_read_patterns.md
#include <cstdio>
#include <cstdint>
#include <cstdlib>
#include <cuda_runtime.h>

#define CK(x) do { cudaError_t e = (x); if (e != cudaSuccess) { printf("ERR %s at %d\n", cudaGetErrorString(e), __LINE__); exit(1);} } while (0)

__device__ __forceinline__ double2 ldnc(const double* p) {
    double2 r;
    asm volatile("ld.global.nc.L1::no_allocate.v2.f64 {%0, %1}, [%2];" : "=d"(r.x), "=d"(r.y) : "l"(p));
    return r;
}
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// P0: linear grid-stride, UNROLL independent 16-B loads per thread
template <int U>
__global__ void __launch_bounds__(256) k_linear(const double* __restrict__ a, long long n2, double* out) {
    long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long stride = (long long)gridDim.x * blockDim.x;
    double s0 = 0, s1 = 0;
    for (; i + (U - 1) * stride < n2; i += U * stride) {
        double2 x[U];
#pragma unroll
        for (int u = 0; u < U; ++u) x[u] = ldnc(a + 2 * (i + u * stride));
#pragma unroll
        for (int u = 0; u < U; ++u) { s0 += x[u].x; s1 += x[u].y; }
    }
    for (; i < n2; i += stride) { double2 x = ldnc(a + 2 * i); s0 += x.x; s1 += x.y; }
    double s = warp_sum(s0 + s1);
    if ((threadIdx.x & 31) == 0 && s == 1.2345) out[0] = s;
}

// P1: column blocks (colsum-like): CTA = (kblock of 512 doubles, split of rows), U rows in flight
template <int U>
__global__ void __launch_bounds__(256) k_column(const double* __restrict__ a, int N, int K, int nkb, int nsplit, double* out) {
    const int kb = blockIdx.x % nkb, sp = blockIdx.x / nkb;
    const int rb = (int)((long long)N * sp / nsplit), re = (int)((long long)N * (sp + 1) / nsplit);
    const int k = (kb * 256 + threadIdx.x) * 2;
    if (k >= K) return;
    const double* col = a + k;
    double s0 = 0, s1 = 0;
    for (int m = rb; m < re; m += U) {
        double2 x[U];
#pragma unroll
        for (int u = 0; u < U; ++u) x[u] = ldnc(col + (long long)min(m + u, re - 1) * K);
#pragma unroll
        for (int u = 0; u < U; ++u) { s0 += x[u].x; s1 += x[u].y; }
    }
    if (s0 + s1 == 1.2345) out[0] = s0;
}

// P2: warp-row pieces with explicit register double buffering.  Unit = (chunk of KC doubles, row).
// CTA gets contiguous unit range (chunk-major); warp w takes rows rb+w, rb+w+8, ...
template <int KC, int U, bool LOCKSTEP>
__global__ void __launch_bounds__(256) k_warprow(const double* __restrict__ a, int N, int K, double* out) {
    const int nch = (K + KC - 1) / KC;
    const long long units = (long long)nch * N;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const long long u0 = units * blockIdx.x / gridDim.x, u1 = units * (blockIdx.x + 1) / gridDim.x;
    double tot = 0;
    for (long long u = u0 + warp; u < u1; u += 8) {
        const int chunk = (int)(u / N), row = (int)(u % N);
        const int k0 = chunk * KC, klen = min(KC, K - k0);
        const double* rp = a + (long long)row * K + k0;
        const int nvec = klen / 2;
        double s0 = 0, s1 = 0;
        int v = lane;
        for (; v + 32 * (U - 1) < nvec; v += 32 * U) {
            double2 x[U];
#pragma unroll
            for (int q = 0; q < U; ++q) x[q] = ldnc(rp + 2 * (v + 32 * q));
#pragma unroll
            for (int q = 0; q < U; ++q) { s0 += x[q].x; s1 += x[q].y; }
        }
        for (; v < nvec; v += 32) { double2 x = ldnc(rp + 2 * v); s0 += x.x; s1 += x.y; }
        tot += warp_sum(s0 + s1);
    }
    if (tot == 1.2345) out[0] = tot;
}

// ---- bulk copy ring per warp
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) { asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) { asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory"); }
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile("{\n.reg .pred p;\nW_%=:\nmbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n@p bra D_%=;\nbra W_%=;\nD_%=:\n}\n" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}

// P3: per-warp ring. piece = PB bytes of one row; stage = RPS rows; DEPTH stages.  Each warp owns a contiguous
// unit range (chunk-major).  WARPS per CTA = blockDim/32.
template <int PB, int RPS, int DEPTH>
__global__ void k_bulkwarp(const double* __restrict__ a, int N, int K, double* out) {
    extern __shared__ __align__(128) unsigned char sm[];
    constexpr int KC = PB / 8;
    const int nwarps = blockDim.x >> 5;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    unsigned char* ring = sm + warp * (DEPTH * RPS * PB);
    uint32_t ring_s = smem_u32(ring);
    uint32_t bars_s = smem_u32(sm + nwarps * (DEPTH * RPS * PB)) + warp * DEPTH * 8;
    if (lane == 0) {
        for (int s = 0; s < DEPTH; ++s) mbar_init(bars_s + 8 * s, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const int nch = (K + KC - 1) / KC;
    const long long units = (long long)nch * N;
    const long long W = (long long)gridDim.x * nwarps, w = (long long)blockIdx.x * nwarps + warp;
    const int u0 = (int)(units * w / W), u1 = (int)(units * (w + 1) / W);  // 32-bit from here on: no 64-bit divides in the loop
    // stage t covers units [u0 + t*RPS, +RPS) clipped to u1 (may straddle chunk boundary: handled per row)
    const int nst = (u1 - u0 + RPS - 1) / RPS;
    auto issue = [&](int t) {
        if (lane == 0) {
            const int slot = (int)(t % DEPTH);
            uint32_t bar = bars_s + 8 * slot;
            uint32_t total = 0;
            for (int q = 0; q < RPS; ++q) {
                int u = u0 + t * RPS + q;
                if (u >= u1) break;
                int chunk = u / N;
                total += (uint32_t)min(KC, K - chunk * KC) * 8;
            }
            mbar_expect_tx(bar, total);
            for (int q = 0; q < RPS; ++q) {
                int u = u0 + t * RPS + q;
                if (u >= u1) break;
                int chunk = u / N, row = u - chunk * N;
                bulk_g2s(ring_s + slot * RPS * PB + q * PB, a + (long long)row * K + (long long)chunk * KC, (uint32_t)min(KC, K - chunk * KC) * 8, bar);
            }
        }
    };
    int issued = 0;
    for (; issued < DEPTH && issued < nst; ++issued) issue(issued);
    double tot = 0;
    for (int t = 0; t < nst; ++t) {
        const int slot = (int)(t % DEPTH);
        mbar_wait(bars_s + 8 * slot, (uint32_t)(t / DEPTH) & 1u);
        double s0 = 0, s1 = 0;
        for (int q = 0; q < RPS; ++q) {
            int u = u0 + t * RPS + q;
            if (u >= u1) break;
            int chunk = u / N;
            int nvec = min(KC, K - chunk * KC) / 2;
            const unsigned char* sb = ring + slot * RPS * PB + q * PB + lane * 16;
#pragma unroll
            for (int vi = 0; vi < PB / 512; ++vi)
                if (vi * 32 + lane < nvec) { double2 x = *reinterpret_cast<const double2*>(sb + vi * 512); s0 += x.x; s1 += x.y; }
        }
        __syncwarp();
        if (issued < nst) { issue(issued); ++issued; }
        tot += warp_sum(s0 + s1);
    }
    if (tot == 1.2345) out[0] = tot;
}

template <typename F>
void run(const char* name, F launch, double bytes) {
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    for (int i = 0; i < 3; ++i) launch();
    CK(cudaDeviceSynchronize());
    cudaEventRecord(e0);
    const int reps = 10;
    for (int r = 0; r < reps; ++r) launch();
    cudaEventRecord(e1);
    cudaEventSynchronize(e1);
    float ms; cudaEventElapsedTime(&ms, e0, e1); ms /= reps;
    printf("%-44s %.1f us  %.0f GB/s  (%s)\n", name, ms * 1e3, bytes / ms / 1e6, cudaGetErrorString(cudaGetLastError()));
    fflush(stdout);
}

template <int PB, int RPS, int DEPTH>
void run_bulk(const char* name, const double* a, int N, int K, double* out, int warps, int ctas_per_sm, double bytes) {
    size_t smem = (size_t)warps * DEPTH * RPS * PB + warps * DEPTH * 8;
    if (smem * ctas_per_sm > 227 * 1024) { printf("%-44s skipped (smem)\n", name); return; }
    CK(cudaFuncSetAttribute(k_bulkwarp<PB, RPS, DEPTH>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    char buf[128];
    snprintf(buf, sizeof buf, "%s PB=%d RPS=%d D=%d w=%d x%d", name, PB, RPS, DEPTH, warps, ctas_per_sm);
    run(buf, [&] { k_bulkwarp<PB, RPS, DEPTH><<<148 * ctas_per_sm, warps * 32, smem>>>(a, N, K, out); }, bytes);
}

int main() {
    const int N = 512, K = 250000;
    const long long n = (long long)N * K;
    double *a, *out;
    CK(cudaMalloc(&a, n * 8));
    CK(cudaMalloc(&out, 64));
    CK(cudaMemset(a, 0, n * 8));
    const double bytes = (double)n * 8;
    run("linear U=4 grid=148*8", [&] { k_linear<4><<<148 * 8, 256>>>(a, n / 2, out); }, bytes);
    run("linear U=8 grid=148*8", [&] { k_linear<8><<<148 * 8, 256>>>(a, n / 2, out); }, bytes);
    run("linear U=8 grid=148*4", [&] { k_linear<8><<<148 * 4, 256>>>(a, n / 2, out); }, bytes);
    run("linear U=16 grid=148*4", [&] { k_linear<16><<<148 * 4, 256>>>(a, n / 2, out); }, bytes);
    for (int nsplit : {1, 2, 4, 8, 16}) {
        char buf[64]; snprintf(buf, sizeof buf, "column U=8 nsplit=%d", nsplit);
        run(buf, [&] { k_column<8><<<489 * nsplit, 256>>>(a, N, K, 489, nsplit, out); }, bytes);
    }
    run("column U=4 nsplit=8", [&] { k_column<4><<<489 * 8, 256>>>(a, N, K, 489, 8, out); }, bytes);
    run("column U=16 nsplit=8", [&] { k_column<16><<<489 * 8, 256>>>(a, N, K, 489, 8, out); }, bytes);
    run("warprow KC=1024 U=4 grid=592", [&] { k_warprow<1024, 4, false><<<592, 256>>>(a, N, K, out); }, bytes);
    run("warprow KC=1024 U=8 grid=592", [&] { k_warprow<1024, 8, false><<<592, 256>>>(a, N, K, out); }, bytes);
    run("warprow KC=1024 U=16 grid=592", [&] { k_warprow<1024, 16, false><<<592, 256>>>(a, N, K, out); }, bytes);
    run("warprow KC=2048 U=16 grid=592", [&] { k_warprow<2048, 16, false><<<592, 256>>>(a, N, K, out); }, bytes);
    run("warprow KC=1024 U=8 grid=1184", [&] { k_warprow<1024, 8, false><<<1184, 256>>>(a, N, K, out); }, bytes);
    run("warprow KC=1024 U=8 grid=4736", [&] { k_warprow<1024, 8, false><<<4736, 256>>>(a, N, K, out); }, bytes);
    run_bulk<4096, 2, 3>("bulk", a, N, K, out, 8, 1, bytes);
    run_bulk<4096, 1, 2>("bulk", a, N, K, out, 8, 1, bytes);
    run_bulk<4096, 1, 3>("bulk", a, N, K, out, 8, 1, bytes);
    run_bulk<4096, 1, 6>("bulk", a, N, K, out, 8, 1, bytes);
    run_bulk<4096, 1, 2>("bulk", a, N, K, out, 4, 1, bytes);
    run_bulk<4096, 1, 4>("bulk", a, N, K, out, 4, 1, bytes);
    run_bulk<4096, 1, 2>("bulk", a, N, K, out, 8, 2, bytes);
    run_bulk<4096, 1, 3>("bulk", a, N, K, out, 8, 2, bytes);
    run_bulk<2048, 1, 3>("bulk", a, N, K, out, 8, 2, bytes);
    run_bulk<2048, 1, 6>("bulk", a, N, K, out, 8, 2, bytes);
    run_bulk<8192, 1, 2>("bulk", a, N, K, out, 8, 1, bytes);
    run_bulk<8192, 1, 3>("bulk", a, N, K, out, 8, 1, bytes);
    run_bulk<16384, 1, 2>("bulk", a, N, K, out, 4, 1, bytes);
    run_bulk<16384, 1, 3>("bulk", a, N, K, out, 4, 1, bytes);
    run_bulk<4096, 1, 3>("bulk", a, N, K, out, 16, 1, bytes);
    return 0;
}
