// fk_dis_direct.cuh -- small DIS tables at R >> 1 in ONE launch (SURVEY 8(a) rows a4 + a5; BASELINE.json config 1 at
// R = 100: N = 2048, K = nA*nx = 450, a 7.4 MB table that is latency-bound, not pipe-bound).
//
//   Sigma[n][r] = sum_k FK[n][k] * f[r][slot(k)],   k = c*nx + i (PACKED order),  slot(k) = flav_c*nx + i
//
// The general R >> 1 path (fk_gemm_dis_ws_kernel) is three launches: transpose f, split-K contraction, reduction of
// the split-K partials.  On a table this small those are three latencies for a few microseconds of FP64 tensor work.
// Here both operands are K-MAJOR as they lie in memory -- a row of the table, and for one replica the run
// f[r][flav_c][0..nx) of every active flavour c -- so both go to shared memory by bulk async copies with no
// transposed copy of f:  the B tile Bs[col][k] of a CTA's replica columns is copied once (nA pieces of nx doubles per
// replica; runs of consecutive flavours merged), the A tile streams through a ring of [64 datapoints][64 k] stages (four
// producer warps: the issue cost of a bulk copy is per warp, profiles/r02_bulk_copy_issue.md).  Four consumer warps hold 16 datapoints
// x (<= 4) 8-replica fragments each and run the plain DMMA loop over the whole K, so there is no split-K and the
// accumulators go straight to sigma.  K <= 512 keeps every accumulation chain within the 512 FMAs the tolerance
// derivation assumes.  Bitwise repeatable: fixed k order per output.
#pragma once

#include "fk_common.cuh"
#include "fk_gemm.cuh"
#include "fk_gemm_ws.cuh"

namespace fk {

constexpr int DD_TM = 64;                 // datapoints per CTA (4 consumer warps x 16)
constexpr int DD_NFC = 4;                 // 8-replica fragments per CTA at most
constexpr int DD_KT = 64;                 // k per stage of the A ring
constexpr int DD_SA = DD_KT + 4;          // row pitch of an A stage (pitch mod 16 == 4: conflict-free fragment loads)
constexpr int DD_STAGES = 3;
constexpr int DD_CONSUMERS = 4;
constexpr int DD_PRODUCERS = 4;            // a bulk copy costs its warp ~57 cycles of issue: ~800 pieces per CTA need four warps
constexpr int DD_THREADS = (DD_CONSUMERS + DD_PRODUCERS) * 32;
constexpr int DD_MAX_K = 512;
constexpr size_t DD_STATIC_SMEM = 2048;    // the kernel's static shared memory (run list), rounded up

// row pitch of the B tile: K rounded up to 16 (the consumers walk whole groups of 4 MMA k-steps; the tail is zero) + 4,
// so that pitch mod 16 == 4 (conflict-free fragment loads)
constexpr int DD_KG = 16;                 // k per group of 4 MMA k-steps
__host__ __device__ inline int dd_pitch_b(int K) { return (K + DD_KG - 1) / DD_KG * DD_KG + 4; }
__host__ __device__ inline size_t dd_smem_bytes(int K, int stages) {
    return (size_t)(stages * DD_TM * DD_SA + DD_NFC * 8 * dd_pitch_b(K)) * 8 + (2 * DD_STAGES + 1) * 8;
}

struct DisDirectParams {
    TableDesc desc;
    ChannelList chan;
    const double* f;    // [R][nfl][nx]
    double* sigma;      // [N][R] (+ out_off * R)
    int R, nfrag, ncs;  // fragments of all R replicas; column groups (gridDim.y)
    int stages;         // stages of the A ring: DD_STAGES, or 2 when the B tile of a K near 512 leaves no room for three
};

__global__ void __launch_bounds__(DD_THREADS, 1)
fk_dis_direct_kernel(const __grid_constant__ DisDirectParams p) {
    pdl_trigger();
    extern __shared__ __align__(128) unsigned char fk_smem[];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const TableDesc& d = p.desc;
    const int K = d.K, nx = d.nx, PB = dd_pitch_b(K);
    const int m0 = blockIdx.x * DD_TM;
    const int f0 = (int)((long long)p.nfrag * blockIdx.y / p.ncs), f1 = (int)((long long)p.nfrag * (blockIdx.y + 1) / p.ncs);
    const int nf = f1 - f0, ncols = nf * 8, rbase = f0 * 8;
    const int nst = (K + DD_KT - 1) / DD_KT, NS = p.stages;

    double* As = reinterpret_cast<double*>(fk_smem);           // [NS][64][68]
    double* Bs = As + NS * DD_TM * DD_SA;                      // [32][PB]   f[rbase + col][slot(k)]
    const uint32_t As_s = (uint32_t)__cvta_generic_to_shared(As), Bs_s = (uint32_t)__cvta_generic_to_shared(Bs);
    const uint32_t bar0 = Bs_s + (uint32_t)(DD_NFC * 8 * PB * 8);
    auto bar_full = [&](int s) { return bar0 + 8u * s; };
    auto bar_empty = [&](int s) { return bar0 + 8u * (DD_STAGES + s); };
    const uint32_t bar_b = bar0 + 8u * (2 * DD_STAGES);
    // zeros once: the k past the end of K in the last group of k-steps, the B rows past this CTA's columns, the rows of a
    // partial datapoint tile, whatever a short last stage leaves
    for (int t = tid; t < NS * DD_TM * DD_SA + DD_NFC * 8 * PB; t += DD_THREADS) As[t] = 0.0;
    // runs of consecutive flavours in the (usually sorted) active list: their nx-runs of f are contiguous both in f and
    // in the B tile, so a run is ONE copy (config 1: 5 runs for 9 flavours)
    __shared__ short run_c0[MAX_NFL], run_len[MAX_NFL];
    __shared__ int nruns_s;
    if (tid == 0) {
        int nr = 0;
        for (int c = 0; c < d.C;) {
            int e = c + 1;
            while (e < d.C && (int)p.chan.a[e] == (int)p.chan.a[e - 1] + 1) ++e;
            run_c0[nr] = (short)c;
            run_len[nr] = (short)(e - c);
            ++nr;
            c = e;
        }
        nruns_s = nr;
        for (int s = 0; s < NS; ++s) {
            mbar_init(bar_full(s), DD_PRODUCERS);   // one arrive.expect_tx per producer warp
            mbar_init(bar_empty(s), DD_CONSUMERS);
        }
        mbar_init(bar_b, DD_PRODUCERS);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // the zeros before any bulk copy lands
    __syncthreads();
    const int rows_valid = min(DD_TM, d.N - m0);

    if (warp >= DD_CONSUMERS) {
        // ================================ producer warps ================================
        // warp pw copies the datapoints 16*pw .. 16*pw + 15 of every A stage and every fourth piece of the B tile
        const int pw = warp - DD_CONSUMERS;
        constexpr int RPW = DD_TM / DD_PRODUCERS;
        const double* __restrict__ fk = reinterpret_cast<const double*>(d.fk);
        const int my_rows = max(0, min(RPW, rows_valid - RPW * pw));
        auto issue_a = [&](int it) {
            const int stage = it % NS, k0 = it * DD_KT;
            const int len = min(DD_KT, K - k0), lenc = (len + 1) & ~1;   // whole 16-byte pieces (K is even: nx is)
            mbar_wait(bar_empty(stage), ((it / NS) & 1) ^ 1);
            if (lane == 0) mbar_expect_tx(bar_full(stage), (uint32_t)(my_rows * lenc * 8));
            __syncwarp();
            const int row = RPW * pw + lane;
            if (lane < my_rows)
                bulk_g2s(As_s + (uint32_t)((stage * DD_TM * DD_SA + row * DD_SA) * 8), fk + (long long)(m0 + row) * d.row_stride + k0,
                         (uint32_t)(lenc * 8), bar_full(stage));
        };
        // the table does not depend on the call before this one: its first stage goes out before the wait
        issue_a(0);
        pdl_wait();   // f may have been written by the kernel before this one in the stream
        // B tile: for every replica column of this CTA, the f-run of every run of active flavours
        const int slots = d.nfl * nx, nruns = nruns_s, npieces = ncols * nruns;
        int my_bytes = 0;
        for (int q = pw * 32 + lane; q < npieces; q += 32 * DD_PRODUCERS) my_bytes += (int)run_len[q % nruns] * nx * 8;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) my_bytes += __shfl_xor_sync(0xffffffffu, my_bytes, o);
        if (lane == 0) mbar_expect_tx(bar_b, (uint32_t)my_bytes);
        __syncwarp();
        for (int q = pw * 32 + lane; q < npieces; q += 32 * DD_PRODUCERS) {
            const int col = q / nruns, run = q - col * nruns, c = run_c0[run];
            const int r = min(rbase + col, p.R - 1);   // columns past R repeat the last replica (never stored)
            bulk_g2s(Bs_s + (uint32_t)((col * PB + c * nx) * 8), p.f + (long long)r * slots + (int)p.chan.a[c] * nx,
                     (uint32_t)((int)run_len[run] * nx * 8), bar_b);
        }
        for (int it = 1; it < nst; ++it) issue_a(it);
        return;
    }

    // ================================ consumer warps: 16 datapoints x nf fragments ================================
    double acc[2][DD_NFC][2];
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
        for (int j = 0; j < DD_NFC; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
    mbar_wait(bar_b, 0);
    // Whole groups of 4 MMA k-steps with all 24 fragment loads ahead of the 32 DMMAs and no branch in between (one warp
    // per scheduler: every exposed shared-memory latency is idle tensor time).  All DD_NFC fragments are computed whatever
    // nf is: the rows of Bs past this CTA's columns are zero, and the slowest CTA (nf = DD_NFC) sets the time of the call.
    const double* Bt = Bs + (lane >> 2) * PB + (lane & 3);
    for (int it = 0; it < nst; ++it) {
        const int stage = it % NS, k0 = it * DD_KT;
        const int ngroups = (min(DD_KT, K - k0) + DD_KG - 1) / DD_KG;
        mbar_wait(bar_full(stage), (it / NS) & 1);
        const double* At = As + stage * DD_TM * DD_SA + (warp * 16 + (lane >> 2)) * DD_SA + (lane & 3);
        const double* Btk = Bt + k0;
        for (int g = 0; g < ngroups; ++g) {
            double a[4][2], b[4][DD_NFC];
#pragma unroll
            for (int s = 0; s < 4; ++s) {
                a[s][0] = At[g * DD_KG + s * 4];
                a[s][1] = At[8 * DD_SA + g * DD_KG + s * 4];
#pragma unroll
                for (int j = 0; j < DD_NFC; ++j) b[s][j] = Btk[j * 8 * PB + g * DD_KG + s * 4];
            }
#pragma unroll
            for (int s = 0; s < 4; ++s)
#pragma unroll
                for (int j = 0; j < DD_NFC; ++j) {
                    dmma884(acc[0][j][0], acc[0][j][1], a[s][0], b[s][j]);
                    dmma884(acc[1][j][0], acc[1][j][1], a[s][1], b[s][j]);
                }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_empty(stage));
    }
    // C fragment: row = lane >> 2, columns 2*(lane & 3) + {0, 1}
    double* sig = p.sigma + d.out_off * p.R;
#pragma unroll
    for (int i = 0; i < 2; ++i) {
        const int n = m0 + warp * 16 + i * 8 + (lane >> 2);
        if (n >= d.N) continue;
#pragma unroll
        for (int j = 0; j < DD_NFC; ++j) {
            const int r = rbase + j * 8 + 2 * (lane & 3);
            if (j < nf) {
                if (r < p.R) sig[(long long)n * p.R + r] = acc[i][j][0];
                if (r + 1 < p.R) sig[(long long)n * p.R + r + 1] = acc[i][j][1];
            }
        }
    }
}

}  // namespace fk
