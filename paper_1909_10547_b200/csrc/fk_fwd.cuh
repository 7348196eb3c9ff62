// fk_fwd.cuh -- bandwidth-bound forward path (R <= 4 per pass).
//
//   sigma[n][r] = sum_k FK[n][k] * L[k][r],   L[k][r] = f[r][a_c][i] * f[r][b_c][j]      Eq. (1)
//
// "Column" decomposition, chosen from the read-pattern measurements in profiles/r01_read_patterns.md:
// a CTA owns a block of FWD_THREADS * VEC consecutive k (4 KB of every row) and a range of datapoints.
//   a1  each thread keeps the luminosity of ITS k (VEC values per replica) in registers for the whole
//       CTA: the luminosity is built once per CTA straight from f and never touches HBM;
//   a2  the CTA walks down its datapoints U rows at a time: U independent, fully coalesced 128-bit
//       no-allocate loads per thread are in flight (the CTA reads U x 4 KB contiguous pieces), each
//       FK element is multiplied by the thread's L values -- per-thread chains are VEC FMAs long;
//   a3  level 1: the U row sums of a warp are folded together in one multi-value xor-butterfly
//       (U-1 + log2(32/U) shuffles for U rows), the 8 warp results are added in a fixed order through
//       shared memory -> ONE partial per (row, k-block); level 2: fk_reduce_chunks_kernel adds the
//       k-blocks of a row in a fixed order.  No atomics anywhere: results are bitwise repeatable.
// The grid is the list of (k-block, datapoint range) pairs -- for a grouped launch the host-built list
// over all tables -- several waves of small CTAs that the hardware scheduler balances.
#pragma once

#include "fk_common.cuh"

namespace fk {

struct FwdParams {
    TableDesc desc;           // single-table launch
    ChannelList chan;         // single-table launch
    const TableDesc* descs;   // grouped launch (device)
    const ColSeg* segs;       // grouped launch (device), one per CTA
    const void* f;            // f[R][nfl][nx] or f_cat
    double* part;             // level-1 partials [row][replica][k-block]
    void* sigma;              // direct output for tables with a single k-block
    int R, r0;                // replicas, first replica of this pass
    int* cnt;                 // tickets per datapoint range (resident tables / groups; zero between launches), or null:
                              // the CTA that completes a range also runs its level-2 reduction (no second launch)
};

constexpr int FWD_THREADS = 256;
constexpr int FWD_WARPS = FWD_THREADS / 32;

// a3 level 2 for up to 4 outputs (n, r) at once: per output the fixed order of the level-2 kernel (four lane-strided
// chains per lane, combined pairwise, then the xor butterfly); the outputs' loads are interleaved so that a warp has up to
// 16 of them in flight.  Partials are read past L1 (they were written by other SMs).
template <int NO>
__device__ __forceinline__ void reduce_chunks_rows(const double* (&src)[NO], int nch, int lane, double (&out)[NO]) {
    double a[NO][4];
#pragma unroll
    for (int q = 0; q < NO; ++q) a[q][0] = a[q][1] = a[q][2] = a[q][3] = 0.0;
    int c = lane;
    for (; c + 96 < nch; c += 128) {
#pragma unroll
        for (int q = 0; q < NO; ++q) {
            a[q][0] += __ldcg(src[q] + c);
            a[q][1] += __ldcg(src[q] + c + 32);
            a[q][2] += __ldcg(src[q] + c + 64);
            a[q][3] += __ldcg(src[q] + c + 96);
        }
    }
    for (; c < nch; c += 32) {
#pragma unroll
        for (int q = 0; q < NO; ++q) a[q][0] += __ldcg(src[q] + c);
    }
#pragma unroll
    for (int q = 0; q < NO; ++q) out[q] = warp_sum((a[q][0] + a[q][1]) + (a[q][2] + a[q][3]));
}

// Folds U per-lane values (one per row) across the warp: afterwards lane l holds the warp total of
// row l >> (5 - log2 U).  Fixed tree; a+b and b+a give the same bits, so every lane agrees.
template <int U>
__device__ __forceinline__ double fold_rows(double (&p)[U], int lane) {
    int off = 16;
#pragma unroll
    for (int n = U; n > 1; n >>= 1, off >>= 1) {
        const bool hi = (lane & off) != 0;
#pragma unroll
        for (int i = 0; i < n / 2; ++i) {
            const double send = hi ? p[i] : p[i + n / 2];
            const double keep = hi ? p[i + n / 2] : p[i];
            p[i] = keep + __shfl_xor_sync(0xffffffffu, send, off);
        }
    }
    double s = p[0];
#pragma unroll
    for (; off > 0; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
    return s;
}

// TS = storage type of the table (float for the fp32-storage variants), T = type of f, sigma and of the arithmetic
template <typename T, int VEC, int RT, int U, bool GROUPED, typename TS = T>
__global__ void __launch_bounds__(FWD_THREADS, RT == 1 ? 4 : RT <= 4 ? 3 : 2)   // R = 1: at most 64 registers, four CTAs per SM
fk_fwd_column_kernel(const __grid_constant__ FwdParams p) {
    pdl_trigger();   // first kernel of a call (normal launch): lets the level-2 reduction be scheduled under this grid's last wave
    using V = Vec<TS, VEC>;
    constexpr int LPR = 32 / U;  // lanes that end up holding the same row
    __shared__ double red[2][FWD_WARPS][U][RT];

    const TableDesc* dp = &p.desc;
    const uint8_t* __restrict__ ca = p.chan.a;
    const uint8_t* __restrict__ cb = p.chan.b;
    int kblock, split;
    if constexpr (GROUPED) {
        const ColSeg sg = p.segs[blockIdx.x];
        dp = &p.descs[sg.table];
        ca = dp->chan_a;
        cb = dp->chan_b;
        kblock = sg.kblock;
        split = sg.split;
    } else {
        kblock = blockIdx.x % p.desc.nchunks;
        split = blockIdx.x / p.desc.nchunks;
    }
    const TableDesc& d = *dp;
    const int R = p.R;
    const int rb = (int)((long long)d.N * split / d.fsplit);
    const int re = (int)((long long)d.N * (split + 1) / d.fsplit);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    // a1: this thread's luminosity values
    const int k = (kblock * FWD_THREADS + threadIdx.x) * VEC;
    const bool kin = k < d.K;  // VEC > 1: rows are padded to a multiple of VEC, so the whole vector is readable
    T L[RT][VEC];
    {
        const int fstride = d.nfl * d.nx;
        const T* __restrict__ f = reinterpret_cast<const T*>(p.f) + d.f_off * R;
#pragma unroll
        for (int e = 0; e < VEC; ++e) {
            int ia = 0, ib = -1;
            bool in = k + e < d.K;
            if (in) decode_k(d, ca, cb, k + e, ia, ib);
            in = in && ia >= 0;
#pragma unroll
            for (int r = 0; r < RT; ++r) {
                const int rr = p.r0 + r;
                T l = T(0);
                if (in && rr < R) {
                    l = __ldg(f + (long long)rr * fstride + ia);
                    if (ib >= 0) l *= __ldg(f + (long long)rr * fstride + ib);
                }
                L[r][e] = l;
            }
        }
    }
    const TS* __restrict__ col = reinterpret_cast<const TS*>(d.fk) + (kin ? k : 0);

    int buf = 0;
    for (int m = rb; m < re; m += U, buf ^= 1) {
        // a2: U rows in flight
        V x[U];
#pragma unroll
        for (int u = 0; u < U; ++u) x[u] = ld_stream(col + (long long)min(m + u, re - 1) * d.row_stride, (V*)nullptr);
        double pr[RT][U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const bool live = kin && (m + u < re);
#pragma unroll
            for (int r = 0; r < RT; ++r) {
                T s = (T)x[u].v[0] * L[r][0];
#pragma unroll
                for (int e = 1; e < VEC; ++e) s = fma((T)x[u].v[e], L[r][e], s);
                pr[r][u] = live ? (double)s : 0.0;
            }
        }
        // a3 level 1: warp fold, then the 8 warps in a fixed order
#pragma unroll
        for (int r = 0; r < RT; ++r) {
            const double s = fold_rows<U>(pr[r], lane);
            if ((lane & (LPR - 1)) == 0) red[buf][warp][lane / LPR][r] = s;
        }
        __syncthreads();
        if (threadIdx.x < U * RT) {
            const int u = threadIdx.x / RT, r = threadIdx.x - u * RT;
            double s = red[buf][0][u][r];
#pragma unroll
            for (int w = 1; w < FWD_WARPS; ++w) s += red[buf][w][u][r];
            const int n = m + u, rr = p.r0 + r;
            if (n < re && rr < R) {
                if (d.nchunks == 1)
                    reinterpret_cast<T*>(p.sigma)[d.out_off * R + (long long)n * R + rr] = (T)s;
                else
                    p.part[d.part_off * R + ((long long)n * R + rr) * d.nchunks + kblock] = s;
            }
        }
    }
    // a3 level 2 without a second launch: the CTA that hands in the last k-block of its datapoint range sums the range's
    // partials (same arithmetic and order as fk_reduce_chunks_kernel, whoever runs it: bitwise the same result)
    if (p.cnt != nullptr && d.nchunks > 1) {
        __shared__ int s_last;
        __threadfence();   // this CTA's partials before its ticket
        __syncthreads();
        if (threadIdx.x == 0) s_last = atomicAdd(p.cnt + d.cnt_off + split, 1) == d.nchunks - 1;
        __syncthreads();
        if (s_last) {
            __threadfence();
            const int nout = (re - rb) * RT;
            for (int o0 = warp * 4; o0 < nout; o0 += FWD_WARPS * 4) {
                const double* src[4];
                int nn[4], rq[4];
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const int o = min(o0 + q, nout - 1);
                    nn[q] = rb + o / RT;
                    rq[q] = min(p.r0 + o % RT, R - 1);
                    src[q] = p.part + d.part_off * R + ((long long)nn[q] * R + rq[q]) * d.nchunks;
                }
                double sum[4];
                reduce_chunks_rows<4>(src, d.nchunks, lane, sum);
#pragma unroll
                for (int q = 0; q < 4; ++q)
                    if (lane == 0 && o0 + q < nout && p.r0 + (o0 + q) % RT < R)
                        reinterpret_cast<T*>(p.sigma)[d.out_off * R + (long long)nn[q] * R + rq[q]] = (T)sum[q];
            }
            if (threadIdx.x == 0) p.cnt[d.cnt_off + split] = 0;   // ready for the next launch
        }
    }
}

// ---- few datapoints, very long rows (the paper's N = 8 shapes of Table 3): with one batch of U rows
// per (k-block, range) the column kernel above would launch ~K/512 CTAs that live for one round trip each, and
// the CTA launch rate, not HBM, sets the pace (3.3 TB/s at K = 1e8).  Here a CTA walks k-blocks blockIdx.x,
// blockIdx.x + gridDim.x, ... of its datapoint range and adds their CTA sums in walk order: same per-thread
// arithmetic, one level-1 partial per CTA (a fixed grid: bitwise repeatable), same level 2.
template <typename T, int VEC, int RT, int U, typename TS = T>
__global__ void __launch_bounds__(FWD_THREADS)
fk_fwd_fewrows_kernel(const __grid_constant__ FwdParams p) {
    pdl_trigger();
    using V = Vec<TS, VEC>;
    constexpr int LPR = 32 / U;
    __shared__ double red[2][FWD_WARPS][U][RT];
    const TableDesc& d = p.desc;
    const uint8_t* __restrict__ ca = p.chan.a;
    const uint8_t* __restrict__ cb = p.chan.b;
    const int split = blockIdx.y, R = p.R;
    const int rb = (int)((long long)d.N * split / d.fsplit);
    const int re = (int)((long long)d.N * (split + 1) / d.fsplit);  // re - rb <= U
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int fstride = d.nfl * d.nx;
    const T* __restrict__ f = reinterpret_cast<const T*>(p.f);
    int buf = 0;
    double tot = 0.0;  // threads < U * RT: this CTA's sum over its k-blocks, in walk order (one partial per CTA)
    for (int kblock = blockIdx.x; kblock < d.nchunks; kblock += gridDim.x, buf ^= 1) {
        const int k = (kblock * FWD_THREADS + threadIdx.x) * VEC;
        const bool kin = k < d.K;
        const TS* __restrict__ col = reinterpret_cast<const TS*>(d.fk) + (kin ? k : 0);
        V x[U];
#pragma unroll
        for (int u = 0; u < U; ++u) x[u] = ld_stream(col + (long long)min(rb + u, re - 1) * d.row_stride, (V*)nullptr);
        T L[RT][VEC];
#pragma unroll
        for (int e = 0; e < VEC; ++e) {
            int ia = 0, ib = -1;
            bool in = k + e < d.K;
            if (in) decode_k(d, ca, cb, k + e, ia, ib);
            in = in && ia >= 0;
#pragma unroll
            for (int r = 0; r < RT; ++r) {
                const int rr = p.r0 + r;
                T l = T(0);
                if (in && rr < R) {
                    l = __ldg(f + (long long)rr * fstride + ia);
                    if (ib >= 0) l *= __ldg(f + (long long)rr * fstride + ib);
                }
                L[r][e] = l;
            }
        }
        double pr[RT][U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const bool live = kin && (rb + u < re);
#pragma unroll
            for (int r = 0; r < RT; ++r) {
                T s = (T)x[u].v[0] * L[r][0];
#pragma unroll
                for (int e = 1; e < VEC; ++e) s = fma((T)x[u].v[e], L[r][e], s);
                pr[r][u] = live ? (double)s : 0.0;
            }
        }
#pragma unroll
        for (int r = 0; r < RT; ++r) {
            const double s = fold_rows<U>(pr[r], lane);
            if ((lane & (LPR - 1)) == 0) red[buf][warp][lane / LPR][r] = s;
        }
        __syncthreads();
        if (threadIdx.x < U * RT) {
            const int u = threadIdx.x / RT, r = threadIdx.x - u * RT;
            double s = red[buf][0][u][r];
#pragma unroll
            for (int w = 1; w < FWD_WARPS; ++w) s += red[buf][w][u][r];
            tot += s;
        }
    }
    if (threadIdx.x < U * RT) {
        const int u = threadIdx.x / RT, r = threadIdx.x - u * RT;
        const int n = rb + u, rr = p.r0 + r;
        if (n < re && rr < R) p.part[((long long)n * R + rr) * gridDim.x + blockIdx.x] = tot;
    }
}

// ---- one read of FK for both passes: when the upstream gradient g[n][r] is known before the
// forward pass (a loss linear in sigma, e.g. config 4's seeded weights), the column kernel also accumulates
// VJP stage 1, G[split][r][k] = sum_{n in range} g[n][r] FK[n][k], from the registers that already hold the row
// pieces.  Same decomposition, same level-1 partials, same fixed orders as the two separate kernels; stage 2 of
// the VJP (fk_vjp_foldk_kernel) and level 2 of the forward (fk_reduce_chunks_kernel) follow unchanged.
struct FusedParams {
    FwdParams fwd;
    const void* g;   // g[N][R]
    double* G;       // [fsplit][R][K] column sums, one slice per datapoint range
};

// (R = 1: capped at 51 registers so that five CTAs stay resident per SM; 54 cost one CTA and 6 % of the bandwidth)
template <typename T, int VEC, int RT, int U, bool GROUPED, typename TS = T>
__global__ void __launch_bounds__(FWD_THREADS, RT == 1 ? (sizeof(T) == sizeof(TS) ? 5 : 4) : 1)
fk_fused_column_kernel(const __grid_constant__ FusedParams q) {
    pdl_trigger();
    using V = Vec<TS, VEC>;
    constexpr int LPR = 32 / U;
    constexpr int MAX_ROWS = 64;  // datapoints per range (the plan uses <= 32)
    __shared__ double red[2][FWD_WARPS][U][RT];
    __shared__ T gs[(MAX_ROWS + U) * RT];
    const FwdParams& p = q.fwd;
    const TableDesc* dp = &p.desc;
    const uint8_t* __restrict__ ca = p.chan.a;
    const uint8_t* __restrict__ cb = p.chan.b;
    int kblock, split;
    if constexpr (GROUPED) {   // grouped: static list of (table, k-block, datapoint range) CTAs; descs carry the fused splits
        const ColSeg sg = p.segs[blockIdx.x];
        dp = &p.descs[sg.table];
        ca = dp->chan_a;
        cb = dp->chan_b;
        kblock = sg.kblock;
        split = sg.split;
    } else {
        kblock = blockIdx.x % p.desc.nchunks;
        split = blockIdx.x / p.desc.nchunks;
    }
    const TableDesc& d = *dp;
    const int R = p.R;
    const int rb = (int)((long long)d.N * split / d.fsplit);
    const int re = (int)((long long)d.N * (split + 1) / d.fsplit);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    {   // g tile of this datapoint range, zero padded to a multiple of U rows
        const T* __restrict__ g = reinterpret_cast<const T*>(q.g) + d.out_off * R;
        const int rows = re - rb, rows_pad = (rows + U - 1) / U * U;
        for (int t = threadIdx.x; t < rows_pad * RT; t += FWD_THREADS) {
            const int m = t / RT, r = t - m * RT, rr = p.r0 + r;
            gs[t] = (m < rows && rr < R) ? __ldg(g + (long long)(rb + m) * R + rr) : T(0);
        }
    }
    const int k = (kblock * FWD_THREADS + threadIdx.x) * VEC;
    const bool kin = k < d.K;
    T L[RT][VEC];
    {
        const int fstride = d.nfl * d.nx;
        const T* __restrict__ f = reinterpret_cast<const T*>(p.f) + d.f_off * R;
#pragma unroll
        for (int e = 0; e < VEC; ++e) {
            int ia = 0, ib = -1;
            bool in = k + e < d.K;
            if (in) decode_k(d, ca, cb, k + e, ia, ib);
            in = in && ia >= 0;
#pragma unroll
            for (int r = 0; r < RT; ++r) {
                const int rr = p.r0 + r;
                T l = T(0);
                if (in && rr < R) {
                    l = __ldg(f + (long long)rr * fstride + ia);
                    if (ib >= 0) l *= __ldg(f + (long long)rr * fstride + ib);
                }
                L[r][e] = l;
            }
        }
    }
    T cs[2][RT][VEC];  // two interleaved column-sum chains
#pragma unroll
    for (int a = 0; a < 2; ++a)
#pragma unroll
        for (int r = 0; r < RT; ++r)
#pragma unroll
            for (int e = 0; e < VEC; ++e) cs[a][r][e] = T(0);
    const TS* __restrict__ col = reinterpret_cast<const TS*>(d.fk) + (kin ? k : 0);
    __syncthreads();

    int buf = 0;
    for (int m = rb; m < re; m += U, buf ^= 1) {
        V x[U];
#pragma unroll
        for (int u = 0; u < U; ++u) x[u] = ld_stream(col + (long long)min(m + u, re - 1) * d.row_stride, (V*)nullptr);
        double pr[RT][U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const bool live = kin && (m + u < re);
#pragma unroll
            for (int r = 0; r < RT; ++r) {
                T s = (T)x[u].v[0] * L[r][0];
#pragma unroll
                for (int e = 1; e < VEC; ++e) s = fma((T)x[u].v[e], L[r][e], s);
                pr[r][u] = live ? (double)s : 0.0;
                const T gv = gs[(m - rb + u) * RT + r];  // 0 on the padded rows
#pragma unroll
                for (int e = 0; e < VEC; ++e) cs[u & 1][r][e] = fma(gv, (T)x[u].v[e], cs[u & 1][r][e]);
            }
        }
#pragma unroll
        for (int r = 0; r < RT; ++r) {
            const double s = fold_rows<U>(pr[r], lane);
            if ((lane & (LPR - 1)) == 0) red[buf][warp][lane / LPR][r] = s;
        }
        __syncthreads();
        if (threadIdx.x < U * RT) {
            const int u = threadIdx.x / RT, r = threadIdx.x - u * RT;
            double s = red[buf][0][u][r];
#pragma unroll
            for (int w = 1; w < FWD_WARPS; ++w) s += red[buf][w][u][r];
            const int n = m + u, rr = p.r0 + r;
            if (n < re && rr < R) {
                if (d.nchunks == 1)
                    reinterpret_cast<T*>(p.sigma)[d.out_off * R + (long long)n * R + rr] = (T)s;
                else
                    p.part[d.part_off * R + ((long long)n * R + rr) * d.nchunks + kblock] = s;
            }
        }
    }
    if (kin) {
#pragma unroll
        for (int r = 0; r < RT; ++r) {
            const int rr = p.r0 + r;
            if (rr >= R) continue;
#pragma unroll
            for (int e = 0; e < VEC; ++e)
                if (k + e < d.K) q.G[d.g_off * R + ((long long)split * R + rr) * d.K + k + e] = (double)cs[0][r][e] + (double)cs[1][r][e];
        }
    }
}

// ---- a3 level 2: sigma[n][r] = sum over k-blocks, fixed order (lane-strided chains + butterfly) ----
struct ReduceParams {
    TableDesc desc;           // single
    const TableDesc* descs;   // grouped (device)
    const int* row_prefix;    // grouped (device) [T+1]: first global row of each table
    int T;
    const double* part;
    void* sigma;
    long long rows;           // total rows (single: N)
    int R;
};

template <typename T, bool GROUPED>
__global__ void __launch_bounds__(256) fk_reduce_chunks_kernel(const __grid_constant__ ReduceParams p) {
    pdl_trigger();
    pdl_wait();   // the level-1 partials of the whole forward grid
    const int lane = threadIdx.x & 31;
    const long long warp0 = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const long long nwarps = ((long long)gridDim.x * blockDim.x) >> 5;
    const long long total = p.rows * p.R;
    for (long long o = warp0; o < total; o += nwarps) {
        const long long grow = o / p.R;
        const int r = (int)(o - grow * p.R);
        const TableDesc* d = &p.desc;
        long long n = grow;
        if constexpr (GROUPED) {
            int lo = 0, hi = p.T;  // last table with row_prefix[t] <= grow
            while (hi - lo > 1) {
                const int mid = (lo + hi) >> 1;
                if (p.row_prefix[mid] <= grow) lo = mid; else hi = mid;
            }
            d = &p.descs[lo];
            n = grow - p.row_prefix[lo];
        }
        const int nch = d->nchunks;
        if (nch == 1) continue;  // written directly by the column kernel
        const double* src = p.part + d->part_off * p.R + (n * p.R + r) * nch;
        const double* srcs[1] = {src};
        double s1[1];
        reduce_chunks_rows<1>(srcs, nch, lane, s1);
        if (lane == 0) reinterpret_cast<T*>(p.sigma)[d->out_off * p.R + n * p.R + r] = (T)s1[0];
    }
}

}  // namespace fk
