// fk_stream.cuh -- bandwidth-bound forward path (R <= 4 per pass).
//
//   sigma[n][r] = sum_k FK[n][k] * L[k][r],   L[k][r] = f[r][a_c][i] * f[r][b_c][j]      Eq. (1)
//
// Work unit = (K-chunk, datapoint row): `kc` consecutive k of one row (8 KB).  Units are ordered
// chunk-major and dealt to a persistent grid in equal contiguous ranges (single table) or by a
// host-built, byte-balanced segment list (grouped launch).  Per (table, chunk) segment a CTA
//   1. builds the luminosity tile L[RT][kc] in shared memory straight from f (never in HBM),
//   2. lets every warp stream whole rows of FK with coalesced 128-bit no-allocate loads, RPW rows at
//      a time sharing the L registers, UNROLL*RPW loads in flight per lane, per-lane chains <= kc/64,
//   3. reduces each row with a fixed xor-butterfly and writes ONE level-1 partial per (row, chunk).
// A second tiny kernel sums the chunk partials of each (n, r) in a fixed order -> bitwise repeatable.
#pragma once

#include "fk_common.cuh"

namespace fk {

struct Segment {       // grouped work list entry: rows [row_begin, row_end) of one (table, chunk)
    int table, chunk, row_begin, row_end;
};

struct StreamParams {
    TableDesc desc;            // single-table launch
    ChannelList chan;          // single-table launch
    const TableDesc* descs;    // grouped launch (device)
    const Segment* segs;       // grouped launch (device)
    const int* cta_seg_start;  // grouped launch (device) [gridDim.x + 1]
    const void* f;             // f[R][nfl][nx] or f_cat
    double* part;              // level-1 partials
    void* sigma;               // direct output for tables with a single chunk
    long long units;           // single table: nchunks * N
    int R, r0;                 // replicas, first replica of this pass
    int kc_stride;             // shared-memory stride of one replica's L tile (>= every table's kc)
};

constexpr int STREAM_THREADS = 256;

template <typename T, int VEC, int RT, int RPW, int UNROLL>
__device__ __forceinline__ void stream_segment(const TableDesc& d, const uint8_t* __restrict__ ca,
                                               const uint8_t* __restrict__ cb, int chunk, int rb, int re,
                                               const StreamParams& p, T* __restrict__ Lt) {
    using V = Vec<T, VEC>;
    const int kc = d.kc, ls = p.kc_stride;
    const int k0 = chunk * kc;
    const int klen = min(kc, d.K - k0);
    const int R = p.R;
    const int fstride = d.nfl * d.nx;
    const T* __restrict__ f = reinterpret_cast<const T*>(p.f) + d.f_off * R;

    __syncthreads();  // the previous segment's readers are done with Lt
    // a1: luminosity tile, zero-padded to kc so the vector loop needs no predicate on L
    for (int k = threadIdx.x; k < kc; k += STREAM_THREADS) {
        int ia = 0, ib = -1;
        const bool in = k < klen;
        if (in) decode_k(d, ca, cb, k0 + k, ia, ib);
#pragma unroll
        for (int r = 0; r < RT; ++r) {
            const int rr = p.r0 + r;
            T l = T(0);
            if (in && rr < R) {
                l = __ldg(f + (long long)rr * fstride + ia);
                if (ib >= 0) l *= __ldg(f + (long long)rr * fstride + ib);
            }
            Lt[r * ls + k] = l;
        }
    }
    __syncthreads();

    // a2: stream the rows
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    constexpr int NWARPS = STREAM_THREADS / 32;
    const int nvec = (klen + VEC - 1) / VEC;  // VEC > 1 implies padded, 16-byte aligned rows
    const T* __restrict__ base = reinterpret_cast<const T*>(d.fk) + k0;

    for (int row = rb + warp * RPW; row < re; row += NWARPS * RPW) {
        const T* rp[RPW];
#pragma unroll
        for (int q = 0; q < RPW; ++q) rp[q] = base + (long long)min(row + q, re - 1) * d.row_stride;

        T acc[RPW][RT][VEC];
#pragma unroll
        for (int q = 0; q < RPW; ++q)
#pragma unroll
            for (int r = 0; r < RT; ++r)
#pragma unroll
                for (int e = 0; e < VEC; ++e) acc[q][r][e] = T(0);

        int v = lane;
        for (; v + 32 * (UNROLL - 1) < nvec; v += 32 * UNROLL) {
            V x[RPW][UNROLL];
#pragma unroll
            for (int u = 0; u < UNROLL; ++u)
#pragma unroll
                for (int q = 0; q < RPW; ++q) x[q][u] = ld_stream(rp[q] + (v + 32 * u) * VEC, (V*)nullptr);
#pragma unroll
            for (int u = 0; u < UNROLL; ++u)
#pragma unroll
                for (int r = 0; r < RT; ++r) {
                    const V l = *reinterpret_cast<const V*>(Lt + r * ls + (v + 32 * u) * VEC);
#pragma unroll
                    for (int q = 0; q < RPW; ++q)
#pragma unroll
                        for (int e = 0; e < VEC; ++e) acc[q][r][e] = fma(x[q][u].v[e], l.v[e], acc[q][r][e]);
                }
        }
        if (v < nvec) {  // ragged tail of the chunk: same shape, loads clamped, L zeroed past the end
            V x[RPW][UNROLL];
#pragma unroll
            for (int u = 0; u < UNROLL; ++u) {
                const int vv = min(v + 32 * u, nvec - 1);
#pragma unroll
                for (int q = 0; q < RPW; ++q) x[q][u] = ld_stream(rp[q] + vv * VEC, (V*)nullptr);
            }
#pragma unroll
            for (int u = 0; u < UNROLL; ++u) {
                const bool ok = v + 32 * u < nvec;
                const int vv = min(v + 32 * u, nvec - 1);
#pragma unroll
                for (int r = 0; r < RT; ++r) {
                    V l = *reinterpret_cast<const V*>(Lt + r * ls + vv * VEC);
#pragma unroll
                    for (int q = 0; q < RPW; ++q)
#pragma unroll
                        for (int e = 0; e < VEC; ++e)
                            acc[q][r][e] = fma(x[q][u].v[e], ok ? l.v[e] : T(0), acc[q][r][e]);
                }
            }
        }

        // a3 level 1: lane partials -> one value per (row, replica), fixed butterfly
#pragma unroll
        for (int q = 0; q < RPW; ++q)
#pragma unroll
            for (int r = 0; r < RT; ++r) {
                double s = (double)acc[q][r][0];
#pragma unroll
                for (int e = 1; e < VEC; ++e) s += (double)acc[q][r][e];
                s = warp_sum(s);
                const int n = row + q, rr = p.r0 + r;
                if (lane == 0 && n < re && rr < R) {
                    if (d.nchunks == 1)
                        reinterpret_cast<T*>(p.sigma)[d.out_off * R + (long long)n * R + rr] = (T)s;
                    else
                        p.part[d.part_off * R + ((long long)n * R + rr) * d.nchunks + chunk] = s;
                }
            }
    }
}

template <typename T, int VEC, int RT, int RPW, int UNROLL, bool GROUPED>
__global__ void __launch_bounds__(STREAM_THREADS)
fk_stream_kernel(const __grid_constant__ StreamParams p) {
    extern __shared__ __align__(16) unsigned char fk_smem[];
    T* Lt = reinterpret_cast<T*>(fk_smem);
    if constexpr (!GROUPED) {
        const long long u0 = p.units * blockIdx.x / gridDim.x;
        const long long u1 = p.units * (blockIdx.x + 1) / gridDim.x;
        if (u0 >= u1) return;
        const int N = p.desc.N;
        const int c0 = (int)(u0 / N), c1 = (int)((u1 - 1) / N);
        for (int chunk = c0; chunk <= c1; ++chunk) {
            const long long lo = (long long)chunk * N;
            const int rb = (int)(max(u0, lo) - lo);
            const int re = (int)(min(u1, lo + N) - lo);
            stream_segment<T, VEC, RT, RPW, UNROLL>(p.desc, p.chan.a, p.chan.b, chunk, rb, re, p, Lt);
        }
    } else {
        const int s0 = p.cta_seg_start[blockIdx.x], s1 = p.cta_seg_start[blockIdx.x + 1];
        for (int s = s0; s < s1; ++s) {
            const Segment sg = p.segs[s];
            const TableDesc& d = p.descs[sg.table];
            stream_segment<T, VEC, RT, RPW, UNROLL>(d, d.chan_a, d.chan_b, sg.chunk, sg.row_begin, sg.row_end, p, Lt);
        }
    }
}

// ---- a3 level 2: sigma[n][r] = sum over chunks, fixed order (lane-strided chains + butterfly) ----
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
        if (nch == 1) continue;  // written directly by the stream kernel
        const double* src = p.part + d->part_off * p.R + (n * p.R + r) * nch;
        double s = 0.0;
        for (int c = lane; c < nch; c += 32) s += src[c];
        s = warp_sum(s);
        if (lane == 0) reinterpret_cast<T*>(p.sigma)[d->out_off * p.R + n * p.R + r] = (T)s;
    }
}

}  // namespace fk
