// fk_vjp.cuh -- gradient of the convolution as a VJP, minimal-flop order:
//
//   stage 1 (one FK pass, bandwidth-bound):  G[r][k] = sum_n g[n][r] * FK[n][k]
//   stage 2 (tiny, gather form, no atomics): df[r][alpha][i] =
//        sum_{c: a_c = alpha} sum_j G[r][k(i,j,c)] * f[r][b_c][j]
//      + sum_{c: b_c = alpha} sum_j G[r][k(j,i,c)] * f[r][a_c][j]          (hadronic; the a_c == b_c,
//        i == j diagonal gets both terms because both sums visit it)
//      DIS: df[r][alpha][i] = sum_{c: flav_c = alpha} G[r][k(i,c)]
//
// Stage 1: a thread owns VEC consecutive k and walks down the datapoints of its split with UNROLL
// independent 128-bit loads in flight; no cross-thread reduction at all.  Datapoints are cut into
// `nsplit` fixed ranges for parallelism; stage 2 adds the splits in a fixed order.
#pragma once

#include "fk_common.cuh"

namespace fk {

struct ColsumParams {
    TableDesc desc;           // single-table launch
    const TableDesc* descs;   // grouped (device)
    const ColSeg* segs;    // grouped (device), one per CTA
    const void* g;            // g[N][R] or g_cat
    double* G;                // [nsplit][R][K] per table
    int R, r0;
    int nkb;                  // single: k-blocks per split
};

constexpr int COLSUM_THREADS = 256;
constexpr int COLSUM_MAX_ROWS = 512;  // datapoints per split (bounds the g tile in shared memory)

template <typename T, int VEC, int RT, int UNROLL, bool GROUPED, typename TS = T>
__global__ void __launch_bounds__(COLSUM_THREADS, RT == 1 ? 4 : 1)   // R = 1: at most 64 registers, four CTAs per SM
fk_colsum_kernel(const __grid_constant__ ColsumParams p) {
    pdl_trigger();
    pdl_wait();
    using V = Vec<TS, VEC>;
    constexpr int NACC = (RT == 1) ? 4 : 2;
    __shared__ T gs[(COLSUM_MAX_ROWS + UNROLL) * RT];

    const TableDesc* dp = &p.desc;
    int kblock, split;
    if constexpr (GROUPED) {
        const ColSeg sg = p.segs[blockIdx.x];
        dp = &p.descs[sg.table];
        kblock = sg.kblock;
        split = sg.split;
    } else {
        kblock = blockIdx.x % p.nkb;
        split = blockIdx.x / p.nkb;
    }
    const TableDesc& d = *dp;
    const int R = p.R;
    const int rb = (int)((long long)d.N * split / d.nsplit);
    const int re = (int)((long long)d.N * (split + 1) / d.nsplit);
    const int rows = re - rb;

    // g tile [rows rounded up to UNROLL][RT], zero padded
    const T* __restrict__ g = reinterpret_cast<const T*>(p.g) + d.out_off * R;
    const int rows_pad = (rows + UNROLL - 1) / UNROLL * UNROLL;
    for (int t = threadIdx.x; t < rows_pad * RT; t += COLSUM_THREADS) {
        const int m = t / RT, r = t - m * RT;
        const int rr = p.r0 + r;
        gs[t] = (m < rows && rr < R) ? __ldg(g + (long long)(rb + m) * R + rr) : T(0);
    }
    __syncthreads();

    const int k = (kblock * COLSUM_THREADS + threadIdx.x) * VEC;
    if (k >= d.K) return;
    const TS* __restrict__ col = reinterpret_cast<const TS*>(d.fk) + k;

    T acc[NACC][RT][VEC];
#pragma unroll
    for (int a = 0; a < NACC; ++a)
#pragma unroll
        for (int r = 0; r < RT; ++r)
#pragma unroll
            for (int e = 0; e < VEC; ++e) acc[a][r][e] = T(0);

    for (int m = 0; m < rows_pad; m += UNROLL) {
        V x[UNROLL];
#pragma unroll
        for (int u = 0; u < UNROLL; ++u)
            x[u] = ld_stream(col + (long long)(rb + min(m + u, rows - 1)) * d.row_stride, (V*)nullptr);
#pragma unroll
        for (int u = 0; u < UNROLL; ++u)
#pragma unroll
            for (int r = 0; r < RT; ++r) {
                const T gv = gs[(m + u) * RT + r];  // broadcast; 0 on the padded rows
#pragma unroll
                for (int e = 0; e < VEC; ++e)
                    acc[u % NACC][r][e] = fma(gv, (T)x[u].v[e], acc[u % NACC][r][e]);
            }
    }

    double* __restrict__ G = p.G + d.g_off * R;
#pragma unroll
    for (int r = 0; r < RT; ++r) {
        const int rr = p.r0 + r;
        if (rr >= R) continue;
#pragma unroll
        for (int e = 0; e < VEC; ++e) {
            if (k + e >= d.K) continue;
            double s = (double)acc[0][r][e];
#pragma unroll
            for (int a = 1; a < NACC; ++a) s += (double)acc[a][r][e];
            G[((long long)split * R + rr) * d.K + k + e] = s;
        }
    }
}

// ---- stage 2: one CTA per (table, alpha, i), replicas on blockIdx.y -----------------------------
struct GatherParams {
    TableDesc desc;           // single
    ChannelList chan;         // single
    const TableDesc* descs;   // grouped (device)
    const int* ai_prefix;     // grouped (device) [T+1]: first (alpha, i) slot of each table
    int T;
    const void* f;
    const double* G;
    void* df;
    int R;
};

constexpr int GATHER_THREADS = 128;

template <typename T, bool GROUPED>
__global__ void __launch_bounds__(GATHER_THREADS)
fk_vjp_gather_kernel(const __grid_constant__ GatherParams p) {
    __shared__ short listA[MAX_C], listB[MAX_C];
    __shared__ int cnt[2];
    __shared__ double wsum[GATHER_THREADS / 32];

    const TableDesc* dp = &p.desc;
    const uint8_t* __restrict__ ca = p.chan.a;
    const uint8_t* __restrict__ cb = p.chan.b;
    int slot = blockIdx.x;
    if constexpr (GROUPED) {
        int lo = 0, hi = p.T;
        while (hi - lo > 1) {
            const int mid = (lo + hi) >> 1;
            if (p.ai_prefix[mid] <= slot) lo = mid; else hi = mid;
        }
        dp = &p.descs[lo];
        slot -= p.ai_prefix[lo];
        ca = dp->chan_a;
        cb = dp->chan_b;
    }
    const TableDesc& d = *dp;
    const int nx = d.nx, C = d.C, R = p.R;
    const int alpha = slot / nx, i = slot - alpha * nx;
    const int r = blockIdx.y;
    const bool had = d.kind == KIND_HADRONIC;

    if (threadIdx.x == 0) {  // channel lists of this flavour, in channel order (fixed)
        int na = 0, nb = 0;
        for (int c = 0; c < C; ++c) {
            if (ca[c] == alpha) listA[na++] = (short)c;
            if (had && cb[c] == alpha) listB[nb++] = (short)c;
        }
        cnt[0] = na;
        cnt[1] = nb;
    }
    __syncthreads();
    const int na = cnt[0], nb = cnt[1];

    const T* __restrict__ f = reinterpret_cast<const T*>(p.f) + d.f_off * R + (long long)r * d.nfl * nx;
    const double* __restrict__ G = p.G + d.g_off * R + (long long)r * d.K;
    const long long split_stride = (long long)R * d.K;
    const int nsplit = d.nsplit;

    double acc = 0.0;
    if (had) {
        const int items = (na + nb) * nx;
        for (int t = threadIdx.x; t < items; t += GATHER_THREADS) {
            const int q = t / nx, j = t - q * nx;
            int k, fo;
            if (q < na) {
                const int c = listA[q];
                k = encode_k(d, i, j, c);
                fo = (int)cb[c] * nx + j;
            } else {
                const int c = listB[q - na];
                k = encode_k(d, j, i, c);
                fo = (int)ca[c] * nx + j;
            }
            double gk = 0.0;
            for (int s = 0; s < nsplit; ++s) gk += G[s * split_stride + k];
            acc = fma(gk, (double)f[fo], acc);
        }
    } else {
        for (int t = threadIdx.x; t < na; t += GATHER_THREADS) {
            const int k = encode_k(d, i, 0, listA[t]);
            double gk = 0.0;
            for (int s = 0; s < nsplit; ++s) gk += G[s * split_stride + k];
            acc += gk;
        }
    }
    acc = warp_sum(acc);
    if ((threadIdx.x & 31) == 0) wsum[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = wsum[0];
#pragma unroll
        for (int w = 1; w < GATHER_THREADS / 32; ++w) s += wsum[w];
        reinterpret_cast<T*>(p.df)[d.f_off * R + ((long long)r * d.nfl + alpha) * nx + i] = (T)s;
    }
}

// ---- stage 2 for hadronic tables, small R: one pass over the column sums, both legs at once -----------
//   A[r][c][i] = sum_j G[r][k(i,j,c)] f[r][b_c][j]      B[r][c][j] = sum_i G[r][k(i,j,c)] f[r][a_c][i]
//   df[r][alpha][x] = sum_{c: a_c = alpha} A[r][c][x] + sum_{c: b_c = alpha} B[r][c][x]
// fk_vjp_foldk_kernel: CTA = (channel, replica).  The channel's nx x nx block of G (the datapoint splits added
// in a fixed order) goes to shared memory with coalesced loads, rows padded to an odd stride; thread x < nx
// then sums row x (A) and thread nx + x sums column x (B), each a sequential chain in index order.  The gather
// kernel above reads G twice with a stride and rebuilds the channel lists in every CTA; it stays for DIS.
struct FoldKParams {
    TableDesc desc;           // single
    ChannelList chan;         // single
    const TableDesc* descs;   // grouped (device)
    const ColSeg* items;      // grouped fold launch: {table, kblock = channel}
    const int* ai_prefix;     // grouped final launch [T+1]
    int T;
    const void* f;
    const double* G;
    double* PA;               // [R][cx_total]: (cx_off + c*nx + x)
    double* PB;               // [R][nchunk][cx_total]
    long long cx_total;
    int nchunk;               // x-row chunks per channel (B partials per chunk)
    void* df;
    int R;
};

constexpr int FOLDK_THREADS = 256;

template <typename T, bool GROUPED>
__global__ void __launch_bounds__(FOLDK_THREADS)
fk_vjp_foldk_kernel(const __grid_constant__ FoldKParams p) {
    pdl_trigger();
    pdl_wait();   // the column sums G of the whole stage-1 grid
    extern __shared__ __align__(128) unsigned char fk_smem[];
    double* Gs = reinterpret_cast<double*>(fk_smem);  // [nx][nx | 1]
    const TableDesc* dp = &p.desc;
    const uint8_t* __restrict__ ca = p.chan.a;
    const uint8_t* __restrict__ cb = p.chan.b;
    int c = blockIdx.x / p.nchunk;
    const int chunk = blockIdx.x % p.nchunk;
    if constexpr (GROUPED) {
        const ColSeg it = p.items[c];
        dp = &p.descs[it.table];
        ca = dp->chan_a;
        cb = dp->chan_b;
        c = it.kblock;
    }
    const TableDesc& d = *dp;
    const int nx = d.nx, R = p.R, r = blockIdx.y, ld = nx | 1;
    const int i0 = (int)((long long)nx * chunk / p.nchunk), i1 = (int)((long long)nx * (chunk + 1) / p.nchunk);
    const double* __restrict__ G = p.G + d.g_off * R + (long long)r * d.K;
    const long long split_stride = (long long)R * d.K;
    for (int t = threadIdx.x + i0 * nx; t < i1 * nx; t += FOLDK_THREADS) {
        const int i = t / nx, j = t - i * nx;
        const int k = encode_k(d, i, j, c);
        double v = 0.0;
        for (int s0 = 0; s0 < d.nsplit; s0 += 8) {  // eight independent loads in flight, added in index order
            double w[8];
#pragma unroll
            for (int q = 0; q < 8; ++q) w[q] = s0 + q < d.nsplit ? G[(long long)(s0 + q) * split_stride + k] : 0.0;
#pragma unroll
            for (int q = 0; q < 8; ++q) v += w[q];
        }
        Gs[(i - i0) * ld + j] = v;
    }
    __syncthreads();
    const T* __restrict__ f = reinterpret_cast<const T*>(p.f) + d.f_off * R + (long long)r * d.nfl * nx;
    const long long o = (long long)r * p.cx_total + d.cx_off + (long long)c * nx;
    const int ni = i1 - i0;
    for (int t = threadIdx.x; t < ni + nx; t += FOLDK_THREADS) {
        double acc = 0.0;
        if (t < ni) {
            const T* fb = f + (int)cb[c] * nx;
            for (int j = 0; j < nx; ++j) acc = fma(Gs[t * ld + j], (double)fb[j], acc);
            p.PA[o + i0 + t] = acc;
        } else {
            const int x = t - ni;
            const T* fa = f + (int)ca[c] * nx + i0;
            for (int i = 0; i < ni; ++i) acc = fma(Gs[i * ld + x], (double)fa[i], acc);
            p.PB[o + ((long long)r * (p.nchunk - 1) + chunk) * p.cx_total + x] = acc;
        }
    }
}

// one warp per (PDF slot, replica): lane l adds the channels l, l + 32, ... of this flavour in index order, then a
// fixed xor butterfly
template <typename T, bool GROUPED>
__global__ void __launch_bounds__(256)
fk_vjp_foldk_final_kernel(const __grid_constant__ FoldKParams p, long long slots_total) {
    pdl_wait();   // PA / PB of the whole fold grid
    const long long gs = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (gs >= slots_total) return;
    const TableDesc* dp = &p.desc;
    const uint8_t* __restrict__ ca = p.chan.a;
    const uint8_t* __restrict__ cb = p.chan.b;
    int slot = (int)gs;
    if constexpr (GROUPED) {
        int lo = 0, hi = p.T;
        while (hi - lo > 1) {
            const int mid = (lo + hi) >> 1;
            if (p.ai_prefix[mid] <= gs) lo = mid; else hi = mid;
        }
        dp = &p.descs[lo];
        slot = (int)(gs - p.ai_prefix[lo]);
        ca = dp->chan_a;
        cb = dp->chan_b;
    }
    const TableDesc& d = *dp;
    const int nx = d.nx, R = p.R, r = blockIdx.y;
    const int alpha = slot / nx, x = slot - alpha * nx;
    const double* __restrict__ PA = p.PA + (long long)r * p.cx_total + d.cx_off + x;
    const double* __restrict__ PB = p.PB + (long long)r * p.nchunk * p.cx_total + d.cx_off + x;
    double s = 0.0;
    for (int c = lane; c < d.C; c += 32) {
        if (ca[c] == alpha) s += PA[c * nx];
        if (cb[c] == alpha)
            for (int ch = 0; ch < p.nchunk; ++ch) s += PB[ch * p.cx_total + c * nx];
    }
    s = warp_sum(s);
    if (lane == 0) reinterpret_cast<T*>(p.df)[d.f_off * R + ((long long)r * d.nfl + alpha) * nx + x] = (T)s;
}

}  // namespace fk
