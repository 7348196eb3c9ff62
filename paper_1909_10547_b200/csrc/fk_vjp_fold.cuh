// fk_vjp_fold.cuh -- VJP stage 2 for R >> 1 on PACKED hadronic tables: ONE streaming pass
// over the replica-innermost column sums G[k][r] (k = c*cstride + i*nx + j) that serves both legs of the
// derivative of Eq. (1):
//
//   A[c][i][r] = sum_j G[(c,i,j)][r] * f[r][b_c][j]        -> df[r][a_c][i]
//   B[c][j][r] = sum_i G[(c,i,j)][r] * f[r][a_c][i]        -> df[r][b_c][j]
//   df[r][alpha][x] = sum_{c: a_c = alpha} A[c][x][r] + sum_{c: b_c = alpha} B[c][x][r]
//
// fk_vjp_fold_kernel: CTA = (channel c, chunk of x-rows i); 256 threads = 4 j-classes (j mod 4) x 64 replica
// pairs.  A thread walks its rows i, loads its <= 16 values of j as independent 128-bit streaming loads (the
// CTA reads every (c, i) row of G as one contiguous nx*RP*8-byte piece), keeps f[b_c][j] and the B sums of
// its j in registers, and writes one A partial per (i, j-class) and one B partial per (chunk, j).  No shared
// memory, no barrier, no atomics; every G element is read exactly once (the gather form reads it twice
// with a stride).  fk_vjp_fold_final_kernel adds the partials of a PDF slot in a fixed order.
#pragma once

#include "fk_common.cuh"
#include "fk_gemm.cuh"

namespace fk {

constexpr int FOLD_THREADS = 256;
constexpr int FOLD_JQ = 4;        // j-classes (threadIdx.x >> 6)
constexpr int FOLD_NXQ = 16;      // j values per thread: supports nx <= 64
constexpr int FOLD_MAX_NX = FOLD_JQ * FOLD_NXQ;

struct FoldParams {
    TableDesc desc;        // single-table launch
    ChannelList chan;      // single-table launch
    const double* fT;      // [slots][RP] replica-innermost f (grouped: + f_off * RP)
    const double* G;       // [K][RP] (grouped: + k_off * RP)
    double* PA;            // [(cx_off + c*nx + i)][FOLD_JQ][RP]
    double* PB;            // [(cx_off + c*nx) * nchunk + chunk*nx + j][RP]
    void* df;              // final kernel: [R][nfl][nx] (grouped: + f_off * R)
    int R, r0, RP, nchunk;
    const TableDesc* descs;  // grouped launch
    const ColSeg* items;     // grouped fold launch: {table, kblock = channel, split = chunk}
    const int* ai_prefix;    // grouped final launch: first (alpha, x) slot of each table
    int T;
};

__device__ __forceinline__ double2 ld_stream2(const double* p) {
    double2 r;
    asm volatile("ld.global.nc.L1::no_allocate.v2.f64 {%0, %1}, [%2];" : "=d"(r.x), "=d"(r.y) : "l"(p));
    return r;
}

template <bool GROUPED>
__global__ void __launch_bounds__(FOLD_THREADS)
fk_vjp_fold_kernel(const __grid_constant__ FoldParams p) {
    const TableDesc* dp = &p.desc;
    const uint8_t* __restrict__ ca = p.chan.a;
    const uint8_t* __restrict__ cb = p.chan.b;
    const double* __restrict__ fT = p.fT;
    const double* __restrict__ G = p.G;
    int c, chunk;
    if constexpr (GROUPED) {
        const ColSeg it = p.items[blockIdx.x];
        dp = &p.descs[it.table];
        ca = dp->chan_a;
        cb = dp->chan_b;
        fT += dp->f_off * p.RP;
        G += dp->k_off * p.RP;
        c = it.kblock;
        chunk = it.split;
    } else {
        c = blockIdx.x / p.nchunk;
        chunk = blockIdx.x - c * p.nchunk;
    }
    const TableDesc& d = *dp;
    const int nx = d.nx, RP = p.RP;
    const int col = 2 * (threadIdx.x & 63), jq = threadIdx.x >> 6;
    if (col >= RP) return;
    const int i0 = (int)((long long)nx * chunk / p.nchunk), i1 = (int)((long long)nx * (chunk + 1) / p.nchunk);

    double2 fb[FOLD_NXQ], sb[FOLD_NXQ];
    {
        const double* src = fT + ((long long)cb[c] * nx + jq) * RP + col;
#pragma unroll
        for (int m = 0; m < FOLD_NXQ; ++m) {
            fb[m] = jq + FOLD_JQ * m < nx ? *reinterpret_cast<const double2*>(src + (long long)FOLD_JQ * m * RP) : make_double2(0.0, 0.0);
            sb[m] = make_double2(0.0, 0.0);
        }
    }
    const double* __restrict__ fa_col = fT + (long long)ca[c] * nx * RP + col;
    const double* __restrict__ Gc = G + ((long long)c * d.cstride + jq) * RP + col;
    const long long cx = d.cx_off + (long long)c * nx;
    double* __restrict__ PA = p.PA + (cx * FOLD_JQ + jq) * RP + col;

    for (int i = i0; i < i1; ++i) {
        const double* row = Gc + (long long)i * nx * RP;
        double2 v[FOLD_NXQ];
#pragma unroll
        for (int m = 0; m < FOLD_NXQ; ++m)
            v[m] = jq + FOLD_JQ * m < nx ? ld_stream2(row + (long long)FOLD_JQ * m * RP) : make_double2(0.0, 0.0);
        const double2 fa = *reinterpret_cast<const double2*>(fa_col + (long long)i * RP);
        double2 s = make_double2(0.0, 0.0);
#pragma unroll
        for (int m = 0; m < FOLD_NXQ; ++m) {
            s.x = fma(v[m].x, fb[m].x, s.x);
            s.y = fma(v[m].y, fb[m].y, s.y);
            sb[m].x = fma(v[m].x, fa.x, sb[m].x);
            sb[m].y = fma(v[m].y, fa.y, sb[m].y);
        }
        *reinterpret_cast<double2*>(PA + (long long)i * FOLD_JQ * RP) = s;
    }
    double* __restrict__ PB = p.PB + ((cx * p.nchunk + (long long)chunk * nx) + jq) * RP + col;
#pragma unroll
    for (int m = 0; m < FOLD_NXQ; ++m)
        if (jq + FOLD_JQ * m < nx) *reinterpret_cast<double2*>(PB + (long long)FOLD_JQ * m * RP) = sb[m];
}

// one CTA per PDF slot (alpha, x), one thread per replica of the pass: channels in list order, partials in index
// order.  The channels of this flavour are compacted into shared memory first so that the partial loads of
// FOLD_FU channels are independent and in flight together.
constexpr int FOLD_FU = 4;

template <typename T, bool GROUPED>
__global__ void __launch_bounds__(GEMM_BN)
fk_vjp_fold_final_kernel(const __grid_constant__ FoldParams p) {
    __shared__ short listA[MAX_C], listB[MAX_C];
    __shared__ int cnt[2];
    const TableDesc* dp = &p.desc;
    const uint8_t* __restrict__ ca = p.chan.a;
    const uint8_t* __restrict__ cb = p.chan.b;
    int slot = blockIdx.x;
    if constexpr (GROUPED) {
        const int tb = table_of(p.ai_prefix, p.T, slot);
        dp = &p.descs[tb];
        slot -= p.ai_prefix[tb];
        ca = dp->chan_a;
        cb = dp->chan_b;
    }
    const TableDesc& d = *dp;
    const int nx = d.nx, RP = p.RP, nchunk = p.nchunk;
    const int alpha = slot / nx, x = slot - alpha * nx;
    if (threadIdx.x < 32) {  // warp 0: ordered compaction by ballot
        int na = 0, nb = 0;
        for (int c0 = 0; c0 < d.C; c0 += 32) {
            const int c = c0 + threadIdx.x;
            const bool ma = c < d.C && ca[c] == alpha, mb = c < d.C && cb[c] == alpha;
            const unsigned ba = __ballot_sync(0xffffffffu, ma), bb = __ballot_sync(0xffffffffu, mb);
            const unsigned below = (1u << threadIdx.x) - 1u;
            if (ma) listA[na + __popc(ba & below)] = (short)c;
            if (mb) listB[nb + __popc(bb & below)] = (short)c;
            na += __popc(ba);
            nb += __popc(bb);
        }
        if (threadIdx.x == 0) { cnt[0] = na; cnt[1] = nb; }
    }
    __syncthreads();
    const int col = threadIdx.x;
    if (col >= RP || p.r0 + col >= p.R) return;
    const int na = cnt[0], nb = cnt[1];
    double s = 0.0;
    for (int q0 = 0; q0 < na; q0 += FOLD_FU) {
        double t[FOLD_FU][FOLD_JQ];
#pragma unroll
        for (int u = 0; u < FOLD_FU; ++u) {
            const int c = listA[min(q0 + u, na - 1)];
            const double* q = p.PA + (d.cx_off + (long long)c * nx + x) * FOLD_JQ * RP + col;
#pragma unroll
            for (int e = 0; e < FOLD_JQ; ++e) t[u][e] = q[e * RP];
        }
#pragma unroll
        for (int u = 0; u < FOLD_FU; ++u)
            if (q0 + u < na) s += (t[u][0] + t[u][1]) + (t[u][2] + t[u][3]);
    }
    for (int q0 = 0; q0 < nb; q0 += FOLD_FU) {
        double t[FOLD_FU];
#pragma unroll
        for (int u = 0; u < FOLD_FU; ++u) {
            const int c = listB[min(q0 + u, nb - 1)];
            const double* q = p.PB + ((d.cx_off + (long long)c * nx) * nchunk + x) * RP + col;
            double v = q[0];
            for (int ch = 1; ch < nchunk; ++ch) v += q[(long long)ch * nx * RP];
            t[u] = v;
        }
#pragma unroll
        for (int u = 0; u < FOLD_FU; ++u)
            if (q0 + u < nb) s += t[u];
    }
    reinterpret_cast<T*>(p.df)[d.f_off * p.R + ((long long)(p.r0 + col) * d.nfl + alpha) * nx + x] = (T)s;
}

}  // namespace fk
