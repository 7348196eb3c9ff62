// fk_vjp_fold.cuh -- VJP stage 2 for R >> 1 on PACKED hadronic tables: ONE streaming pass
// over the replica-innermost column sums G[k][r] (k = c*cstride + i*nx + j) that serves both legs of the
// derivative of Eq. (1):
//
//   A[c][i][r] = sum_j G[(c,i,j)][r] * f[r][b_c][j]        -> df[r][a_c][i]
//   B[c][j][r] = sum_i G[(c,i,j)][r] * f[r][a_c][i]        -> df[r][b_c][j]
//   df[r][alpha][x] = sum_{c: a_c = alpha} A[c][x][r] + sum_{c: b_c = alpha} B[c][x][r]
//
// fk_vjp_fold_kernel: CTA = (channel c, chunk of x-rows i); 256 threads = 4 j-classes (j mod 4) x 64 replica
// pairs.  Every (c, i) row of G is one contiguous nx*RP*8-byte piece: it arrives in a shared-memory ring by ONE
// bulk async copy (cp.async.bulk, mbarrier completion), several rows ahead of the threads that use it.  A
// thread keeps f[b_c][j] and the B sums of its <= 16 values of j in registers and writes one A partial per
// (i, j-class) and one B partial per (chunk, j).  No atomics; every G element crosses HBM exactly once (the
// gather form reads it twice with a stride).  fk_vjp_fold_final_kernel adds the partials of a PDF slot in a fixed order.
#pragma once

#include "fk_common.cuh"
#include "fk_gemm.cuh"
#include "fk_gemm_ws.cuh"

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
    int nslots;            // fold kernel: rows of G in the shared-memory ring (>= 2)
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

// shared memory: a ring of FOLD_SLOTS (c, i) rows of G ([nx][RP] doubles each) + 2 mbarriers per slot
constexpr int FOLD_MAX_SLOTS = 4;
__host__ __device__ inline int fold_slots(int nx, int RP, size_t max_bytes) {
    const size_t row = (size_t)nx * RP * 8;
    int s = (int)((max_bytes - 2 * FOLD_MAX_SLOTS * 8) / row);
    return s > FOLD_MAX_SLOTS ? FOLD_MAX_SLOTS : s;
}

template <bool GROUPED>
__global__ void __launch_bounds__(FOLD_THREADS)
fk_vjp_fold_kernel(const __grid_constant__ FoldParams p) {
    extern __shared__ __align__(128) unsigned char fk_smem[];
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
    const int nx = d.nx, RP = p.RP, S = p.nslots;
    const int col = 2 * (threadIdx.x & 63), jq = threadIdx.x >> 6, lane = threadIdx.x & 31;
    const int i0 = (int)((long long)nx * chunk / p.nchunk), i1 = (int)((long long)nx * (chunk + 1) / p.nchunk);
    const uint32_t row_bytes = (uint32_t)(nx * RP * 8);

    // ring of (c, i) rows: each row of G is ONE contiguous piece, fetched by one bulk copy that completes on the
    // slot's mbarrier; up to S rows are in flight per SM whatever the consumers do
    double* ring = reinterpret_cast<double*>(fk_smem);
    const uint32_t ring_s = (uint32_t)__cvta_generic_to_shared(ring);
    const uint32_t bar0 = ring_s + (uint32_t)S * row_bytes;
    auto bar_full = [&](int s) { return bar0 + 8u * s; };
    auto bar_empty = [&](int s) { return bar0 + 8u * (FOLD_MAX_SLOTS + s); };
    if (threadIdx.x == 0) {
        for (int s = 0; s < S; ++s) {
            mbar_init(bar_full(s), 1);
            mbar_init(bar_empty(s), FOLD_THREADS / 32);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const double* __restrict__ Gc = G + (long long)c * d.cstride * RP;
    auto issue = [&](int i) {  // thread 0 only: row i -> slot (i - i0) % S
        const int q = i - i0, s = q % S;
        mbar_wait(bar_empty(s), ((q / S) & 1) ^ 1);
        mbar_expect_tx(bar_full(s), row_bytes);
        bulk_g2s(ring_s + (uint32_t)s * row_bytes, Gc + (long long)i * d.jp * RP, row_bytes, bar_full(s));   // x-rows are jp apart (fp32 tables pad them)
    };
    if (threadIdx.x == 0)
        for (int i = i0; i < min(i1, i0 + S - 1); ++i) issue(i);

    const bool active = col < RP;
    double2 fb[FOLD_NXQ], sb[FOLD_NXQ];
    {
        const double* src = fT + ((long long)cb[c] * nx + jq) * RP + col;
#pragma unroll
        for (int m = 0; m < FOLD_NXQ; ++m) {
            fb[m] = (active && jq + FOLD_JQ * m < nx) ? *reinterpret_cast<const double2*>(src + (long long)FOLD_JQ * m * RP) : make_double2(0.0, 0.0);
            sb[m] = make_double2(0.0, 0.0);
        }
    }
    const double* __restrict__ fa_col = fT + (long long)ca[c] * nx * RP + col;
    const long long cx = d.cx_off + (long long)c * nx;
    double* __restrict__ PA = p.PA + (cx * FOLD_JQ + jq) * RP + col;

    // f[a_c][i] of the next row is fetched one row ahead: the L2 round trip is off the per-row critical path
    double2 fa_next = active ? *reinterpret_cast<const double2*>(fa_col + (long long)i0 * RP) : make_double2(0.0, 0.0);
    for (int i = i0; i < i1; ++i) {
        const int q = i - i0, s = q % S;
        if (threadIdx.x == 0 && i + S - 1 < i1) issue(i + S - 1);  // its slot was left by every warp after row i - 1
        __syncwarp();
        const double2 fa = fa_next;
        if (active && i + 1 < i1) fa_next = *reinterpret_cast<const double2*>(fa_col + (long long)(i + 1) * RP);
        mbar_wait(bar_full(s), (q / S) & 1);
        if (active) {
            const double* row = ring + (size_t)s * nx * RP + jq * RP + col;
            double2 a = make_double2(0.0, 0.0);
#pragma unroll
            for (int m = 0; m < FOLD_NXQ; ++m) {
                if (jq + FOLD_JQ * m < nx) {
                    const double2 v = *reinterpret_cast<const double2*>(row + FOLD_JQ * m * RP);
                    a.x = fma(v.x, fb[m].x, a.x);
                    a.y = fma(v.y, fb[m].y, a.y);
                    sb[m].x = fma(v.x, fa.x, sb[m].x);
                    sb[m].y = fma(v.y, fa.y, sb[m].y);
                }
            }
            *reinterpret_cast<double2*>(PA + (long long)i * FOLD_JQ * RP) = a;
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_empty(s));
    }
    if (active) {
        double* __restrict__ PB = p.PB + ((cx * p.nchunk + (long long)chunk * nx) + jq) * RP + col;
#pragma unroll
        for (int m = 0; m < FOLD_NXQ; ++m)
            if (jq + FOLD_JQ * m < nx) *reinterpret_cast<double2*>(PB + (long long)FOLD_JQ * m * RP) = sb[m];
    }
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
