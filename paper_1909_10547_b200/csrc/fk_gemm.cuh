// fk_gemm.cuh -- R >> 1 dense contraction (the paper's flat view FK[N x K] . PDF[K x R],
// PAPER.md:83-100) on the FP64 tensor-core path (mma.sync.m8n8k4.f64 = DMMA.8x8x4), fp64 only.
//
//   Sigma[n][r] = sum_k FK[n][k] * L[k][r],   L[k][r] = f[r][a_c][i] * f[r][b_c][j]     Eq. (1)
//
// The output is tiny (N x R) and K is huge, so all parallelism is split-K: CTA = (128-datapoint tile,
// K range).  Per K-tile of 32:
//   * the FK tile [128 n][32 k] streams global -> shared with 16-byte cp.async, 3 stages deep
//     (FK is read exactly once: every (n, k) belongs to one CTA);
//   * the luminosity tile L[32 k][<=128 r] is BUILT ON THE FLY from the replica-innermost copy fT of f
//     (gathered through the table's k -> (slot a, slot b) codes), one K-tile ahead in registers, and put
//     in shared memory; it never exists in HBM (the custom operator's memory saving);
//   * 8 warps (4 along n x 2 along r) run DMMA on 32 x (8..64) warp tiles; the +4 padding of both
//     shared tiles makes every fragment load conflict-free.
// Level 1 writes one partial tile per K range; fk_gemm_reduce_kernel adds the ranges in a fixed order:
// no atomics, bitwise repeatable.  B200 has the same FP64 peak on DFMA and DMMA (37.2 TFLOP/s,
// profiles/r01_fp64_peak.md); DMMA is used because it needs 8x fewer issue slots and 4x less
// shared-memory operand traffic than a DFMA register tile.  tcgen05 has no f64 kind.
#pragma once

#include "fk_common.cuh"

namespace fk {

constexpr int GEMM_THREADS = 256;
constexpr int GEMM_BM = 128;               // datapoints per CTA tile
constexpr int GEMM_KT = 32;                // k per pipeline stage
constexpr int GEMM_SA = GEMM_KT + 4;       // shared row stride of the FK tile (doubles): conflict-free A fragments
constexpr int GEMM_BN = 128;               // replicas per pass
constexpr int GEMM_SB = GEMM_BN + 4;       // shared row stride of the L tile
constexpr int GEMM_STAGES = 3;
constexpr int GEMM_FLUSH = 16;             // K-tiles between flushes of the register tile (chain <= 512 FMAs)
constexpr int GEMM_SMEM_BYTES = (GEMM_STAGES * GEMM_BM * GEMM_SA + 2 * GEMM_KT * GEMM_SB) * 8;
constexpr uint32_t KDEC_NONE = 0xffffu;    // DIS: no second factor

// padded replica count of a pass over `r` replicas, at most GEMM_BN.  Forward kernels: a multiple of 16 (two warp
// columns of the same whole number of 8-replica MMA fragments: one instruction stream for all consumer warps).
__host__ __device__ inline int gemm_rp(int r) {
    const int rp = (r + 15) / 16 * 16;
    return rp < GEMM_BN ? rp : GEMM_BN;
}
// VJP contraction and fold: whole fragments, at least two; an odd count gives warp column 0 one fragment more than
// column 1 (the columns share the schedulers pairwise, so the odd fragment costs half a slot, not a whole one)
__host__ __device__ inline int gemm_rp8(int r) {
    const int rp = (r + 7) / 8 * 8;
    return rp < 16 ? 16 : rp < GEMM_BN ? rp : GEMM_BN;
}
// shared row stride of a [k][RP] tile whose rows are read by the 4 k-lanes of a B fragment: == 4 (mod 16) doubles
__host__ __device__ inline int gemm_sb(int RP) { return RP + (RP % 16 ? 12 : 4); }

struct GemmFwdParams {
    TableDesc desc;
    const uint32_t* kdec;  // [K]: slot_a | slot_b << 16, slot = flavour * nx + x  (slot_b = KDEC_NONE for DIS)
    const double* fT;      // [nfl*nx][RP]: f transposed, replica innermost, zero padded to RP
    double* gpart;         // [ksplit][N][RP] level-1 partials
    int RP;                // padded replicas of this pass = 8 * nfrag
    int nfrag;             // 8-replica fragments in use (<= 16)
    int nfw;               // fragments per warp column (2 warp columns; <= 8)
    int ksplit, kper;      // K ranges and their length (multiple of GEMM_KT)
    // grouped launch: one CTA per item (table, datapoint tile, K range); per-table kdec / offsets in descs
    const TableDesc* descs;
    const ColSeg* items;   // {table, kblock = datapoint tile, split = K range}
};

__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src, uint32_t src_bytes) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async8(uint32_t dst, const void* src, uint32_t src_bytes) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(dst), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
        : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// k -> (slot a, slot b) codes of a table, built once per table (or per stateless call)
__global__ void __launch_bounds__(256) fk_kdec_kernel(TableDesc d, ChannelList chan, uint32_t* __restrict__ kdec) {
    for (int k = blockIdx.x * blockDim.x + threadIdx.x; k < d.K; k += gridDim.x * blockDim.x) {
        int ia, ib;
        decode_k(d, chan.a, chan.b, k, ia, ib);
        // padding (ia < 0): FK is exactly 0 there, any finite luminosity will do -> slots (0, 0)
        kdec[k] = ia < 0 ? 0u : ((uint32_t)ia | ((ib >= 0 ? (uint32_t)ib : KDEC_NONE) << 16));
    }
}

// fT[slot][r - r0] = f[r][slot] for r in [r0, r0 + RP), zero beyond R
template <typename T, typename O = double>
__global__ void __launch_bounds__(256) fk_transpose_f_kernel(const T* __restrict__ f, O* __restrict__ fT, int slots,
                                                              int R, int r0, int RP) {
    pdl_trigger();   // first kernel of a call: the contraction behind it may start its prologue and table loads now
    const long long total = (long long)slots * RP;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const int s = (int)(t / RP), c = (int)(t - (long long)s * RP);
        const int r = r0 + c;
        fT[t] = r < R ? (O)f[(long long)r * slots + s] : O(0);
    }
}

template <int VEC, bool GROUPED>
__global__ void __launch_bounds__(GEMM_THREADS, 1)
fk_gemm_fwd_kernel(const __grid_constant__ GemmFwdParams p) {
    pdl_trigger();
    pdl_wait();   // fT of the transpose kernel launched just before (a programmatic dependent launch, fk_common.cuh)
    extern __shared__ __align__(128) unsigned char fk_smem[];
    double* As = reinterpret_cast<double*>(fk_smem);                  // [STAGES][BM][SA]
    double* Ls = As + GEMM_STAGES * GEMM_BM * GEMM_SA;                 // [2][KT][SB]
    const uint32_t As_s = (uint32_t)__cvta_generic_to_shared(As);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const TableDesc* dp = &p.desc;
    const uint32_t* __restrict__ kdec = p.kdec;
    const double* __restrict__ fT = p.fT;
    double* gpart = p.gpart;
    int mt, ks, kper;
    if constexpr (GROUPED) {
        const ColSeg it = p.items[blockIdx.x];
        dp = &p.descs[it.table];
        kdec = dp->kdec;
        fT += dp->f_off * p.RP;
        gpart += dp->gp_off * p.RP;
        mt = it.kblock;
        ks = it.split;
        kper = dp->gkper;
    } else {
        const int mtiles = (p.desc.N + GEMM_BM - 1) / GEMM_BM;
        mt = blockIdx.x % mtiles;
        ks = blockIdx.x / mtiles;
        kper = p.kper;
    }
    const TableDesc& d = *dp;
    const int m0 = mt * GEMM_BM;
    const int kbeg = ks * kper;
    const int kend = min(d.K, kbeg + kper);
    const int nk = kend > kbeg ? (kend - kbeg + GEMM_KT - 1) / GEMM_KT : 0;
    const bool had = d.kind == KIND_HADRONIC;

    // ---- producers -------------------------------------------------------------------------------
    auto load_fk = [&](int t) {  // FK tile of K-tile t -> stage t % STAGES (zero filled outside the table)
        const int slot = t % GEMM_STAGES;
        const int kt0 = kbeg + t * GEMM_KT;
        constexpr int CH = GEMM_KT / VEC;  // chunks per row
#pragma unroll
        for (int j = 0; j < GEMM_BM * CH / GEMM_THREADS; ++j) {
            const int q = tid + j * GEMM_THREADS;
            const int row = q / CH, cc = q - row * CH;
            const int n = m0 + row, k = kt0 + cc * VEC;
            const bool ok = n < d.N && k < kend;
            const double* src = reinterpret_cast<const double*>(d.fk) + (long long)(ok ? n : 0) * d.row_stride + (ok ? k : 0);
            const uint32_t dst = As_s + (uint32_t)(((slot * GEMM_BM + row) * GEMM_SA + cc * VEC) * 8);
            if constexpr (VEC == 2) cp_async16(dst, src, ok ? 16u : 0u);
            else cp_async8(dst, src, ok ? 8u : 0u);
        }
    };
    // luminosity: thread owns the replica pair (2*c2, 2*c2+1) of K-tile rows kq, kq+4, ..., kq+28
    const int c2 = tid & 63, kq = tid >> 6;
    const bool ccol = 2 * c2 < p.RP;
    double2 la[GEMM_KT / 4], lb[GEMM_KT / 4];
    auto load_L = [&](int t) {
        const int kt0 = kbeg + t * GEMM_KT;
#pragma unroll
        for (int j = 0; j < GEMM_KT / 4; ++j) {
            const int k = kt0 + kq + 4 * j;
            la[j] = make_double2(0.0, 0.0);
            lb[j] = make_double2(1.0, 1.0);
            if (ccol && k < kend) {
                const uint32_t code = __ldg(kdec + k);
                la[j] = __ldg(reinterpret_cast<const double2*>(fT + (long long)(code & 0xffffu) * p.RP) + c2);
                if (had) lb[j] = __ldg(reinterpret_cast<const double2*>(fT + (long long)(code >> 16) * p.RP) + c2);
            }
        }
    };
    auto store_L = [&](int t) {
        double* Lb = Ls + (t & 1) * GEMM_KT * GEMM_SB;
        if (ccol) {
#pragma unroll
            for (int j = 0; j < GEMM_KT / 4; ++j)
                *reinterpret_cast<double2*>(Lb + (kq + 4 * j) * GEMM_SB + 2 * c2) =
                    make_double2(la[j].x * lb[j].x, la[j].y * lb[j].y);
        }
    };

    // ---- consumers: warp tile 32 datapoints x (8 * nfw) replicas --------------------------------------
    const int wm = warp & 3, wn = warp >> 2;
    const int nfw = min(p.nfw, max(0, p.nfrag - wn * p.nfw));  // fragments of this warp column
    const int cb = wn * p.nfw * 8;
    double acc[4][8][2];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 8; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

    // ---- level-1 partial tile gpart[ks][n][c] (+)= acc, acc = 0 ----------------------------------------
    double* out = gpart + (long long)ks * d.N * p.RP;
    auto flush = [&](bool first) {
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int n = m0 + wm * 32 + i * 8 + (lane >> 2);
            double2* q = reinterpret_cast<double2*>(out + (long long)n * p.RP + cb + 2 * (lane & 3));
            double2 o[8];  // all loads of a row first: one L2 round trip per row, not per fragment
#pragma unroll
            for (int j = 0; j < 8; ++j) o[j] = (!first && j < nfw && n < d.N) ? q[j * 4] : make_double2(0.0, 0.0);
#pragma unroll
            for (int j = 0; j < 8; ++j)
                if (j < nfw && n < d.N) {
                    q[j * 4] = make_double2(acc[i][j][0] + o[j].x, acc[i][j][1] + o[j].y);
                    acc[i][j][0] = acc[i][j][1] = 0.0;
                }
        }
    };

#pragma unroll
    for (int s = 0; s < GEMM_STAGES - 1; ++s) {
        if (s < nk) load_fk(s);
        cp_async_commit();
    }
    if (nk > 0) {
        load_L(0);
        store_L(0);
    }
    for (int t = 0; t < nk; ++t) {
        cp_async_wait<GEMM_STAGES - 2>();
        __syncthreads();  // stage t has landed and L tile t is stored; everyone is done with K-tile t-1
        if (t + GEMM_STAGES - 1 < nk) load_fk(t + GEMM_STAGES - 1);
        cp_async_commit();
        if (t + 1 < nk) load_L(t + 1);

        const double* At = As + ((t % GEMM_STAGES) * GEMM_BM + wm * 32 + (lane >> 2)) * GEMM_SA + (lane & 3);
        const double* Bt = Ls + (t & 1) * GEMM_KT * GEMM_SB + (lane & 3) * GEMM_SB + cb + (lane >> 2);
#pragma unroll
        for (int k4 = 0; k4 < GEMM_KT / 4; ++k4) {
            double a[4], b[8];
#pragma unroll
            for (int i = 0; i < 4; ++i) a[i] = At[i * 8 * GEMM_SA + k4 * 4];
#pragma unroll
            for (int j = 0; j < 8; ++j) b[j] = j < nfw ? Bt[k4 * 4 * GEMM_SB + j * 8] : 0.0;
#pragma unroll
            for (int j = 0; j < 8; ++j)
                if (j < nfw) {
#pragma unroll
                    for (int i = 0; i < 4; ++i) dmma884(acc[i][j][0], acc[i][j][1], a[i], b[j]);
                }
        }
        if (t + 1 < nk) store_L(t + 1);
        // bounded chains: every GEMM_FLUSH K-tiles (512 FMAs per accumulator) the register tile is added
        // into this CTA's partial tile in gpart (thread-private addresses, L2-resident) and cleared, so a
        // same-sign sum cannot build up a long serial rounding bias
        if ((t + 1) % GEMM_FLUSH == 0 && t + 1 < nk) {
            flush(t + 1 == GEMM_FLUSH);
        }
    }
    flush(nk <= GEMM_FLUSH);
}

// level 2: sigma[n][r0 + c] = sum over K ranges, fixed order
// level 2: sigma[n][r0 + c] = sum over K ranges, fixed order
constexpr int GEMM_REDUCE_QUAD = 16;   // from this many K ranges on, four threads share an output
template <typename T, typename P = double>
__global__ void __launch_bounds__(256) fk_gemm_reduce_kernel(const P* __restrict__ gpart, T* __restrict__ sigma,
                                                              long long out_off, int N, int R, int r0, int RP, int ksplit) {
    pdl_wait();   // the level-1 partials of the whole contraction grid (no-op in a normal launch)
    const long long total = (long long)N * RP;
    if (ksplit < GEMM_REDUCE_QUAD) {   // few slices: one thread per output, all loads in flight
        for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
            const int n = (int)(t / RP), c = (int)(t - (long long)n * RP);
            if (r0 + c >= R) continue;
            double w[GEMM_REDUCE_QUAD], s = 0.0;
#pragma unroll
            for (int e = 0; e < GEMM_REDUCE_QUAD; ++e) w[e] = e < ksplit ? (double)gpart[(long long)e * total + t] : 0.0;
#pragma unroll
            for (int e = 0; e < GEMM_REDUCE_QUAD; ++e) s += w[e];
            sigma[out_off + (long long)n * R + r0 + c] = (T)s;
        }
        return;
    }
    // four threads per output: thread q adds the slices q, q + 4, ... in index order (all its loads in flight: at most 16
    // slices per thread per round), then the quad is combined by a fixed xor butterfly -- one latency round instead of
    // ksplit / 8
    const int q = threadIdx.x & 3;
    for (long long t = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 2; t < ((total + 63) & ~63LL); t += ((long long)gridDim.x * blockDim.x) >> 2) {
        const bool live = t < total;
        const long long tt = live ? t : total - 1;
        double s = 0.0;
        for (int k0 = q; k0 < ksplit; k0 += 64) {
            double w[16];
#pragma unroll
            for (int e = 0; e < 16; ++e) w[e] = k0 + 4 * e < ksplit ? (double)gpart[(long long)(k0 + 4 * e) * total + tt] : 0.0;
#pragma unroll
            for (int e = 0; e < 16; ++e) s += w[e];
        }
        s += __shfl_xor_sync(0xffffffffu, s, 1);
        s += __shfl_xor_sync(0xffffffffu, s, 2);
        const int n = (int)(tt / RP), c = (int)(tt - (long long)n * RP);
        if (live && q == 0 && r0 + c < R) sigma[out_off + (long long)n * R + r0 + c] = (T)s;
    }
}

// last table t with prefix[t] <= x  (prefix has T + 1 entries)
__device__ __forceinline__ int table_of(const int* __restrict__ prefix, int T, long long x) {
    int lo = 0, hi = T;
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (prefix[mid] <= x) lo = mid; else hi = mid;
    }
    return lo;
}

// grouped: fT_cat[global slot][c] = f_cat[f_off_t * R + (r0 + c) * slots_t + slot]
template <typename T, typename O = double>
__global__ void __launch_bounds__(256) fk_transpose_f_grouped_kernel(const T* __restrict__ f_cat, O* __restrict__ fT,
                                                                      const int* __restrict__ ai_prefix, int ntab,
                                                                      long long slots_total, int R, int r0, int RP) {
    const long long total = slots_total * RP;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const long long gs = t / RP;
        const int c = (int)(t - gs * RP), r = r0 + c;
        const int tb = table_of(ai_prefix, ntab, gs);
        const long long base = ai_prefix[tb], slots = ai_prefix[tb + 1] - base;
        fT[t] = r < R ? (O)f_cat[base * R + (long long)r * slots + (gs - base)] : O(0);
    }
}

// grouped level 2: sigma_cat[global row][r0 + c] = sum over the K ranges of the row's table, fixed order
// TC: the partials of the tcgen05 contraction (fk_tc32.cu: TableDesc::tc_gp_off, tc_ksplit), else of the DMMA one
template <typename T, typename P = double, bool TC = false>
__global__ void __launch_bounds__(256) fk_gemm_reduce_grouped_kernel(const P* __restrict__ gpart, T* __restrict__ sigma,
                                                                      const TableDesc* __restrict__ descs,
                                                                      const int* __restrict__ row_prefix, int ntab,
                                                                      long long rows_total, int R, int r0, int RP) {
    pdl_wait();   // the level-1 partials of the whole contraction grid (no-op in a normal launch)
    const long long total = rows_total * RP;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const long long grow = t / RP;
        const int c = (int)(t - grow * RP);
        if (r0 + c >= R) continue;
        const int tb = table_of(row_prefix, ntab, grow);
        const TableDesc& d = descs[tb];
        const long long n = grow - row_prefix[tb];
        const P* src = gpart + ((TC ? d.tc_gp_off : d.gp_off) + n) * RP + c;
        const long long stride = (long long)d.N * RP;
        const int nsl = TC ? d.tc_ksplit : d.gksplit;
        double s = 0.0;
        for (int k0 = 0; k0 < nsl; k0 += 8) {  // eight loads in flight, added in index order
            double w[8];
#pragma unroll
            for (int q = 0; q < 8; ++q) w[q] = k0 + q < nsl ? (double)src[(k0 + q) * stride] : 0.0;
#pragma unroll
            for (int q = 0; q < 8; ++q) s += w[q];
        }
        sigma[grow * R + r0 + c] = (T)s;
    }
}

// ---------------------------------------------------------------------------------------------------
// VJP stage 1 for R >> 1 (minimal-flop order): G[k][c] = sum_n FK[n][k] * g[n][r0 + c].
// Same machinery with the FK tile used transposed: CTA = 128 consecutive k (1 KB of every row), the
// contraction runs over ALL datapoints in steps of 32 (no split: one CTA owns its G tile, fixed order),
// both operands arrive by cp.async (FK tile [32 n][128 k], upstream-gradient tile [32 n][RP]).
struct GemmVjpParams {
    TableDesc desc;
    const double* gP;   // [N][RP]: g of this pass, replica innermost, zero padded
    double* G;          // [K][RP] column sums, replica innermost
    int RP, nfrag, nfw;
    const TableDesc* descs;  // grouped launch: one CTA per item {table, kblock = 128-k tile}
    const ColSeg* items;
};

constexpr int GEMMV_BK = 128;                // k per CTA tile (the M dimension of the MMA)
constexpr int GEMMV_NT = 32;                 // datapoints per pipeline stage
constexpr int GEMMV_S = GEMMV_BK + 4;        // shared row stride of both tiles
constexpr int GEMMV_STAGES = 3;
constexpr int GEMMV_SMEM_BYTES = GEMMV_STAGES * 2 * GEMMV_NT * GEMMV_S * 8;

template <int VEC, bool GROUPED>
__global__ void __launch_bounds__(GEMM_THREADS, 1)
fk_gemm_vjp_kernel(const __grid_constant__ GemmVjpParams p) {
    extern __shared__ __align__(128) unsigned char fk_smem[];
    double* As = reinterpret_cast<double*>(fk_smem);            // [STAGES][NT][S]  FK tile, k innermost
    double* Bs = As + GEMMV_STAGES * GEMMV_NT * GEMMV_S;         // [STAGES][NT][S]  g tile, replica innermost
    const uint32_t As_s = (uint32_t)__cvta_generic_to_shared(As), Bs_s = (uint32_t)__cvta_generic_to_shared(Bs);

    const TableDesc* dp = &p.desc;
    const double* __restrict__ gP = p.gP;
    double* __restrict__ G = p.G;
    int kt = blockIdx.x;
    if constexpr (GROUPED) {
        const ColSeg it = p.items[blockIdx.x];
        dp = &p.descs[it.table];
        gP += dp->out_off * p.RP;
        G += dp->k_off * p.RP;
        kt = it.kblock;
    }
    const TableDesc& d = *dp;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int k0 = kt * GEMMV_BK;
    const int nt = (d.N + GEMMV_NT - 1) / GEMMV_NT;

    auto load_stage = [&](int t) {
        const int slot = t % GEMMV_STAGES;
        const int n0 = t * GEMMV_NT;
        {   // FK tile: NT rows x BK k
            constexpr int CH = GEMMV_BK / VEC;
#pragma unroll
            for (int j = 0; j < GEMMV_NT * CH / GEMM_THREADS; ++j) {
                const int q = tid + j * GEMM_THREADS;
                const int row = q / CH, cc = q - row * CH;
                const int n = n0 + row, k = k0 + cc * VEC;
                const bool ok = n < d.N && k < d.K;
                const double* src = reinterpret_cast<const double*>(d.fk) + (long long)(ok ? n : 0) * d.row_stride + (ok ? k : 0);
                const uint32_t dst = As_s + (uint32_t)(((slot * GEMMV_NT + row) * GEMMV_S + cc * VEC) * 8);
                if constexpr (VEC == 2) cp_async16(dst, src, ok ? 16u : 0u);
                else cp_async8(dst, src, ok ? 8u : 0u);
            }
        }
        {   // g tile: NT rows x RP replicas (RP is a multiple of 8: 16-byte chunks)
            const int CH = p.RP / 2;
            for (int q = tid; q < GEMMV_NT * CH; q += GEMM_THREADS) {
                const int row = q / CH, cc = q - row * CH;
                const int n = n0 + row;
                const bool ok = n < d.N;
                const double* src = gP + (long long)(ok ? n : 0) * p.RP + cc * 2;
                cp_async16(Bs_s + (uint32_t)(((slot * GEMMV_NT + row) * GEMMV_S + cc * 2) * 8), src, ok ? 16u : 0u);
            }
        }
    };

    const int wm = warp & 3, wn = warp >> 2;
    const int nfw = min(p.nfw, max(0, p.nfrag - wn * p.nfw));
    const int cb = wn * p.nfw * 8;
    double acc[4][8][2];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 8; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

#pragma unroll
    for (int s = 0; s < GEMMV_STAGES - 1; ++s) {
        if (s < nt) load_stage(s);
        cp_async_commit();
    }
    // bounded chains: every GEMM_FLUSH stages (512 datapoints) the register tile is added into this CTA's own G tile
    auto flushG = [&](bool first) {
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int k = k0 + wm * 32 + i * 8 + (lane >> 2);
#pragma unroll
            for (int j = 0; j < 8; ++j)
                if (j < nfw) {
                    if (k < d.K) {
                        double2* q = reinterpret_cast<double2*>(G + (long long)k * p.RP + cb + j * 8 + 2 * (lane & 3));
                        const double2 o = first ? make_double2(0.0, 0.0) : *q;
                        *q = make_double2(acc[i][j][0] + o.x, acc[i][j][1] + o.y);
                    }
                    acc[i][j][0] = acc[i][j][1] = 0.0;
                }
        }
    };
    bool flushed = false;
    for (int t = 0; t < nt; ++t) {
        cp_async_wait<GEMMV_STAGES - 2>();
        __syncthreads();
        if (t + GEMMV_STAGES - 1 < nt) load_stage(t + GEMMV_STAGES - 1);
        cp_async_commit();
        // A fragment: row m = k (lane >> 2), col = datapoint (lane & 3)  ->  As[n][k]
        const double* At = As + ((t % GEMMV_STAGES) * GEMMV_NT + (lane & 3)) * GEMMV_S + wm * 32 + (lane >> 2);
        const double* Bt = Bs + ((t % GEMMV_STAGES) * GEMMV_NT + (lane & 3)) * GEMMV_S + cb + (lane >> 2);
#pragma unroll
        for (int n4 = 0; n4 < GEMMV_NT / 4; ++n4) {
            double a[4], b[8];
#pragma unroll
            for (int i = 0; i < 4; ++i) a[i] = At[n4 * 4 * GEMMV_S + i * 8];
#pragma unroll
            for (int j = 0; j < 8; ++j) b[j] = j < nfw ? Bt[n4 * 4 * GEMMV_S + j * 8] : 0.0;
#pragma unroll
            for (int j = 0; j < 8; ++j)
                if (j < nfw) {
#pragma unroll
                    for (int i = 0; i < 4; ++i) dmma884(acc[i][j][0], acc[i][j][1], a[i], b[j]);
                }
        }
        if ((t + 1) % GEMM_FLUSH == 0 && t + 1 < nt) {
            flushG(!flushed);
            flushed = true;
        }
    }
    flushG(!flushed);
}

// gP[n][c] = g[n][r0 + c] (zero beyond R)
template <typename T>
__global__ void __launch_bounds__(256) fk_pad_g_kernel(const T* __restrict__ g, double* __restrict__ gP, int N, int R, int r0, int RP) {
    const long long total = (long long)N * RP;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const int n = (int)(t / RP), c = (int)(t - (long long)n * RP);
        gP[t] = r0 + c < R ? (double)g[(long long)n * R + r0 + c] : 0.0;
    }
}

// VJP stage 2 for the replica-innermost G: one CTA per (alpha, i), one thread per replica of the pass.
//   df[r][alpha][i] = sum_{c: a_c = alpha} sum_j G[k(i,j,c)][r] f[r][b_c][j] + sum_{c: b_c = alpha} sum_j G[k(j,i,c)][r] f[r][a_c][j]
// Every load is coalesced along r; 4 interleaved chains per thread, combined in a fixed order.
struct GatherRParams {
    TableDesc desc;
    ChannelList chan;
    const double* fT;   // [slots][RP]
    const double* G;    // [K][RP]
    void* df;           // [R][nfl][nx]
    int R, r0, RP;
    const TableDesc* descs;  // grouped launch: blockIdx.x = global (alpha, i) slot
    const int* ai_prefix;
    int T;
};

template <typename T, bool GROUPED>
__global__ void __launch_bounds__(128) fk_vjp_gather_r_kernel(const __grid_constant__ GatherRParams p) {
    __shared__ short listA[MAX_C], listB[MAX_C];
    __shared__ uint8_t other[2][MAX_C];  // flavour of the opposite leg of every listed channel
    __shared__ int cnt[2];
    const TableDesc* dp = &p.desc;
    const uint8_t* __restrict__ ca = p.chan.a;
    const uint8_t* __restrict__ cb = p.chan.b;
    const double* __restrict__ G = p.G;
    const double* __restrict__ fT = p.fT;
    int slot = blockIdx.x;
    if constexpr (GROUPED) {
        const int tb = table_of(p.ai_prefix, p.T, slot);
        dp = &p.descs[tb];
        slot -= p.ai_prefix[tb];
        ca = dp->chan_a;
        cb = dp->chan_b;
        G += dp->k_off * p.RP;
        fT += dp->f_off * p.RP;
    }
    const TableDesc& d = *dp;
    const int nx = d.nx, C = d.C;
    const int alpha = slot / nx, i = slot - alpha * nx;
    const bool had = d.kind == KIND_HADRONIC;
    if (threadIdx.x == 0) {
        int na = 0, nb = 0;
        for (int c = 0; c < C; ++c) {
            if (ca[c] == alpha) { other[0][na] = cb[c]; listA[na++] = (short)c; }
            if (had && cb[c] == alpha) { other[1][nb] = ca[c]; listB[nb++] = (short)c; }
        }
        cnt[0] = na;
        cnt[1] = nb;
    }
    __syncthreads();
    const int na = cnt[0], nb = cnt[1];
    const int c0 = blockIdx.y * blockDim.x + threadIdx.x;  // replica column of this pass
    if (c0 >= p.RP || p.r0 + c0 >= p.R) return;
    G += c0;
    fT += c0;
    double acc[4] = {0.0, 0.0, 0.0, 0.0};
    if (had) {
        for (int q = 0; q < na; ++q) {
            const int c = listA[q];
            const long long fo = (long long)other[0][q] * nx;
            for (int j = 0; j < nx; ++j) {
                const int k = encode_k(d, i, j, c);
                acc[j & 3] = fma(G[(long long)k * p.RP], fT[(fo + j) * p.RP], acc[j & 3]);
            }
        }
        for (int q = 0; q < nb; ++q) {
            const int c = listB[q];
            const long long fo = (long long)other[1][q] * nx;
            for (int j = 0; j < nx; ++j) {
                const int k = encode_k(d, j, i, c);
                acc[j & 3] = fma(G[(long long)k * p.RP], fT[(fo + j) * p.RP], acc[j & 3]);
            }
        }
    } else {
        for (int q = 0; q < na; ++q) acc[q & 3] += G[(long long)encode_k(d, i, 0, listA[q]) * p.RP];
    }
    const double s = (acc[0] + acc[1]) + (acc[2] + acc[3]);
    reinterpret_cast<T*>(p.df)[d.f_off * p.R + ((long long)(p.r0 + c0) * d.nfl + alpha) * nx + i] = (T)s;
}

}  // namespace fk
