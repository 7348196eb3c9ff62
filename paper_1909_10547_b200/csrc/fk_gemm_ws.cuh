// fk_gemm_ws.cuh -- R >> 1 dense contraction for PACKED hadronic tables, warp-specialised (SURVEY 8(a) rows a1 + a4).
//
//   Sigma[n][r] = sum_k FK[n][k] * L[k][r],   L[(c,i,j)][r] = f[r][a_c][i] * f[r][b_c][j]       Eq. (1)
//
// What differs from the generic kernel in fk_gemm.cuh (which stays for logical-layout and DIS tables):
//   * one PRODUCER warp moves data with bulk async copies (cp.async.bulk, UBLKCP) that complete on
//     mbarriers; eight CONSUMER warps do nothing but shared-memory fragment loads and DMMA.  The consumers
//     never compute a global address and never meet at a CTA-wide barrier, so the FP64 tensor pipe does not
//     drain once per K-tile while every warp plays producer (ncu on the generic kernel: 2 warps per
//     scheduler stall together at each stage hand-over).
//   * the luminosity tile is never built.  In the packed order k = c*cstride + i*nx + j the factor
//     f[b_c][j] of a whole channel is one contiguous [nx][RP] block of the replica-innermost copy fT: it is
//     bulk-copied into shared memory once per channel (double buffered) and serves nx*nx values of k;
//     the other factor f[a_c][i] changes every nx steps of k and lives in 8 registers per thread.  The B
//     fragment of an MMA k-step is formed at load time: b = fB[j][r] * fA[i][r]  (8 DMUL per 32 DMMA).
//     No k -> (slot, slot) codes, no gathers, no luminosity tile in shared memory or HBM.
//   * FK tiles [128 n][32 k] arrive as one 256-byte bulk copy per datapoint row into rows padded to 36
//     doubles (conflict-free A fragments); channel blocks are padded to 4 elements by the pack kernel, so an
//     MMA k-step never straddles a channel and every copy is 32-byte aligned.
// Split-K partials, the periodic flush that bounds the accumulation chains, and the fixed-order level-2
// reduction are those of fk_gemm.cuh.  Results are bitwise repeatable.
#pragma once

#include <type_traits>

#include "fk_common.cuh"
#include "fk_gemm.cuh"

namespace fk {

constexpr int WS_CONSUMER_WARPS = 8;
constexpr int WS_THREADS = (WS_CONSUMER_WARPS + 4) * 32;  // + the producer's warpgroup (1 working warp): register
                                                          // reallocation (setmaxnreg) works on whole warpgroups.
                                                          // (9 warps would not help: registers are per scheduler,
                                                          // 3 warps on one of them still cap a thread at 170.)
constexpr int WS_PRODUCER_WARPS = 4;
constexpr int WS_STAGES = 3;
constexpr int WS_STAGE_DOUBLES = GEMM_BM * GEMM_SA;        // FK tile [128][36]
constexpr int WS_NBAR = 2 * WS_STAGES + 4;                 // full[S], empty[S], fb_full[2], fb_empty[2]

__host__ __device__ inline size_t ws_smem_bytes(int nx, int RP) {
    return (size_t)(WS_STAGES * WS_STAGE_DOUBLES + 2 * nx * gemm_sb(RP)) * 8 + WS_NBAR * 8;
}

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n.reg .pred p;\nW_%=:\nmbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n@p bra D_%=;\nbra W_%=;\nD_%=:\n}\n" ::"r"(bar),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst), "l"(src),
                 "r"(bytes), "r"(bar)
                 : "memory");
}

// The forward kernel reads the table once: its bulk copies carry an L2 evict-first policy, so that the streamed rows do not
// push the small, re-read operands (the level-1 partial tiles that are read-modified-written at every flush, fT) out of L2
// (config 3 forward 1.069 -> 1.057 ms).  The VJP kernel keeps the default policy (1.082 ms; 1.097 with the hint).
__device__ __forceinline__ uint64_t l2_evict_first_policy() {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ void bulk_g2s_stream(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar, uint64_t pol) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(dst), "l"(src),
                 "r"(bytes), "r"(bar), "l"(pol)
                 : "memory");
}

// Same fields as GemmFwdParams where they mean the same thing.
struct WsFwdParams {
    TableDesc desc;        // single-table launch
    ChannelList chan;      // single-table launch
    const double* fT;      // [nfl*nx][RP] replica-innermost f (grouped: + desc.f_off * RP)
    double* gpart;         // [ksplit][N][RP] level-1 partials (grouped: + desc.gp_off * RP)
    int RP;                // padded replicas of this pass = 8 * NFRAG
    int ksplit, kper;      // single-table launch: K ranges (a multiple of ksub_rem) and their length
    int ksub_rem;          // single-table launch: k sub-splits (1, 2, 4) of the last, partial datapoint tile
    const TableDesc* descs;  // grouped launch
    const ColSeg* items;     // grouped launch {table, kblock = first datapoint, split = K range of the item, pad_ = k sub-splits}
};

// Ragged datapoint counts: a tile of TM = 128 / KSUB datapoints (KSUB = 1, 2, 4) keeps all 8 consumer warps on
// real rows.  The 4 warp rows become (TM / 32) row blocks x KSUB k sub-splits: sub-split q takes the MMA
// k-steps q, q + KSUB, ... of a stage that is KSUB times longer in k ([TM][32 * KSUB] doubles, the same bytes),
// covers KSUB base K ranges per item and writes its own level-1 partial slice, so an item costs the same
// DMMA time and the reduction sees the same number of slices whatever the tile height.
__host__ __device__ inline int ws_ksub_for_rows(int rows) { return rows <= 32 ? 4 : rows <= 64 ? 2 : 1; }

// NFRAG = 8-replica fragments of the pass = RP / 8, even here: each of the two warp columns takes NFRAG / 2.  (An
// uneven split, as in the VJP kernel below, was measured slower for this kernel: two instruction streams of this
// size per SM.)  The fragment count of a warp is a compile-time constant: the 4 x NF DMMAs of a k-step
// carry no predicates, so ptxas is free to batch the fragment loads and the DMULs ahead of them.
// TS = storage type of the table: float for FK_F32S64 tables, whose tiles are copied as stored (half the bytes, the same
// byte pitch per shared-memory row) and widened to double when the A fragments are loaded.
template <int NFRAG, bool GROUPED, typename TS = double>
__global__ void __launch_bounds__(WS_THREADS, 1)
fk_gemm_fwd_ws_kernel(const __grid_constant__ WsFwdParams p) {
    constexpr int ESZ = (int)sizeof(TS);
    pdl_trigger();
    pdl_wait();   // fT of the transpose kernel launched just before (a programmatic dependent launch, fk_common.cuh)
    extern __shared__ __align__(128) unsigned char fk_smem[];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;

    const TableDesc* dp = &p.desc;
    const uint8_t* __restrict__ cha = p.chan.a;
    const uint8_t* __restrict__ chb = p.chan.b;
    const double* __restrict__ fT = p.fT;
    double* gpart = p.gpart;
    int m0, ks, kper, KSUB;
    if constexpr (GROUPED) {
        const ColSeg it = p.items[blockIdx.x];
        dp = &p.descs[it.table];
        cha = dp->chan_a;
        chb = dp->chan_b;
        fT += dp->f_off * p.RP;
        gpart += dp->gp_off * p.RP;
        m0 = it.kblock;
        ks = it.split;
        KSUB = it.pad_;
        kper = dp->gkper;
    } else {
        const int nfull = p.desc.N / GEMM_BM, nb_full = nfull * p.ksplit;
        if ((int)blockIdx.x < nb_full) {
            m0 = ((int)blockIdx.x % nfull) * GEMM_BM;
            ks = (int)blockIdx.x / nfull;
            KSUB = 1;
        } else {
            m0 = nfull * GEMM_BM;
            ks = (int)blockIdx.x - nb_full;
            KSUB = p.ksub_rem;
        }
        kper = p.kper;
    }
    const TableDesc& d = *dp;
    const int nx = d.nx, RP = p.RP, SB = gemm_sb(RP), cstride = d.cstride;
    constexpr int NFW0 = NFRAG / 2;
    const int TM = GEMM_BM / KSUB, KTv = GEMM_KT * KSUB, SAv = KTv + 4;  // tile rows, k per stage, shared row stride
    const int kbeg = min(d.K, ks * kper * KSUB), kend = min(d.K, kbeg + kper * KSUB);
    // an empty K range (more slices than K-tiles) still writes its zero partials
    const int c0 = kbeg / cstride, c1 = kbeg < kend ? (kend - 1) / cstride : c0 - 1;

    double* As = reinterpret_cast<double*>(fk_smem);       // [STAGES][128][36]
    double* Bs = As + WS_STAGES * WS_STAGE_DOUBLES;         // [2][nx][SB]   f[b_c][j][r] of two channels
    const uint32_t As_s = (uint32_t)__cvta_generic_to_shared(As);
    const uint32_t Bs_s = (uint32_t)__cvta_generic_to_shared(Bs);
    const uint32_t bar0 = Bs_s + (uint32_t)(2 * nx * SB * 8);
    auto bar_full = [&](int s) { return bar0 + 8u * s; };
    auto bar_empty = [&](int s) { return bar0 + 8u * (WS_STAGES + s); };
    auto bar_fbfull = [&](int b) { return bar0 + 8u * (2 * WS_STAGES + b); };
    auto bar_fbempty = [&](int b) { return bar0 + 8u * (2 * WS_STAGES + 2 + b); };
    if (tid == 0) {
        for (int s = 0; s < WS_STAGES; ++s) {
            mbar_init(bar_full(s), WS_PRODUCER_WARPS);   // one arrive.expect_tx per producer warp
            mbar_init(bar_empty(s), WS_CONSUMER_WARPS);
        }
        for (int b = 0; b < 2; ++b) {
            mbar_init(bar_fbfull(b), 1);
            mbar_init(bar_fbempty(b), WS_CONSUMER_WARPS);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp >= WS_CONSUMER_WARPS) {
        // ================================ producer warp ================================
        // 384 threads cap the kernel at 168 registers; the producer warpgroup hands its share to the consumers:
        // 256 x 232 + 128 x 40 = 384 x 168 exactly (asking for more than the CTA owns would block forever)
        asm volatile("setmaxnreg.dec.sync.aligned.u32 40;" ::: "memory");
        // All four warps of the producer warpgroup issue copies: a bulk copy costs its warp ~57 cycles of issue whatever
        // its size (measured, profiles/r02_bulk_copy_issue.md), so ONE warp needs 7 300 cycles for the 128 row pieces
        // of a stage that the consumers finish in 8 192 -- any hiccup of the producer then stalls the tensor pipe.  Warp pw
        // takes the datapoints 32*pw .. 32*pw + 31 of every stage and arrives on the stage's barrier with its own byte count.
        const int pw = warp - WS_CONSUMER_WARPS;
        const TS* __restrict__ fk = reinterpret_cast<const TS*>(d.fk);
        const uint64_t pol = l2_evict_first_policy();
        const int rows_valid = min(TM, d.N - m0);
        const int my_rows = max(0, min(32, rows_valid - 32 * pw));
        auto issue_fb = [&](int c, int ccn) {  // f[b_c][.][.] of channel c -> buffer ccn & 1 (producer warp 0)
            if (pw != 0) return;
            const int buf = ccn & 1;
            mbar_wait(bar_fbempty(buf), ((ccn >> 1) & 1) ^ 1);
            if (lane == 0) mbar_expect_tx(bar_fbfull(buf), (uint32_t)(nx * RP * 8));
            __syncwarp();
            const double* src = fT + (long long)chb[c] * nx * RP;
            for (int row = lane; row < nx; row += 32)
                bulk_g2s(Bs_s + (uint32_t)((buf * nx + row) * SB * 8), src + (long long)row * RP, (uint32_t)(RP * 8), bar_fbfull(buf));
        };
        int it = 0, cc = 0;
        if (c0 <= c1) issue_fb(c0, 0);
        for (int c = c0; c <= c1; ++c, ++cc) {
            const int sb = max(kbeg, c * cstride), se = min(kend, (c + 1) * cstride);
            bool next_issued = c == c1;
            int tiles = 0;
            for (int k0 = sb; k0 < se; k0 += KTv, ++it, ++tiles) {
                // the buffer of channel c + 1 was released when the consumers left channel c - 1, which they
                // had to do before tile WS_STAGES of this channel can be issued: this wait never blocks here
                if (!next_issued && tiles == WS_STAGES) {
                    issue_fb(c + 1, cc + 1);
                    next_issued = true;
                }
                const int len = min(KTv, se - k0);
                const int stage = it % WS_STAGES;
                mbar_wait(bar_empty(stage), ((it / WS_STAGES) & 1) ^ 1);
                if (lane == 0) mbar_expect_tx(bar_full(stage), (uint32_t)(my_rows * len * ESZ));
                __syncwarp();
                const int row = lane + 32 * pw;
                if (lane < my_rows)
                    bulk_g2s_stream(As_s + (uint32_t)((stage * WS_STAGE_DOUBLES + row * SAv) * 8),
                                    fk + (long long)(m0 + row) * d.row_stride + k0, (uint32_t)(len * ESZ), bar_full(stage), pol);
            }
            if (!next_issued) issue_fb(c + 1, cc + 1);
        }
        return;
    }

    // ================================ consumer warps: warp tile 32 datapoints x (8 * nfw) replicas ================================
    asm volatile("setmaxnreg.inc.sync.aligned.u32 232;" ::: "memory");
    auto consume = [&](auto ks_tag, auto nf_tag) {
        constexpr int NFW = decltype(nf_tag)::value;           // fragments of this warp's column
        const int wm = warp & 3, wn = warp >> 2;
        constexpr int KS = decltype(ks_tag)::value;            // compile-time k sub-splits: immediate shared-memory offsets
        constexpr int KTc = GEMM_KT * KS, SAc = KTc + 4;
        const int rb = wm % (4 / KS), ksub = wm / (4 / KS);    // row block and k sub-split of this warp row
        constexpr int kst = 4 * KS;                            // k between consecutive MMA k-steps of this warp
        const int cbcol = wn * NFW0 * 8;
        double acc[4][NFW][2];
    #pragma unroll
        for (int i = 0; i < 4; ++i)
    #pragma unroll
            for (int j = 0; j < NFW; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

        // level-1 partial tile gpart[ks][n][c] (+)= acc, acc = 0   (thread-private addresses, L2 resident)
        double* out = gpart + (long long)(ks * KS + ksub) * d.N * RP;
        auto flush = [&](bool first) {
    #pragma unroll
            for (int i = 0; i < 4; ++i) {
                const int n = m0 + rb * 32 + i * 8 + (lane >> 2);
                double2* q = reinterpret_cast<double2*>(out + (long long)n * RP + cbcol + 2 * (lane & 3));
                double2 o[NFW];
    #pragma unroll
                for (int j = 0; j < NFW; ++j) o[j] = (!first && n < d.N) ? q[j * 4] : make_double2(0.0, 0.0);
    #pragma unroll
                for (int j = 0; j < NFW; ++j) {
                    if (n < d.N) q[j * 4] = make_double2(acc[i][j][0] + o[j].x, acc[i][j][1] + o[j].y);
                    acc[i][j][0] = acc[i][j][1] = 0.0;
                }
            }
        };

        int it = 0, cc = 0;
        bool flushed = false;
        for (int c = c0; c <= c1; ++c, ++cc) {
            const int sb = max(kbeg, c * cstride), se = min(kend, (c + 1) * cstride);
            const int buf = cc & 1;
            mbar_wait(bar_fbfull(buf), (cc >> 1) & 1);
            const double* Bt = Bs + (long long)buf * nx * SB + cbcol + (lane >> 2);
            const double* __restrict__ fa_base = fT + (long long)cha[c] * nx * RP + cbcol + (lane >> 2);
            // this lane's k of every MMA k-step is 4*step + (lane & 3): its own (i, j), walked incrementally
            int i, j;
            {
                const int kl = sb - c * cstride + ksub * 4 + (lane & 3);
                i = kl / nx;
                j = kl - i * nx;
            }
            // f[a_c][i][r] for the 8 replica columns of this lane's B fragments, and the same for row i + 1,
            // fetched one x-row (nx values of k) ahead so that the row switch never waits for L2
            double fa[NFW], fan[NFW];
            auto load_row = [&](double (&dst)[NFW], int row) {
                const double* src = fa_base + (long long)min(row, nx - 1) * RP;  // row >= nx only on the zero padding
    #pragma unroll
                for (int j8 = 0; j8 < NFW; ++j8) dst[j8] = __ldg(src + j8 * 8);
            };
            load_row(fa, i);
            load_row(fan, i + 1);
            for (int k0 = sb; k0 < se; k0 += KTc, ++it) {
                const int nsteps = max(0, ((min(KTc, se - k0) >> 2) - ksub + KS - 1) / KS);
                const int stage = it % WS_STAGES;
                mbar_wait(bar_full(stage), (it / WS_STAGES) & 1);
                constexpr int PSc = SAc * 8 / ESZ;   // row pitch in elements of TS
                const TS* At = reinterpret_cast<const TS*>(As + stage * WS_STAGE_DOUBLES) + (rb * 32 + (lane >> 2)) * PSc + ksub * 4 + (lane & 3);
    #pragma unroll
                for (int s = 0; s < GEMM_KT / 4; ++s) {
                    if (s < nsteps) {
                        double a[4], b[NFW];
    #pragma unroll
                        for (int i4 = 0; i4 < 4; ++i4) a[i4] = (double)At[i4 * 8 * PSc + s * kst];
    #pragma unroll
                        for (int j8 = 0; j8 < NFW; ++j8) b[j8] = Bt[j * SB + j8 * 8] * fa[j8];
    #pragma unroll
                        for (int j8 = 0; j8 < NFW; ++j8)
    #pragma unroll
                            for (int i4 = 0; i4 < 4; ++i4) dmma884(acc[i4][j8][0], acc[i4][j8][1], a[i4], b[j8]);
                        j += kst;
                        if (j >= nx) {
                            j -= nx;
                            ++i;
                            if (j < nx) {
    #pragma unroll
                                for (int j8 = 0; j8 < NFW; ++j8) fa[j8] = fan[j8];
                            } else {  // nx < 4: more than one row per MMA k-step
                                do {
                                    j -= nx;
                                    ++i;
                                } while (j >= nx);
                                load_row(fa, i);
                            }
                            load_row(fan, i + 1);
                        }
                        __syncwarp();
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(bar_empty(stage));
                // the two warp columns share the SM's four schedulers pairwise: they flush half a period apart, so one
                // warp of a scheduler keeps the FP64 pipe busy while the other waits for its partials from L2
                if ((it + 1 + wn * (GEMM_FLUSH / 2)) % GEMM_FLUSH == 0) {
                    flush(!flushed);
                    flushed = true;
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_fbempty(buf));
        }
        flush(!flushed);
    };
    static_assert(NFRAG % 2 == 0, "the forward kernel takes whole pairs of fragments (RP a multiple of 16)");
    switch (KSUB) {
        case 1: consume(std::integral_constant<int, 1>{}, std::integral_constant<int, NFW0>{}); break;
        case 2: consume(std::integral_constant<int, 2>{}, std::integral_constant<int, NFW0>{}); break;
        default: consume(std::integral_constant<int, 4>{}, std::integral_constant<int, NFW0>{}); break;
    }
}

}  // namespace fk

namespace fk {

// ---------------------------------------------------------------------------------------------------
// VJP stage 1 for R >> 1, warp-specialised and persistent:  G[k][c] = sum_n FK[n][k] * g[n][r0 + c]
// (the same contraction as fk_gemm_vjp_kernel in fk_gemm.cuh, which stays for tables
// whose rows cannot be bulk-copied).  A CTA walks the 128-k tiles  first, first + grid, ...  of the launch;
// its producer warp streams [32 n][128 k] FK pieces and [32 n][RP] upstream-gradient pieces through a ring of
// mbarrier-completed bulk copies and runs ahead across tile boundaries, so the consumers' FP64 tensor pipe
// only drains for the register -> HBM store of a finished G tile.  Shared memory is zeroed once: rows a
// short last stage does not copy hold finite stale values and are masked on the g side.
struct WsVjpParams {
    TableDesc desc;     // single-table launch
    const double* gP;   // [N][RP]: g of this pass, replica innermost, zero padded (grouped: + out_off * RP)
    double* G;          // [K][RP] column sums (grouped: + k_off * RP)
    int RP, ntiles;     // ntiles: work items of the launch: 128-k tiles (single-table: + the column parts of the tail tiles) or grouped items
    int nwhole, nparts; // single-table launch: items [0, nwhole) are whole tiles; item nwhole + s is column part s % nparts of tile
                        // nwhole + s / nparts.  The tiles left over after the last full round of the persistent grid are cut
                        // into 2 or 4 column parts (disjoint outputs, nothing to add up): the last round lasts 1/2 or 1/4 tile.
    const TableDesc* descs;  // grouped launch
    const ColSeg* items;     // grouped launch {table, kblock = 128-k tile}
};

constexpr int WSV_STAGE_DOUBLES = 2 * GEMMV_NT * GEMMV_S;   // FK piece + g piece
constexpr size_t WSV_SMEM_BYTES = (size_t)GEMMV_STAGES * WSV_STAGE_DOUBLES * 8 + 2 * GEMMV_STAGES * 8;

// TS = storage type of the table: float for the fp32-stored tables (FK_F32, FK_F32S64), whose pieces are copied as they are
// (half the bytes) and widened to double when the A fragments are loaded; everything else is fp64 either way.
template <int NFRAG, bool GROUPED, typename TS = double>
__global__ void __launch_bounds__(WS_THREADS, 1)
fk_gemm_vjp_ws_kernel(const __grid_constant__ WsVjpParams p) {
    constexpr int PS = GEMMV_S * 8 / (int)sizeof(TS);    // row pitch of the FK piece in elements (same byte pitch for both types)
    constexpr int VEL = 16 / (int)sizeof(TS);            // elements per 16-byte piece of a bulk copy
    extern __shared__ __align__(128) unsigned char fk_smem[];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    double* Sm = reinterpret_cast<double*>(fk_smem);  // [STAGES][2][NT][S]
    const uint32_t Sm_s = (uint32_t)__cvta_generic_to_shared(Sm);
    const uint32_t bar0 = Sm_s + (uint32_t)(GEMMV_STAGES * WSV_STAGE_DOUBLES * 8);
    auto bar_full = [&](int s) { return bar0 + 8u * s; };
    auto bar_empty = [&](int s) { return bar0 + 8u * (GEMMV_STAGES + s); };
    for (int q = tid; q < GEMMV_STAGES * WSV_STAGE_DOUBLES; q += WS_THREADS) Sm[q] = 0.0;
    if (tid == 0) {
        for (int s = 0; s < GEMMV_STAGES; ++s) {
            mbar_init(bar_full(s), 1);
            mbar_init(bar_empty(s), WS_CONSUMER_WARPS);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");  // the zeros are ordered before the bulk copies
    __syncthreads();
    const int RP = p.RP;

    auto tile_of = [&](int t, const TableDesc*& d, const double*& gP, double*& G, int& kt, int& part) {
        part = -1;   // whole tile
        if constexpr (GROUPED) {
            const ColSeg it = p.items[t];
            d = &p.descs[it.table];
            gP = p.gP + d->out_off * RP;
            G = p.G + d->k_off * RP;
            kt = it.kblock;
        } else {
            d = &p.desc;
            gP = p.gP;
            G = p.G;
            kt = t;
            if (t >= p.nwhole) {
                const int sidx = t - p.nwhole;
                kt = p.nwhole + sidx / p.nparts;
                part = sidx % p.nparts;
            }
        }
    };

    if (warp >= WS_CONSUMER_WARPS) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 40;" ::: "memory");
        if (warp != WS_CONSUMER_WARPS) return;
        int it = 0;
        for (int t = blockIdx.x; t < p.ntiles; t += gridDim.x) {
            const TableDesc* d;
            const double* gP;
            double* G;
            int kt, part;
            tile_of(t, d, gP, G, kt, part);
            const int k0 = kt * GEMMV_BK, klen = min(GEMMV_BK, d->K - k0);
            const int klenc = (klen + VEL - 1) / VEL * VEL;   // whole 16-byte pieces: the pad elements of a packed row are 0
            const TS* __restrict__ fk = reinterpret_cast<const TS*>(d->fk) + k0;
            for (int n0 = 0; n0 < d->N; n0 += GEMMV_NT, ++it) {
                const int stage = it % GEMMV_STAGES, rows = min(GEMMV_NT, d->N - n0);
                mbar_wait(bar_empty(stage), ((it / GEMMV_STAGES) & 1) ^ 1);
                if (lane == 0) mbar_expect_tx(bar_full(stage), (uint32_t)(rows * (klenc * (int)sizeof(TS) + RP * 8)));
                __syncwarp();
                if (lane < rows) {
                    const uint32_t dstA = Sm_s + (uint32_t)((stage * WSV_STAGE_DOUBLES + lane * GEMMV_S) * 8);
                    bulk_g2s(dstA, fk + (long long)(n0 + lane) * d->row_stride, (uint32_t)(klenc * (int)sizeof(TS)), bar_full(stage));
                    bulk_g2s(dstA + (uint32_t)(GEMMV_NT * GEMMV_S * 8), gP + (long long)(n0 + lane) * RP, (uint32_t)(RP * 8), bar_full(stage));
                }
            }
        }
        return;
    }

    asm volatile("setmaxnreg.inc.sync.aligned.u32 232;" ::: "memory");
    constexpr int NFW0 = (NFRAG + 1) / 2, NFW1 = NFRAG / 2;
    const int wm = warp & 3, wn = warp >> 2;
    int it = 0;
    // one tile (or one column part of a tile): this warp's 32 k x (8 * NFW) replica columns from column cbcol on
    auto run_tile = [&](auto nf_tag, const int cbcol, const TableDesc* d, double* G, const int kt) {
        constexpr int NFW = decltype(nf_tag)::value;  // fragments of this warp
        double acc[4][NFW][2];
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < NFW; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
        // bounded chains: every GEMM_FLUSH stages (512 datapoints) the register tile is added
        // into this CTA's own G tile (thread-private addresses, L2 resident) and cleared, as the forward kernel does
        const int k0 = kt * GEMMV_BK;
        auto flushG = [&](bool first) {
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const int k = k0 + wm * 32 + i * 8 + (lane >> 2);
#pragma unroll
                for (int j = 0; j < NFW; ++j) {
                    if (k < d->K) {
                        double2* q = reinterpret_cast<double2*>(G + (long long)k * RP + cbcol + j * 8 + 2 * (lane & 3));
                        const double2 o = first ? make_double2(0.0, 0.0) : *q;
                        *q = make_double2(acc[i][j][0] + o.x, acc[i][j][1] + o.y);
                    }
                    acc[i][j][0] = acc[i][j][1] = 0.0;
                }
            }
        };
        bool flushed = false;
        int nst = 0;
        for (int n0 = 0; n0 < d->N; n0 += GEMMV_NT, ++it, ++nst) {
            const int stage = it % GEMMV_STAGES, rows = min(GEMMV_NT, d->N - n0);
            mbar_wait(bar_full(stage), (it / GEMMV_STAGES) & 1);
            // A fragment: row m = k (lane >> 2), col = datapoint (lane & 3)  ->  As[n][k]
            const TS* At = reinterpret_cast<const TS*>(Sm + stage * WSV_STAGE_DOUBLES) + (lane & 3) * PS + wm * 32 + (lane >> 2);
            const double* Bt = Sm + stage * WSV_STAGE_DOUBLES + GEMMV_NT * GEMMV_S + (lane & 3) * GEMMV_S + cbcol + (lane >> 2);
            if (rows == GEMMV_NT) {
#pragma unroll
                for (int n4 = 0; n4 < GEMMV_NT / 4; ++n4) {
                    double a[4], b[NFW];
#pragma unroll
                    for (int i = 0; i < 4; ++i) a[i] = (double)At[n4 * 4 * PS + i * 8];
#pragma unroll
                    for (int j = 0; j < NFW; ++j) b[j] = Bt[n4 * 4 * GEMMV_S + j * 8];
#pragma unroll
                    for (int j = 0; j < NFW; ++j)
#pragma unroll
                        for (int i = 0; i < 4; ++i) dmma884(acc[i][j][0], acc[i][j][1], a[i], b[j]);
                }
            } else {
                for (int n4 = 0; n4 * 4 < rows; ++n4) {
                    const bool live = n4 * 4 + (lane & 3) < rows;
                    double a[4], b[NFW];
#pragma unroll
                    for (int i = 0; i < 4; ++i) a[i] = (double)At[n4 * 4 * PS + i * 8];
#pragma unroll
                    for (int j = 0; j < NFW; ++j) b[j] = live ? Bt[n4 * 4 * GEMMV_S + j * 8] : 0.0;
#pragma unroll
                    for (int j = 0; j < NFW; ++j)
#pragma unroll
                        for (int i = 0; i < 4; ++i) dmma884(acc[i][j][0], acc[i][j][1], a[i], b[j]);
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_empty(stage));
            if ((nst + 1) % GEMM_FLUSH == 0 && n0 + GEMMV_NT < d->N) {
                flushG(!flushed);
                flushed = true;
            }
        }
        flushG(!flushed);
    };
    for (int t = blockIdx.x; t < p.ntiles; t += gridDim.x) {
        const TableDesc* d;
        const double* gP;
        double* G;
        int kt, part;
        tile_of(t, d, gP, G, kt, part);
        if (part < 0) {
            if (wn == 0) run_tile(std::integral_constant<int, NFW0>{}, 0, d, G, kt);
            else run_tile(std::integral_constant<int, NFW1>{}, NFW0 * 8, d, G, kt);
        } else if constexpr (!GROUPED && NFRAG % 4 == 0) {
            // column part of a tail tile: NFRAG / nparts fragments, half of them per warp column
            if constexpr (NFRAG % 8 == 0) {
                if (p.nparts == 4) {
                    constexpr int Q = NFRAG / 8;
                    run_tile(std::integral_constant<int, Q>{}, (part * 2 + wn) * Q * 8, d, G, kt);
                    continue;
                }
            }
            constexpr int H = NFRAG / 4;
            run_tile(std::integral_constant<int, H>{}, (part * 2 + wn) * H * 8, d, G, kt);
        }
    }
}


}  // namespace fk

namespace fk {

// ---------------------------------------------------------------------------------------------------
// R >> 1 contraction for DIS tables (SURVEY 8(a) rows a4 + a5; the paper's flat operation of Table 3,
// PAPER.md:83-100, is this with one pseudo-flavour):  Sigma[n][r] = sum_k FK[n][k] * f[r][slot(k)],
// slot(k) = flav_c * nx + i.  The luminosity of a DIS table is a ROW of the replica-innermost copy fT, so the
// B tile of a stage is 32 bulk copies of fT rows (any k-order: the producer decodes k); no luminosity is built and
// the consumers run the plain DMMA loop.  Same producer / consumer split, mbarrier ring, split-K partials, periodic
// flush and level-2 reduction as fk_gemm_fwd_ws_kernel; tiles of 128 datapoints (a partial last tile computes on
// stale rows that are never stored).  Shared memory is zeroed once, so a k-step that reaches past the end of a K
// range multiplies zeroed B rows with finite stale A columns.
constexpr int WSD_STAGES = 3;
__host__ __device__ inline size_t wsd_smem_bytes(int RP) {
    return (size_t)WSD_STAGES * (WS_STAGE_DOUBLES + GEMM_KT * gemm_sb(RP)) * 8 + 2 * WSD_STAGES * 8;
}

template <int NFRAG>
__global__ void __launch_bounds__(WS_THREADS, 1)
fk_gemm_dis_ws_kernel(const __grid_constant__ WsFwdParams p) {
    pdl_trigger();
    extern __shared__ __align__(128) unsigned char fk_smem[];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const TableDesc& d = p.desc;
    const int RP = p.RP, SB = gemm_sb(RP);
    constexpr int NFW = NFRAG / 2;
    const int mtiles = (d.N + GEMM_BM - 1) / GEMM_BM;
    const int m0 = ((int)blockIdx.x % mtiles) * GEMM_BM, ks = (int)blockIdx.x / mtiles;
    const int kbeg = min(d.K, ks * p.kper), kend = min(d.K, kbeg + p.kper);
    const int nst = (kend - kbeg + GEMM_KT - 1) / GEMM_KT;

    double* As = reinterpret_cast<double*>(fk_smem);               // [STAGES][128][36]
    double* Bs = As + WSD_STAGES * WS_STAGE_DOUBLES;                // [STAGES][32][SB]   fT rows of the stage's k
    const uint32_t As_s = (uint32_t)__cvta_generic_to_shared(As), Bs_s = (uint32_t)__cvta_generic_to_shared(Bs);
    const uint32_t bar0 = Bs_s + (uint32_t)(WSD_STAGES * GEMM_KT * SB * 8);
    auto bar_full = [&](int s) { return bar0 + 8u * s; };
    auto bar_empty = [&](int s) { return bar0 + 8u * (WSD_STAGES + s); };
    for (int t = tid; t < WSD_STAGES * (WS_STAGE_DOUBLES + GEMM_KT * SB); t += WS_THREADS) As[t] = 0.0;
    if (tid == 0) {
        for (int s = 0; s < WSD_STAGES; ++s) {
            mbar_init(bar_full(s), WS_PRODUCER_WARPS);   // one arrive.expect_tx per producer warp
            mbar_init(bar_empty(s), WS_CONSUMER_WARPS);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // the zeros before any bulk copy lands
    __syncthreads();
    pdl_wait();   // fT of the transpose kernel launched just before

    if (warp >= WS_CONSUMER_WARPS) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 40;" ::: "memory");
        // four producer warps (a bulk copy costs its warp ~57 cycles of issue, fk_gemm_fwd_ws_kernel): warp pw copies the
        // datapoints 32*pw .. 32*pw + 31 of the FK tile, warp 0 also the 32 fT rows of the stage
        const int pw = warp - WS_CONSUMER_WARPS;
        const double* __restrict__ fk = reinterpret_cast<const double*>(d.fk);
        const uint64_t pol = l2_evict_first_policy();
        const int rows_valid = min(GEMM_BM, d.N - m0);
        const int my_rows = max(0, min(32, rows_valid - 32 * pw));
        for (int it = 0; it < nst; ++it) {
            const int stage = it % WSD_STAGES, k0 = kbeg + it * GEMM_KT;
            const int len = min(GEMM_KT, kend - k0), lenc = (len + 1) & ~1;   // whole 16-byte pieces: the pad element of a row is 0
            mbar_wait(bar_empty(stage), ((it / WSD_STAGES) & 1) ^ 1);
            // rows of fT for the k of this stage; rows past the end of the range are zeroed by this lane
            const uint32_t brow = Bs_s + (uint32_t)((stage * GEMM_KT + lane) * SB * 8);
            if (pw == 0 && lane >= len)
                for (int c = 0; c < RP; c += 2) asm volatile("st.shared.v2.f64 [%0], {%1, %1};" ::"r"(brow + (uint32_t)c * 8u), "d"(0.0) : "memory");
            __syncwarp();
            if (lane == 0) mbar_expect_tx(bar_full(stage), (uint32_t)((my_rows * lenc + (pw == 0 ? len * RP : 0)) * 8));
            __syncwarp();
            if (pw == 0 && lane < len) {
                int ia, ib;
                decode_k(d, p.chan.a, p.chan.b, k0 + lane, ia, ib);
                bulk_g2s(brow, p.fT + (long long)ia * RP, (uint32_t)(RP * 8), bar_full(stage));
            }
            const int row = lane + 32 * pw;
            if (lane < my_rows)
                bulk_g2s_stream(As_s + (uint32_t)((stage * WS_STAGE_DOUBLES + row * GEMM_SA) * 8),
                                fk + (long long)(m0 + row) * d.row_stride + k0, (uint32_t)(lenc * 8), bar_full(stage), pol);
        }
        return;
    }

    // consumers: warp tile 32 datapoints x (8 * NFW) replicas, plain DMMA loop
    asm volatile("setmaxnreg.inc.sync.aligned.u32 232;" ::: "memory");
    const int wm = warp & 3, wn = warp >> 2, cbcol = wn * NFW * 8;
    double acc[4][NFW][2];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < NFW; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
    double* out = p.gpart + (long long)ks * d.N * RP;
    auto flush = [&](bool first) {
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int n = m0 + wm * 32 + i * 8 + (lane >> 2);
            double2* q = reinterpret_cast<double2*>(out + (long long)n * RP + cbcol + 2 * (lane & 3));
            double2 o[NFW];
#pragma unroll
            for (int j = 0; j < NFW; ++j) o[j] = (!first && n < d.N) ? q[j * 4] : make_double2(0.0, 0.0);
#pragma unroll
            for (int j = 0; j < NFW; ++j) {
                if (n < d.N) q[j * 4] = make_double2(acc[i][j][0] + o[j].x, acc[i][j][1] + o[j].y);
                acc[i][j][0] = acc[i][j][1] = 0.0;
            }
        }
    };
    bool flushed = false;
    for (int it = 0; it < nst; ++it) {
        const int stage = it % WSD_STAGES;
        const int nsteps = (min(GEMM_KT, kend - (kbeg + it * GEMM_KT)) + 3) >> 2;
        mbar_wait(bar_full(stage), (it / WSD_STAGES) & 1);
        const double* At = As + stage * WS_STAGE_DOUBLES + (wm * 32 + (lane >> 2)) * GEMM_SA + (lane & 3);
        const double* Bt = Bs + (stage * GEMM_KT + (lane & 3)) * SB + cbcol + (lane >> 2);
#pragma unroll
        for (int s = 0; s < GEMM_KT / 4; ++s) {
            if (s < nsteps) {
                double a[4], b[NFW];
#pragma unroll
                for (int i4 = 0; i4 < 4; ++i4) a[i4] = At[i4 * 8 * GEMM_SA + s * 4];
#pragma unroll
                for (int j8 = 0; j8 < NFW; ++j8) b[j8] = Bt[s * 4 * SB + j8 * 8];
#pragma unroll
                for (int j8 = 0; j8 < NFW; ++j8)
#pragma unroll
                    for (int i4 = 0; i4 < 4; ++i4) dmma884(acc[i4][j8][0], acc[i4][j8][1], a[i4], b[j8]);
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_empty(stage));
        if ((it + 1 + wn * (GEMM_FLUSH / 2)) % GEMM_FLUSH == 0) {
            flush(!flushed);
            flushed = true;
        }
    }
    flush(!flushed);
}

}  // namespace fk
