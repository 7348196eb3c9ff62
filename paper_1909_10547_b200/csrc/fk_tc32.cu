// fk_tc32.cu -- R >> 1 dense contraction of the fp32 variant on the 5th-generation tensor cores (tcgen05, sm_100a).
//
//   sigma[n][r] = sum_{c,i} f[r][a_c][i] * T[n][(c,i)][r],   T[n][(c,i)][r] = sum_j FK[n][c][i][j] * f[r][b_c][j]     Eq. (1)
//
// BASELINE.json config 3 ("the dense contraction case where tensor cores may apply", fp32 variant), SURVEY 8(a) row
// a4 / 8(f).3; the paper's own observation that the GPU wins in the large N x R rows (Table 3).
// tcgen05 has no f64 kind, so only the fp32 variant (reading R18: fp32 table, fp32 f, 1e-5 of sum|terms|)
// can use it; a single TF32 pass misses that tolerance (1.7e-5), so every fp32 operand x is split
// exactly into x = hi + lo, hi = x with the 13 low mantissa bits cleared (what kind::tf32 reads of an fp32 word),
// lo = x - hi (exact in fp32), and three products are accumulated in fp32:  fb_hi FK_hi + fb_lo FK + fb FK_lo.  The first
// runs as kind::tf32; the two correction products are 2^-11 of the result, so 8-bit operands suffice for them and they run
// as kind::f16 on bf16 roundings of fb_lo, FK, fb, FK_lo (twice the MMA rate, half the shared-memory bytes): each
// rounding costs <= 2^-9 of a 2^-11 term, like the dropped lo x lo term <= 2^-20 of |term|.
//
// The contraction is done in the factored order above, which the flat GEMM view hides: the inner sum over j has
// the SAME right-hand factor f[b_c][.][r] for every x-row i and every datapoint n of a channel, so the tensor-core operand
// built from f changes once per CHANNEL (not once per k), and the outer factor f[a_c][i][r] is one scalar per accumulator
// row, applied by the epilogue in full fp32.  No luminosity tile is ever formed, in HBM or on chip.
//
//   D^T[r][n] = sum_j fb[r][j] * FK[n][(c,i)][j]          one tcgen05.mma chain per (c, i) row: M = 128 replicas (TMEM lanes),
//                                                         N = 128 datapoints, K = nx rounded up to 8
//   A operand  fb_hi (tf32), bf16(fb_lo), bf16(fb) of channel c, [128 r][K], in TENSOR MEMORY (tcgen05.st, double
//              buffered per channel): shared memory carries only the table;
//   B operand  FK rows [128 n][K] of (c, i): raw tile by TMA (cp.async.bulk.tensor, 128-byte swizzle, box 32 k x 128 n,
//              two boxes; a box must start on 16 bytes, which is why fp32 tables are packed with x-rows padded to a
//              multiple of 4 elements (TableDesc::jp); k beyond nx meets zero rows of fb), bf16(FK) and bf16(FK_lo)
//              tiles ([128 n][64 bf16], one swizzle row each) by 4 splitter warps;
//   epilogue   acc[n] += f[a_c][i][r] * D^T[r][n]  (tcgen05.ld, lane = replica r), two-level fp32 sums (x-rows of a channel, then channels);
//              at the end the partial tile goes to gpart[range][n][r] (split level 1).
// One CTA = one item (128-datapoint tile, range of (c, i) rows), warp-specialised: warp 0 TMA producer, warp 1 MMA
// issuer, warp 2 TMEM allocator, warps 4-7 splitter + fb operand, warps 8-15 epilogue.  Level 2 (fixed-order sum over
// the ranges, in fp64) is fk_gemm_reduce_kernel.  No atomics: bitwise repeatable.
#include "fk_tc32.h"

#include <cuda.h>
#include <cuda_bf16.h>

#include <cstdio>
#include <cstring>
#include <mutex>

namespace fk {

namespace {

constexpr int TC_THREADS = 512;            // 4 warpgroups: control, splitter, 2 x epilogue
constexpr int TC_SPLIT_WARPS = 4;
constexpr int TC_EPI_WARPS = 8;
constexpr int TC_RAW_STAGES = 3;           // TMA ring of raw FK tiles
constexpr int TC_LO_STAGES = 2;            // FK_lo tiles
constexpr int TC_BOX_BYTES = TC_BN * 32 * 4;      // one TMA box: 128 rows x 32 fp32 = 16 KB
constexpr int TC_STAGE_BYTES = 2 * TC_BOX_BYTES;  // K extent <= 64: two boxes
constexpr int TC_TMEM_COLS = 512;          // D: 2 x 128 columns; fb operand: 2 buffers x (tf32 hi 64 + bf16 lo 32 + bf16 full 32)
constexpr uint32_t TC_TMEM_A = 256, TC_A_LO_BF = 64, TC_A_FULL_BF = 96;
constexpr uint32_t TF32_MASK = 0xffffe000u;

// ---- PTX wrappers (one instruction each) -------------------------------------------------------------------------
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
// Every wait of this kernel is bounded: a protocol error (or a fault in an asynchronous copy that never signals its
// barrier) traps after ~10^7 polls instead of hanging the device (the launch then fails with an error the C-ABI call
// reports); -DFK_TC32_DEBUG prints which waiter it was.
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity, int what = 0) {
    uint32_t done = 0;
    for (uint32_t spins = 0; !done; ++spins) {
        asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}\n"
                     : "=r"(done)
                     : "r"(bar), "r"(parity)
                     : "memory");
        if (!done && spins > (1u << 24)) {
#ifdef FK_TC32_DEBUG
            printf("fk_tc32: barrier wait timed out (waiter %d, block %d, thread %d, barrier 0x%x, parity %u)\n", what, (int)blockIdx.x,
                   (int)threadIdx.x, bar, parity);
            asm volatile("exit;");   // every waiter times out in turn and the kernel ends: the messages get flushed
#endif
            asm volatile("trap;");
        }
    }
}
#ifdef FK_TC32_TIMING
// debug build only: cycles spent in a wait, added to `acc`
#define FK_TWAIT(ACC, ...) do { const long long t0_ = clock64(); mbar_wait(__VA_ARGS__); ACC += clock64() - t0_; } while (0)
#else
#define FK_TWAIT(ACC, ...) mbar_wait(__VA_ARGS__)
#endif
// one lane of a converged warp (the same one every time): control flow stays warp-uniform around the single-thread
// instructions (TMA, tcgen05.mma, tcgen05.commit), so their operands live in uniform registers
__device__ __forceinline__ bool elect_one() {
    uint32_t pred;
    asm volatile("{\n.reg .pred P;\nelect.sync _|P, 0xffffffff;\nselp.u32 %0, 1, 0, P;\n}\n" : "=r"(pred));
    return pred != 0;
}
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const void* tmap, int c0, int c1, uint32_t bar) {
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];" ::"r"(dst),
                 "l"(tmap), "r"(bar), "r"(c0), "r"(c1)
                 : "memory");
}
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
// D[tmem] (+)= A[tmem] . B[smem desc]^T, kind::tf32, issued by one thread for the CTA
__device__ __forceinline__ void tc_mma_tf32_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\ntcgen05.mma.cta_group::1.kind::tf32 [%0], [%1], %2, %3, p;\n}\n" ::"r"(d_tmem),
        "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate)
        : "memory");
}
// D[tmem] += A[tmem] . B[smem desc]^T, kind::f16 on bf16 operands (K = 16 per instruction)
__device__ __forceinline__ void tc_mma_bf16_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\ntcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n}\n" ::"r"(d_tmem),
        "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate)
        : "memory");
}
__device__ __forceinline__ void tc_ld16(uint32_t taddr, float (&v)[16]) {
    uint32_t r[16];
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]),
          "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
        : "r"(taddr));
#pragma unroll
    for (int e = 0; e < 16; ++e) v[e] = __uint_as_float(r[e]);
}
__device__ __forceinline__ void tc_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tc_st8(uint32_t taddr, const float (&v)[8]) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"r"(taddr), "r"(__float_as_uint(v[0])),
                 "r"(__float_as_uint(v[1])), "r"(__float_as_uint(v[2])), "r"(__float_as_uint(v[3])), "r"(__float_as_uint(v[4])),
                 "r"(__float_as_uint(v[5])), "r"(__float_as_uint(v[6])), "r"(__float_as_uint(v[7]))
                 : "memory");
}
__device__ __forceinline__ void tc_st4(uint32_t taddr, const uint32_t (&v)[4]) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};" ::"r"(taddr), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]) : "memory");
}
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {   // element k (even) in the low half, k + 1 in the high half
    const __nv_bfloat162 b = __floats2bfloat162_rn(lo, hi);
    return *reinterpret_cast<const uint32_t*>(&b);
}
__device__ __forceinline__ void tc_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

// UMMA shared-memory descriptor, K-major operand in the 128-byte-swizzle canonical layout (rows of 128 bytes, 8-row
// groups 1024 bytes apart): start address >> 4 | LBO (unused for swizzled K-major) | SBO = 1024 >> 4 | version 1 |
// layout type 2 (SWIZZLE_128B).  Advancing k by 8 fp32 inside the swizzle row = start address + 32 bytes.
__device__ __forceinline__ uint64_t umma_desc_sw128(uint32_t smem_addr) {
    return (uint64_t)((smem_addr & 0x3ffffu) >> 4) | (1ull << 16) | ((uint64_t)(1024 >> 4) << 32) | (1ull << 46) | (2ull << 61);
}
// UMMA instruction descriptor: D fp32, A and B tf32, both K-major, no negate / sparsity / saturate
__host__ __device__ constexpr uint32_t umma_idesc_tf32(int M, int N) {
    return (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}
// the same with bf16 operands (kind::f16)
__host__ __device__ constexpr uint32_t umma_idesc_bf16(int M, int N) {
    return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}

// barrier slots
enum { BAR_FK_FULL = 0, BAR_FK_FREE = 4, BAR_LO_FULL = 8, BAR_LO_FREE = 10, BAR_A_FULL = 12, BAR_A_FREE = 14, BAR_ACC_FULL = 16, BAR_ACC_FREE = 18, BAR_COUNT = 20 };

constexpr size_t TC_SMEM_BYTES = (size_t)(TC_RAW_STAGES + TC_LO_STAGES) * TC_STAGE_BYTES + 8 * BAR_COUNT + 16 + 1024;   // + alignment slack

template <bool GROUPED>
__global__ void __launch_bounds__(TC_THREADS, 1)
fk_tc32_fwd_kernel(const __grid_constant__ Tc32Params p) {
    extern __shared__ unsigned char fk_smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31;
    const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);   // provably warp-uniform: role branches do not diverge
    pdl_trigger();   // the level-2 reduction may be scheduled under this grid's tail (it waits for the partials itself)
#ifdef FK_TC32_TIMING
    long long tw[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    const long long t_start = clock64();
#else
    long long tw[1];   // unused: FK_TWAIT ignores it
    (void)tw;
#endif

    const TableDesc* dp = &p.desc;
    const uint8_t* __restrict__ cha = p.chan.a;
    const uint8_t* __restrict__ chb = p.chan.b;
    const float* __restrict__ fT = p.fT;
    float* gpart = p.gpart;
    const void* tmap = p.tmap;
    const int RP = p.RP;
    int n0, ks, tper;
    if constexpr (GROUPED) {
        const ColSeg it = p.items[blockIdx.x];
        dp = &p.descs[it.table];
        cha = dp->chan_a;
        chb = dp->chan_b;
        fT += dp->f_off * RP;
        gpart += dp->tc_gp_off * RP;
        tmap = dp->tmap;
        n0 = it.kblock;
        ks = it.split;
        tper = dp->tc_kper;
    } else {
        const int ntiles = (p.desc.N + TC_BN - 1) / TC_BN;
        n0 = ((int)blockIdx.x % ntiles) * TC_BN;
        ks = (int)blockIdx.x / ntiles;
        tper = p.tper;
    }
    const TableDesc& d = *dp;
    const int nx = d.nx, cstride = d.cstride, jp = d.jp;
    const int nk8 = (nx + 7) >> 3;                    // tf32 MMA steps of 8 k per (c, i) row
    const int nk16 = (nk8 + 1) >> 1;                  // bf16 MMA steps of 16 k
    const int T = d.C * nx;                           // (c, i) rows of the table
    const int t0 = min(T, ks * tper), ntl = min(T, t0 + tper) - t0;
    const int rows = min(TC_BN, d.N - n0), NT = (rows + 15) & ~15;   // UMMA N
    const int c_first = t0 / nx, i_first = t0 - c_first * nx;
    const int c_last = ntl > 0 ? (t0 + ntl - 1) / nx : c_first;

    const uint32_t base = ((uint32_t)__cvta_generic_to_shared(fk_smem_raw) + 1023u) & ~1023u;
    const uint32_t sm_raw = base, sm_lo = base + TC_RAW_STAGES * TC_STAGE_BYTES;
    const uint32_t sm_bars = sm_lo + TC_LO_STAGES * TC_STAGE_BYTES, sm_tmem_slot = sm_bars + 8u * BAR_COUNT;
    auto bar = [&](int slot) { return sm_bars + 8u * (uint32_t)slot; };

    if (tid == 0) {
        for (int s = 0; s < 4; ++s) {
            mbar_init(bar(BAR_FK_FULL + s), 1);
            mbar_init(bar(BAR_FK_FREE + s), 1);
        }
        for (int s = 0; s < 2; ++s) {
            mbar_init(bar(BAR_LO_FULL + s), TC_SPLIT_WARPS);
            mbar_init(bar(BAR_LO_FREE + s), 1);
            mbar_init(bar(BAR_A_FULL + s), TC_SPLIT_WARPS);
            mbar_init(bar(BAR_A_FREE + s), 1);
            mbar_init(bar(BAR_ACC_FULL + s), 1);
            mbar_init(bar(BAR_ACC_FREE + s), TC_EPI_WARPS);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    // the bf16 tiles are written up to k = 8 nk8; a last k-step of 16 reads 8 more: zero them once (they meet zero rows of
    // the fb operand, but 0 x NaN of stale shared memory would still poison the accumulator)
    for (uint32_t o = (uint32_t)tid * 16u; o < (uint32_t)(TC_LO_STAGES * TC_STAGE_BYTES); o += TC_THREADS * 16u)
        asm volatile("st.shared.v4.u32 [%0], {%1, %1, %1, %1};" ::"r"(sm_lo + o), "r"(0u) : "memory");
    fence_async_smem();
    if (warp == 2) {   // TMEM: all 512 columns (one CTA per SM by shared memory), address written to shared memory
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(sm_tmem_slot), "r"(TC_TMEM_COLS) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    uint32_t tmem_base;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(sm_tmem_slot));

    if (warp < 4) {
        // ============================ control warpgroup ============================
        asm volatile("setmaxnreg.dec.sync.aligned.u32 40;" ::: "memory");
        if (warp == 0) {
            // ---- TMA producer: the raw FK rows of (c, i) for 128 datapoints -> ring slot t % TC_RAW_STAGES
            const bool leader = elect_one();
            const uint32_t tx = nk8 > 4 ? TC_STAGE_BYTES : TC_BOX_BYTES;
            int c = c_first, i = i_first;
            for (int t = 0; t < ntl; ++t) {
                const int slot = t % TC_RAW_STAGES;
                FK_TWAIT(tw[6], bar(BAR_FK_FREE + slot), ((t / TC_RAW_STAGES) & 1) ^ 1, 1);
                const int k0 = c * cstride + i * jp;   // 16-byte aligned: jp and cstride are multiples of 4
                const uint32_t dst = sm_raw + (uint32_t)slot * TC_STAGE_BYTES;
                if (leader) {
                    mbar_expect_tx(bar(BAR_FK_FULL + slot), tx);
                    tma_load_2d(dst, tmap, k0, n0, bar(BAR_FK_FULL + slot));
                    if (nk8 > 4) tma_load_2d(dst + TC_BOX_BYTES, tmap, k0 + 32, n0, bar(BAR_FK_FULL + slot));
                }
                __syncwarp();
                if (++i == nx) { i = 0; ++c; }
            }
        } else if (warp == 1) {
            // ---- MMA issuer: the whole warp walks the loop, one elected lane issues
            const bool leader = elect_one();
            const uint32_t idesc = umma_idesc_tf32(128, NT), idesc_bf = umma_idesc_bf16(128, NT);
            int i = i_first, cc = 0;
            bool newch = true;
            for (int t = 0; t < ntl; ++t) {
                const int slot = t % TC_RAW_STAGES, ls = t & 1, buf = t & 1, abuf = cc & 1;
                if (newch) {
                    mbar_wait(bar(BAR_A_FULL + abuf), (cc >> 1) & 1, 2);
                    newch = false;
                }
                FK_TWAIT(tw[0], bar(BAR_ACC_FREE + buf), ((t >> 1) & 1) ^ 1, 3);
                FK_TWAIT(tw[1], bar(BAR_FK_FULL + slot), (t / TC_RAW_STAGES) & 1, 4);
                tc_fence_after();
                const uint32_t d_acc = tmem_base + (uint32_t)buf * 128u;
                const uint32_t a_hi = tmem_base + TC_TMEM_A + (uint32_t)abuf * 128u;
                // 8 fp32 = 16 bf16 = 32 bytes (descriptor + 2) along the swizzle row; the second fp32 box holds k 32..63
                const uint64_t braw = umma_desc_sw128(sm_raw + (uint32_t)slot * TC_STAGE_BYTES);
                const uint64_t bfk = umma_desc_sw128(sm_lo + (uint32_t)ls * TC_STAGE_BYTES);                  // bf16(FK)
                const uint64_t blo = umma_desc_sw128(sm_lo + (uint32_t)ls * TC_STAGE_BYTES + TC_BOX_BYTES);   // bf16(FK_lo)
                if (leader) {
#pragma unroll
                    for (int k8 = 0; k8 < 8; ++k8) {
                        if (k8 < nk8) {
                            const uint64_t b = braw + (uint64_t)((k8 >> 2) * (TC_BOX_BYTES >> 4) + (k8 & 3) * 2);
                            tc_mma_tf32_ts(d_acc, a_hi + 8u * (uint32_t)k8, b, idesc, k8 > 0 ? 1u : 0u);
                        }
                    }
                }
                __syncwarp();
                FK_TWAIT(tw[2], bar(BAR_LO_FULL + ls), (t >> 1) & 1, 5);
                tc_fence_after();
                if (leader) {
#pragma unroll
                    for (int k16 = 0; k16 < 4; ++k16) {
                        if (k16 < nk16) {
                            tc_mma_bf16_ts(d_acc, a_hi + TC_A_LO_BF + 8u * (uint32_t)k16, bfk + (uint64_t)(k16 * 2), idesc_bf, 1u);
                            tc_mma_bf16_ts(d_acc, a_hi + TC_A_FULL_BF + 8u * (uint32_t)k16, blo + (uint64_t)(k16 * 2), idesc_bf, 1u);
                        }
                    }
                    tc_commit(bar(BAR_FK_FREE + slot));
                    tc_commit(bar(BAR_LO_FREE + ls));
                    tc_commit(bar(BAR_ACC_FULL + buf));
                }
                if (++i == nx) {   // last row of the channel: its fb operand buffer goes back to the builders
                    i = 0;
                    if (leader) tc_commit(bar(BAR_A_FREE + abuf));
                    ++cc;
                    newch = true;
                }
                __syncwarp();
            }
        }
    } else if (warp < 4 + TC_SPLIT_WARPS) {
        // ============================ splitter + fb operand ============================
        asm volatile("setmaxnreg.dec.sync.aligned.u32 96;" ::: "memory");
        const int st = tid - 128;                  // datapoint row of the tile (splitter) = replica lane (fb operand)
        const uint32_t lane_addr = (uint32_t)((warp & 3) * 32) << 16;
        // fb_hi / fb_lo of channel c -> TMEM operand buffer cc & 1: lane r, column j (zero for j >= nx and r >= RP)
        auto build_a = [&](int cc, int c) {
            const int abuf = cc & 1;
            mbar_wait(bar(BAR_A_FREE + abuf), ((cc >> 1) & 1) ^ 1, 6);
            tc_fence_after();
            const float* src = fT + (long long)chb[c] * nx * RP + st;
            const uint32_t a_hi = tmem_base + lane_addr + TC_TMEM_A + (uint32_t)abuf * 128u;
            for (int j0 = 0; j0 < 16 * nk16; j0 += 8) {   // the bf16 operands span whole k-steps of 16: zero beyond nx
                float hi[8];
                uint32_t lob[4], fullb[4];
#pragma unroll
                for (int e = 0; e < 8; e += 2) {
                    const float v0 = (j0 + e < nx && st < RP) ? __ldg(src + (long long)(j0 + e) * RP) : 0.f;
                    const float v1 = (j0 + e + 1 < nx && st < RP) ? __ldg(src + (long long)(j0 + e + 1) * RP) : 0.f;
                    hi[e] = __uint_as_float(__float_as_uint(v0) & TF32_MASK);
                    hi[e + 1] = __uint_as_float(__float_as_uint(v1) & TF32_MASK);
                    lob[e >> 1] = pack_bf16(v0 - hi[e], v1 - hi[e + 1]);
                    fullb[e >> 1] = pack_bf16(v0, v1);
                }
                tc_st8(a_hi + (uint32_t)j0, hi);
                tc_st4(a_hi + TC_A_LO_BF + (uint32_t)(j0 >> 1), lob);
                tc_st4(a_hi + TC_A_FULL_BF + (uint32_t)(j0 >> 1), fullb);
            }
            tc_wait_st();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(bar(BAR_A_FULL + abuf));
        };
        int c = c_first, i = i_first, cc = 0;
        pdl_wait();   // fT is written by the transpose kernel just before this launch (the table itself is not: TMA runs ahead)
        if (ntl > 0) build_a(0, c);
        bool build_next = c < c_last;   // the next channel's operand is built under the first row of this one
        for (int t = 0; t < ntl; ++t) {
            const int slot = t % TC_RAW_STAGES, ls = t & 1;
            FK_TWAIT(tw[3], bar(BAR_LO_FREE + ls), ((t >> 1) & 1) ^ 1, 7);
            FK_TWAIT(tw[4], bar(BAR_FK_FULL + slot), (t / TC_RAW_STAGES) & 1, 8);
#ifdef FK_TC32_TIMING
            const long long ts0 = clock64();
#endif
            if (st < NT) {
                // bf16(FK) and bf16(FK_lo), FK_lo = x - tf32(x): logical fp32 chunk q of row st sits at 16-byte position
                // (q & 7) ^ (st & 7) of the row's 128 bytes in box q >> 3; two fp32 chunks make bf16 chunk m = q / 2 at
                // position m ^ (st & 7) of the row's 128 bytes in its tile
                const uint32_t src = sm_raw + (uint32_t)slot * TC_STAGE_BYTES + (uint32_t)st * 128u;
                const uint32_t dst = sm_lo + (uint32_t)ls * TC_STAGE_BYTES + (uint32_t)st * 128u;
                // all loads of the row first (volatile asm keeps program order: loads interleaved with the stores of the
                // previous chunk would make every chunk wait out a full shared-memory round trip under the tensor core's own
                // traffic), then the arithmetic and the stores
                float x[8][8];
#pragma unroll
                for (int m = 0; m < 8; ++m) {
                    if (m < nk8) {
#pragma unroll
                        for (int h = 0; h < 2; ++h) {
                            const int q = 2 * m + h;
                            const uint32_t o = (uint32_t)(q >> 3) * TC_BOX_BYTES + (uint32_t)(((q & 7) ^ (st & 7)) << 4);
                            asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(x[m][4 * h]), "=f"(x[m][4 * h + 1]), "=f"(x[m][4 * h + 2]), "=f"(x[m][4 * h + 3]) : "r"(src + o));
                        }
                    }
                }
#pragma unroll
                for (int m = 0; m < 8; ++m) {
                    if (m < nk8) {
                        uint32_t fb4[4], lo4[4];
#pragma unroll
                        for (int e = 0; e < 8; e += 2) {
                            const float l0 = x[m][e] - __uint_as_float(__float_as_uint(x[m][e]) & TF32_MASK);
                            const float l1 = x[m][e + 1] - __uint_as_float(__float_as_uint(x[m][e + 1]) & TF32_MASK);
                            fb4[e >> 1] = pack_bf16(x[m][e], x[m][e + 1]);
                            lo4[e >> 1] = pack_bf16(l0, l1);
                        }
                        const uint32_t od = (uint32_t)((m ^ (st & 7)) << 4);
                        asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(dst + od), "r"(fb4[0]), "r"(fb4[1]), "r"(fb4[2]), "r"(fb4[3]) : "memory");
                        asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(dst + TC_BOX_BYTES + od), "r"(lo4[0]), "r"(lo4[1]), "r"(lo4[2]), "r"(lo4[3]) : "memory");
                    }
                }
            }
#ifdef FK_TC32_TIMING
            const long long ts1 = clock64();
#endif
            fence_async_smem();   // generic-proxy stores -> visible to the tensor core (async proxy)
            __syncwarp();
            if (lane == 0) mbar_arrive(bar(BAR_LO_FULL + ls));
#ifdef FK_TC32_TIMING
            tw[7] += ts1 - ts0;
            tw[5] += clock64() - ts1;
#endif
            if (build_next) {
                build_a(cc + 1, c + 1);
                build_next = false;
            }
            if (++i == nx) {
                i = 0;
                ++c;
                ++cc;
                build_next = c < c_last;
            }
        }
    } else {
        // ============================ epilogue ============================
        // the CTA owns 512 x 128 registers: 128 x 40 (control) + 128 x 96 (splitter) + 256 x 168 (here) fits
        asm volatile("setmaxnreg.inc.sync.aligned.u32 168;" ::: "memory");
        const int q = warp & 3, h = (warp - 4 - TC_SPLIT_WARPS) >> 2;   // TMEM lane quarter = warp % 4, column half
        const int r = q * 32 + lane;                                     // replica of this thread's TMEM lane
        const bool live = h * 64 < NT;
        // two-level fp32 accumulation: `acc` over the x-rows of one channel (<= TC_MAX_NX terms), `tot` over channels
        float acc[64], tot[64];
#pragma unroll
        for (int e = 0; e < 64; ++e) acc[e] = tot[e] = 0.f;
        int c = c_first, i = i_first;
        auto load_fa = [&](int cq, int iq) { return r < RP ? __ldg(fT + ((long long)cha[cq] * nx + iq) * RP + r) : 0.f; };
        pdl_wait();   // fT (see the builders); also orders the final gpart stores after the previous call's readers
        float fa_next = ntl > 0 ? load_fa(c, i) : 0.f;
        for (int t = 0; t < ntl; ++t) {
            const int buf = t & 1;
            const float fa = fa_next;
            const bool chan_end = ++i == nx;
            if (chan_end) { i = 0; ++c; }
            if (t + 1 < ntl) fa_next = load_fa(c, i);
            FK_TWAIT(tw[5], bar(BAR_ACC_FULL + buf), (t >> 1) & 1, 9);
            tc_fence_after();
            if (live) {
                const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(buf * 128 + h * 64);
#pragma unroll
                for (int g = 0; g < 4; ++g) {
                    if (h * 64 + g * 16 < NT) {   // warp-uniform
                        float v[16];
                        tc_ld16(taddr + (uint32_t)(g * 16), v);
                        tc_wait_ld();
#pragma unroll
                        for (int e = 0; e < 16; ++e) acc[g * 16 + e] = fmaf(fa, v[e], acc[g * 16 + e]);
                    }
                }
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(bar(BAR_ACC_FREE + buf));
            if (chan_end || t == ntl - 1) {
#pragma unroll
                for (int e = 0; e < 64; ++e) { tot[e] += acc[e]; acc[e] = 0.f; }
            }
        }
        if (live && r < RP) {
            float* out = gpart + ((long long)ks * d.N + n0 + h * 64) * RP + r;
#pragma unroll
            for (int e = 0; e < 64; ++e)
                if (h * 64 + e < rows) out[(long long)e * RP] = tot[e];
        }
    }
#ifdef FK_TC32_TIMING
    if (blockIdx.x == 5 && lane == 0 && (warp == 0 || warp == 1 || warp == 4 || warp == 8))
        printf("tc32 timing block %d warp %d: total %lld | issuer waits ACC_FREE %lld FK_FULL %lld LO_FULL %lld | splitter waits LO_FREE %lld FK_FULL %lld | "
               "epilogue waits ACC_FULL (splitter: fence+arrive) %lld | tma waits FK_FREE %lld | splitter work %lld\n", (int)blockIdx.x, warp, clock64() - t_start, tw[0], tw[1], tw[2], tw[3], tw[4], tw[5], tw[6], tw[7]);
#endif
    tc_fence_before();
    __syncthreads();
    if (warp == 2) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(TC_TMEM_COLS) : "memory");
    }
}

}  // namespace

size_t tc32_smem_bytes() { return TC_SMEM_BYTES; }

bool tc32_encode_tensor_map(void* out_host, const void* fk_dev, long long row_stride, int K, int N) {
    typedef CUresult (*EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                 const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                 CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    static std::once_flag once;
    static EncodeFn fn = nullptr;
    std::call_once(once, [] {
        void* sym = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &sym, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess)
            fn = (EncodeFn)sym;
    });
    if (!fn) return false;
    static_assert(sizeof(CUtensorMap) == TC_TMAP_BYTES, "tensor map size");
    alignas(64) CUtensorMap tm;
    const cuuint64_t gdim[2] = {(cuuint64_t)K, (cuuint64_t)N};
    const cuuint64_t gstr[1] = {(cuuint64_t)row_stride * 4u};
    const cuuint32_t box[2] = {32, TC_BN};
    const cuuint32_t estr[2] = {1, 1};
    const CUresult rc = fn(&tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<void*>(fk_dev), gdim, gstr, box, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (rc != CUDA_SUCCESS) return false;
    memcpy(out_host, &tm, sizeof tm);
    return true;
}

cudaError_t tc32_fwd_launch(const Tc32Params& p, int grid, bool grouped, bool pdl, cudaStream_t s) {
    auto kern = grouped ? fk_tc32_fwd_kernel<true> : fk_tc32_fwd_kernel<false>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TC_SMEM_BYTES);
    if (e != cudaSuccess) return e;
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof cfg);
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(TC_THREADS);
    cfg.dynamicSmemBytes = TC_SMEM_BYTES;
    cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;   // fk_common.cuh, pdl_wait
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, p);
}

}  // namespace fk
