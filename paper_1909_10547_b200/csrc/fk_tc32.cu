// fk_tc32.cu -- R >> 1 dense contraction of the fp32 variant on the 5th-generation tensor cores (tcgen05, sm_100a).
//
//   Sigma[n][r] = sum_k FK[n][k] * L[k][r],   L[(c,i,j)][r] = f[r][a_c][i] * f[r][b_c][j]       Eq. (1)
//
// BASELINE.json config 3 ("the dense contraction case where tensor cores may apply", fp32 variant), SURVEY 8(a) row
// a4 / 8(f).3; the paper's own observation that the GPU wins in the large N x R rows (Table 3).
// tcgen05 has no f64 kind, so only the fp32 variant (reading R18: fp32 table, fp32 f, 1e-5 of sum|terms|)
// can use it; a single TF32 pass misses that tolerance (1.7e-5), so every fp32 operand x is split
// exactly into x = hi + lo, hi = x with the 13 low mantissa bits cleared (what kind::tf32 reads of an fp32 word),
// lo = x - hi (exact in fp32), and three products are accumulated in fp32:  FK_hi L_hi + FK_hi L_lo + FK_lo L_hi
// (the dropped lo x lo term and the truncation of lo to 11 bits are each <= 2^-20 of |term|).
//
// One CTA = one item (128-datapoint tile, K range), persistent for its K range, warp-specialised:
//   warp 0      TMA producer: FK tiles [128 n][32 k] fp32 straight from the packed table through a tensor map
//               (cp.async.bulk.tensor, 128-byte swizzle, rows beyond N and k beyond K zero-filled) into a 3-4 stage ring;
//   warp 1      bulk-copies, once per channel, the [nx][RP] block of the replica-innermost f[b_c] (double buffered);
//   warp 2      issues tcgen05.mma (kind::tf32, M = 128, cta_group::1), per 8 k:
//                 D[:, 0:2RP]   (+)= FK_raw  . [L_hi ; L_lo]^T     (N = 2 RP: the L tiles are stacked, FK is read once)
//                 D[:, RP:2RP]   += FK_lo   . L_hi^T               (N = RP)
//               accumulators live in TMEM (2 x 256 columns, double buffered); tcgen05.commit releases the stages;
//   warps 4-11  builders: the luminosity tile is built ON THE FLY (never in HBM): thread = (replica r,
//               k chunk) multiplies the shared f[b_c][j][r] by f[a_c][i][r] (prefetched one stage ahead), splits into
//               hi / lo and stores both tiles in the UMMA K-major 128-byte-swizzle layout; the same warps split the
//               raw FK tile (FK_lo = x - hi(x), element-wise, layout-agnostic);
//   warps 12-19 epilogue: every TC_FLUSH stages the finished accumulator is drained with tcgen05.ld and added, in
//               fp32 round-to-nearest, into per-thread register accumulators, which bounds the chain the tensor core
//               accumulates with its own rounding; at the end the partial tile goes to gpart[ks][n][r] (split-K level 1).
// Level 2 (fixed-order sum over the K ranges, in fp64) is fk_gemm_reduce_kernel.  No atomics: bitwise repeatable.
#include "fk_tc32.h"

#include <cuda.h>

#include <cstdio>
#include <cstring>
#include <mutex>

namespace fk {

namespace {

constexpr int TC_THREADS = 640;            // 5 warpgroups: control, 2 x builders, 2 x epilogue
constexpr int TC_BUILD_WARPS = 8;
constexpr int TC_EPI_WARPS = 8;
constexpr int TC_B_STAGES = 2;             // FK_lo / L tile ring
constexpr int TC_FK_TILE = TC_BM * TC_KT * 4;   // 16 KB
constexpr int TC_TMEM_COLS = 512;
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
// barrier) traps after ~10^7 polls instead of hanging the device; `what` identifies the waiter in the message.
__device__ __noinline__ void mbar_timeout(int what, uint32_t bar, uint32_t parity) {
    printf("fk_tc32: barrier wait timed out (waiter %d, block %d, thread %d, barrier 0x%x, parity %u)\n", what, (int)blockIdx.x,
           (int)threadIdx.x, bar, parity);
    __trap();
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity, int what = 0) {
    uint32_t done = 0;
    for (uint32_t spins = 0; !done; ++spins) {
        asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}\n"
                     : "=r"(done)
                     : "r"(bar), "r"(parity)
                     : "memory");
        if (!done && spins > (1u << 24)) mbar_timeout(what, bar, parity);
    }
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst), "l"(src),
                 "r"(bytes), "r"(bar)
                 : "memory");
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
// D[tmem] (+)= A[smem desc] . B[smem desc]^T, kind::tf32, issued by one thread for the CTA
__device__ __forceinline__ void tc_mma_tf32(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\ntcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n}\n" ::"r"(d_tmem),
        "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate)
        : "memory");
}
__device__ __forceinline__ void tc_ld8(uint32_t taddr, float (&v)[8]) {
    uint32_t r0, r1, r2, r3, r4, r5, r6, r7;
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                 : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3), "=r"(r4), "=r"(r5), "=r"(r6), "=r"(r7)
                 : "r"(taddr));
    v[0] = __uint_as_float(r0); v[1] = __uint_as_float(r1); v[2] = __uint_as_float(r2); v[3] = __uint_as_float(r3);
    v[4] = __uint_as_float(r4); v[5] = __uint_as_float(r5); v[6] = __uint_as_float(r6); v[7] = __uint_as_float(r7);
}
__device__ __forceinline__ void tc_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

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

struct Smem {
    uint32_t fk_raw, fk_lo, ltile, fb, bars, tmem_slot;   // shared-space byte addresses
    int ltile_bytes, fb_bytes;
};
__host__ __device__ inline size_t tc32_layout(int nx, int RP, int fk_stages, uint32_t base, Smem* out) {
    Smem s;
    s.fk_raw = base;
    s.fk_lo = s.fk_raw + (uint32_t)fk_stages * TC_FK_TILE;
    s.ltile = s.fk_lo + TC_B_STAGES * TC_FK_TILE;
    s.ltile_bytes = 2 * RP * TC_KT * 4;             // L_hi rows then L_lo rows
    s.fb = s.ltile + TC_B_STAGES * (uint32_t)s.ltile_bytes;
    s.fb_bytes = nx * RP * 4;
    s.bars = (s.fb + 2u * (uint32_t)s.fb_bytes + 7u) & ~7u;
    s.tmem_slot = s.bars + 8u * 24u;
    if (out) *out = s;
    return (size_t)(s.tmem_slot + 16u - base);
}

// barrier slots inside Smem::bars
enum { BAR_FK_FULL = 0, BAR_FK_FREE = 4, BAR_BUILT = 8, BAR_SLOT_FREE = 10, BAR_FB_FULL = 12, BAR_FB_FREE = 14, BAR_ACC_FULL = 16, BAR_ACC_FREE = 18 };

template <int NC, bool GROUPED>   // NC = RP / 16: 8-column groups of an epilogue thread
__global__ void __launch_bounds__(TC_THREADS, 1)
fk_tc32_fwd_kernel(const __grid_constant__ Tc32Params p) {
    extern __shared__ unsigned char fk_smem_raw[];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    constexpr int RP = NC * 16;

    const TableDesc* dp = &p.desc;
    const uint8_t* __restrict__ cha = p.chan.a;
    const uint8_t* __restrict__ chb = p.chan.b;
    const float* __restrict__ fT = p.fT;
    float* gpart = p.gpart;
    const void* tmap = p.tmap;
    int m0, ks, kper;
    if constexpr (GROUPED) {
        const ColSeg it = p.items[blockIdx.x];
        dp = &p.descs[it.table];
        cha = dp->chan_a;
        chb = dp->chan_b;
        fT += dp->f_off * RP;
        gpart += dp->tc_gp_off * RP;
        tmap = dp->tmap;
        m0 = it.kblock;
        ks = it.split;
        kper = dp->tc_kper;
    } else {
        const int mtiles = (p.desc.N + TC_BM - 1) / TC_BM;
        m0 = ((int)blockIdx.x % mtiles) * TC_BM;
        ks = (int)blockIdx.x / mtiles;
        kper = p.kper;
    }
    const TableDesc& d = *dp;
    const int nx = d.nx, cstride = d.cstride, S_FK = p.fk_stages;
    const int kbeg = min(d.K, ks * kper), kend = min(d.K, kbeg + kper);
    const int nst = (kend - kbeg + TC_KT - 1) / TC_KT;   // stages of this item (0: an empty range still writes zeros)
    const int c0 = kbeg / cstride, c1 = kbeg < kend ? (kend - 1) / cstride : c0 - 1;

    Smem sm;
    const uint32_t base = ((uint32_t)__cvta_generic_to_shared(fk_smem_raw) + 1023u) & ~1023u;
    tc32_layout(nx, RP, S_FK, base, &sm);
    auto bar = [&](int slot) { return sm.bars + 8u * (uint32_t)slot; };

    if (tid == 0) {
        for (int s = 0; s < 4; ++s) {
            mbar_init(bar(BAR_FK_FULL + s), 1);
            mbar_init(bar(BAR_FK_FREE + s), 1);
        }
        for (int s = 0; s < 2; ++s) {
            mbar_init(bar(BAR_BUILT + s), TC_BUILD_WARPS);
            mbar_init(bar(BAR_SLOT_FREE + s), 1);
            mbar_init(bar(BAR_FB_FULL + s), 1);
            mbar_init(bar(BAR_FB_FREE + s), TC_BUILD_WARPS);
            mbar_init(bar(BAR_ACC_FULL + s), 1);
            mbar_init(bar(BAR_ACC_FREE + s), TC_EPI_WARPS);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 3) {   // TMEM: all 512 columns (one CTA per SM by shared memory), address written to shared memory
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(sm.tmem_slot), "r"(TC_TMEM_COLS) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    uint32_t tmem_base;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(sm.tmem_slot));

    if (warp < 4) {
        // ============================ control warpgroup ============================
        asm volatile("setmaxnreg.dec.sync.aligned.u32 40;" ::: "memory");
        if (warp == 0 && lane == 0) {
            // ---- TMA producer: FK tile of stage s -> ring slot s % S_FK
            for (int s = 0; s < nst; ++s) {
                const int slot = s % S_FK;
                mbar_wait(bar(BAR_FK_FREE + slot), ((s / S_FK) & 1) ^ 1, 1);
                mbar_expect_tx(bar(BAR_FK_FULL + slot), TC_FK_TILE);
                tma_load_2d(sm.fk_raw + (uint32_t)slot * TC_FK_TILE, tmap, kbeg + s * TC_KT, m0, bar(BAR_FK_FULL + slot));
            }
        } else if (warp == 1 && lane == 0) {
            // ---- f[b_c][.][.] of channel c -> buffer (c - c0) & 1
            for (int c = c0, cc = 0; c <= c1; ++c, ++cc) {
                const int buf = cc & 1;
                mbar_wait(bar(BAR_FB_FREE + buf), ((cc >> 1) & 1) ^ 1, 2);
                mbar_expect_tx(bar(BAR_FB_FULL + buf), (uint32_t)sm.fb_bytes);
                bulk_g2s(sm.fb + (uint32_t)buf * sm.fb_bytes, fT + (long long)chb[c] * nx * RP, (uint32_t)sm.fb_bytes, bar(BAR_FB_FULL + buf));
            }
        } else if (warp == 2 && lane == 0) {
            // ---- MMA issuer
            constexpr uint32_t idesc_stacked = umma_idesc_tf32(TC_BM, 2 * RP), idesc_single = umma_idesc_tf32(TC_BM, RP);
            for (int s = 0; s < nst; ++s) {
                const int fl = s / TC_FLUSH, a = fl & 1;
                const bool fresh = s % TC_FLUSH == 0;
                if (fresh) mbar_wait(bar(BAR_ACC_FREE + a), ((fl >> 1) & 1) ^ 1, 3);
                const int bs = s % TC_B_STAGES, fs = s % S_FK;
                mbar_wait(bar(BAR_BUILT + bs), (s / TC_B_STAGES) & 1, 4);
                mbar_wait(bar(BAR_FK_FULL + fs), (s / S_FK) & 1, 5);
                tc_fence_after();
                const uint32_t d_acc = tmem_base + (uint32_t)a * 256u;
                const uint64_t a_raw = umma_desc_sw128(sm.fk_raw + (uint32_t)fs * TC_FK_TILE);
                const uint64_t a_lo = umma_desc_sw128(sm.fk_lo + (uint32_t)bs * TC_FK_TILE);
                const uint64_t b_l = umma_desc_sw128(sm.ltile + (uint32_t)bs * sm.ltile_bytes);
#pragma unroll
                for (int k8 = 0; k8 < TC_KT / 8; ++k8) {
                    const uint64_t adv = (uint64_t)(k8 * 32 >> 4);   // 8 fp32 = 32 bytes along the swizzle row
                    tc_mma_tf32(d_acc, a_raw + adv, b_l + adv, idesc_stacked, (fresh && k8 == 0) ? 0u : 1u);
                    tc_mma_tf32(d_acc + RP, a_lo + adv, b_l + adv, idesc_single, 1u);
                }
                tc_commit(bar(BAR_FK_FREE + fs));
                tc_commit(bar(BAR_SLOT_FREE + bs));
                if ((s + 1) % TC_FLUSH == 0 || s == nst - 1) tc_commit(bar(BAR_ACC_FULL + a));
            }
        }
    } else if (warp < 4 + TC_BUILD_WARPS) {
        // ============================ builders ============================
        const int bt = tid - 128, r = bt & 127, half = bt >> 7;
        const bool rlive = r < RP;
        const uint32_t magic = (uint32_t)((0x100000000ull + (uint64_t)nx - 1) / (uint64_t)nx);   // ceil(2^32 / nx)
        const int nxnx = nx * nx;
        int c_lo = c0, cbase = c0 * cstride;   // channel of the first k of the current stage
        int cc_ready = -1;                     // channels (relative to c0) whose f[b_c] block has been waited for
        // coordinates of the chunk starting at k: channel c, position rem inside it
        auto coords = [&](int k, int clo, int cb, int& c, int& rem) {
            const bool nxt = k >= cb + cstride;
            c = clo + (nxt ? 1 : 0);
            rem = k - cb - (nxt ? cstride : 0);
        };
        // f[a_c][i][r] and f[a_c][i + 1][r] of the 4 chunks of a stage
        float fa_cur[4][2], fa_nxt[4][2];
        auto load_fa = [&](float (&dst)[4][2], int k0, int clo, int cb) {
#pragma unroll
            for (int m = 0; m < 4; ++m) {
                const int k = k0 + 4 * half + 8 * m;
                dst[m][0] = dst[m][1] = 0.f;
                if (rlive && k < kend) {
                    int c, rem;
                    coords(k, clo, cb, c, rem);
                    const int i = (int)__umulhi((uint32_t)rem, magic);
                    const float* src = fT + ((long long)cha[c] * nx) * RP + r;
                    dst[m][0] = __ldg(src + (long long)min(i, nx - 1) * RP);
                    dst[m][1] = __ldg(src + (long long)min(i + 1, nx - 1) * RP);
                }
            }
        };
        if (nst > 0) load_fa(fa_cur, kbeg, c_lo, cbase);
        for (int s = 0; s < nst; ++s) {
            const int k0 = kbeg + s * TC_KT;
            const int bs = s % TC_B_STAGES, fs = s % S_FK;
            // next stage's channel bookkeeping and f[a_c] prefetch
            int c_lo_n = c_lo, cbase_n = cbase;
            if (k0 + TC_KT >= cbase + cstride) { ++c_lo_n; cbase_n += cstride; }
            if (s + 1 < nst) load_fa(fa_nxt, k0 + TC_KT, c_lo_n, cbase_n);

            mbar_wait(bar(BAR_SLOT_FREE + bs), ((s / TC_B_STAGES) & 1) ^ 1, 6);
            const int c_hi = min(c1, (k0 + TC_KT - 1) / cstride) - c0;
            while (cc_ready < c_hi) {
                ++cc_ready;
                mbar_wait(bar(BAR_FB_FULL + (cc_ready & 1)), (cc_ready >> 1) & 1, 7);
            }
            if (rlive) {
                const uint32_t lt = sm.ltile + (uint32_t)bs * sm.ltile_bytes;
#pragma unroll
                for (int m = 0; m < 4; ++m) {
                    const int q = half + 2 * m, k = k0 + 4 * q;
                    float hi[4] = {0.f, 0.f, 0.f, 0.f}, lo[4] = {0.f, 0.f, 0.f, 0.f};
                    if (k < kend) {
                        int c, rem;
                        coords(k, c_lo, cbase, c, rem);
                        const int i = (int)__umulhi((uint32_t)rem, magic), j = rem - i * nx;
                        const uint32_t fbb = sm.fb + (uint32_t)((c - c0) & 1) * sm.fb_bytes + (uint32_t)r * 4u;
#pragma unroll
                        for (int e = 0; e < 4; ++e) {
                            const bool wrap = j + e >= nx;
                            const int je = j + e - (wrap ? nx : 0);
                            float fb;
                            asm volatile("ld.shared.f32 %0, [%1];" : "=f"(fb) : "r"(fbb + (uint32_t)(je * RP) * 4u));
                            const float L = (rem + e < nxnx) ? fb * (wrap ? fa_cur[m][1] : fa_cur[m][0]) : 0.f;   // channel padding: 0
                            hi[e] = __uint_as_float(__float_as_uint(L) & TF32_MASK);
                            lo[e] = L - hi[e];
                        }
                    }
                    // UMMA K-major, 128-byte swizzle: row r, 16-byte chunk q at position q ^ (r & 7); L_lo rows follow L_hi rows
                    const uint32_t off = (uint32_t)r * 128u + (uint32_t)((q ^ (r & 7)) << 4);
                    asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(lt + off), "f"(hi[0]), "f"(hi[1]), "f"(hi[2]), "f"(hi[3]) : "memory");
                    asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(lt + (uint32_t)RP * 128u + off), "f"(lo[0]), "f"(lo[1]), "f"(lo[2]), "f"(lo[3]) : "memory");
                }
            }
            // FK_lo = x - hi(x) over the raw tile (element-wise: the swizzle is the same on both sides)
            mbar_wait(bar(BAR_FK_FULL + fs), (s / S_FK) & 1, 8);
            {
                const uint32_t src = sm.fk_raw + (uint32_t)fs * TC_FK_TILE, dst = sm.fk_lo + (uint32_t)bs * TC_FK_TILE;
#pragma unroll
                for (int m = 0; m < TC_FK_TILE / 16 / (TC_BUILD_WARPS * 32); ++m) {
                    const uint32_t o = (uint32_t)(bt + m * TC_BUILD_WARPS * 32) * 16u;
                    float x0, x1, x2, x3;
                    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(x0), "=f"(x1), "=f"(x2), "=f"(x3) : "r"(src + o));
                    x0 -= __uint_as_float(__float_as_uint(x0) & TF32_MASK);
                    x1 -= __uint_as_float(__float_as_uint(x1) & TF32_MASK);
                    x2 -= __uint_as_float(__float_as_uint(x2) & TF32_MASK);
                    x3 -= __uint_as_float(__float_as_uint(x3) & TF32_MASK);
                    asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(dst + o), "f"(x0), "f"(x1), "f"(x2), "f"(x3) : "memory");
                }
            }
            fence_async_smem();   // generic-proxy stores -> visible to the tensor core (async proxy)
            __syncwarp();
            if (lane == 0) mbar_arrive(bar(BAR_BUILT + bs));
            // a channel whose last k lies in this stage is finished: its f[b_c] buffer goes back to the loader
            if (k0 + TC_KT >= cbase + cstride && c_lo < c1) {
                if (lane == 0) mbar_arrive(bar(BAR_FB_FREE + ((c_lo - c0) & 1)));
            }
            c_lo = c_lo_n;
            cbase = cbase_n;
#pragma unroll
            for (int m = 0; m < 4; ++m) { fa_cur[m][0] = fa_nxt[m][0]; fa_cur[m][1] = fa_nxt[m][1]; }
        }
    } else {
        // ============================ epilogue ============================
        // the CTA owns 640 x 96 registers: 128 x 40 (control) + 256 x 96 (builders) + 256 x 120 (here) fits, more would block forever
        asm volatile("setmaxnreg.inc.sync.aligned.u32 120;" ::: "memory");
        const int ew = warp - 4 - TC_BUILD_WARPS, q = warp & 3, h = ew >> 2;   // TMEM lane quarter = warp % 4, column half
        float acc[NC * 8];
#pragma unroll
        for (int e = 0; e < NC * 8; ++e) acc[e] = 0.f;
        const int nflush = (nst + TC_FLUSH - 1) / TC_FLUSH;
        for (int fl = 0; fl < nflush; ++fl) {
            const int a = fl & 1;
            mbar_wait(bar(BAR_ACC_FULL + a), (fl >> 1) & 1, 9);
            tc_fence_after();
            const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(a * 256 + h * (RP / 2));
#pragma unroll
            for (int g = 0; g < NC; ++g) {
                float v[8], w[8];
                tc_ld8(taddr + (uint32_t)(g * 8), v);          // FK_hi L_hi
                tc_ld8(taddr + (uint32_t)(RP + g * 8), w);     // FK_hi L_lo + FK_lo L_hi
                tc_wait_ld();
#pragma unroll
                for (int e = 0; e < 8; ++e) acc[g * 8 + e] += v[e] + w[e];
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(bar(BAR_ACC_FREE + a));
        }
        const int n = m0 + q * 32 + lane;
        if (n < d.N) {
            float4* out = reinterpret_cast<float4*>(gpart + ((long long)ks * d.N + n) * RP + h * (RP / 2));
#pragma unroll
            for (int g = 0; g < NC * 2; ++g) out[g] = make_float4(acc[4 * g], acc[4 * g + 1], acc[4 * g + 2], acc[4 * g + 3]);
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 3) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(TC_TMEM_COLS) : "memory");
    }
}

}  // namespace

size_t tc32_smem_bytes(int nx, int RP, int* fk_stages) {
    for (int st = 4; st >= 3; --st) {
        const size_t need = tc32_layout(nx, RP, st, 0, nullptr) + 1024;   // + alignment slack
        if (need <= 232448) {
            if (fk_stages) *fk_stages = st;
            return need;
        }
    }
    return 0;
}

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
    const cuuint32_t box[2] = {TC_KT, TC_BM};
    const cuuint32_t estr[2] = {1, 1};
    const CUresult rc = fn(&tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<void*>(fk_dev), gdim, gstr, box, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (rc != CUDA_SUCCESS) return false;
    memcpy(out_host, &tm, sizeof tm);
    return true;
}

cudaError_t tc32_fwd_launch(const Tc32Params& p, int grid, bool grouped, size_t smem, cudaStream_t s) {
#define FK_TC_CASE(NCv)                                                                                                      \
    case NCv: {                                                                                                              \
        auto kern = grouped ? fk_tc32_fwd_kernel<NCv, true> : fk_tc32_fwd_kernel<NCv, false>;                                \
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);                  \
        if (e != cudaSuccess) return e;                                                                                      \
        kern<<<grid, TC_THREADS, smem, s>>>(p);                                                                              \
        break;                                                                                                               \
    }
    switch (p.RP / 16) {
        FK_TC_CASE(1) FK_TC_CASE(2) FK_TC_CASE(3) FK_TC_CASE(4) FK_TC_CASE(5) FK_TC_CASE(6) FK_TC_CASE(7) FK_TC_CASE(8)
        default: return cudaErrorInvalidValue;
    }
#undef FK_TC_CASE
    return cudaGetLastError();
}

}  // namespace fk
