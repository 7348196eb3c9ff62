// fk_sparse.cuh -- element-sparse storage of an FK table (FK_STORE_SPARSE; "element-sparse FK for tables
// with many stored zeros", BASELINE config 1's 30 %).  Not storing what is absent is the method's own idea one level up
// (only the active flavour combinations are stored); real FK tables are zero wherever the kinematics
// forbid an (x_i, x_j) pair.  The R = 1 convolution and its VJP are HBM-bound (2 flop per 8 bytes), so bytes not stored
// are time not spent.
//
// Layout (fp64, packed k-order of fk_common.cuh: channel-major, x innermost), per datapoint row n and per block of
// SP_BLOCK = 512 consecutive k (the k-block of one column-kernel CTA):
//   blk[n][kb]       {off: index of the block's first value in vals; wpre: seven 9-bit counts of the nonzeros before
//                     words 1..7; mask[8]: bit (k % 64) of word (k % 512) / 64 is set iff FK[n][k] != 0}     80 bytes
//   vals[]           the nonzero values of all blocks, in (n, kb, k) order                                  8 bytes each
// i.e. 8 bytes per nonzero + 0.156 bytes per element: 72 % of the dense bytes at 30 % zeros, 52 % at 50 %.
//
// Kernels: thread (warp w, lane l) of a CTA owns k = kb*512 + 64 w + l and k + 32 -- bits l and l + 32 of ITS warp's mask
// word.  A CTA first brings the 80-byte index records of its rows into shared memory with coalesced 128-bit loads (so the
// dependent step index -> value costs its latency once per CTA, not once per batch of rows), then every warp finds its
// value positions with two popcounts and its lanes read consecutive values (coalesced), U rows in flight.  Everything after the load is the dense column kernel's arithmetic: luminosity in
// registers, multi-value butterfly, fixed-order CTA sum, level-1 partials; level 2 and the VJP stage 2 are the dense
// kernels (the column sums G[k] are dense).  Fixed orders, no atomics: bitwise repeatable.
#pragma once

#include "fk_common.cuh"
#include "fk_fwd.cuh"
#include "fk_vjp.cuh"

namespace fk {

constexpr int SP_BLOCK = 512;   // = FWD_THREADS * 2: the k-blocks of the plan (fk_api.cu make_plan) are the sparse blocks

struct SparseBlk {
    unsigned long long off;
    unsigned long long wpre;
    unsigned long long mask[8];
};
static_assert(sizeof(SparseBlk) == 80, "SparseBlk is five 16-byte pieces");
constexpr int SP_CHUNK = 64;   // rows whose index records a CTA stages at a time

// logical index of packed position kp (hadronic: channel blocks of cstride, x-rows jp apart; DIS: c * nx + i), -1: padding
__device__ __forceinline__ long long sp_klog(int kind, int nx, int C, int cstride, int jp, int K, int kp) {
    if (kp >= K) return -1;
    if (kind == KIND_HADRONIC) {
        const int c = kp / cstride, rem = kp - c * cstride;
        const int i = rem / jp, j = rem - i * jp;
        return (i < nx && j < nx) ? ((long long)i * nx + j) * C + c : -1;
    }
    const int c = kp / nx, i = kp - c * nx;
    return (long long)i * C + c;
}

// Pass 1 (FILL = false): masks and the nonzero count of every (n, kb) block.  Pass 2 (FILL = true), after the host's
// exclusive scan of the counts into hdr[].off: the per-word prefix counts and the values.  One CTA of 256 threads per block.
template <bool FILL>
__global__ void __launch_bounds__(256)
fk_sparse_build_kernel(const double* __restrict__ in, int kind, int N, int nx, int C, int K, int cstride, int jp, int nkb,
                       unsigned int* __restrict__ count, SparseBlk* __restrict__ sblk, double* __restrict__ vals) {
    __shared__ unsigned int wcnt[8];
    const long long blk = blockIdx.x;
    const int n = (int)(blk / nkb), kb = (int)(blk - (long long)n * nkb);
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    const long long klen = kind == KIND_HADRONIC ? (long long)C * nx * nx : (long long)C * nx;
    const int ka = kb * SP_BLOCK + 64 * w + l;
    const long long la = sp_klog(kind, nx, C, cstride, jp, K, ka), lb = sp_klog(kind, nx, C, cstride, jp, K, ka + 32);
    const double va = la >= 0 ? in[(long long)n * klen + la] : 0.0, vb = lb >= 0 ? in[(long long)n * klen + lb] : 0.0;
    const unsigned int ma = __ballot_sync(0xffffffffu, va != 0.0), mb = __ballot_sync(0xffffffffu, vb != 0.0);
    if (l == 0) wcnt[w] = __popc(ma) + __popc(mb);
    __syncthreads();
    if (!FILL) {
        if (l == 0) sblk[blk].mask[w] = (unsigned long long)ma | ((unsigned long long)mb << 32);
        if (threadIdx.x == 0) {
            unsigned int tot = 0;
            for (int q = 0; q < 8; ++q) tot += wcnt[q];
            count[blk] = tot;
        }
        return;
    }
    unsigned int pre = 0;
    for (int q = 0; q < w; ++q) pre += wcnt[q];
    const unsigned long long off = sblk[blk].off;
    if (va != 0.0) vals[off + pre + __popc(ma & ((1u << l) - 1u))] = va;
    if (vb != 0.0) vals[off + pre + __popc(ma) + __popc(mb & ((1u << l) - 1u))] = vb;
    if (threadIdx.x == 0) {
        unsigned long long wp = 0, run = 0;
        for (int q = 1; q < 8; ++q) {
            run += wcnt[q - 1];
            wp |= run << (9 * (q - 1));
        }
        sblk[blk].wpre = wp;
    }
}

// index records of rows [r0, r0 + nrows) of k-block kb -> shared memory (five 16-byte pieces each)
__device__ __forceinline__ void sp_stage_index(const TableDesc& d, int nkb, int kb, int r0, int nrows, SparseBlk* dst, int tid, int nthreads) {
    for (int t = tid; t < nrows * 5; t += nthreads) {
        const int m = t / 5, q = t - m * 5;
        const uint4* src = reinterpret_cast<const uint4*>(reinterpret_cast<const SparseBlk*>(d.sp_blk) + ((long long)(r0 + m) * nkb + kb)) + q;
        reinterpret_cast<uint4*>(dst + m)[q] = __ldg(src);
    }
}
// The two values of this thread in the row whose staged index record is `b` (0 where the bit is clear or `live` is
// false).  wsh = 9 * (w - 1) (w > 0), lt = (1 << lane) - 1.  The loads are predicated (no select afterwards) and the asm
// is not volatile: the table is read-only, so the compiler is free to issue the U rows' index reads first and their
// value loads back to back.
__device__ __forceinline__ void sp_load_pair(const double* __restrict__ vals, const SparseBlk& b, int w, uint32_t wsh, uint32_t lt, int lane,
                                             bool live, double& xa, double& xb) {
    const uint2 m = *reinterpret_cast<const uint2*>(&b.mask[w]);   // bits l and l + 32 of this warp's word
    const unsigned int ma = m.x, mb = m.y, lbit = lt + 1u;
    const unsigned int wp = w ? (unsigned int)(b.wpre >> wsh) & 0x1ffu : 0u;
    const double* vp = vals + (b.off + wp);
    const unsigned int ia = __popc(ma & lt), ib = __popc(ma) + __popc(mb & lt);
    const unsigned int pa = live ? ma & lbit : 0u, pb = live ? mb & lbit : 0u;
    xa = xb = 0.0;
    const uint64_t pol = stream_policy();   // L2 evict-first: the values are read once
    asm("{\n.reg .pred p;\nsetp.ne.u32 p, %2, 0;\n@p ld.global.nc.L1::no_allocate.L2::cache_hint.f64 %0, [%1], %3;\n}\n" : "+d"(xa) : "l"(vp + ia), "r"(pa), "l"(pol));
    asm("{\n.reg .pred p;\nsetp.ne.u32 p, %2, 0;\n@p ld.global.nc.L1::no_allocate.L2::cache_hint.f64 %0, [%1], %3;\n}\n" : "+d"(xb) : "l"(vp + ib), "r"(pb), "l"(pol));
}

// a1 + a2 + a3 level 1 over a sparse table: same CTA decomposition (k-block x datapoint range), same partials as
// fk_fwd_column_kernel
template <int RT, int U>
__global__ void __launch_bounds__(FWD_THREADS)
fk_fwd_sparse_kernel(const __grid_constant__ FwdParams p) {
    pdl_trigger();
    constexpr int LPR = 32 / U;
    __shared__ double red[2][FWD_WARPS][U][RT];
    __shared__ __align__(16) SparseBlk sblk[SP_CHUNK];
    const TableDesc& d = p.desc;
    const int kblock = blockIdx.x % d.nchunks, split = blockIdx.x / d.nchunks;
    const int R = p.R;
    const int rb = (int)((long long)d.N * split / d.fsplit);
    const int re = (int)((long long)d.N * (split + 1) / d.fsplit);   // the plan gives <= 32 rows per range (fk_api.cu)
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int ka = kblock * SP_BLOCK + 64 * warp + lane;
    sp_stage_index(d, d.nchunks, kblock, rb, min(re - rb, SP_CHUNK), sblk, threadIdx.x, FWD_THREADS);

    double L[RT][2];
    {
        const int fstride = d.nfl * d.nx;
        const double* __restrict__ f = reinterpret_cast<const double*>(p.f);
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            const int k = ka + 32 * e;
            int ia = 0, ib = -1;
            bool in = k < d.K;
            if (in) decode_k(d, p.chan.a, p.chan.b, k, ia, ib);
            in = in && ia >= 0;
#pragma unroll
            for (int r = 0; r < RT; ++r) {
                const int rr = p.r0 + r;
                double lum = 0.0;
                if (in && rr < R) {
                    lum = __ldg(f + (long long)rr * fstride + ia);
                    if (ib >= 0) lum *= __ldg(f + (long long)rr * fstride + ib);
                }
                L[r][e] = lum;
            }
        }
    }
    __syncthreads();
    const double* __restrict__ vals = reinterpret_cast<const double*>(d.fk);
    const uint32_t wsh = warp ? 9u * (uint32_t)(warp - 1) : 0u, lt = (1u << lane) - 1u;
    int buf = 0;
    for (int m = rb; m < re; m += U, buf ^= 1) {
        if (m > rb && (m - rb) % SP_CHUNK == 0) {   // ranges longer than a chunk (not planned today): restage
            __syncthreads();
            sp_stage_index(d, d.nchunks, kblock, m, min(re - m, SP_CHUNK), sblk, threadIdx.x, FWD_THREADS);
            __syncthreads();
        }
        const int mrel = (m - rb) % SP_CHUNK, nlive = re - m;   // U divides SP_CHUNK: a batch never straddles chunks
        double xa[U], xb[U];
        const SparseBlk* rec = sblk + mrel;
        if (nlive >= U) {   // whole batch: immediate offsets, no selects
#pragma unroll
            for (int u = 0; u < U; ++u) sp_load_pair(vals, rec[u], warp, wsh, lt, lane, true, xa[u], xb[u]);
        } else {
#pragma unroll
            for (int u = 0; u < U; ++u) sp_load_pair(vals, rec[u < nlive ? u : 0], warp, wsh, lt, lane, u < nlive, xa[u], xb[u]);
        }
        double pr[RT][U];
#pragma unroll
        for (int u = 0; u < U; ++u)
#pragma unroll
            for (int r = 0; r < RT; ++r) pr[r][u] = fma(xb[u], L[r][1], xa[u] * L[r][0]);
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
            for (int wq = 1; wq < FWD_WARPS; ++wq) s += red[buf][wq][u][r];
            const int n = m + u, rr = p.r0 + r;
            if (n < re && rr < R) {
                if (d.nchunks == 1)
                    reinterpret_cast<double*>(p.sigma)[(long long)n * R + rr] = s;
                else
                    p.part[((long long)n * R + rr) * d.nchunks + kblock] = s;
            }
        }
    }
}

// a6 stage 1 over a sparse table: G[split][r][k] = sum_{n in range} g[n][r] FK[n][k] (dense column sums)
template <int RT, int U>
__global__ void __launch_bounds__(COLSUM_THREADS)
fk_colsum_sparse_kernel(const __grid_constant__ ColsumParams p) {
    pdl_trigger();
    pdl_wait();
    __shared__ double gs[(COLSUM_MAX_ROWS + U) * RT];
    __shared__ __align__(16) SparseBlk sblk[2][SP_CHUNK];   // double buffered: the next chunk's records load under this chunk's values
    const TableDesc& d = p.desc;
    const int kblock = blockIdx.x % p.nkb, split = blockIdx.x / p.nkb;
    const int R = p.R;
    const int rb = (int)((long long)d.N * split / d.nsplit);
    const int re = (int)((long long)d.N * (split + 1) / d.nsplit);
    const int rows = re - rb;
    const double* __restrict__ g = reinterpret_cast<const double*>(p.g);
    const int rows_pad = (rows + U - 1) / U * U;
    for (int t = threadIdx.x; t < rows_pad * RT; t += COLSUM_THREADS) {
        const int m = t / RT, r = t - m * RT, rr = p.r0 + r;
        gs[t] = (m < rows && rr < R) ? __ldg(g + (long long)(rb + m) * R + rr) : 0.0;
    }
    __syncthreads();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int ka = kblock * SP_BLOCK + 64 * warp + lane;
    double acc[2][RT][2];   // two interleaved chains
#pragma unroll
    for (int a = 0; a < 2; ++a)
#pragma unroll
        for (int r = 0; r < RT; ++r) acc[a][r][0] = acc[a][r][1] = 0.0;
    static_assert(SP_CHUNK % U == 0, "whole batches per chunk");
    const double* __restrict__ vals = reinterpret_cast<const double*>(d.fk);
    const uint32_t wsh = warp ? 9u * (uint32_t)(warp - 1) : 0u, lt = (1u << lane) - 1u;
    sp_stage_index(d, p.nkb, kblock, rb, min(rows, SP_CHUNK), sblk[0], threadIdx.x, COLSUM_THREADS);
    __syncthreads();
    for (int c0 = 0, cb = 0; c0 < rows; c0 += SP_CHUNK, cb ^= 1) {
        // the next chunk's index records: loaded into registers now, stored after this chunk's arithmetic
        uint4 nxt[2];
        const int nrows_next = min(rows - (c0 + SP_CHUNK), SP_CHUNK);
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int t = threadIdx.x + h * COLSUM_THREADS;
            if (t < nrows_next * 5) {
                const int m = t / 5, q = t - m * 5;
                nxt[h] = __ldg(reinterpret_cast<const uint4*>(reinterpret_cast<const SparseBlk*>(d.sp_blk) + ((long long)(rb + c0 + SP_CHUNK + m) * p.nkb + kblock)) + q);
            }
        }
        const int mend = min(rows_pad, c0 + SP_CHUNK);
        for (int m = c0; m < mend; m += U) {
            const int nlive = rows - m;
            double xa[U], xb[U];
            const SparseBlk* rec = &sblk[cb][m - c0];
            if (nlive >= U) {   // whole batch: immediate offsets, no selects
#pragma unroll
                for (int u = 0; u < U; ++u) sp_load_pair(vals, rec[u], warp, wsh, lt, lane, true, xa[u], xb[u]);
            } else {
#pragma unroll
                for (int u = 0; u < U; ++u) sp_load_pair(vals, rec[u < nlive ? u : 0], warp, wsh, lt, lane, u < nlive, xa[u], xb[u]);
            }
#pragma unroll
            for (int u = 0; u < U; ++u)
#pragma unroll
                for (int r = 0; r < RT; ++r) {
                    const double gv = gs[(m + u) * RT + r];   // 0 on the padded rows
                    acc[u & 1][r][0] = fma(gv, xa[u], acc[u & 1][r][0]);
                    acc[u & 1][r][1] = fma(gv, xb[u], acc[u & 1][r][1]);
                }
        }
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int t = threadIdx.x + h * COLSUM_THREADS;
            if (t < nrows_next * 5) reinterpret_cast<uint4*>(&sblk[cb ^ 1][t / 5])[t % 5] = nxt[h];
        }
        __syncthreads();
    }
#pragma unroll
    for (int r = 0; r < RT; ++r) {
        const int rr = p.r0 + r;
        if (rr >= R) continue;
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            const int k = ka + 32 * e;
            if (k < d.K) p.G[((long long)split * R + rr) * d.K + k] = acc[0][r][e] + acc[1][r][e];
        }
    }
}

}  // namespace fk
