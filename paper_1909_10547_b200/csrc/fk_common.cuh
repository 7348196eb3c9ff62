// fk_common.cuh -- descriptors, index decode and small device helpers shared by the kernels.
// Hand-written for sm_100a.  Nothing here is shared with oracle/ (see include/fkconv.h for the maths).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

namespace fk {

constexpr int KIND_DIS = 0;
constexpr int KIND_HADRONIC = 1;
constexpr int LAYOUT_LOGICAL = 0;  // hadronic k = (i*nx + j)*C + c ; DIS k = i*nA + c   (BASELINE.json order)
constexpr int LAYOUT_PACKED = 1;   // hadronic k = c*cstride + i*jp + j, cstride = nx*jp rounded up to 4 (zero padded) ; DIS k = c*nx + i
                                   // (jp = nx, except fp32 tables: nx rounded up to 4, so that every x-row starts on 16 bytes: TMA)

// Programmatic dependent launch (PDL): the later kernels of a compute call are launched with
// cudaLaunchAttributeProgrammaticStreamSerialization (fk_api.cu, launch_pdl).  A kernel calls pdl_trigger() first thing, so
// that its successor's CTAs are scheduled (and run their prologue) as soon as every CTA of this grid has STARTED, and
// pdl_wait() before its first access to global memory that a predecessor in the stream may write or still read: the wait
// returns once the whole predecessor grid has completed and its memory is visible.  Both are no-ops in a normal launch.
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

constexpr int MAX_C = 1024;   // active flavour pairs / flavours per table
constexpr int MAX_NFL = 256;  // flavour indices are stored as uint8

// Flavour indices of the active channels, passed BY VALUE in kernel-parameter space for single-table
// launches (no H2D copy, no allocation, graph-capturable).  Grouped launches read them from HBM.
struct ChannelList {
    uint8_t a[MAX_C];  // a_c  (DIS: flav_c)
    uint8_t b[MAX_C];  // b_c  (DIS: unused)
};

// One FK table as the kernels see it.
struct TableDesc {
    const void* fk;       // device; datapoint n starts at fk + n*row_stride elements
    long long row_stride; // elements (>= K; PACK pads it to a 16-byte multiple)
    int K;                // contraction length per datapoint: C*nx*nx (hadronic) or nA*nx (DIS)
    int N, nx, nfl, C;
    int cstride;          // PACKED hadronic: elements per channel block (nx*jp rounded up to a multiple of 4)
    int jp;               // PACKED hadronic: elements between consecutive x-rows i of a channel block (>= nx; the gap is zero)
    int kind, layout;
    int vec_ok;           // rows are 16-byte aligned -> 128-bit loads
    int store32;          // the table is stored in fp32 (FK_F32, FK_F32S64)
    // grouped launches only
    const uint8_t* chan_a;   // device copies of the channel list (a_c / b_c)
    const uint8_t* chan_b;
    long long f_off;         // element offset of f_t / df_t inside f_cat for R = 1 (scaled by R)
    long long out_off;       // element offset of sigma_t / g_t inside sigma_cat for R = 1 (scaled by R)
    long long part_off;      // element offset of this table's level-1 partials for R = 1 (scaled by R)
    long long cnt_off;       // first ticket counter of this table (FwdParams::cnt), one per forward datapoint range
    long long g_off;         // element offset of this table's column sums G for R = 1 (scaled by R)
    int nchunks;             // forward: number of k-blocks (= level-1 partials per row)
    int fsplit;              // forward: number of datapoint ranges per k-block
    int nsplit;              // VJP stage 1: number of datapoint ranges per k-block
    // R >> 1 contraction (fk_gemm.cuh), grouped launches only
    const uint32_t* kdec;    // device [K]: k -> (slot a, slot b) codes
    long long gp_off;        // row offset of this table's split-K partial tiles (sum over earlier tables of ksplit * N)
    long long k_off;         // offset of this table's column sums inside G_cat (sum of K over earlier tables)
    int gksplit, gkper;      // K ranges of the forward contraction and their length
    long long cx_off;        // sum of C * nx over earlier tables: first (channel, x) slot of the VJP fold partials
    // tcgen05 contraction of fp32 tables (fk_tc32.cu)
    const void* tmap;        // device copy of the table's CUtensorMap (null: the table cannot take that path)
    // element-sparse storage (fk_sparse.cuh): fk = the nonzero values; null sp_blk: dense
    const void* sp_blk;                   // [N][nchunks] SparseBlk: value offset, per-word prefix counts, bit masks
    int tc_ksplit, tc_kper;  // grouped launches: K ranges of the tcgen05 contraction and their length (multiple of 32)
    long long tc_gp_off;     // grouped launches: row offset of this table's tcgen05 split-K partials
};

// Work list entry of the column kernels (forward and VJP stage 1): one CTA = one (k-block, datapoint range).
struct ColSeg {
    int table, kblock, split, pad_;
};

// Offsets (inside one replica's f[nfl][nx]) of the two PDF factors of contraction index k.
// Hadronic: L[k] = f[ia] * f[ib];  DIS: L[k] = f[ia] (ib = -1);  ia = -1: padding, L[k] = 0.
__device__ __forceinline__ void decode_k(const TableDesc& d, const uint8_t* __restrict__ ca,
                                         const uint8_t* __restrict__ cb, int k, int& ia, int& ib) {
    const int nx = d.nx;
    if (d.kind == KIND_HADRONIC) {
        int c, i, j;
        if (d.layout == LAYOUT_LOGICAL) {
            c = k % d.C;
            const int p = k / d.C;
            i = p / nx;
            j = p - i * nx;
        } else {
            c = k / d.cstride;
            const int rem = k - c * d.cstride;
            i = rem / d.jp;
            j = rem - i * d.jp;
            if (i >= nx || j >= nx) {  // zero padding at the end of an x-row or of a channel block: no luminosity
                ia = ib = -1;
                return;
            }
        }
        ia = (int)ca[c] * nx + i;
        ib = (int)cb[c] * nx + j;
    } else {
        int c, i;
        if (d.layout == LAYOUT_LOGICAL) {
            i = k / d.C;
            c = k - i * d.C;
        } else {
            c = k / nx;
            i = k - c * nx;
        }
        ia = (int)ca[c] * nx + i;
        ib = -1;
    }
}

// Contraction index of (i, j, c) resp. (i, c) in the table's k-order (inverse of decode_k).
__device__ __forceinline__ int encode_k(const TableDesc& d, int i, int j, int c) {
    if (d.kind == KIND_HADRONIC)
        return d.layout == LAYOUT_LOGICAL ? (i * d.nx + j) * d.C + c : c * d.cstride + i * d.jp + j;
    return d.layout == LAYOUT_LOGICAL ? i * d.C + c : c * d.nx + i;
}

// ---- streaming loads: FK is read once, keep it out of L1 -------------------------------------
// L2 evict-first policy for the table stream (not volatile: one createpolicy per thread, hoisted out of the loops): the
// small operands that ARE re-read -- level-1 partials, column sums G, f -- stay in L2 while the table passes through
__device__ __forceinline__ uint64_t stream_policy() {
    uint64_t pol;
    asm("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
template <typename T, int VEC> struct Vec;
template <> struct Vec<double, 2> { double v[2]; };
template <> struct Vec<double, 1> { double v[1]; };
template <> struct Vec<float, 4> { float v[4]; };
template <> struct Vec<float, 1> { float v[1]; };

__device__ __forceinline__ Vec<double, 2> ld_stream(const double* p, Vec<double, 2>*) {
    Vec<double, 2> r;
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.v2.f64 {%0, %1}, [%2], %3;" : "=d"(r.v[0]), "=d"(r.v[1]) : "l"(p), "l"(stream_policy()));
    return r;
}
__device__ __forceinline__ Vec<double, 1> ld_stream(const double* p, Vec<double, 1>*) {
    Vec<double, 1> r;
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.f64 %0, [%1], %2;" : "=d"(r.v[0]) : "l"(p), "l"(stream_policy()));
    return r;
}
__device__ __forceinline__ Vec<float, 4> ld_stream(const float* p, Vec<float, 4>*) {
    Vec<float, 4> r;
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.v4.f32 {%0, %1, %2, %3}, [%4], %5;"
                 : "=f"(r.v[0]), "=f"(r.v[1]), "=f"(r.v[2]), "=f"(r.v[3]) : "l"(p), "l"(stream_policy()));
    return r;
}
__device__ __forceinline__ Vec<float, 1> ld_stream(const float* p, Vec<float, 1>*) {
    Vec<float, 1> r;
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.f32 %0, [%1], %2;" : "=f"(r.v[0]) : "l"(p), "l"(stream_policy()));
    return r;
}

// ---- fixed-order warp tree (xor butterfly): every lane ends with the same bits ------------------
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

template <typename T> struct VecWidth;
template <> struct VecWidth<double> { static constexpr int value = 2; };
template <> struct VecWidth<float> { static constexpr int value = 4; };

}  // namespace fk
