// fk_api.cu -- the C-ABI of include/fkconv.h: argument validation, table / group handles, launch plans.
// Host logic only; every step of the path runs in the kernels of fk_fwd.cuh / fk_vjp.cuh / fk_vjp_fold.cuh /
// fk_gemm.cuh / fk_gemm_ws.cuh.  There is no CPU fallback anywhere in this file.
#include "../../include/fkconv.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <mutex>
#include <new>
#include <string>
#include <type_traits>
#include <vector>

#include "fk_common.cuh"
#include "fk_gemm.cuh"
#include "fk_gemm_ws.cuh"
#include "fk_vjp_fold.cuh"
#include "fk_pack.cuh"
#include "fk_fwd.cuh"
#include "fk_vjp.cuh"
#include "fk_chi2.cuh"
#include "fk_tc32.h"
#include "fk_sparse.cuh"
#include "fk_dis_direct.cuh"

namespace {

thread_local std::string g_err;

int fail(int code, const char* fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    g_err = buf;
    return code;
}

#define FK_CUDA(call)                                                                              \
    do {                                                                                           \
        cudaError_t e_ = (call);                                                                   \
        if (e_ != cudaSuccess)                                                                     \
            return fail(e_ == cudaErrorMemoryAllocation ? FK_ERR_ALLOC : FK_ERR_CUDA, "%s: %s",    \
                        #call, cudaGetErrorString(e_));                                            \
    } while (0)

// ---- plan constants (frozen from the round-1 sweeps; nothing is read from the environment) ----
constexpr int FWD_ROWS_F64 = 32;           // datapoints per forward CTA, fp64 table
constexpr int FWD_ROWS_F32 = 64;           // fp32-stored table: 4 luminosity values per thread to amortise
constexpr int FWD_MIN_CTAS_PER_SM = 8;     // small tables: cut finer until the grid covers the GPU this often
constexpr int COLSUM_CTAS_PER_SM = 24;     // VJP stage 1: CTAs wanted per SM
constexpr int GROUP_GEMM_WAVES = 16;       // grouped R >> 1 forward: waves of equal-cost items

// ---- process-wide options (fk_set_option, include/fkconv.h): path selection only ----
int g_opt[FK_OPT_COUNT_] = {
    /* FK_OPT_GEMM_MIN_R  */ 0,   // 0 = built-in threshold (5 on the warp-specialised path, 13 otherwise)
    /* FK_OPT_WARP_SPEC   */ 1,
    /* FK_OPT_FOLD        */ 1,
    /* FK_OPT_FOLDK       */ 1,
    /* FK_OPT_FUSED       */ 1,
    /* FK_OPT_FEWROWS     */ 1,
    /* FK_OPT_TC32        */ 1,
    /* FK_OPT_TC32_MIN_R  */ 0,
    /* FK_OPT_PDL         */ 1,
    /* FK_OPT_FUSE_L2     */ 1,
    /* FK_OPT_DIS_DIRECT  */ 80,  // smallest R that takes fk_dis_direct_kernel (0 = never): its time barely depends on R, the split-K chain's does
};
inline int opt(int o) { return g_opt[o]; }

int sm_count() {
    static std::mutex mu;
    static std::map<int, int> cache;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return 0;
    std::lock_guard<std::mutex> lk(mu);
    auto it = cache.find(dev);
    if (it != cache.end()) return it->second;
    int n = 0;
    if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) n = 0;
    cache[dev] = n;
    return n;
}

// cudaFuncSetAttribute is per DEVICE: the opt-in to more than 48 KB of dynamic shared memory is cached per
// (device, kernel), so a process that drives several GPUs sets it on each of them.
bool ensure_dyn_smem(const void* func, size_t bytes) {
    static std::mutex mu;
    static std::map<std::pair<int, const void*>, size_t> done;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return false;
    std::lock_guard<std::mutex> lk(mu);
    auto it = done.find({dev, func});
    if (it != done.end() && it->second >= bytes) return true;
    if (cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes) != cudaSuccess) return false;
    done[{dev, func}] = bytes;
    return true;
}
template <typename F> bool ensure_dyn_smem(F* func, size_t bytes) { return ensure_dyn_smem((const void*)func, bytes); }

// ---- kernel timing hook (fk_profile_enable / fk_profile_read / fk_profile_report) ----
// While enabled, every kernel launch of a compute call is bracketed by an event pair on the caller's stream, keyed by a
// short kernel name (FK_TIMED below).  Off by default: the pairs serialise neighbouring launches.
struct Profiler {
    std::mutex mu;
    bool on = false;
    struct Rec { cudaEvent_t a, b; const char* name; };
    std::vector<Rec> recs;
    size_t used = 0;
    bool begin(cudaStream_t s, size_t& slot, const char* name) {
        std::lock_guard<std::mutex> lk(mu);
        if (!on) return false;
        if (used == recs.size()) {
            Rec r{nullptr, nullptr, name};
            if (cudaEventCreate(&r.a) != cudaSuccess || cudaEventCreate(&r.b) != cudaSuccess) return false;
            recs.push_back(r);
        }
        slot = used++;
        recs[slot].name = name;
        cudaEventRecord(recs[slot].a, s);
        return true;
    }
    void end(cudaStream_t s, size_t slot) {
        std::lock_guard<std::mutex> lk(mu);
        cudaEventRecord(recs[slot].b, s);
    }
} g_prof;
struct ProfScope {
    cudaStream_t s;
    size_t slot = 0;
    bool on;
    ProfScope(cudaStream_t s_, const char* name) : s(s_) { on = g_prof.begin(s, slot, name); }
    ~ProfScope() { if (on) g_prof.end(s, slot); }
    ProfScope(const ProfScope&) = delete;
};
// FK_TIMED("name", stream) statement;   -- the statement's launches are one timed record (no dangling-else hazard)
#define FK_TIMED(NAME, S) switch (ProfScope fk_ps_{S, NAME}; 0) default:

// Launch of a LATER kernel of a compute call with programmatic stream serialisation (fk_common.cuh, pdl_wait): its CTAs
// may be scheduled while the preceding kernel of the same call drains; the kernel itself waits (griddepcontrol.wait)
// before it touches memory.  The first kernel of every call is a normal launch, so the caller's own preceding work
// (which produced f, g) is complete and visible as usual.
template <typename... KArgs, typename... Args>
cudaError_t launch_pdl(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t s, Args&&... args) {
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof cfg);
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = opt(FK_OPT_PDL) ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, KArgs(std::forward<Args>(args))...);
}

template <typename T> constexpr int dtype_of();
template <> constexpr int dtype_of<double>() { return FK_F64; }
template <> constexpr int dtype_of<float>() { return FK_F32; }
size_t dtype_size(int dtype) { return dtype == FK_F64 ? 8 : 4; }     // storage element of the table
size_t io_size(int dtype) { return dtype == FK_F32 ? 4 : 8; }        // element of f, sigma, g, df

// ------------------------------------------------------------------------------------------------
// plans
// ------------------------------------------------------------------------------------------------
// Both bandwidth-bound kernels (forward, VJP stage 1) cut a table into CTAs of one k-block
// (256 * VEC consecutive k: 4 KB of every row) times one datapoint range.
struct Plan {
    int nkb = 0;      // k-blocks per row
    int fsplit = 0;   // forward: datapoint ranges
    int nsplit = 0;   // VJP stage 1: datapoint ranges
};

constexpr int FWD_U = 8;  // rows in flight per thread of the forward column kernel

void make_plan(fk::TableDesc& d, int dtype, Plan& pl) {
    const int vecw = dtype == FK_F64 ? 2 : 4;
    const int vec = d.vec_ok ? vecw : 1;
    pl.nkb = (d.K + fk::FWD_THREADS * vec - 1) / (fk::FWD_THREADS * vec);
    const int sms = std::max(1, sm_count());

    // forward: ~32 datapoints per CTA (finer for small tables so that the grid still covers the GPU a few
    // times over), never fewer than one batch of FWD_U rows
    int rows = dtype == FK_F64 ? FWD_ROWS_F64 : FWD_ROWS_F32;
    const long long want_f = (long long)FWD_MIN_CTAS_PER_SM * sms;
    while (rows > FWD_U && (long long)pl.nkb * ((d.N + rows - 1) / rows) < want_f) rows /= 2;
    rows = std::max(rows, 1);
    pl.fsplit = std::max(1, std::min(d.N, (d.N + rows - 1) / rows));

    // VJP stage 1: fewer, longer ranges (every range writes K column sums that stage 2 adds up)
    // CTAs wanted for stage 1; a k-block of an fp32-stored table is twice as many k (1024), so the same CTA count would
    // halve the rows per CTA and double the column-sum slices: ask for half as many
    const int want = COLSUM_CTAS_PER_SM * sms / (dtype == FK_F64 ? 1 : 2);
    int nsplit = (want + pl.nkb - 1) / pl.nkb;
    nsplit = std::min(nsplit, std::max(1, d.N / 16));                  // >= 16 datapoints per split
    nsplit = std::max(nsplit, (d.N + fk::COLSUM_MAX_ROWS - 1) / fk::COLSUM_MAX_ROWS);
    nsplit = std::max(1, std::min(nsplit, d.N));
    pl.nsplit = nsplit;

    d.nchunks = pl.nkb;
    d.fsplit = pl.fsplit;
    d.nsplit = pl.nsplit;
}

size_t part_elems_per_replica(const fk::TableDesc& d) { return d.nchunks > 1 ? (size_t)d.N * d.nchunks : 0; }
size_t G_elems_per_replica(const fk::TableDesc& d) { return (size_t)d.nsplit * d.K; }
// small-R VJP stage 2 in one pass over G (fk_vjp_foldk_kernel): hadronic tables whose nx x nx block fits shared memory
bool foldk_ok(const fk::TableDesc& d) { return d.kind == fk::KIND_HADRONIC && d.nx <= 128 && opt(FK_OPT_FOLDK); }
size_t foldk_smem(int nx) { return (size_t)nx * (nx | 1) * 8; }
constexpr int FOLDK_MAX_CHUNKS = 8;
// x-row chunks per channel so that a table (or group) with few channels still covers the GPU about twice
int foldk_chunks(long long channels) {
    const long long want = 2LL * std::max(1, sm_count());
    return (int)std::max<long long>(1, std::min<long long>(FOLDK_MAX_CHUNKS, (want + channels - 1) / std::max<long long>(1, channels)));
}
size_t foldk_elems_per_replica(const fk::TableDesc& d) { return foldk_ok(d) ? (1 + FOLDK_MAX_CHUNKS) * (size_t)d.C * d.nx : 0; }

// ------------------------------------------------------------------------------------------------
// validation
// ------------------------------------------------------------------------------------------------
int check_dims(const char* who, int kind, int N, int nx, int nfl, int C, int R) {
    if (N <= 0 || nx <= 0 || nfl <= 0 || C <= 0 || R <= 0)
        return fail(FK_ERR_INVALID_ARG, "%s: non-positive size (N=%d nx=%d nfl=%d C=%d R=%d)", who, N, nx, nfl, C, R);
    if (nfl > fk::MAX_NFL || C > fk::MAX_C)
        return fail(FK_ERR_UNSUPPORTED, "%s: nfl=%d > %d or C=%d > %d", who, nfl, fk::MAX_NFL, C, fk::MAX_C);
    const long long K = kind == FK_KIND_HADRONIC ? (long long)C * ((long long)nx * (nx + 3) + 3) : (long long)C * nx;   // padded x-rows (packed_jp)
    if (K >= (1LL << 31) - 4096) return fail(FK_ERR_UNSUPPORTED, "%s: K=%lld does not fit 31 bits", who, K);
    if ((long long)nfl * nx >= (1LL << 31) - 4096) return fail(FK_ERR_UNSUPPORTED, "%s: nfl*nx does not fit 31 bits", who);
    if (kind == FK_KIND_DIS && C > nfl)
        return fail(FK_ERR_INVALID_ARG, "%s: nA=%d > nfl=%d", who, C, nfl);
    return FK_OK;
}

int fill_channels(const char* who, int kind, const int32_t* idx, int nfl, int C, fk::ChannelList& ch) {
    memset(&ch, 0, sizeof ch);
    for (int c = 0; c < C; ++c) {
        const int a = kind == FK_KIND_HADRONIC ? idx[2 * c] : idx[c];
        const int b = kind == FK_KIND_HADRONIC ? idx[2 * c + 1] : 0;
        if (a < 0 || a >= nfl || b < 0 || b >= nfl)
            return fail(FK_ERR_INVALID_ARG, "%s: flavour index out of [0,%d) at channel %d: (%d,%d)", who, nfl, c, a, b);
        ch.a[c] = (uint8_t)a;
        ch.b[c] = (uint8_t)b;
    }
    return FK_OK;
}

// x-row pitch of a packed hadronic table: fp32 tables (FK_F32) pad nx to a multiple of 4, so that every (c, i) row starts
// on a 16-byte boundary -- what a TMA box needs (fk_tc32.cu); all others are dense (jp = nx)
int packed_jp(int kind, int nx, int dtype) { return (kind == FK_KIND_HADRONIC && dtype == FK_F32) ? (nx + 3) / 4 * 4 : nx; }

fk::TableDesc make_desc(int kind, int layout, const void* fkp, int N, int nx, int nfl, int C, long long row_stride,
                        int dtype) {
    fk::TableDesc d;
    memset(&d, 0, sizeof d);
    d.fk = fkp;
    d.jp = layout == fk::LAYOUT_PACKED ? packed_jp(kind, nx, dtype) : nx;
    d.cstride = (layout == fk::LAYOUT_PACKED && kind == FK_KIND_HADRONIC) ? (nx * d.jp + 3) / 4 * 4 : nx * nx;
    d.K = kind == FK_KIND_HADRONIC ? C * d.cstride : C * nx;
    d.row_stride = row_stride > 0 ? row_stride : d.K;
    d.N = N; d.nx = nx; d.nfl = nfl; d.C = C;
    d.kind = kind == FK_KIND_HADRONIC ? fk::KIND_HADRONIC : fk::KIND_DIS;
    d.layout = layout;
    const int vecw = dtype == FK_F64 ? 2 : 4;
    d.vec_ok = ((uintptr_t)fkp % 16 == 0) && (d.row_stride % vecw == 0);
    d.store32 = dtype != FK_F64;
    return d;
}

// ------------------------------------------------------------------------------------------------
// launchers
// ------------------------------------------------------------------------------------------------
// picks the replica tile for a pass starting at r0
inline int pick_rt(int remaining) { return remaining >= 3 ? 4 : remaining; }

template <typename T, bool GROUPED, typename TS = T>
cudaError_t fwd_dispatch(bool vec_ok, int rt, const fk::FwdParams& p, int grid, cudaStream_t s) {
    constexpr int VW = fk::VecWidth<TS>::value;
#define FK_FWD(V, RTv) FK_TIMED("fk_fwd_column", s) fk::fk_fwd_column_kernel<T, V, RTv, FWD_U, GROUPED, TS><<<grid, fk::FWD_THREADS, 0, s>>>(p)
    if constexpr (!GROUPED && std::is_same<T, double>::value && std::is_same<TS, double>::value) {
        if (rt == 8) {   // 5..12 replicas on tables without a dense path (DIS, logical layout): 8 per read, 4 rows in flight
            if (vec_ok) FK_TIMED("fk_fwd_column", s) fk::fk_fwd_column_kernel<T, VW, 8, 4, false, TS><<<grid, fk::FWD_THREADS, 0, s>>>(p);
            else FK_TIMED("fk_fwd_column", s) fk::fk_fwd_column_kernel<T, 1, 8, 4, false, TS><<<grid, fk::FWD_THREADS, 0, s>>>(p);
            return cudaGetLastError();
        }
    }
    if (vec_ok) {
        if (rt == 1) FK_FWD(VW, 1); else if (rt == 2) FK_FWD(VW, 2); else FK_FWD(VW, 4);
    } else {
        if (rt == 1) FK_FWD(1, 1); else if (rt == 2) FK_FWD(1, 2); else FK_FWD(1, 4);
    }
#undef FK_FWD
    return cudaGetLastError();
}

template <typename T, bool GROUPED, typename TS = T>
cudaError_t colsum_dispatch(bool vec_ok, int rt, const fk::ColsumParams& p, int grid, cudaStream_t s) {
    constexpr int VW = fk::VecWidth<TS>::value;
    constexpr int U = 8;
#define FK_COLSUM(V, RTv) FK_TIMED("fk_colsum", s) fk::fk_colsum_kernel<T, V, RTv, U, GROUPED, TS><<<grid, fk::COLSUM_THREADS, 0, s>>>(p)
    if (vec_ok) {
        if (rt == 1) FK_COLSUM(VW, 1); else if (rt == 2) FK_COLSUM(VW, 2); else FK_COLSUM(VW, 4);
    } else {
        if (rt == 1) FK_COLSUM(1, 1); else if (rt == 2) FK_COLSUM(1, 2); else FK_COLSUM(1, 4);
    }
#undef FK_COLSUM
    return cudaGetLastError();
}

// ---- R >> 1: FP64 tensor-core contraction (fk_gemm.cuh) ---------------------------------------------
struct GemmPlan {
    int ksplit, kper, RPmax, ksub_rem;
};

template <typename T>
bool gemm_wanted(const fk::TableDesc& d, int R) {
    if (dtype_of<T>() != FK_F64 || d.store32 || d.sp_blk) return false;  // fp32 variants (reading R18) and sparse tables: column kernels
    if ((long long)d.nfl * d.nx >= (long long)fk::KDEC_NONE) return false;
    // packed hadronic tables take the warp-specialised kernel, which beats the <= 4-replica column passes from
    // R = 5 on; the generic cp.async kernel (DIS, logical layout) streams FK at ~2 TB/s and only wins once the
    // column kernel would need more than 3 passes
    const bool ws = d.kind == fk::KIND_HADRONIC && d.layout == fk::LAYOUT_PACKED && d.vec_ok;
    return R >= (opt(FK_OPT_GEMM_MIN_R) > 0 ? opt(FK_OPT_GEMM_MIN_R) : ws ? 5 : 13);
}

GemmPlan gemm_plan(const fk::TableDesc& d, int R) {
    GemmPlan gp;
    const int mtiles = (d.N + fk::GEMM_BM - 1) / fk::GEMM_BM;
    const int target = std::max(1, sm_count());  // one wave of equal items
    int ksplit = std::max(1, target / mtiles);
    gp.kper = ((d.K + ksplit - 1) / ksplit + fk::GEMM_KT - 1) / fk::GEMM_KT * fk::GEMM_KT;
    gp.ksplit = (d.K + gp.kper - 1) / gp.kper;
    // a partial last datapoint tile is cut into k sub-splits (fk_gemm_ws.cuh): whole groups of K ranges
    gp.ksub_rem = d.N % fk::GEMM_BM ? fk::ws_ksub_for_rows(d.N % fk::GEMM_BM) : 1;
    gp.ksplit = (gp.ksplit + gp.ksub_rem - 1) / gp.ksub_rem * gp.ksub_rem;
    gp.RPmax = fk::gemm_rp(R);
    return gp;
}

// doubles: fT [slots][RPmax] + level-1 partials [ksplit][N][RPmax] (+ k codes when the caller has none)
size_t gemm_fwd_scratch_elems(const fk::TableDesc& d, int R, bool with_kdec) {
    const GemmPlan gp = gemm_plan(d, R);
    return (size_t)d.nfl * d.nx * gp.RPmax + (size_t)gp.ksplit * d.N * gp.RPmax + (with_kdec ? ((size_t)d.K + 1) / 2 : 0);
}

constexpr size_t MAX_DYN_SMEM = 232448;  // 227 KB per CTA on sm_100a

// the warp-specialised kernel (fk_gemm_ws.cuh) serves packed hadronic tables whose f[b_c] tiles fit next to the FK ring
bool ws_ok(const fk::TableDesc& d, int RP) {
    return d.kind == fk::KIND_HADRONIC && d.layout == fk::LAYOUT_PACKED && d.vec_ok && d.jp == d.nx && opt(FK_OPT_WARP_SPEC) &&
           fk::ws_smem_bytes(d.nx, RP) <= MAX_DYN_SMEM;
}

// RP = 8 * NFRAG (fk::gemm_rp: a multiple of 16), NFRAG = 2, 4, ..., 16: one instantiation per fragment count
template <bool GROUPED, typename TS = double>
bool ws_launch(const fk::WsFwdParams& w, int grid, size_t smem, cudaStream_t s) {
    switch (w.RP / 8) {
#define FK_WS_CASE(NFW) case NFW: if (!ensure_dyn_smem(fk::fk_gemm_fwd_ws_kernel<NFW, GROUPED, TS>, MAX_DYN_SMEM)) return false; \
                                  FK_TIMED("fk_gemm_fwd_ws", s) launch_pdl(fk::fk_gemm_fwd_ws_kernel<NFW, GROUPED, TS>, grid, fk::WS_THREADS, smem, s, w); break
        FK_WS_CASE(2); FK_WS_CASE(4); FK_WS_CASE(6); FK_WS_CASE(8); FK_WS_CASE(10); FK_WS_CASE(12); FK_WS_CASE(14);
        default: FK_WS_CASE(16);
#undef FK_WS_CASE
    }
    return true;
}

// FK_F32S64 tables (fp32 storage, fp64 f / sigma and arithmetic) at R >> 1: the warp-specialised FP64 contraction over the
// table as stored.  The DMMA work is that of the fp64 table; it replaces ceil(R / 4) column passes over half the bytes.
constexpr int FWD32_DEFAULT_MIN_R = 9;
bool fwd32_wanted(const fk::TableDesc& d, int R) {
    if (!d.store32 || d.sp_blk || !ws_ok(d, fk::gemm_rp(R))) return false;
    if ((long long)d.nfl * d.nx >= (long long)fk::KDEC_NONE) return false;
    return R >= (opt(FK_OPT_GEMM_MIN_R) > 0 ? opt(FK_OPT_GEMM_MIN_R) : FWD32_DEFAULT_MIN_R);
}

// DIS tables (any k-order): the warp-specialised kernel whose B tile is 32 fT rows per stage (fk_gemm_dis_ws_kernel)
bool wsd_ok(const fk::TableDesc& d, int RP) {
    return d.kind == fk::KIND_DIS && d.vec_ok && opt(FK_OPT_WARP_SPEC) && fk::wsd_smem_bytes(RP) <= MAX_DYN_SMEM;
}
bool wsd_launch(const fk::WsFwdParams& w, int grid, cudaStream_t s) {
    const size_t smem = fk::wsd_smem_bytes(w.RP);
    switch (w.RP / 8) {
#define FK_WSD_CASE(NFW) case NFW: if (!ensure_dyn_smem(fk::fk_gemm_dis_ws_kernel<NFW>, MAX_DYN_SMEM)) return false; \
                                   FK_TIMED("fk_gemm_dis_ws", s) launch_pdl(fk::fk_gemm_dis_ws_kernel<NFW>, grid, fk::WS_THREADS, smem, s, w); break
        FK_WSD_CASE(2); FK_WSD_CASE(4); FK_WSD_CASE(6); FK_WSD_CASE(8); FK_WSD_CASE(10); FK_WSD_CASE(12); FK_WSD_CASE(14);
        default: FK_WSD_CASE(16);
#undef FK_WSD_CASE
    }
    return true;
}

// Small packed DIS tables at R >> 1 (config 1 at R = 100): one launch, no transposed copy of f, no split-K partials
// (fk_dis_direct.cuh).  "Small" = the table stays in L2 while every column group of CTAs reads it, and the grid is a few
// waves at most; larger tables keep the split-K kernel, which reads FK once with 128-datapoint tiles.
bool dis_direct_wanted(const fk::TableDesc& d, int R, const void* f) {
    if (d.kind != fk::KIND_DIS || d.layout != fk::LAYOUT_PACKED || !d.vec_ok || d.store32 || d.sp_blk || !opt(FK_OPT_DIS_DIRECT)) return false;
    if (d.nx % 2 || d.K > fk::DD_MAX_K || d.K != d.C * d.nx || (reinterpret_cast<uintptr_t>(f) & 15)) return false;   // 16-byte pieces of f
    if (R > 512 || (long long)d.N * d.K * 8 > (64LL << 20) || fk::dd_smem_bytes(d.K, 2) > MAX_DYN_SMEM - fk::DD_STATIC_SMEM) return false;
    return R >= std::max(13, opt(FK_OPT_DIS_DIRECT));   // never below the dense threshold of DIS tables
}

int run_conv_dis_direct(const fk::TableDesc& d, const fk::ChannelList& ch, const double* f, double* sigma, int R, cudaStream_t s, int* launches) {
    fk::DisDirectParams p;
    memset(&p, 0, sizeof p);
    p.desc = d;
    p.chan = ch;
    p.f = f;
    p.sigma = sigma;
    p.R = R;
    p.nfrag = (R + 7) / 8;
    p.ncs = (p.nfrag + fk::DD_NFC - 1) / fk::DD_NFC;
    p.stages = fk::dd_smem_bytes(d.K, fk::DD_STAGES) <= MAX_DYN_SMEM - fk::DD_STATIC_SMEM ? fk::DD_STAGES : 2;
    const size_t smem = fk::dd_smem_bytes(d.K, p.stages);
    if (!ensure_dyn_smem(fk::fk_dis_direct_kernel, smem)) return fail(FK_ERR_CUDA, "dis direct: cannot reserve %zu bytes of shared memory", smem);
    const dim3 grid((d.N + fk::DD_TM - 1) / fk::DD_TM, p.ncs);
    FK_TIMED("fk_dis_direct", s) fk::fk_dis_direct_kernel<<<grid, fk::DD_THREADS, smem, s>>>(p);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(FK_ERR_CUDA, "dis direct launch failed: %s", cudaGetErrorString(e));
    if (launches) *launches = 1;
    return FK_OK;
}

// the persistent warp-specialised VJP contraction needs 16-byte aligned, 16-byte multiple row pieces
// fp32-stored rows: vec_ok makes row_stride a multiple of 4, so the copies rounded up to 16 bytes stay inside the row
bool wsv_ok(const fk::TableDesc& d) { return d.vec_ok && (d.store32 || d.K % 2 == 0) && opt(FK_OPT_WARP_SPEC); }

template <bool GROUPED, typename TS = double>
bool wsv_launch(const fk::WsVjpParams& w0, cudaStream_t s) {
    fk::WsVjpParams w = w0;
    const int sms = std::max(1, sm_count());
    if (!GROUPED) {
        // the tiles left over after the last full round of the persistent grid become 2 or 4 column parts each when that
        // still fits one round: the last round then lasts a half or a quarter of a tile (config 3: 30 of 1954 tiles -> 120 parts)
        const int tiles = w.ntiles, nfrag = w.RP / 8;
        w.nwhole = tiles / sms * sms;
        const int left = tiles - w.nwhole;
        w.nparts = (left > 0 && nfrag % 8 == 0 && 4 * left <= sms) ? 4 : (left > 0 && nfrag % 4 == 0 && 2 * left <= sms) ? 2 : 1;
        if (w.nparts == 1) w.nwhole = tiles;
        w.ntiles = w.nwhole + (tiles - w.nwhole) * w.nparts;
    }
    const int grid = std::max(1, std::min(w.ntiles, sms));
    switch (w.RP / 8) {
#define FK_WSV_CASE(NFW) case NFW: if (!ensure_dyn_smem(fk::fk_gemm_vjp_ws_kernel<NFW, GROUPED, TS>, fk::WSV_SMEM_BYTES)) return false; \
                                   FK_TIMED("fk_gemm_vjp_ws", s) fk::fk_gemm_vjp_ws_kernel<NFW, GROUPED, TS><<<grid, fk::WS_THREADS, fk::WSV_SMEM_BYTES, s>>>(w); break
        FK_WSV_CASE(2); FK_WSV_CASE(3); FK_WSV_CASE(4); FK_WSV_CASE(5); FK_WSV_CASE(6); FK_WSV_CASE(7); FK_WSV_CASE(8); FK_WSV_CASE(9);
        FK_WSV_CASE(10); FK_WSV_CASE(11); FK_WSV_CASE(12); FK_WSV_CASE(13); FK_WSV_CASE(14); FK_WSV_CASE(15);
        default: FK_WSV_CASE(16);
#undef FK_WSV_CASE
    }
    return true;
}

// TS = storage type of the table; float (FK_F32S64) only with the warp-specialised kernel (fwd32_wanted)
template <typename TS = double>
int run_conv_gemm(const fk::TableDesc& d, const fk::ChannelList& ch, const uint32_t* kdec, const double* f,
                  double* sigma, int R, double* scratch, cudaStream_t s, int* launches) {
    const GemmPlan gp = gemm_plan(d, R);
    const int slots = d.nfl * d.nx;
    double* fT = scratch;
    double* gpart = fT + (size_t)slots * gp.RPmax;
    int nl = 0;
    const bool ws = ws_ok(d, gp.RPmax);
    const bool wsd = !ws && wsd_ok(d, gp.RPmax);
    if (!std::is_same<TS, double>::value && !ws) return fail(FK_ERR_UNSUPPORTED, "gemm: fp32-stored table without the packed bulk-copy layout");
    if (!kdec && !ws && !wsd) {
        uint32_t* kd = reinterpret_cast<uint32_t*>(gpart + (size_t)gp.ksplit * d.N * gp.RPmax);
        FK_TIMED("fk_kdec", s) fk::fk_kdec_kernel<<<std::min(1024, (d.K + 255) / 256), 256, 0, s>>>(d, ch, kd);
        ++nl;
        kdec = kd;
    }
    if (!ws && !wsd && !(ensure_dyn_smem(fk::fk_gemm_fwd_kernel<2, false>, fk::GEMM_SMEM_BYTES) &&
                 ensure_dyn_smem(fk::fk_gemm_fwd_kernel<1, false>, fk::GEMM_SMEM_BYTES)))
        return fail(FK_ERR_CUDA, "gemm: cannot reserve %d bytes of shared memory", fk::GEMM_SMEM_BYTES);
    const int mtiles = (d.N + fk::GEMM_BM - 1) / fk::GEMM_BM;
    for (int r0 = 0; r0 < R; r0 += fk::GEMM_BN) {
        fk::GemmFwdParams p;
        memset(&p, 0, sizeof p);
        p.desc = d;
        p.kdec = kdec;
        p.fT = fT;
        p.gpart = gpart;
        p.RP = fk::gemm_rp(R - r0);
        p.nfrag = p.RP / 8;
        p.nfw = (p.nfrag + 1) / 2;
        p.ksplit = gp.ksplit;
        p.kper = gp.kper;
        const long long tot = (long long)slots * p.RP;
        FK_TIMED("fk_transpose_f", s) fk::fk_transpose_f_kernel<double><<<(int)std::min<long long>(2048, (tot + 255) / 256), 256, 0, s>>>(f, fT, slots, R, r0, p.RP);
        if (ws) {
            fk::WsFwdParams w;
            memset(&w, 0, sizeof w);
            w.desc = d;
            w.chan = ch;
            w.fT = fT;
            w.gpart = gpart;
            w.RP = p.RP;
            w.ksplit = gp.ksplit;
            w.kper = gp.kper;
            w.ksub_rem = gp.ksub_rem;
            const int nfull = d.N / fk::GEMM_BM;
            if (!ws_launch<false, TS>(w, nfull * gp.ksplit + (d.N % fk::GEMM_BM ? gp.ksplit / gp.ksub_rem : 0), fk::ws_smem_bytes(d.nx, p.RP), s))
                return fail(FK_ERR_CUDA, "gemm: cannot reserve %zu bytes of shared memory", MAX_DYN_SMEM);
        } else if (wsd) {
            fk::WsFwdParams w;
            memset(&w, 0, sizeof w);
            w.desc = d;
            w.chan = ch;
            w.fT = fT;
            w.gpart = gpart;
            w.RP = p.RP;
            w.ksplit = gp.ksplit;
            w.kper = gp.kper;
            if (!wsd_launch(w, mtiles * gp.ksplit, s)) return fail(FK_ERR_CUDA, "gemm: cannot reserve %zu bytes of shared memory", MAX_DYN_SMEM);
        } else if (d.vec_ok) FK_TIMED("fk_gemm_fwd", s) launch_pdl(fk::fk_gemm_fwd_kernel<2, false>, mtiles * gp.ksplit, fk::GEMM_THREADS, fk::GEMM_SMEM_BYTES, s, p);
        else FK_TIMED("fk_gemm_fwd", s) launch_pdl(fk::fk_gemm_fwd_kernel<1, false>, mtiles * gp.ksplit, fk::GEMM_THREADS, fk::GEMM_SMEM_BYTES, s, p);
        const long long outs = (long long)d.N * p.RP;
        FK_TIMED("fk_gemm_reduce", s) launch_pdl(fk::fk_gemm_reduce_kernel<double>, (int)std::min<long long>(16384, ((gp.ksplit < fk::GEMM_REDUCE_QUAD ? 1 : 4) * outs + 255) / 256), 256, 0, s,
                                                 gpart, sigma, d.out_off * R, d.N, R, r0, p.RP, gp.ksplit);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return fail(FK_ERR_CUDA, "gemm forward launch failed: %s", cudaGetErrorString(e));
        nl += 3;
    }
    if (launches) *launches = nl;
    return FK_OK;
}

// the single-pass fold (fk_vjp_fold.cuh) serves packed hadronic tables with nx <= 64; others take the gather
bool fold_ok(const fk::TableDesc& d) {
    return d.kind == fk::KIND_HADRONIC && d.layout == fk::LAYOUT_PACKED && d.nx <= fk::FOLD_MAX_NX && opt(FK_OPT_FOLD);
}
// x-row chunks per channel: the CTA count (channels x chunks) that fills whole waves best (1 CTA of 256 threads
// per SM by registers), preferring fewer chunks (each chunk writes its own B partial)
int fold_chunks(long long channels) {
    const long long slots = std::max(1, sm_count());
    int best = 1;
    double best_eff = 0.0;
    for (int n = 1; n <= 8; ++n) {
        const long long ctas = channels * n, waves = (ctas + slots - 1) / slots;
        const double eff = (double)ctas / (double)(waves * slots) - 0.03 * n;  // every CTA pays its own ring fill
        if (eff > best_eff) { best_eff = eff; best = n; }
    }
    return best;
}
constexpr int FOLD_MAX_CHUNKS = 8;

// doubles: fT [slots][RPmax] + gP [N][RPmax] + G [K][RPmax] + fold partials [C*nx][4 + chunks][RPmax]
size_t gemm_vjp_scratch_elems(const fk::TableDesc& d, int R) {
    const size_t RPmax = fk::gemm_rp(R);
    return ((size_t)d.nfl * d.nx + (size_t)d.N + (size_t)d.K + (size_t)d.C * d.nx * (fk::FOLD_JQ + FOLD_MAX_CHUNKS)) * RPmax;
}

// T = type of f, g and df; TS = storage type of the table (float: FK_F32 and FK_F32S64 tables, widened to double in the
// A-fragment loads of the warp-specialised kernel).  The contraction, G and the fold are fp64 for every variant.
// fp32-stored tables (FK_F32, FK_F32S64) at R >> 1: the same FP64 contraction over the table as it is stored (half the
// bytes); G = FK^T g in fp64 costs the same DMMA work whatever the storage, and replaces ceil(R / 4) column passes.
constexpr int VJP32_DEFAULT_MIN_R = 9;   // from 3 column passes of <= 4 replicas on
bool vjp32_wanted(const fk::TableDesc& d, int R) {
    if (!d.store32 || d.sp_blk || !wsv_ok(d)) return false;
    if ((long long)d.nfl * d.nx >= (long long)fk::KDEC_NONE) return false;
    return R >= (opt(FK_OPT_GEMM_MIN_R) > 0 ? opt(FK_OPT_GEMM_MIN_R) : VJP32_DEFAULT_MIN_R);
}

template <typename T, typename TS>
int run_vjp_gemm(const fk::TableDesc& d, const fk::ChannelList& ch, const T* f, const T* g, T* df,
                 int R, double* scratch, cudaStream_t s, int* launches) {
    const int RPmax = fk::gemm_rp8(R);
    const int slots = d.nfl * d.nx;
    double* fT = scratch;
    double* gP = fT + (size_t)slots * RPmax;
    double* G = gP + (size_t)d.N * RPmax;
    if (!std::is_same<TS, double>::value && !wsv_ok(d)) return fail(FK_ERR_UNSUPPORTED, "gemm vjp: fp32-stored table without 16-byte aligned rows");
    if (!wsv_ok(d) && !(ensure_dyn_smem(fk::fk_gemm_vjp_kernel<2, false>, fk::GEMMV_SMEM_BYTES) &&
                        ensure_dyn_smem(fk::fk_gemm_vjp_kernel<1, false>, fk::GEMMV_SMEM_BYTES)))
        return fail(FK_ERR_CUDA, "gemm vjp: cannot reserve %d bytes of shared memory", fk::GEMMV_SMEM_BYTES);
    int nl = 0;
    for (int r0 = 0; r0 < R; r0 += fk::GEMM_BN) {
        const int RP = fk::gemm_rp8(R - r0);
        const long long tf = (long long)slots * RP, tg = (long long)d.N * RP;
        FK_TIMED("fk_transpose_f", s) fk::fk_transpose_f_kernel<T, double><<<(int)std::min<long long>(2048, (tf + 255) / 256), 256, 0, s>>>(f, fT, slots, R, r0, RP);
        FK_TIMED("fk_pad_g", s) fk::fk_pad_g_kernel<T><<<(int)std::min<long long>(2048, (tg + 255) / 256), 256, 0, s>>>(g + d.out_off * R, gP, d.N, R, r0, RP);
        fk::GemmVjpParams p;
        memset(&p, 0, sizeof p);
        p.desc = d;
        p.gP = gP;
        p.G = G;
        p.RP = RP;
        p.nfrag = RP / 8;
        p.nfw = (p.nfrag + 1) / 2;
        const int grid = (d.K + fk::GEMMV_BK - 1) / fk::GEMMV_BK;
        if (wsv_ok(d)) {
            fk::WsVjpParams w;
            memset(&w, 0, sizeof w);
            w.desc = d;
            w.gP = gP;
            w.G = G;
            w.RP = RP;
            w.ntiles = grid;
            if (!wsv_launch<false, TS>(w, s)) return fail(FK_ERR_CUDA, "gemm vjp: cannot reserve %zu bytes of shared memory", fk::WSV_SMEM_BYTES);
        } else if (d.vec_ok) FK_TIMED("fk_gemm_vjp", s) fk::fk_gemm_vjp_kernel<2, false><<<grid, fk::GEMM_THREADS, fk::GEMMV_SMEM_BYTES, s>>>(p);
        else FK_TIMED("fk_gemm_vjp", s) fk::fk_gemm_vjp_kernel<1, false><<<grid, fk::GEMM_THREADS, fk::GEMMV_SMEM_BYTES, s>>>(p);
        if (fold_ok(d)) {
            fk::FoldParams q;
            memset(&q, 0, sizeof q);
            q.desc = d;
            q.desc.cx_off = 0;
            q.chan = ch;
            q.fT = fT;
            q.G = G;
            q.PA = G + (size_t)d.K * RPmax;
            q.PB = q.PA + (size_t)d.C * d.nx * fk::FOLD_JQ * RPmax;
            q.df = df;
            q.R = R;
            q.r0 = r0;
            q.RP = RP;
            q.nchunk = fold_chunks(d.C);
            q.nslots = fk::fold_slots(d.nx, RP, MAX_DYN_SMEM);
            if (!ensure_dyn_smem(fk::fk_vjp_fold_kernel<false>, MAX_DYN_SMEM) || q.nslots < 1) return fail(FK_ERR_CUDA, "gemm vjp: cannot reserve shared memory for the fold ring");
            FK_TIMED("fk_vjp_fold", s) fk::fk_vjp_fold_kernel<false><<<d.C * q.nchunk, fk::FOLD_THREADS,
                                            (size_t)q.nslots * d.nx * RP * 8 + 2 * fk::FOLD_MAX_SLOTS * 8, s>>>(q);
            FK_TIMED("fk_vjp_fold_final", s) fk::fk_vjp_fold_final_kernel<T, false><<<slots, fk::GEMM_BN, 0, s>>>(q);
            ++nl;
        } else {
            fk::GatherRParams q;
            memset(&q, 0, sizeof q);
            q.desc = d;
            q.chan = ch;
            q.fT = fT;
            q.G = G;
            q.df = df;
            q.R = R;
            q.r0 = r0;
            q.RP = RP;
            FK_TIMED("fk_vjp_gather_r", s) fk::fk_vjp_gather_r_kernel<T, false><<<dim3(slots, (RP + 127) / 128), 128, 0, s>>>(q);
        }
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return fail(FK_ERR_CUDA, "gemm vjp launch failed: %s", cudaGetErrorString(e));
        nl += 4;
    }
    if (launches) *launches = nl;
    return FK_OK;
}

// ---- fp32 variant at R >> 1: tcgen05 3xTF32 contraction (fk_tc32.cu) ------------------------------------------------
constexpr int TC32_DEFAULT_MIN_R = 5;   // from 2 column passes of <= 4 replicas on
struct Tc32Plan {
    int ksplit, tper, RPmax;
};
bool tc32_wanted(const fk::TableDesc& d, int R) {
    if (!opt(FK_OPT_TC32) || !d.tmap || d.kind != fk::KIND_HADRONIC || d.layout != fk::LAYOUT_PACKED || d.nx > fk::TC_MAX_NX || d.jp % 4) return false;
    return R >= (opt(FK_OPT_TC32_MIN_R) > 0 ? opt(FK_OPT_TC32_MIN_R) : TC32_DEFAULT_MIN_R);
}
Tc32Plan tc32_plan(const fk::TableDesc& d, int R) {
    Tc32Plan tp;
    tp.RPmax = fk::tc_rp(R);
    const int ntiles = fk::tc32_ntiles(d.N), T = d.C * d.nx;   // datapoint tiles, (c, i) rows
    int ksplit = std::max(1, std::min(T, std::max(1, sm_count()) / ntiles));   // one wave of equal items, one CTA per SM
    ksplit = std::max(ksplit, (T + fk::TC_MAX_TILES - 1) / fk::TC_MAX_TILES);   // bounded fp32 chains in the epilogue
    tp.tper = (T + ksplit - 1) / ksplit;
    tp.ksplit = (T + tp.tper - 1) / tp.tper;
    return tp;
}
// scratch in doubles: fT32 [slots][RPmax] floats + level-1 partials [ksplit][N][RPmax] floats
size_t tc32_scratch_elems(const fk::TableDesc& d, int R) {
    const Tc32Plan tp = tc32_plan(d, R);
    return ((size_t)d.nfl * d.nx * tp.RPmax + (size_t)tp.ksplit * d.N * tp.RPmax + 1) / 2 + 64;
}

int run_conv_tc32(const fk::TableDesc& d, const fk::ChannelList& ch, const float* f, float* sigma, int R, double* scratch,
                  cudaStream_t s, int* launches) {
    const Tc32Plan tp = tc32_plan(d, R);
    const int slots = d.nfl * d.nx;
    float* fT = reinterpret_cast<float*>(scratch);
    float* gpart = fT + ((size_t)slots * tp.RPmax + 31) / 32 * 32;   // 128-byte aligned
    int nl = 0;
    for (int r0 = 0; r0 < R; r0 += fk::TC_MAX_RP) {
        fk::Tc32Params p;
        memset(&p, 0, sizeof p);
        p.desc = d;
        p.chan = ch;
        p.tmap = d.tmap;
        p.fT = fT;
        p.gpart = gpart;
        p.RP = fk::tc_rp(R - r0);
        p.ksplit = tp.ksplit;
        p.tper = tp.tper;
        const long long tot = (long long)slots * p.RP;
        FK_TIMED("fk_transpose_f", s) fk::fk_transpose_f_kernel<float, float><<<(int)std::min<long long>(2048, (tot + 255) / 256), 256, 0, s>>>(f, fT, slots, R, r0, p.RP);
        cudaError_t e = cudaSuccess;
        FK_TIMED("fk_tc32_fwd", s) e = fk::tc32_fwd_launch(p, fk::tc32_ntiles(d.N) * tp.ksplit, false, opt(FK_OPT_PDL) != 0, s);
        if (e != cudaSuccess) return fail(FK_ERR_CUDA, "tcgen05 forward launch failed: %s", cudaGetErrorString(e));
        const long long outs = (long long)d.N * p.RP;
        FK_TIMED("fk_gemm_reduce", s) launch_pdl(fk::fk_gemm_reduce_kernel<float, float>, (int)std::min<long long>(16384, ((tp.ksplit < fk::GEMM_REDUCE_QUAD ? 1 : 4) * outs + 255) / 256), 256, 0, s,
                                                 gpart, sigma, d.out_off * R, d.N, R, r0, p.RP, tp.ksplit);
        e = cudaGetLastError();
        if (e != cudaSuccess) return fail(FK_ERR_CUDA, "tcgen05 forward reduce launch failed: %s", cudaGetErrorString(e));
        nl += 3;
    }
    if (launches) *launches = nl;
    return FK_OK;
}

// One table, any R.  `part` holds >= part_elems_per_replica * R doubles (may be null if nchunks == 1).
template <typename T, typename TS = T>
int run_conv_single(const fk::TableDesc& d, const fk::ChannelList& ch, const Plan& pl, const uint32_t* kdec,
                    const T* f, T* sigma, int R, double* part, cudaStream_t s, int* launches, int* cnt = nullptr) {
    int nl = 0;
    if constexpr (std::is_same<T, double>::value) {
        if constexpr (std::is_same<TS, float>::value) {
            if (fwd32_wanted(d, R)) return run_conv_gemm<float>(d, ch, kdec, f, sigma, R, part, s, launches);
        }
        if constexpr (std::is_same<TS, double>::value) {
            if (dis_direct_wanted(d, R, f)) return run_conv_dis_direct(d, ch, f, sigma, R, s, launches);
        }
        if (gemm_wanted<T>(d, R)) return run_conv_gemm<double>(d, ch, kdec, f, sigma, R, part, s, launches);
    }
    if constexpr (std::is_same<T, float>::value && std::is_same<TS, float>::value) {
        if (tc32_wanted(d, R)) return run_conv_tc32(d, ch, f, sigma, R, part, s, launches);
    }
    fk::FwdParams p;
    memset(&p, 0, sizeof p);
    p.desc = d;
    p.chan = ch;
    p.f = f;
    p.part = part;
    p.sigma = sigma;
    p.R = R;
    const int fgrid = pl.nkb * pl.fsplit;
    // few datapoints per range and very many k-blocks: CTAs that walk the k-blocks (fk_fwd_fewrows_kernel)
    const bool fewrows = (d.N + pl.fsplit - 1) / pl.fsplit <= FWD_U && pl.nkb >= 64 * std::max(1, sm_count()) &&
                         d.vec_ok && !d.sp_blk && opt(FK_OPT_FEWROWS);
    // resident tables whose forward grid is one wave or less (latency-bound, L2-resident: configs 0 and 1): the column
    // kernel's last CTA per datapoint range runs the level-2 reduction itself and the second launch goes away.  On large
    // tables the ticket's round trip at the end of EVERY CTA costs more occupancy than the launch (measured: config 2
    // forward 0.160 -> 0.166 ms, config 4 2.16 -> 2.77 ms), so they keep the separate kernel.
    const bool l2_in_kernel = cnt != nullptr && !fewrows && !d.sp_blk && opt(FK_OPT_FUSE_L2) &&
                              (long long)pl.nkb * pl.fsplit <= 8LL * std::max(1, sm_count());
    p.cnt = l2_in_kernel ? cnt : nullptr;
    for (int r0 = 0; r0 < R;) {
        int rt = pick_rt(R - r0);
        if (R - r0 >= 5 && !fewrows && !d.sp_blk && std::is_same<T, double>::value && std::is_same<TS, double>::value) rt = 8;
        p.r0 = r0;
        cudaError_t e;
        if (fewrows) {
            constexpr int VW = fk::VecWidth<TS>::value;
            const dim3 grid(std::max(1, sm_count()) * 16, pl.fsplit);
            if (rt == 1) FK_TIMED("fk_fwd_fewrows", s) fk::fk_fwd_fewrows_kernel<T, VW, 1, FWD_U, TS><<<grid, fk::FWD_THREADS, 0, s>>>(p);
            else if (rt == 2) FK_TIMED("fk_fwd_fewrows", s) fk::fk_fwd_fewrows_kernel<T, VW, 2, FWD_U, TS><<<grid, fk::FWD_THREADS, 0, s>>>(p);
            else FK_TIMED("fk_fwd_fewrows", s) fk::fk_fwd_fewrows_kernel<T, VW, 4, FWD_U, TS><<<grid, fk::FWD_THREADS, 0, s>>>(p);
            e = cudaGetLastError();
        } else if (d.sp_blk) {
            if constexpr (std::is_same<T, double>::value && std::is_same<TS, double>::value) {
                if (rt == 1) FK_TIMED("fk_fwd_sparse", s) fk::fk_fwd_sparse_kernel<1, FWD_U><<<fgrid, fk::FWD_THREADS, 0, s>>>(p);
                else if (rt == 2) FK_TIMED("fk_fwd_sparse", s) fk::fk_fwd_sparse_kernel<2, FWD_U><<<fgrid, fk::FWD_THREADS, 0, s>>>(p);
                else FK_TIMED("fk_fwd_sparse", s) fk::fk_fwd_sparse_kernel<4, FWD_U><<<fgrid, fk::FWD_THREADS, 0, s>>>(p);
            }
            e = cudaGetLastError();
        } else
            e = fwd_dispatch<T, false, TS>(d.vec_ok, rt, p, fgrid, s);
        if (e != cudaSuccess) return fail(FK_ERR_CUDA, "forward kernel launch failed: %s", cudaGetErrorString(e));
        ++nl;
        r0 += std::min(rt, R - r0);
    }
    if (pl.nkb > 1 && !l2_in_kernel) {
        fk::ReduceParams q;
        memset(&q, 0, sizeof q);
        q.desc = d;
        if (fewrows) q.desc.nchunks = std::max(1, sm_count()) * 16;  // one partial per CTA of the few-rows kernel
        q.part = part;
        q.sigma = sigma;
        q.rows = d.N;
        q.R = R;
        const long long outs = (long long)d.N * R;
        const int grid = (int)std::min<long long>((outs + 7) / 8, (long long)sm_count() * 8);
        FK_TIMED("fk_reduce_chunks", s) launch_pdl(fk::fk_reduce_chunks_kernel<T, false>, std::max(1, grid), 256, 0, s, q);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return fail(FK_ERR_CUDA, "reduce kernel launch failed: %s", cudaGetErrorString(e));
        ++nl;
    }
    if (launches) *launches = nl;
    return FK_OK;
}

// `G` holds >= G_elems_per_replica * R doubles.
template <typename T, typename TS = T>
int run_vjp_single(const fk::TableDesc& d, const fk::ChannelList& ch, const Plan& pl, const T* f, const T* g, T* df,
                   int R, double* G, cudaStream_t s, int* launches) {
    int nl = 0;
    if constexpr (std::is_same<TS, double>::value) {
        if (gemm_wanted<T>(d, R)) return run_vjp_gemm<T, TS>(d, ch, f, g, df, R, G, s, launches);
    } else {
        if (vjp32_wanted(d, R)) return run_vjp_gemm<T, TS>(d, ch, f, g, df, R, G, s, launches);
    }
    {
        fk::ColsumParams p;
        memset(&p, 0, sizeof p);
        p.desc = d;
        p.g = g;
        p.G = G;
        p.R = R;
        p.nkb = pl.nkb;
        for (int r0 = 0; r0 < R;) {
            const int rt = pick_rt(R - r0);
            p.r0 = r0;
            cudaError_t e;
            if (d.sp_blk) {
                if constexpr (std::is_same<T, double>::value && std::is_same<TS, double>::value) {
                    const int cgrid = pl.nkb * pl.nsplit;
                    if (rt == 1) FK_TIMED("fk_colsum_sparse", s) fk::fk_colsum_sparse_kernel<1, 8><<<cgrid, fk::COLSUM_THREADS, 0, s>>>(p);
                    else if (rt == 2) FK_TIMED("fk_colsum_sparse", s) fk::fk_colsum_sparse_kernel<2, 8><<<cgrid, fk::COLSUM_THREADS, 0, s>>>(p);
                    else FK_TIMED("fk_colsum_sparse", s) fk::fk_colsum_sparse_kernel<4, 8><<<cgrid, fk::COLSUM_THREADS, 0, s>>>(p);
                }
                e = cudaGetLastError();
            } else
                e = colsum_dispatch<T, false, TS>(d.vec_ok, rt, p, pl.nkb * pl.nsplit, s);
            if (e != cudaSuccess) return fail(FK_ERR_CUDA, "colsum kernel launch failed: %s", cudaGetErrorString(e));
            ++nl;
            r0 += rt;
        }
    }
    if (foldk_ok(d)) {
        if (!ensure_dyn_smem(fk::fk_vjp_foldk_kernel<T, false>, foldk_smem(128)))
            return fail(FK_ERR_CUDA, "vjp: cannot reserve %zu bytes of shared memory", foldk_smem(128));
        fk::FoldKParams q;
        memset(&q, 0, sizeof q);
        q.desc = d;
        q.desc.cx_off = 0;
        q.chan = ch;
        q.f = f;
        q.G = G;
        q.cx_total = (long long)d.C * d.nx;
        q.PA = G + G_elems_per_replica(d) * R;
        q.PB = q.PA + q.cx_total * R;
        q.nchunk = foldk_chunks(d.C);
        q.df = df;
        q.R = R;
        const long long slots = (long long)d.nfl * d.nx;
        FK_TIMED("fk_vjp_foldk", s) launch_pdl(fk::fk_vjp_foldk_kernel<T, false>, dim3(d.C * q.nchunk, R), fk::FOLDK_THREADS, foldk_smem(d.nx), s, q);
        FK_TIMED("fk_vjp_foldk_final", s) launch_pdl(fk::fk_vjp_foldk_final_kernel<T, false>, dim3((unsigned)((slots + 7) / 8), R), 256, 0, s, q, slots);
        ++nl;
    } else {
        fk::GatherParams q;
        memset(&q, 0, sizeof q);
        q.desc = d;
        q.chan = ch;
        q.f = f;
        q.G = G;
        q.df = df;
        q.R = R;
        FK_TIMED("fk_vjp_gather", s) fk::fk_vjp_gather_kernel<T, false><<<dim3(d.nfl * d.nx, R), fk::GATHER_THREADS, 0, s>>>(q);
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(FK_ERR_CUDA, "gather kernel launch failed: %s", cudaGetErrorString(e));
    ++nl;
    if (launches) *launches = nl;
    return FK_OK;
}

// forward + VJP from one read of FK (fk_fused_column_kernel), small R, hadronic tables.
// scratch: part [N][R][nchunks] | G [fsplit][R][K] | fold partials
template <typename T>
bool fused_ok(const fk::TableDesc& d, int R) {
    return !gemm_wanted<T>(d, R) && !vjp32_wanted(d, R) && !d.sp_blk && foldk_ok(d) && (d.N + d.fsplit - 1) / d.fsplit <= 64 && opt(FK_OPT_FUSED);
}
size_t fused_scratch_elems(const fk::TableDesc& d, int R) {
    return (part_elems_per_replica(d) + (size_t)d.fsplit * d.K + (1 + FOLDK_MAX_CHUNKS) * (size_t)d.C * d.nx) * R;
}

template <typename T, typename TS = T>
int run_conv_vjp_fused(const fk::TableDesc& d0, const fk::ChannelList& ch, const Plan& pl, const T* f, const T* g,
                       T* sigma, T* df, int R, double* scratch, cudaStream_t s, int* launches) {
    constexpr int VW = fk::VecWidth<TS>::value;
    fk::TableDesc d = d0;
    // up to 64 datapoints per CTA (the forward alone takes ~32): half as many column-sum slices to write and to fold
    d.fsplit = std::max(1, std::min(d0.fsplit, (d0.N + 63) / 64));
    d.nsplit = d.fsplit;  // the column sums are cut into the forward's datapoint ranges
    double* part = scratch;
    double* G = part + part_elems_per_replica(d) * R;
    int nl = 0;
    fk::FusedParams p;
    memset(&p, 0, sizeof p);
    p.fwd.desc = d;
    p.fwd.chan = ch;
    p.fwd.f = f;
    p.fwd.part = part;
    p.fwd.sigma = sigma;
    p.fwd.R = R;
    p.g = g;
    p.G = G;
    const int grid = pl.nkb * d.fsplit;
    for (int r0 = 0; r0 < R;) {
        const int rt = pick_rt(R - r0);
        p.fwd.r0 = r0;
#define FK_FUSED(V, RTv) FK_TIMED("fk_fused_column", s) fk::fk_fused_column_kernel<T, V, RTv, FWD_U, false, TS><<<grid, fk::FWD_THREADS, 0, s>>>(p)
        if (d.vec_ok) {
            if (rt == 1) FK_FUSED(VW, 1); else if (rt == 2) FK_FUSED(VW, 2); else FK_FUSED(VW, 4);
        } else {
            if (rt == 1) FK_FUSED(1, 1); else if (rt == 2) FK_FUSED(1, 2); else FK_FUSED(1, 4);
        }
#undef FK_FUSED
        ++nl;
        r0 += rt;
    }
    if (pl.nkb > 1) {
        fk::ReduceParams q;
        memset(&q, 0, sizeof q);
        q.desc = d;
        q.part = part;
        q.sigma = sigma;
        q.rows = d.N;
        q.R = R;
        const long long outs = (long long)d.N * R;
        const int rgrid = (int)std::min<long long>((outs + 7) / 8, (long long)sm_count() * 8);
        FK_TIMED("fk_reduce_chunks", s) launch_pdl(fk::fk_reduce_chunks_kernel<T, false>, std::max(1, rgrid), 256, 0, s, q);
        ++nl;
    }
    if (!ensure_dyn_smem(fk::fk_vjp_foldk_kernel<T, false>, foldk_smem(128)))
        return fail(FK_ERR_CUDA, "conv_vjp: cannot reserve %zu bytes of shared memory", foldk_smem(128));
    fk::FoldKParams q;
    memset(&q, 0, sizeof q);
    q.desc = d;
    q.desc.cx_off = 0;
    q.chan = ch;
    q.f = f;
    q.G = G;
    q.cx_total = (long long)d.C * d.nx;
    q.PA = G + (size_t)d.fsplit * d.K * R;
    q.PB = q.PA + q.cx_total * R;
    q.nchunk = foldk_chunks(d.C);
    q.df = df;
    q.R = R;
    const long long slots = (long long)d.nfl * d.nx;
    FK_TIMED("fk_vjp_foldk", s) launch_pdl(fk::fk_vjp_foldk_kernel<T, false>, dim3(d.C * q.nchunk, R), fk::FOLDK_THREADS, foldk_smem(d.nx), s, q);
    FK_TIMED("fk_vjp_foldk_final", s) launch_pdl(fk::fk_vjp_foldk_final_kernel<T, false>, dim3((unsigned)((slots + 7) / 8), R), 256, 0, s, q, slots);
    nl += 2;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(FK_ERR_CUDA, "fused forward + VJP launch failed: %s", cudaGetErrorString(e));
    if (launches) *launches = nl;
    return FK_OK;
}

template <typename T>
size_t conv_scratch_elems(const fk::TableDesc& d, int R, bool with_kdec) {
    if (gemm_wanted<T>(d, R)) return gemm_fwd_scratch_elems(d, R, with_kdec);
    size_t need = part_elems_per_replica(d) * R;
    if (fwd32_wanted(d, R)) need = std::max(need, gemm_fwd_scratch_elems(d, R, false));   // FK_F32S64 handles size with T = float
    if (std::is_same<T, float>::value && d.tmap && d.kind == fk::KIND_HADRONIC && d.nx <= fk::TC_MAX_NX)   // either fp32 path may be selected later
        need = std::max(need, tc32_scratch_elems(d, R));
    return need;
}
template <typename T>
size_t vjp_scratch_elems(const fk::TableDesc& d, int R) {
    if (gemm_wanted<T>(d, R) || vjp32_wanted(d, R)) return gemm_vjp_scratch_elems(d, R);
    return (G_elems_per_replica(d) + foldk_elems_per_replica(d)) * R;
}

// stateless front end shared by the fp64 / fp32 entry points
template <typename T>
int stateless(const char* who, int kind, bool vjp, const T* fkp, const int32_t* idx, const T* f, const T* g, T* out,
              int N, int nx, int nfl, int C, int R, void* stream) {
    g_err.clear();
    if (!fkp || !idx || !f || !out || (vjp && !g)) return fail(FK_ERR_INVALID_ARG, "%s: null pointer", who);
    int rc = check_dims(who, kind, N, nx, nfl, C, R);
    if (rc) return rc;
    if ((uintptr_t)fkp % sizeof(T) || (uintptr_t)f % sizeof(T) || (uintptr_t)out % sizeof(T))
        return fail(FK_ERR_INVALID_ARG, "%s: misaligned pointer", who);
    fk::ChannelList ch;
    rc = fill_channels(who, kind, idx, nfl, C, ch);
    if (rc) return rc;
    fk::TableDesc d = make_desc(kind, fk::LAYOUT_LOGICAL, fkp, N, nx, nfl, C, 0, dtype_of<T>());
    Plan pl;
    make_plan(d, dtype_of<T>(), pl);
    cudaStream_t s = (cudaStream_t)stream;
    const size_t elems = vjp ? vjp_scratch_elems<T>(d, R) : conv_scratch_elems<T>(d, R, true);
    double* scratch = nullptr;
    if (elems) FK_CUDA(cudaMallocAsync((void**)&scratch, elems * sizeof(double), s));
    rc = vjp ? run_vjp_single<T>(d, ch, pl, f, g, out, R, scratch, s, nullptr)
             : run_conv_single<T>(d, ch, pl, nullptr, f, out, R, scratch, s, nullptr);
    if (scratch) {
        cudaError_t e = cudaFreeAsync(scratch, s);
        if (rc == FK_OK && e != cudaSuccess) return fail(FK_ERR_CUDA, "cudaFreeAsync: %s", cudaGetErrorString(e));
    }
    return rc;
}

}  // namespace

// --------------------------------------------------------------------------------------------------
// handles
// --------------------------------------------------------------------------------------------------
// A handle owns ONE scratch buffer: calls on it are serialised.  Host threads take the handle's mutex for the
// duration of the (asynchronous) call; on the device every call records an event after its last kernel, and a
// call that arrives on a different stream first makes that stream wait for it.  While a stream is being captured
// into a CUDA graph neither happens (one stream per handle inside a capture) and the scratch must not grow.
struct HandleSync {
    std::mutex mu;
    int device = -1;
    cudaEvent_t done = nullptr;
    cudaStream_t last = nullptr;
    bool used = false;
    int init() {
        if (cudaGetDevice(&device) != cudaSuccess) return FK_ERR_CUDA;
        return cudaEventCreateWithFlags(&done, cudaEventDisableTiming) == cudaSuccess ? FK_OK : FK_ERR_CUDA;
    }
    void destroy() {
        if (done) cudaEventDestroy(done);
        done = nullptr;
    }
};

struct fk_table {
    HandleSync sync;
    fk::TableDesc desc;
    fk::ChannelList chan;
    Plan plan;
    int dtype = FK_F64, store = FK_STORE_BORROW, kind = FK_KIND_HADRONIC;
    void* owned_fk = nullptr;
    uint8_t* dev_chan = nullptr;  // [2][C] for grouped launches
    uint32_t* kdec = nullptr;     // [K] k -> (slot a, slot b) codes for the R >> 1 contraction
    void* d_tmap = nullptr;       // device copy of the CUtensorMap of a packed fp32 hadronic table (fk_tc32.cu)
    int* l2cnt = nullptr;         // [fsplit] tickets of the forward kernel's in-kernel level-2 reduction (zero between launches)
    void* sp_blk = nullptr;       // FK_STORE_SPARSE (fk_sparse.cuh): index records; owned_fk holds the nonzero values
    size_t sp_bytes = 0;          // bytes of the sparse table as stored (values + masks + headers)
    double* scratch = nullptr;    // forward partials / VJP column sums (one buffer, used by one call at a time)
    size_t scratch_elems = 0;
    void* h_stage = nullptr;      // pinned host staging for the *_host calls
    void* d_stage = nullptr;
    size_t stage_bytes = 0;
    int last_launches = 0;
};

namespace {

bool stream_capturing(cudaStream_t s) {
    cudaStreamCaptureStatus st = cudaStreamCaptureStatusNone;
    return cudaStreamIsCapturing(s, &st) == cudaSuccess && st != cudaStreamCaptureStatusNone;
}

// Scope of one compute call on a handle (see HandleSync).
struct CallGuard {
    HandleSync& h;
    cudaStream_t s;
    bool capturing = false;
    std::unique_lock<std::mutex> lk;
    CallGuard(HandleSync& h_, cudaStream_t s_) : h(h_), s(s_), lk(h_.mu) {}
    int begin(const char* who) {
        int dev = -1;
        if (cudaGetDevice(&dev) != cudaSuccess) return fail(FK_ERR_CUDA, "%s: no CUDA device", who);
        if (dev != h.device)
            return fail(FK_ERR_INVALID_ARG, "%s: the handle lives on device %d, the current device is %d", who, h.device, dev);
        capturing = stream_capturing(s);
        if (!capturing && h.used && h.last != s) {
            cudaError_t e = cudaStreamWaitEvent(s, h.done, 0);
            if (e != cudaSuccess) return fail(FK_ERR_CUDA, "%s: cudaStreamWaitEvent: %s", who, cudaGetErrorString(e));
        }
        return FK_OK;
    }
    ~CallGuard() {
        if (!capturing && h.done && cudaEventRecord(h.done, s) == cudaSuccess) {
            h.last = s;
            h.used = true;
        }
    }
};

int ensure_scratch(fk_table* t, size_t elems, cudaStream_t s = nullptr) {
    if (elems <= t->scratch_elems) return FK_OK;
    if (stream_capturing(s))
        return fail(FK_ERR_UNSUPPORTED, "the table's scratch must grow to %zu doubles, which cannot happen during stream capture: "
                                        "give R_hint at create or make one call outside the capture first", elems);
    if (t->scratch) cudaFree(t->scratch);
    t->scratch = nullptr;
    t->scratch_elems = 0;
    FK_CUDA(cudaMalloc((void**)&t->scratch, elems * sizeof(double)));
    t->scratch_elems = elems;
    return FK_OK;
}

int ensure_stage(fk_table* t, size_t bytes) {
    if (bytes <= t->stage_bytes) return FK_OK;
    if (t->h_stage) cudaFreeHost(t->h_stage);
    if (t->d_stage) cudaFree(t->d_stage);
    t->h_stage = t->d_stage = nullptr;
    t->stage_bytes = 0;
    FK_CUDA(cudaMallocHost(&t->h_stage, bytes));
    FK_CUDA(cudaMalloc(&t->d_stage, bytes));
    t->stage_bytes = bytes;
    return FK_OK;
}

size_t table_scratch_need(const fk_table* t, int R) {
    const size_t conv = t->dtype == FK_F64 ? conv_scratch_elems<double>(t->desc, R, t->kdec == nullptr)
                                           : conv_scratch_elems<float>(t->desc, R, true);
    const size_t vjp = t->dtype == FK_F64 ? vjp_scratch_elems<double>(t->desc, R) : vjp_scratch_elems<float>(t->desc, R);
    return std::max(conv, vjp);
}

template <typename T, typename TS = T>
int table_conv_t(fk_table* t, const void* f, void* sigma, int R, cudaStream_t s) {
    int rc = ensure_scratch(t, table_scratch_need(t, R), s);
    if (rc) return rc;
    return run_conv_single<T, TS>(t->desc, t->chan, t->plan, t->kdec, (const T*)f, (T*)sigma, R, t->scratch, s,
                              &t->last_launches, t->l2cnt);
}

template <typename T, typename TS = T>
int table_vjp_t(fk_table* t, const void* f, const void* g, void* df, int R, cudaStream_t s) {
    int rc = ensure_scratch(t, table_scratch_need(t, R), s);
    if (rc) return rc;
    return run_vjp_single<T, TS>(t->desc, t->chan, t->plan, (const T*)f, (const T*)g, (T*)df, R, t->scratch, s,
                             &t->last_launches);
}

template <typename T, typename TS = T>
int table_conv_vjp_t(fk_table* t, const void* f, const void* g, void* sigma, void* df, int R, cudaStream_t s) {
    if (!fused_ok<T>(t->desc, R)) {
        int rc = table_conv_t<T, TS>(t, f, sigma, R, s);
        if (rc) return rc;
        const int nl = t->last_launches;
        rc = table_vjp_t<T, TS>(t, f, g, df, R, s);
        t->last_launches += nl;
        return rc;
    }
    int rc = ensure_scratch(t, std::max(table_scratch_need(t, R), fused_scratch_elems(t->desc, R)), s);
    if (rc) return rc;
    return run_conv_vjp_fused<T, TS>(t->desc, t->chan, t->plan, (const T*)f, (const T*)g, (T*)sigma, (T*)df, R, t->scratch, s,
                                 &t->last_launches);
}

}  // namespace

extern "C" {

const char* fk_last_error_string(void) { return g_err.c_str(); }
int fk_version(void) { return 100; }
int fk_compiled_arch(void) { return 100; }

int fk_set_option(int option, int value) {
    if (option < 0 || option >= FK_OPT_COUNT_) return fail(FK_ERR_INVALID_ARG, "fk_set_option: unknown option %d", option);
    g_opt[option] = value;
    return FK_OK;
}
int fk_get_option(int option, int* value) {
    if (option < 0 || option >= FK_OPT_COUNT_ || !value) return fail(FK_ERR_INVALID_ARG, "fk_get_option: bad argument");
    *value = g_opt[option];
    return FK_OK;
}

int fk_profile_enable(int on) {
    std::lock_guard<std::mutex> lk(g_prof.mu);
    g_prof.on = on != 0;
    return FK_OK;
}
// finished records of the current batch, summed per kernel name; clears the batch
static void prof_collect(std::vector<std::pair<const char*, std::pair<int, double>>>& out) {
    for (size_t i = 0; i < g_prof.used; ++i) {
        float ms = 0.f;
        if (cudaEventSynchronize(g_prof.recs[i].b) != cudaSuccess ||
            cudaEventElapsedTime(&ms, g_prof.recs[i].a, g_prof.recs[i].b) != cudaSuccess)
            continue;
        bool found = false;
        for (auto& o : out)
            if (!strcmp(o.first, g_prof.recs[i].name)) { o.second.first++; o.second.second += ms; found = true; break; }
        if (!found) out.push_back({g_prof.recs[i].name, {1, (double)ms}});
    }
    g_prof.used = 0;
}
int fk_profile_read(double* mean_kernel_ms, int* launches) {
    std::lock_guard<std::mutex> lk(g_prof.mu);
    std::vector<std::pair<const char*, std::pair<int, double>>> v;
    prof_collect(v);
    // the record with the largest total time (the dominant kernel of what ran)
    const std::pair<const char*, std::pair<int, double>>* best = nullptr;
    for (auto& o : v)
        if (!best || o.second.second > best->second.second) best = &o;
    if (mean_kernel_ms) *mean_kernel_ms = best ? best->second.second / best->second.first : 0.0;
    if (launches) *launches = best ? best->second.first : 0;
    return FK_OK;
}
int fk_profile_report(char* buf, int capacity) {
    if (!buf || capacity <= 0) return fail(FK_ERR_INVALID_ARG, "fk_profile_report: no buffer");
    std::lock_guard<std::mutex> lk(g_prof.mu);
    std::vector<std::pair<const char*, std::pair<int, double>>> v;
    prof_collect(v);
    int pos = 0;
    buf[0] = 0;
    for (auto& o : v) {
        const int n = snprintf(buf + pos, (size_t)(capacity - pos), "%s\t%d\t%.9g\n", o.first, o.second.first, o.second.second);
        if (n < 0 || n >= capacity - pos) return fail(FK_ERR_INVALID_ARG, "fk_profile_report: buffer of %d bytes is too small", capacity);
        pos += n;
    }
    return FK_OK;
}

// ---- latency floors ("L2 caveat"): an empty launch and a plain read of `bytes` bytes, so that the
// microsecond-scale configs (0 and 1) can be read against what ANY kernel over the same bytes would cost ----
namespace {
__global__ void fk_probe_empty_kernel() {}
__global__ void __launch_bounds__(256) fk_probe_read_kernel(const double2* __restrict__ buf, long long n16, double* __restrict__ sink) {
    double acc = 0.0;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < n16; t += (long long)gridDim.x * blockDim.x) {
        double2 v;
        asm volatile("ld.global.nc.L1::no_allocate.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(buf + t));
        acc += v.x + v.y;
    }
    if (acc == 1.2345e300) *sink = acc;   // keeps the loads alive; never true for finite tables
}
}  // namespace

int fk_probe_launch(int kind, const void* buf, long long bytes, double* sink, void* stream) {
    g_err.clear();
    cudaStream_t s = (cudaStream_t)stream;
    if (kind == 0) {
        fk_probe_empty_kernel<<<1, 32, 0, s>>>();
    } else if (kind == 1) {
        if (!buf || !sink || bytes < 16 || (uintptr_t)buf % 16) return fail(FK_ERR_INVALID_ARG, "fk_probe_launch: needs a 16-byte aligned buffer and a sink");
        const long long n16 = bytes / 16;
        const int grid = (int)std::min<long long>((n16 + 255) / 256, (long long)std::max(1, sm_count()) * 8);
        fk_probe_read_kernel<<<grid, 256, 0, s>>>((const double2*)buf, n16, sink);
    } else
        return fail(FK_ERR_INVALID_ARG, "fk_probe_launch: kind=%d", kind);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(FK_ERR_CUDA, "fk_probe_launch: %s", cudaGetErrorString(e));
    return FK_OK;
}

// ---- two-PDF (p pbar) form: stacked flavours, then the single-PDF path (fk_pack.cuh, fk_stack2_kernel) ----
namespace {
int hadronic2(const char* who, bool vjp, const double* fkp, const int32_t* pairs, const double* f1, const double* f2, const double* g,
              double* out1, double* out2, int N, int nx, int nfl, int C, int R, void* stream) {
    g_err.clear();
    if (!fkp || !pairs || !f1 || !f2 || !out1 || (vjp && (!g || !out2))) return fail(FK_ERR_INVALID_ARG, "%s: null pointer", who);
    int rc = check_dims(who, FK_KIND_HADRONIC, N, nx, nfl, C, R);
    if (rc) return rc;
    if (2 * nfl > fk::MAX_NFL) return fail(FK_ERR_UNSUPPORTED, "%s: 2*nfl=%d > %d", who, 2 * nfl, fk::MAX_NFL);
    std::vector<int32_t> p2(2 * (size_t)C);
    for (int c = 0; c < C; ++c) {
        const int a = pairs[2 * c], b = pairs[2 * c + 1];
        if (a < 0 || a >= nfl || b < 0 || b >= nfl)
            return fail(FK_ERR_INVALID_ARG, "%s: flavour index out of [0,%d) at channel %d: (%d,%d)", who, nfl, c, a, b);
        p2[2 * c] = a;
        p2[2 * c + 1] = nfl + b;
    }
    cudaStream_t s = (cudaStream_t)stream;
    const int slots = nfl * nx;
    const size_t fe = 2 * (size_t)R * slots;
    double* F = nullptr;
    FK_CUDA(cudaMallocAsync((void**)&F, (vjp ? 2 : 1) * fe * sizeof(double), s));
    const int grid = (int)std::min<size_t>(1024, (fe + 255) / 256);
    fk::fk_stack2_kernel<double><<<grid, 256, 0, s>>>(f1, f2, F, R, slots);
    if (vjp) {
        rc = stateless<double>(who, FK_KIND_HADRONIC, true, fkp, p2.data(), F, g, F + fe, N, nx, 2 * nfl, C, R, stream);
        if (rc == FK_OK) fk::fk_unstack2_kernel<double><<<grid, 256, 0, s>>>(F + fe, out1, out2, R, slots);
    } else {
        rc = stateless<double>(who, FK_KIND_HADRONIC, false, fkp, p2.data(), F, nullptr, out1, N, nx, 2 * nfl, C, R, stream);
    }
    const std::string keep = g_err;   // stateless() clears the message on entry only; keep it across the free
    cudaError_t e = cudaGetLastError();
    cudaError_t e2 = cudaFreeAsync(F, s);
    if (rc != FK_OK) { g_err = keep; return rc; }
    if (e != cudaSuccess || e2 != cudaSuccess) return fail(FK_ERR_CUDA, "%s: %s", who, cudaGetErrorString(e != cudaSuccess ? e : e2));
    return FK_OK;
}
}  // namespace

int fk_conv_hadronic2(const double* fk, const int32_t* pairs, const double* f1, const double* f2, double* sigma, int N, int nx,
                      int nfl, int C, int R, void* stream) {
    return hadronic2("fk_conv_hadronic2", false, fk, pairs, f1, f2, nullptr, sigma, nullptr, N, nx, nfl, C, R, stream);
}
int fk_conv_hadronic2_vjp(const double* fk, const int32_t* pairs, const double* f1, const double* f2, const double* g, double* df1,
                          double* df2, int N, int nx, int nfl, int C, int R, void* stream) {
    return hadronic2("fk_conv_hadronic2_vjp", true, fk, pairs, f1, f2, g, df1, df2, N, nx, nfl, C, R, stream);
}

int fk_conv_dis(const double* fk, const int32_t* flav, const double* f, double* sigma, int N, int nx, int nfl, int nA,
                int R, void* stream) {
    return stateless<double>("fk_conv_dis", FK_KIND_DIS, false, fk, flav, f, nullptr, sigma, N, nx, nfl, nA, R, stream);
}
int fk_conv_hadronic(const double* fk, const int32_t* pairs, const double* f, double* sigma, int N, int nx, int nfl,
                     int C, int R, void* stream) {
    return stateless<double>("fk_conv_hadronic", FK_KIND_HADRONIC, false, fk, pairs, f, nullptr, sigma, N, nx, nfl, C, R,
                             stream);
}
// ---- allocation-free forward (include/fkconv.h, fk_conv_hadronic_static) -------------------------------------------
// The scratch of the forward path in a file-scope device array.  In HOST code the name below is a host-side stand-in, not
// a device address: only static_scratch_ptr() may touch it, and kernels get the address cudaGetSymbolAddress returned.
static __device__ __align__(256) unsigned char fk_static_scratch[FK_STATIC_SCRATCH_BYTES];
namespace {
constexpr size_t STATIC_TICKET_BYTES = 4096;   // [1024] tickets of the in-kernel level-2 reduction, ahead of the doubles
constexpr int STATIC_MAX_DEVICES = 64;

// device address of the array on the CURRENT device: looked up once per device, with that device current
int static_scratch_ptr(const char* who, unsigned char** out) {
    static std::mutex mu;
    static unsigned char* ptr[STATIC_MAX_DEVICES] = {};
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(FK_ERR_CUDA, "%s: no CUDA device (%s)", who, cudaGetErrorString(e));
    if (dev < 0 || dev >= STATIC_MAX_DEVICES) return fail(FK_ERR_UNSUPPORTED, "%s: device ordinal %d beyond %d", who, dev, STATIC_MAX_DEVICES - 1);
    std::lock_guard<std::mutex> lk(mu);
    if (!ptr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, fk_static_scratch);
        if (e != cudaSuccess || !p) return fail(FK_ERR_CUDA, "%s: cudaGetSymbolAddress failed on device %d: %s", who, dev, cudaGetErrorString(e));
        ptr[dev] = static_cast<unsigned char*>(p);
    }
    *out = ptr[dev];
    return FK_OK;
}
}  // namespace

int fk_conv_hadronic_static(const double* fkp, const int32_t* pairs, const double* f, double* sigma, int N, int nx, int nfl,
                            int C, int R, void* stream) {
    const char* who = "fk_conv_hadronic_static";
    g_err.clear();
    if (!fkp || !pairs || !f || !sigma) return fail(FK_ERR_INVALID_ARG, "%s: null pointer", who);
    int rc = check_dims(who, FK_KIND_HADRONIC, N, nx, nfl, C, R);
    if (rc) return rc;
    if ((uintptr_t)fkp % sizeof(double) || (uintptr_t)f % sizeof(double) || (uintptr_t)sigma % sizeof(double))
        return fail(FK_ERR_INVALID_ARG, "%s: misaligned pointer", who);
    fk::ChannelList ch;
    rc = fill_channels(who, FK_KIND_HADRONIC, pairs, nfl, C, ch);
    if (rc) return rc;
    fk::TableDesc d = make_desc(FK_KIND_HADRONIC, fk::LAYOUT_LOGICAL, fkp, N, nx, nfl, C, 0, FK_F64);
    Plan pl;
    make_plan(d, FK_F64, pl);
    const size_t need = conv_scratch_elems<double>(d, R, true) * sizeof(double) + STATIC_TICKET_BYTES;
    if (need > (size_t)FK_STATIC_SCRATCH_BYTES)
        return fail(FK_ERR_UNSUPPORTED, "%s: N=%d nx=%d C=%d R=%d needs %zu bytes of scratch, the static array holds %zu "
                                        "(FK_STATIC_SCRATCH_BYTES): use fk_conv_hadronic or a resident table", who, N, nx, C, R, need,
                    (size_t)FK_STATIC_SCRATCH_BYTES);
    unsigned char* base = nullptr;
    rc = static_scratch_ptr(who, &base);
    if (rc) return rc;
    cudaStream_t s = (cudaStream_t)stream;
    int* cnt = nullptr;
    if ((size_t)pl.fsplit * sizeof(int) <= STATIC_TICKET_BYTES) {   // the tickets must start at zero whatever the last call left
        cnt = reinterpret_cast<int*>(base);
        FK_CUDA(cudaMemsetAsync(cnt, 0, (size_t)pl.fsplit * sizeof(int), s));
    }
    return run_conv_single<double>(d, ch, pl, nullptr, f, sigma, R, reinterpret_cast<double*>(base + STATIC_TICKET_BYTES), s, nullptr, cnt);
}

int fk_conv_hadronic_vjp(const double* fk, const int32_t* pairs, const double* f, const double* g, double* df, int N,
                         int nx, int nfl, int C, int R, void* stream) {
    return stateless<double>("fk_conv_hadronic_vjp", FK_KIND_HADRONIC, true, fk, pairs, f, g, df, N, nx, nfl, C, R,
                             stream);
}
int fk_conv_dis_vjp(const double* fk, const int32_t* flav, const double* f, const double* g, double* df, int N, int nx,
                    int nfl, int nA, int R, void* stream) {
    return stateless<double>("fk_conv_dis_vjp", FK_KIND_DIS, true, fk, flav, f, g, df, N, nx, nfl, nA, R, stream);
}
int fk_conv_dis_f32(const float* fk, const int32_t* flav, const float* f, float* sigma, int N, int nx, int nfl, int nA,
                    int R, void* stream) {
    return stateless<float>("fk_conv_dis_f32", FK_KIND_DIS, false, fk, flav, f, nullptr, sigma, N, nx, nfl, nA, R, stream);
}
int fk_conv_hadronic_f32(const float* fk, const int32_t* pairs, const float* f, float* sigma, int N, int nx, int nfl,
                         int C, int R, void* stream) {
    return stateless<float>("fk_conv_hadronic_f32", FK_KIND_HADRONIC, false, fk, pairs, f, nullptr, sigma, N, nx, nfl, C,
                            R, stream);
}
int fk_conv_hadronic_vjp_f32(const float* fk, const int32_t* pairs, const float* f, const float* g, float* df, int N,
                             int nx, int nfl, int C, int R, void* stream) {
    return stateless<float>("fk_conv_hadronic_vjp_f32", FK_KIND_HADRONIC, true, fk, pairs, f, g, df, N, nx, nfl, C, R,
                            stream);
}

// ---------------------------------------------------------------------------------------- tables
int fk_table_create(fk_table** out, int kind, const double* fk_logical, const int32_t* index_list, int N, int nx,
                    int nfl, int C, int dtype, int store, int R_hint) {
    g_err.clear();
    if (!out) return fail(FK_ERR_INVALID_ARG, "fk_table_create: null out");
    *out = nullptr;
    if (!fk_logical || !index_list) return fail(FK_ERR_INVALID_ARG, "fk_table_create: null pointer");
    if (kind != FK_KIND_DIS && kind != FK_KIND_HADRONIC) return fail(FK_ERR_INVALID_ARG, "fk_table_create: bad kind %d", kind);
    if (dtype != FK_F64 && dtype != FK_F32 && dtype != FK_F32S64) return fail(FK_ERR_INVALID_ARG, "fk_table_create: bad dtype %d", dtype);
    if (store != FK_STORE_BORROW && store != FK_STORE_PACK && store != FK_STORE_SPARSE) return fail(FK_ERR_INVALID_ARG, "fk_table_create: bad store %d", store);
    if (store == FK_STORE_SPARSE && dtype != FK_F64) return fail(FK_ERR_UNSUPPORTED, "fk_table_create: sparse storage holds fp64 tables only");
    if (dtype != FK_F64 && store == FK_STORE_BORROW)
        return fail(FK_ERR_INVALID_ARG, "fk_table_create: an fp32 table must be packed (the logical input is fp64)");
    int rc = check_dims("fk_table_create", kind, N, nx, nfl, C, std::max(1, R_hint));
    if (rc) return rc;
    if ((uintptr_t)fk_logical % 8) return fail(FK_ERR_INVALID_ARG, "fk_table_create: misaligned fk pointer");

    fk_table* t = new (std::nothrow) fk_table();
    if (!t) return fail(FK_ERR_ALLOC, "fk_table_create: host allocation failed");
    rc = fill_channels("fk_table_create", kind, index_list, nfl, C, t->chan);
    if (rc) { delete t; return rc; }
    if (t->sync.init() != FK_OK) { delete t; return fail(FK_ERR_CUDA, "fk_table_create: no CUDA device"); }
    t->dtype = dtype; t->store = store; t->kind = kind;

    const int jp = packed_jp(kind, nx, dtype);
    const int cstride = (nx * jp + 3) / 4 * 4;  // packed hadronic channel block (fk_common.cuh)
    const int K = kind == FK_KIND_HADRONIC ? C * (store != FK_STORE_BORROW ? cstride : nx * nx) : C * nx;
    auto bail = [&](int code) { fk_table_destroy(t); return code; };
    if (store == FK_STORE_SPARSE) {
        // two passes over the logical table (one-time): masks + block counts, host scan, values + per-word prefixes
        const int dkind = kind == FK_KIND_HADRONIC ? fk::KIND_HADRONIC : fk::KIND_DIS;
        const int nkb = (K + fk::SP_BLOCK - 1) / fk::SP_BLOCK;
        const long long nblk = (long long)N * nkb;
        if (nblk >= (1LL << 31)) { bail(0); return fail(FK_ERR_UNSUPPORTED, "fk_table_create: sparse table with %lld blocks", nblk); }
        unsigned int* d_count = nullptr;
        cudaError_t e = cudaMalloc(&t->sp_blk, (size_t)nblk * sizeof(fk::SparseBlk));
        if (e == cudaSuccess) e = cudaMalloc((void**)&d_count, (size_t)nblk * sizeof(unsigned int));
        if (e != cudaSuccess) { if (d_count) cudaFree(d_count); bail(0); return fail(FK_ERR_ALLOC, "fk_table_create: sparse index: %s", cudaGetErrorString(e)); }
        fk::fk_sparse_build_kernel<false><<<(unsigned)nblk, 256>>>(fk_logical, dkind, N, nx, C, K, cstride, jp, nkb, d_count,
                                                                   (fk::SparseBlk*)t->sp_blk, nullptr);
        std::vector<unsigned int> cnt((size_t)nblk);
        e = cudaMemcpy(cnt.data(), d_count, (size_t)nblk * sizeof(unsigned int), cudaMemcpyDeviceToHost);
        if (e != cudaSuccess) { cudaFree(d_count); bail(0); return fail(FK_ERR_CUDA, "fk_table_create: sparse pass 1: %s", cudaGetErrorString(e)); }
        // exclusive scan of the block counts on the host (one-time), written into the records' `off` field
        std::vector<unsigned long long> off((size_t)nblk);
        unsigned long long nnz = 0;
        for (long long b = 0; b < nblk; ++b) { off[b] = nnz; nnz += cnt[b]; }
        e = cudaMemcpy2D(t->sp_blk, sizeof(fk::SparseBlk), off.data(), sizeof(unsigned long long), sizeof(unsigned long long), (size_t)nblk,
                         cudaMemcpyHostToDevice);
        cudaFree(d_count);
        if (e == cudaSuccess) e = cudaMalloc(&t->owned_fk, std::max<size_t>(16, (size_t)nnz * sizeof(double)));
        if (e != cudaSuccess) { bail(0); return fail(FK_ERR_ALLOC, "fk_table_create: sparse values (%llu nonzeros): %s", nnz, cudaGetErrorString(e)); }
        fk::fk_sparse_build_kernel<true><<<(unsigned)nblk, 256>>>(fk_logical, dkind, N, nx, C, K, cstride, jp, nkb, nullptr,
                                                                  (fk::SparseBlk*)t->sp_blk, (double*)t->owned_fk);
        e = cudaGetLastError();
        if (e == cudaSuccess) e = cudaDeviceSynchronize();
        if (e != cudaSuccess) { bail(0); return fail(FK_ERR_CUDA, "fk_table_create: sparse pass 2: %s", cudaGetErrorString(e)); }
        t->desc = make_desc(kind, fk::LAYOUT_PACKED, t->owned_fk, N, nx, nfl, C, ((long long)K + 1) / 2 * 2, dtype);
        t->desc.vec_ok = 1;   // the plan's k-blocks are the 512-element sparse blocks
        t->desc.sp_blk = t->sp_blk;
        t->sp_bytes = (size_t)nnz * sizeof(double) + (size_t)nblk * sizeof(fk::SparseBlk);
    } else if (store == FK_STORE_PACK) {
        const int vecw = dtype == FK_F64 ? 2 : 4;
        const long long row_stride = ((long long)K + vecw - 1) / vecw * vecw;
        const size_t bytes = (size_t)N * row_stride * dtype_size(dtype);
        cudaError_t e = cudaMalloc(&t->owned_fk, bytes);
        if (e != cudaSuccess) { bail(0); return fail(FK_ERR_ALLOC, "fk_table_create: cudaMalloc(%zu): %s", bytes, cudaGetErrorString(e)); }
        const long long total = (long long)N * row_stride;
        const int grid = (int)std::min<long long>((total + 255) / 256, 148LL * 64);
        if (dtype == FK_F64)
            fk::fk_pack_kernel<double><<<grid, 256>>>(fk_logical, (double*)t->owned_fk, N, nx, C,
                                                     kind == FK_KIND_HADRONIC ? fk::KIND_HADRONIC : fk::KIND_DIS, K, cstride, jp, row_stride);
        else
            fk::fk_pack_kernel<float><<<grid, 256>>>(fk_logical, (float*)t->owned_fk, N, nx, C,
                                                    kind == FK_KIND_HADRONIC ? fk::KIND_HADRONIC : fk::KIND_DIS, K, cstride, jp, row_stride);
        e = cudaGetLastError();
        if (e == cudaSuccess) e = cudaDeviceSynchronize();
        if (e != cudaSuccess) { bail(0); return fail(FK_ERR_CUDA, "fk_table_create: pack kernel: %s", cudaGetErrorString(e)); }
        t->desc = make_desc(kind, fk::LAYOUT_PACKED, t->owned_fk, N, nx, nfl, C, row_stride, dtype);
    } else {
        t->desc = make_desc(kind, fk::LAYOUT_LOGICAL, fk_logical, N, nx, nfl, C, 0, dtype);
    }
    make_plan(t->desc, dtype, t->plan);

    cudaError_t e = cudaMalloc((void**)&t->l2cnt, std::max(1, t->plan.fsplit) * sizeof(int));
    if (e == cudaSuccess) e = cudaMemset(t->l2cnt, 0, std::max(1, t->plan.fsplit) * sizeof(int));
    if (e != cudaSuccess) { bail(0); return fail(FK_ERR_ALLOC, "fk_table_create: ticket counters: %s", cudaGetErrorString(e)); }
    e = cudaMalloc((void**)&t->dev_chan, 2 * (size_t)C);
    if (e == cudaSuccess) e = cudaMemcpy(t->dev_chan, t->chan.a, C, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(t->dev_chan + C, t->chan.b, C, cudaMemcpyHostToDevice);
    if (e != cudaSuccess) { bail(0); return fail(FK_ERR_CUDA, "fk_table_create: channel upload: %s", cudaGetErrorString(e)); }
    t->desc.chan_a = t->dev_chan;
    t->desc.chan_b = t->dev_chan + C;
    if (dtype == FK_F64 && store != FK_STORE_SPARSE && (long long)nfl * nx < (long long)fk::KDEC_NONE) {
        e = cudaMalloc((void**)&t->kdec, (size_t)K * sizeof(uint32_t));
        if (e == cudaSuccess) {
            fk::fk_kdec_kernel<<<std::min(1024, (K + 255) / 256), 256>>>(t->desc, t->chan, t->kdec);
            e = cudaGetLastError();
            if (e == cudaSuccess) e = cudaDeviceSynchronize();
        }
        if (e != cudaSuccess) { bail(0); return fail(FK_ERR_CUDA, "fk_table_create: k codes: %s", cudaGetErrorString(e)); }
        t->desc.kdec = t->kdec;
    }

    if (dtype == FK_F32 && store == FK_STORE_PACK && kind == FK_KIND_HADRONIC && t->desc.vec_ok) {
        // tensor map for the tcgen05 path; a driver without the entry point simply leaves the table on the column kernels
        alignas(64) unsigned char tm[fk::TC_TMAP_BYTES];
        if (fk::tc32_encode_tensor_map(tm, t->owned_fk, t->desc.row_stride, t->desc.K, N)) {
            e = cudaMalloc(&t->d_tmap, fk::TC_TMAP_BYTES);
            if (e == cudaSuccess) e = cudaMemcpy(t->d_tmap, tm, fk::TC_TMAP_BYTES, cudaMemcpyHostToDevice);
            if (e != cudaSuccess) { bail(0); return fail(FK_ERR_CUDA, "fk_table_create: tensor map upload: %s", cudaGetErrorString(e)); }
            t->desc.tmap = t->d_tmap;
        }
    }
    rc = ensure_scratch(t, table_scratch_need(t, std::max(1, R_hint)));
    if (rc) return bail(rc);
    *out = t;
    return FK_OK;
}

int fk_table_destroy(fk_table* t) {
    if (!t) return FK_OK;
    if (t->owned_fk) cudaFree(t->owned_fk);
    if (t->dev_chan) cudaFree(t->dev_chan);
    if (t->kdec) cudaFree(t->kdec);
    if (t->d_tmap) cudaFree(t->d_tmap);
    if (t->sp_blk) cudaFree(t->sp_blk);
    if (t->l2cnt) cudaFree(t->l2cnt);
    if (t->scratch) cudaFree(t->scratch);
    if (t->h_stage) cudaFreeHost(t->h_stage);
    if (t->d_stage) cudaFree(t->d_stage);
    t->sync.destroy();
    delete t;
    return FK_OK;
}

int fk_table_info(const fk_table* t, int* N, int* nx, int* nfl, int* C, int64_t* K, int64_t* row_stride,
                  int64_t* device_bytes) {
    if (!t) return fail(FK_ERR_INVALID_ARG, "fk_table_info: null table");
    if (N) *N = t->desc.N;
    if (nx) *nx = t->desc.nx;
    if (nfl) *nfl = t->desc.nfl;
    if (C) *C = t->desc.C;
    if (K) *K = t->desc.K;
    if (row_stride) *row_stride = t->desc.row_stride;
    if (device_bytes)
        *device_bytes = (int64_t)((t->sp_blk ? t->sp_bytes : t->owned_fk ? (size_t)t->desc.N * t->desc.row_stride * dtype_size(t->dtype) : 0) +
                                  t->scratch_elems * sizeof(double) + t->stage_bytes + 2 * (size_t)t->desc.C);
    return FK_OK;
}

}  // extern "C"

namespace {
// unguarded bodies (the caller holds the handle's CallGuard)
int table_conv_any(fk_table* t, const void* f, void* sigma, int R, cudaStream_t s) {
    if (t->dtype == FK_F32S64) return table_conv_t<double, float>(t, f, sigma, R, s);
    return t->dtype == FK_F64 ? table_conv_t<double>(t, f, sigma, R, s) : table_conv_t<float>(t, f, sigma, R, s);
}
int table_vjp_any(fk_table* t, const void* f, const void* g, void* df, int R, cudaStream_t s) {
    if (t->dtype == FK_F32S64) return table_vjp_t<double, float>(t, f, g, df, R, s);
    return t->dtype == FK_F64 ? table_vjp_t<double>(t, f, g, df, R, s) : table_vjp_t<float>(t, f, g, df, R, s);
}
int chi2_launch(const double* sigma, const double* data, const double* cinv, double* chi2, double* g, int N, int R, cudaStream_t s) {
    FK_TIMED("fk_chi2_grad", s) fk::fk_chi2_grad_kernel<<<N, dim3(32, 8), 0, s>>>(sigma, data, cinv, g, N, R);
    FK_TIMED("fk_chi2_sum", s) fk::fk_chi2_sum_kernel<<<(R + 7) / 8, 256, 0, s>>>(sigma, data, g, chi2, N, R);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(FK_ERR_CUDA, "fk_chi2 launch failed: %s", cudaGetErrorString(e));
    return FK_OK;
}
}  // namespace

extern "C" {

int fk_table_conv(fk_table* t, const void* f, void* sigma, int R, void* stream) {
    g_err.clear();
    if (!t || !f || !sigma) return fail(FK_ERR_INVALID_ARG, "fk_table_conv: null pointer");
    if (R <= 0) return fail(FK_ERR_INVALID_ARG, "fk_table_conv: R=%d", R);
    CallGuard cg(t->sync, (cudaStream_t)stream);
    if (int rc = cg.begin("fk_table_conv")) return rc;
    return table_conv_any(t, f, sigma, R, (cudaStream_t)stream);
}

int fk_table_vjp(fk_table* t, const void* f, const void* g, void* df, int R, void* stream) {
    g_err.clear();
    if (!t || !f || !g || !df) return fail(FK_ERR_INVALID_ARG, "fk_table_vjp: null pointer");
    if (R <= 0) return fail(FK_ERR_INVALID_ARG, "fk_table_vjp: R=%d", R);
    CallGuard cg(t->sync, (cudaStream_t)stream);
    if (int rc = cg.begin("fk_table_vjp")) return rc;
    return table_vjp_any(t, f, g, df, R, (cudaStream_t)stream);
}

int fk_table_conv_vjp(fk_table* t, const void* f, const void* g, void* sigma, void* df, int R, void* stream) {
    g_err.clear();
    if (!t || !f || !g || !sigma || !df) return fail(FK_ERR_INVALID_ARG, "fk_table_conv_vjp: null pointer");
    if (R <= 0) return fail(FK_ERR_INVALID_ARG, "fk_table_conv_vjp: R=%d", R);
    cudaStream_t s = (cudaStream_t)stream;
    CallGuard cg(t->sync, s);
    if (int rc = cg.begin("fk_table_conv_vjp")) return rc;
    if (t->dtype == FK_F32S64) return table_conv_vjp_t<double, float>(t, f, g, sigma, df, R, s);
    return t->dtype == FK_F64 ? table_conv_vjp_t<double>(t, f, g, sigma, df, R, s)
                              : table_conv_vjp_t<float>(t, f, g, sigma, df, R, s);
}

int fk_chi2(const double* sigma, const double* data, const double* cinv, double* chi2, double* g, int N, int R, void* stream) {
    g_err.clear();
    if (!sigma || !data || !cinv || !chi2 || !g) return fail(FK_ERR_INVALID_ARG, "fk_chi2: null pointer");
    if (N <= 0 || R <= 0) return fail(FK_ERR_INVALID_ARG, "fk_chi2: non-positive size (N=%d R=%d)", N, R);
    return chi2_launch(sigma, data, cinv, chi2, g, N, R, (cudaStream_t)stream);
}

int fk_table_fit_step(fk_table* t, const double* f, const double* data, const double* cinv, double* sigma, double* g,
                      double* chi2, double* df, int R, void* stream) {
    g_err.clear();
    if (!t || !f || !data || !cinv || !sigma || !g || !chi2 || !df) return fail(FK_ERR_INVALID_ARG, "fk_table_fit_step: null pointer");
    if (t->dtype == FK_F32) return fail(FK_ERR_UNSUPPORTED, "fk_table_fit_step: tables with fp64 buffers only (FK_F64, FK_F32S64)");
    if (R <= 0) return fail(FK_ERR_INVALID_ARG, "fk_table_fit_step: R=%d", R);
    cudaStream_t s = (cudaStream_t)stream;
    CallGuard cg(t->sync, s);
    if (int rc = cg.begin("fk_table_fit_step")) return rc;
    int rc = table_conv_any(t, f, sigma, R, s);
    if (rc) return rc;
    const int nl = t->last_launches;
    rc = chi2_launch(sigma, data, cinv, chi2, g, t->desc.N, R, s);
    if (rc) return rc;
    rc = table_vjp_any(t, f, g, df, R, s);
    t->last_launches += nl + 2;
    return rc;
}

int fk_table_conv_host(fk_table* t, const void* f_host, void* sigma_host, int R, void* stream) {
    g_err.clear();
    if (!t || !f_host || !sigma_host) return fail(FK_ERR_INVALID_ARG, "fk_table_conv_host: null pointer");
    if (R <= 0) return fail(FK_ERR_INVALID_ARG, "fk_table_conv_host: R=%d", R);
    const size_t es = io_size(t->dtype);
    const size_t fb = (size_t)R * t->desc.nfl * t->desc.nx * es, sb = (size_t)t->desc.N * R * es;
    const size_t fb_al = (fb + 255) / 256 * 256;
    cudaStream_t s = (cudaStream_t)stream;
    CallGuard cg(t->sync, s);
    if (int rc0 = cg.begin("fk_table_conv_host")) return rc0;
    int rc = ensure_stage(t, 2 * fb_al + 2 * ((sb + 255) / 256 * 256));
    if (rc) return rc;
    char* h = (char*)t->h_stage; char* d = (char*)t->d_stage;
    memcpy(h, f_host, fb);
    FK_CUDA(cudaMemcpyAsync(d, h, fb, cudaMemcpyHostToDevice, s));
    rc = table_conv_any(t, d, d + fb_al, R, s);
    if (rc) return rc;
    FK_CUDA(cudaMemcpyAsync(h + fb_al, d + fb_al, sb, cudaMemcpyDeviceToHost, s));
    FK_CUDA(cudaStreamSynchronize(s));
    memcpy(sigma_host, h + fb_al, sb);
    return FK_OK;
}

int fk_table_vjp_host(fk_table* t, const void* f_host, const void* g_host, void* df_host, int R, void* stream) {
    g_err.clear();
    if (!t || !f_host || !g_host || !df_host) return fail(FK_ERR_INVALID_ARG, "fk_table_vjp_host: null pointer");
    if (R <= 0) return fail(FK_ERR_INVALID_ARG, "fk_table_vjp_host: R=%d", R);
    const size_t es = io_size(t->dtype);
    const size_t fb = (size_t)R * t->desc.nfl * t->desc.nx * es, gb = (size_t)t->desc.N * R * es;
    const size_t fb_al = (fb + 255) / 256 * 256, gb_al = (gb + 255) / 256 * 256;
    cudaStream_t s = (cudaStream_t)stream;
    CallGuard cg(t->sync, s);
    if (int rc0 = cg.begin("fk_table_vjp_host")) return rc0;
    int rc = ensure_stage(t, 2 * fb_al + 2 * gb_al);
    if (rc) return rc;
    char* h = (char*)t->h_stage; char* d = (char*)t->d_stage;
    memcpy(h, f_host, fb);
    memcpy(h + fb_al, g_host, gb);
    FK_CUDA(cudaMemcpyAsync(d, h, fb_al + gb, cudaMemcpyHostToDevice, s));
    rc = table_vjp_any(t, d, d + fb_al, d + fb_al + gb_al, R, s);
    if (rc) return rc;
    FK_CUDA(cudaMemcpyAsync(h + fb_al + gb_al, d + fb_al + gb_al, fb, cudaMemcpyDeviceToHost, s));
    FK_CUDA(cudaStreamSynchronize(s));
    memcpy(df_host, h + fb_al + gb_al, fb);
    return FK_OK;
}

int fk_table_conv_vjp_host(fk_table* t, const void* f_host, const void* g_host, void* sigma_host, void* df_host, int R, void* stream) {
    g_err.clear();
    if (!t || !f_host || !g_host || !sigma_host || !df_host) return fail(FK_ERR_INVALID_ARG, "fk_table_conv_vjp_host: null pointer");
    if (R <= 0) return fail(FK_ERR_INVALID_ARG, "fk_table_conv_vjp_host: R=%d", R);
    const size_t es = io_size(t->dtype);
    const size_t fb = (size_t)R * t->desc.nfl * t->desc.nx * es, gb = (size_t)t->desc.N * R * es;
    const size_t fb_al = (fb + 255) / 256 * 256, gb_al = (gb + 255) / 256 * 256;
    cudaStream_t s = (cudaStream_t)stream;
    CallGuard cg(t->sync, s);
    if (int rc0 = cg.begin("fk_table_conv_vjp_host")) return rc0;
    int rc = ensure_stage(t, 2 * fb_al + 2 * gb_al);   // f | g | sigma | df, one copy in, one copy out
    if (rc) return rc;
    char* h = (char*)t->h_stage; char* d = (char*)t->d_stage;
    memcpy(h, f_host, fb);
    memcpy(h + fb_al, g_host, gb);
    FK_CUDA(cudaMemcpyAsync(d, h, fb_al + gb, cudaMemcpyHostToDevice, s));
    char* d_sig = d + fb_al + gb_al; char* d_df = d_sig + gb_al;
    if (t->dtype == FK_F32S64) rc = table_conv_vjp_t<double, float>(t, d, d + fb_al, d_sig, d_df, R, s);
    else rc = t->dtype == FK_F64 ? table_conv_vjp_t<double>(t, d, d + fb_al, d_sig, d_df, R, s)
                                 : table_conv_vjp_t<float>(t, d, d + fb_al, d_sig, d_df, R, s);
    if (rc) return rc;
    FK_CUDA(cudaMemcpyAsync(h + fb_al + gb_al, d_sig, gb_al + fb, cudaMemcpyDeviceToHost, s));
    FK_CUDA(cudaStreamSynchronize(s));
    memcpy(sigma_host, h + fb_al + gb_al, gb);
    memcpy(df_host, h + fb_al + 2 * gb_al, fb);
    return FK_OK;
}

int fk_table_last_launches(const fk_table* t) { return t ? t->last_launches : 0; }

}  // extern "C"

#include "fk_group.inl"
