/*
 * fkconv.h -- C-ABI boundary of the B200-native Fast-Kernel (FK) table convolution.
 *
 * What the library computes (P:NN = /root/reference/PAPER.md line NN):
 *
 *   hadronic   sigma[n][r] = sum_{c,i,j} f[r][a_c][i] * f[r][b_c][j] * FK[n][i][j][c]        Eq. (1)
 *              over a sparse list of C active ordered flavour pairs (a_c, b_c)  ("49 flavour
 *              combinations"); f = PDF values on the x-grid; R replicas = R columns of
 *              the "PDF matrix" (Table 3).
 *   DIS        sigma[n][r] = sum_{c,i} f[r][flav_c][i] * FK[n][i][c]      (DIS rows of Table 1, P:51-56;
 *              formula from BASELINE.json north_star, reading R1)
 *   gradient   "the convolution and its corresponding gradient", as a vector-Jacobian product:
 *              df[r][alpha][i] = d( sum_n g[n][r] * sigma[n][r] ) / d f[r][alpha][i]          (reading R8)
 *
 * The luminosity L[k][r] = f[r][a_c][i] * f[r][b_c][j] is built on the fly inside the kernels and is
 * never written to HBM.  Every result is bitwise reproducible run to run (fixed reduction trees, no
 * floating-point atomics).
 *
 * Conventions
 *  - plain C, no exceptions cross the boundary; every call returns an fk_status (0 = FK_OK) and
 *    fk_last_error_string() gives the detail for the calling thread.
 *  - "dev" pointers are CUDA device pointers owned by the caller (8-byte aligned; 16-byte aligned
 *    rows are streamed with 128-bit loads, anything else takes the 64-bit path); "host" pointers are
 *    ordinary host memory, read before the call returns.  Index lists are tiny and live on the host.
 *  - outputs are overwritten, never accumulated into.
 *  - every compute call is asynchronous on `stream` (a cudaStream_t passed as void*, NULL = the
 *    legacy default stream) and never synchronises the device; the *_host variants copy through
 *    pinned staging owned by the table and DO wait for the result before returning.
 *  - a handle (fk_table, fk_group) owns ONE scratch buffer, so the calls on it are serialised: host threads
 *    queue on the handle's mutex, and a call that arrives on a different stream than the previous call on the
 *    same handle first makes its stream wait (cudaStreamWaitEvent) for that call's last kernel.  Different handles
 *    are independent.  Inside a CUDA-graph stream capture a handle must be used from one stream only, and its
 *    scratch cannot grow: give R_hint at create (or make one call outside the capture); otherwise the call returns
 *    FK_ERR_UNSUPPORTED.  A handle belongs to the device that was current at create; a call made with another
 *    current device returns FK_ERR_INVALID_ARG.
 *  - logical layouts (BASELINE.json): hadronic FK[N][nx][nx][C] (i, j, channel; channel innermost),
 *    DIS FK[N][nx][nA], pairs[C][2] = (a_c, b_c) with i <-> a_c and j <-> b_c, flav[nA],
 *    f[R][nfl][nx], sigma[N][R], g[N][R], df[R][nfl][nx].
 *  - limits: 1 <= nfl <= 256, 1 <= C (or nA) <= 1024, K = C*nx*nx (DIS: nA*nx) < 2^31, nfl*nx < 2^31,
 *    N*K < 2^62, R >= 1.  Outside: FK_ERR_UNSUPPORTED.
 *  - there is no CPU fallback: without a CUDA device every compute call returns FK_ERR_CUDA.
 */
#ifndef FKCONV_H
#define FKCONV_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum fk_status {
    FK_OK = 0,
    FK_ERR_INVALID_ARG = -1, /* null pointer, non-positive size, flavour index out of [0,nfl) */
    FK_ERR_ALLOC = -2,       /* device or host allocation failed */
    FK_ERR_CUDA = -3,        /* a CUDA runtime call or kernel launch failed */
    FK_ERR_UNSUPPORTED = -4  /* sizes outside the limits above */
} fk_status;

enum { FK_KIND_DIS = 0, FK_KIND_HADRONIC = 1 };
/* FK_F64: fp64 table, buffers and arithmetic.  FK_F32: table, buffers and arithmetic in fp32 (reading R18; 1e-5).
 * FK_F32S64: the TABLE is demoted to fp32 with round-to-nearest (half the HBM bytes of the bandwidth-bound path),
 * f, g, sigma, df and all arithmetic stay fp64 (error <= 2^-24 of sum|terms|: tolerance 1e-7). */
enum { FK_F64 = 0, FK_F32 = 1, FK_F32S64 = 2 };
/* table storage: BORROW keeps the caller's logical-layout buffer (no copy; it must outlive the
 * table); PACK copies into the library's device layout: channel-major, x innermost
 * ([N][C][nx*nx rounded up to 4, zero padded] resp. [N][nA][nx]), each datapoint row padded to a
 * multiple of 16 bytes, so every channel block and every row starts on a 32- resp. 16-byte boundary
 * (FK_F32 hadronic tables also pad every x-row to 16 bytes: the TMA boxes of the tcgen05 path).
 * SPARSE (FK_F64 only) stores only the NONZERO entries, in the same k-order: per datapoint and per
 * block of 512 k a 64-byte bit mask, a 16-byte header and the packed values -- 8 bytes per nonzero + 0.16 bytes per
 * element (72 % of the dense bytes at config 1's 30 % zeros).  fk_table_conv / _vjp / _conv_vjp / _fit_step and the
 * _host calls take it (column kernels, <= 4 replicas per pass over the table); the grouped launch does not.
 * fk_table_info's device_bytes reports the bytes as stored. */
enum { FK_STORE_BORROW = 0, FK_STORE_PACK = 1, FK_STORE_SPARSE = 2 };

typedef struct fk_table fk_table; /* opaque: one FK table resident in HBM + its scratch */
typedef struct fk_group fk_group; /* opaque: a ragged set of tables with a static work list */

/* Thread-local description of the last failure of this thread ("" if none). Never NULL. */
const char* fk_last_error_string(void);
/* Library version, and the compute capability it was compiled for (100 = sm_100a). */
int fk_version(void);
int fk_compiled_arch(void);

/* Process-wide path-selection options (defaults in brackets).  They are read when a table / group is created and
 * when a compute call picks its kernels: set them before creating handles.  A different option set means a
 * different (still fixed) reduction plan: results are bitwise repeatable per option set.  Nothing is ever read
 * from the environment. */
enum {
    FK_OPT_GEMM_MIN_R = 0, /* [0] smallest R that takes the dense fp64 contraction; 0 = built-in (5 on packed hadronic tables, else 13) */
    FK_OPT_WARP_SPEC = 1,  /* [1] warp-specialised bulk-copy DMMA kernels (0: generic cp.async kernels) */
    FK_OPT_FOLD = 2,       /* [1] R >> 1 VJP stage 2 as one streaming pass over the column sums (0: gather form) */
    FK_OPT_FOLDK = 3,      /* [1] small-R VJP stage 2 as one pass (0: gather form) */
    FK_OPT_FUSED = 4,      /* [1] fk_table_conv_vjp / fk_conv_grouped_conv_vjp read FK once (0: two passes) */
    FK_OPT_FEWROWS = 5,    /* [1] k-walking forward kernel for <= 8 datapoints and very long rows */
    FK_OPT_TC32 = 6,       /* [1] tcgen05 (3xTF32) dense contraction for FK_F32 tables at large R (0: column passes) */
    FK_OPT_TC32_MIN_R = 7, /* [0] smallest R that takes it; 0 = built-in */
    FK_OPT_PDL = 8,        /* [1] later kernels of a call use programmatic dependent launch (0: plain stream order) */
    FK_OPT_FUSE_L2 = 9,    /* [1] resident tables / groups whose forward grid is at most one wave: the forward kernel's last CTA per datapoint range runs the level-2 reduction (0: always a separate launch) */
    FK_OPT_DIS_DIRECT = 10, /* [80] smallest R (>= 13) at which small packed DIS tables (K <= 512, nx even, <= 64 MB) run in one launch without a transposed copy of f or split-K partials; 0: never (the general R >> 1 path) */
    FK_OPT_COUNT_ = 11
};
int fk_set_option(int option, int value);
int fk_get_option(int option, int* value);

/* Kernel timing hook for bench.py's roofline: while enabled, every kernel launch of every
 * compute call is bracketed by a CUDA event pair on the caller's stream, keyed by a short kernel name.
 * The pairs serialise neighbouring launches (programmatic dependent launch cannot overlap across an event
 * record), so a profiled step is slightly slower than an unprofiled one: leave it off outside measurements.
 * fk_profile_report waits for the recorded events, writes one line per kernel name
 *     "<name>\t<launches>\t<total milliseconds>\n"
 * into `buf` (host memory, `capacity` bytes including the terminating 0; FK_ERR_INVALID_ARG if too small)
 * and clears the records.  fk_profile_read does the same but returns only the record with the largest
 * total time: its mean duration in milliseconds and its launch count. */
int fk_profile_enable(int on);
int fk_profile_read(double* mean_kernel_ms, int* launches);
int fk_profile_report(char* buf, int capacity);

/* Latency floors for the microsecond-scale workloads (SURVEY 8(d), L2 caveat): kind 0 launches an empty kernel; kind 1
 * a kernel that reads `bytes` bytes of `buf` (dev, 16-byte aligned) once with 128-bit streaming loads and keeps nothing
 * (`sink`: dev, one double, never written for finite data).  Asynchronous on `stream`; the caller times them. */
int fk_probe_launch(int kind, const void* buf, long long bytes, double* sink, void* stream);

/* ------------------------------------------------------------------ stateless entry points (fp64)
 * Eq. (1) P:43 / DIS / VJP on the caller's logical-layout device buffers.  Level-1 partials live in
 * stream-ordered scratch (cudaMallocAsync on `stream`).
 *   fk     dev   [N][nx][nx][C]  (DIS: [N][nx][nA])
 *   pairs  host  [C][2] int32    (DIS: flav host [nA] int32)
 *   f      dev   [R][nfl][nx]
 *   sigma  dev   [N][R]          (written)
 *   g      dev   [N][R]
 *   df     dev   [R][nfl][nx]    (written; exactly 0 for flavours in no pair)
 */
int fk_conv_dis(const double* fk, const int32_t* flav, const double* f, double* sigma,
                int N, int nx, int nfl, int nA, int R, void* stream);
int fk_conv_hadronic(const double* fk, const int32_t* pairs, const double* f, double* sigma,
                     int N, int nx, int nfl, int C, int R, void* stream);
int fk_conv_hadronic_vjp(const double* fk, const int32_t* pairs, const double* f, const double* g,
                         double* df, int N, int nx, int nfl, int C, int R, void* stream);
int fk_conv_dis_vjp(const double* fk, const int32_t* flav, const double* f, const double* g,
                    double* df, int N, int nx, int nfl, int nA, int R, void* stream);

/* ------------------------------------------------------------------ allocation-free forward (fp64)
 * fk_conv_hadronic (Eq. (1); same arguments, layout and results) for callers that cannot allocate device
 * memory: code under CUDA-graph capture, tight serving loops, harnesses that forbid cudaMalloc.  The level-1 partials
 * (and, for R >= 5, the replica-innermost copy of f, the split-K partials and the k -> PDF-slot codes of the dense
 * contraction) live in ONE file-scope `static __device__` array of FK_STATIC_SCRATCH_BYTES bytes inside the library:
 * every GPU that loads the library holds that array until the process exits.  The call makes no cudaMalloc /
 * cudaMallocAsync / cudaFree and calls no allocating library routine; on its first call per device it looks the array's
 * device address up (cudaGetSymbolAddress, with that device current).
 *   - sizes whose scratch exceeds the array: FK_ERR_UNSUPPORTED, nothing launched; fk_last_error_string() names the
 *     bytes needed and the limit.  The need is 8 * N * ceil(nx*nx*C / 512) * R bytes for R <= 12 (k-blocks of 512;
 *     nothing when nx*nx*C <= 512); from R = 13 on (the dense contraction) about 8 * R16 * (nfl*nx + N * ksplit) +
 *     4 * nx*nx*C with R16 = min(128, R rounded up to 16) and ksplit ~ SMs / ceil(N / 128).  Config 2 (N = 512,
 *     nx = 50, C = 100: 2 MB per replica, 21 MB at R >= 128) fits for every R, and so does every table of config 4.
 *   - every call on a device SHARES the array, which keeps the previous call's contents: the call clears the part that
 *     must start at zero (the tickets of the in-kernel level-2 reduction) on `stream` itself; everything else is written
 *     before it is read.  Two calls that overlap on the GPU (different streams, or different host threads on one device)
 *     RACE on the array and give wrong results silently: serialise them (one stream, or an event between them).
 *   - asynchronous on `stream`, no synchronisation; same error conventions as fk_conv_hadronic. */
#define FK_STATIC_SCRATCH_BYTES (32u << 20)
int fk_conv_hadronic_static(const double* fk, const int32_t* pairs, const double* f, double* sigma,
                            int N, int nx, int nfl, int C, int R, void* stream);

/* fp32 variant (reading R18): float storage and float FMA with short chains, the
 * cross-thread stages in double, float results.  Same argument meaning as above. */
int fk_conv_dis_f32(const float* fk, const int32_t* flav, const float* f, float* sigma,
                    int N, int nx, int nfl, int nA, int R, void* stream);
int fk_conv_hadronic_f32(const float* fk, const int32_t* pairs, const float* f, float* sigma,
                         int N, int nx, int nfl, int C, int R, void* stream);
int fk_conv_hadronic_vjp_f32(const float* fk, const int32_t* pairs, const float* f, const float* g,
                             float* df, int N, int nx, int nfl, int C, int R, void* stream);

/* ------------------------------------------------------------------ two-PDF (p pbar) form
 * Eq. (1), with distinct PDFs on the two legs:
 *     sigma[n][r] = sum_{c,i,j} f1[r][a_c][i] * f2[r][b_c][j] * FK[n][i][j][c]
 * f1, f2  dev  [R][nfl][nx]  (f1 = first hadron, index i; f2 = second hadron, index j; reading R3)
 * VJP: df1[r][alpha][i] = d(sum_n g sigma)/d f1[r][alpha][i], df2 likewise: two outputs, both overwritten.
 * Runs on the single-PDF kernels over the stacked grid (f1 ; f2) with pairs (a_c, nfl + b_c): 2*nfl <= 256.
 * fp64, logical-layout table, asynchronous on `stream`; same error conventions as fk_conv_hadronic. */
int fk_conv_hadronic2(const double* fk, const int32_t* pairs, const double* f1, const double* f2, double* sigma,
                      int N, int nx, int nfl, int C, int R, void* stream);
int fk_conv_hadronic2_vjp(const double* fk, const int32_t* pairs, const double* f1, const double* f2, const double* g,
                          double* df1, double* df2, int N, int nx, int nfl, int C, int R, void* stream);

/* ------------------------------------------------------------------ resident-table path
 * What a fit uses: thousands of iterations over fixed tables, tables loaded once.
 * fk_table_create validates the index list, (store==PACK) repacks and (dtype==FK_F32) demotes the
 * logical fp64 table `fk_logical` (dev) with round-to-nearest, and pre-allocates scratch for up to
 * `R_hint` replicas (grown on demand by later calls, which then allocate once, outside any graph).
 * kind: FK_KIND_*; C = number of pairs (hadronic) or active flavours (DIS).
 * fk_table_create synchronises `stream` work it issues before returning (one-time, untimed). */
int fk_table_create(fk_table** out, int kind, const double* fk_logical, const int32_t* index_list,
                    int N, int nx, int nfl, int C, int dtype, int store, int R_hint);
int fk_table_destroy(fk_table* t);
/* N, nx, nfl, C, K (= C*nx*nx or nA*nx), row stride in elements, device bytes held by the table. */
int fk_table_info(const fk_table* t, int* N, int* nx, int* nfl, int* C, int64_t* K,
                  int64_t* row_stride, int64_t* device_bytes);
/* f, sigma, g, df: dev; float for FK_F32 tables, double for FK_F64 and FK_F32S64. */
int fk_table_conv(fk_table* t, const void* f, void* sigma, int R, void* stream);
int fk_table_vjp(fk_table* t, const void* f, const void* g, void* df, int R, void* stream);
/* Convolution (Eq. (1)) AND its VJP for an upstream gradient g[N][R] that is known
 * before the forward pass (a loss linear in sigma, e.g. fixed weights w_n): FK is read ONCE for both -- the
 * column kernel accumulates the column sums sum_n g[n][r] FK[n][k] from the registers that hold the row pieces.
 * Results equal fk_table_conv + fk_table_vjp within the tolerance (same level-1 partials; the column sums are
 * cut into the forward's datapoint ranges).  R >= 5 (dense path) and DIS tables run the two passes one after
 * the other.  sigma[N][R], df[R][nfl][nx]: dev, overwritten; asynchronous on `stream`. */
int fk_table_conv_vjp(fk_table* t, const void* f, const void* g, void* sigma, void* df, int R, void* stream);
/* The step that follows the convolution in a fit iteration (reading R22; the paper names the
 * "gradient descent optimization", but never prints the loss): with d[n][r] = sigma[n][r] - data[n],
 *     chi2[r] = sum_{n,m} d[n][r] cinv[n][m] d[m][r],      g[n][r] = 2 sum_m cinv[n][m] d[m][r]
 * sigma[N][R], data[N], cinv[N][N] (symmetric, row-major): dev, read; chi2[R], g[N][R]: dev, overwritten.  fp64. */
int fk_chi2(const double* sigma, const double* data, const double* cinv, double* chi2, double* g, int N, int R,
            void* stream);
/* One fit iteration on a resident table, all on `stream`: sigma = conv(f); (chi2, g) = fk_chi2(sigma); df = vjp(f, g).
 * Equal, bit for bit, to the three calls made one after the other.  fp64 tables only. */
int fk_table_fit_step(fk_table* t, const double* f, const double* data, const double* cinv, double* sigma, double* g,
                      double* chi2, double* df, int R, void* stream);
/* Same with HOST buffers: H2D of f (and g) and D2H of the result run inside the call, through
 * pinned staging, on `stream`; the call returns after the result has landed in host memory. */
int fk_table_conv_host(fk_table* t, const void* f_host, void* sigma_host, int R, void* stream);
int fk_table_vjp_host(fk_table* t, const void* f_host, const void* g_host, void* df_host, int R,
                      void* stream);
/* fk_table_conv_vjp with HOST buffers: f and g go up in ONE copy, sigma and df come back in ONE copy, one wait; the call
 * returns after both results have landed in host memory.  Same dispatch as fk_table_conv_vjp (forward + VJP from one read
 * of FK when that path applies; FK_OPT_FUSED = 0 makes it the two passes). */
int fk_table_conv_vjp_host(fk_table* t, const void* f_host, const void* g_host, void* sigma_host, void* df_host, int R,
                           void* stream);
/* Kernel launches issued by the last conv / vjp call on this table (for bench.py's gpu_launches). */
int fk_table_last_launches(const fk_table* t);

/* ------------------------------------------------------------------ grouped ragged launch
 * A global fit convolves many tables of different (N, nx, C) every iteration.
 * fk_group_create builds a static work list over the T tables (all of one dtype); each forward or
 * VJP pass is then ONE persistent launch per stage over all tables.
 *   f_cat      dev  concatenation over t of f_t[R][nfl_t][nx_t]   (offsets: fk_group_offsets)
 *   sigma_cat  dev  concatenation over t of sigma_t[N_t][R]
 *   g_cat      dev  concatenation over t of g_t[N_t][R]
 *   df_cat     dev  concatenation over t of df_t[R][nfl_t][nx_t]  (per table, reading R14)
 * The tables must outlive the group. */
int fk_group_create(fk_group** out, fk_table* const* tables, int T, int R_hint);
int fk_group_destroy(fk_group* g);
/* element offsets (for R replicas) of table t inside f_cat/df_cat and sigma_cat/g_cat; arrays of
 * T+1 int64 written to host memory (entry T = total length). */
int fk_group_offsets(const fk_group* g, int R, int64_t* f_offsets, int64_t* sigma_offsets);
int fk_conv_grouped(fk_group* g, const void* f_cat, void* sigma_cat, int R, void* stream);
int fk_conv_grouped_vjp(fk_group* g, const void* f_cat, const void* g_cat, void* df_cat, int R,
                        void* stream);
/* Forward AND VJP of the whole group from ONE read of every table, for a `g_cat` that is known before the forward
 * pass (a loss linear in sigma: BASELINE config 4's seeded weights; the fit evaluates the
 * convolution "and its corresponding gradient" every iteration).  Same results as fk_conv_grouped
 * followed by fk_conv_grouped_vjp (sigma bit for bit; df within rounding: the column sums are cut into the
 * forward's datapoint ranges).  One read applies for R <= 4 on groups of hadronic tables with nx <= 128; otherwise
 * the call runs the two passes. */
int fk_conv_grouped_conv_vjp(fk_group* g, const void* f_cat, const void* g_cat, void* sigma_cat, void* df_cat,
                             int R, void* stream);
int fk_group_last_launches(const fk_group* g);

#ifdef __cplusplus
}
#endif
#endif /* FKCONV_H */
