// fk_tc32.h -- host interface of the tcgen05 dense contraction for fp32 tables (fk_tc32.cu); internal, not part of the
// C-ABI.  The fp32 variant of the R >> 1 convolution (BASELINE.json config 3, "the dense contraction case where tensor
// cores may apply") runs on the 5th-generation tensor cores as a 3xTF32 split.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "fk_common.cuh"

namespace fk {

constexpr int TC_BM = 128;        // datapoints per CTA tile = UMMA M
constexpr int TC_KT = 32;         // k per pipeline stage = one 128-byte swizzle row of fp32
constexpr int TC_MAX_RP = 128;    // padded replicas per pass = UMMA N of the (FK_lo, L_hi) product; the stacked product takes 2 RP
constexpr int TC_FLUSH = 8;       // stages between drains of the TMEM accumulator (chain <= 32 accumulations of 8 k)
constexpr int TC_TMAP_BYTES = 128;  // sizeof(CUtensorMap)

// padded replica count of a pass: a multiple of 16, at most TC_MAX_RP
inline int tc_rp(int r) {
    const int rp = (r + 15) / 16 * 16;
    return rp < TC_MAX_RP ? rp : TC_MAX_RP;
}

struct Tc32Params {
    TableDesc desc;          // single-table launch
    ChannelList chan;        // single-table launch
    const void* tmap;        // single-table launch: device copy of the table's CUtensorMap (grouped: desc.tmap)
    const float* fT;         // [nfl*nx][RP] replica-innermost fp32 copy of f (grouped: + desc.f_off * RP)
    float* gpart;            // [ksplit][N][RP] level-1 partials (grouped: + desc.gp_off * RP)
    int RP;                  // padded replicas of this pass (multiple of 16, <= 128)
    int ksplit, kper;        // single-table launch: K ranges and their length (a multiple of TC_KT)
    int fk_stages;           // TMA ring depth (3 or 4)
    const TableDesc* descs;  // grouped launch
    const ColSeg* items;     // grouped launch {table, kblock = first datapoint, split = K range}
};

// dynamic shared memory of a launch (0: does not fit, take another path)
size_t tc32_smem_bytes(int nx, int RP, int* fk_stages);
// tile / item counts
inline int tc32_mtiles(int N) { return (N + TC_BM - 1) / TC_BM; }
// Writes the 128-byte tensor map of a packed fp32 table [N][row_stride] (box 32 k x 128 rows, 128-byte swizzle,
// zero fill outside the table) to `out_host`.  false: the driver entry point is missing or refused the arguments.
bool tc32_encode_tensor_map(void* out_host, const void* fk_dev, long long row_stride, int K, int N);
// Launches the contraction; grid = datapoint tiles x K ranges (single) or items (grouped).
cudaError_t tc32_fwd_launch(const Tc32Params& p, int grid, bool grouped, size_t smem, cudaStream_t s);

}  // namespace fk
