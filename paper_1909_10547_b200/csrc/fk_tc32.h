// fk_tc32.h -- host interface of the tcgen05 dense contraction for fp32 tables (fk_tc32.cu); internal, not part of the
// C-ABI.  The fp32 variant of the R >> 1 convolution (BASELINE.json config 3, "the dense contraction case where tensor
// cores may apply") runs on the 5th-generation tensor cores as a 3xTF32 split.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "fk_common.cuh"

namespace fk {

constexpr int TC_BN = 128;        // datapoints per CTA tile = UMMA N (partial tiles: rounded up to 16)
constexpr int TC_MAX_RP = 128;    // replicas per pass = UMMA M (the lanes of TMEM)
constexpr int TC_MAX_NX = 64;     // x-grid points: one (c, i) row of the table is one MMA K extent of <= 64
constexpr int TC_MAX_TILES = 2048; // (c, i) rows per item: bounds the second-level fp32 chain of the epilogue (channels of an item)
constexpr int TC_TMAP_BYTES = 128;  // sizeof(CUtensorMap)

// padded replica count of a pass: a multiple of 4 (128-bit rows of fT / gpart), at most TC_MAX_RP
inline int tc_rp(int r) {
    const int rp = (r + 3) / 4 * 4;
    return rp < TC_MAX_RP ? rp : TC_MAX_RP;
}

struct Tc32Params {
    TableDesc desc;          // single-table launch
    ChannelList chan;        // single-table launch
    const void* tmap;        // single-table launch: device copy of the table's CUtensorMap (grouped: desc.tmap)
    const float* fT;         // [nfl*nx][RP] replica-innermost fp32 copy of f (grouped: + desc.f_off * RP)
    float* gpart;            // [ksplit][N][RP] level-1 partials (grouped: + desc.tc_gp_off * RP)
    int RP;                  // padded replicas of this pass
    int ksplit, tper;        // single-table launch: ranges of (c, i) rows and their length
    const TableDesc* descs;  // grouped launch
    const ColSeg* items;     // grouped launch {table, kblock = first datapoint, split = range of (c, i) rows}
};

// dynamic shared memory of a launch
size_t tc32_smem_bytes();
inline int tc32_ntiles(int N) { return (N + TC_BN - 1) / TC_BN; }
// Writes the 128-byte tensor map of a packed fp32 table [N][row_stride] (box 32 k x 128 rows, 128-byte swizzle,
// zero fill outside the table) to `out_host`.  false: the driver entry point is missing or refused the arguments.
bool tc32_encode_tensor_map(void* out_host, const void* fk_dev, long long row_stride, int K, int N);
// Launches the contraction; grid = datapoint tiles x ranges (single) or items (grouped); pdl: as a programmatic
// dependent launch behind the transpose kernel (the kernel waits for fT itself, fk_common.cuh pdl_wait).
cudaError_t tc32_fwd_launch(const Tc32Params& p, int grid, bool grouped, bool pdl, cudaStream_t s);

}  // namespace fk
