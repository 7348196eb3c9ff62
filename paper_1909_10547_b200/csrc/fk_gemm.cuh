// fk_gemm.cuh -- R >> 1 dense contraction -- placeholder until the FP64 split-K
// kernel lands: gemm_wanted() is false, so every R runs through replica tiles of the stream kernel.
#pragma once

#include "fk_common.cuh"

namespace fk {

inline bool gemm_wanted(int) { return false; }
inline int gemm_pick_split(const TableDesc&, int, int) { return 1; }
inline size_t gemm_forward_scratch_elems(const TableDesc&, int, int) { return 0; }

template <typename T>
int gemm_forward_single(const TableDesc&, const ChannelList&, const T*, T*, int, double*, int, cudaStream_t, int*) {
    return (int)cudaErrorNotSupported;
}
template <typename T>
int gemm_colsum_single(const TableDesc&, const T*, double*, int, cudaStream_t, int*) {
    return (int)cudaErrorNotSupported;
}

}  // namespace fk
