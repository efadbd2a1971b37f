// Thread-per-cell colour-pass kernel for BCC / 2 shells / w = 4 / <= 4 species on 2-bit packed
// storage.  (Placeholder until the generic path is validated: reports "not supported".)
#pragma once
#include "smcx_common.cuh"

namespace smcxk {

inline bool thread_kernel_supported(const Geom&) { return false; }
inline int configure_thread_per_cell() { return 0; }
inline int launch_thread_per_cell(const Geom&, uint32_t*, const int32_t*, const uint32_t*, DevState*, int,
                                  cudaStream_t) { return -1; }

}  // namespace smcxk
