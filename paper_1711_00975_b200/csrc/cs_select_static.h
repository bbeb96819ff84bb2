/*
 * cs_select_static.h -- the allocation-free selection call (cs_select_static, include/cs.h): declaration shared by
 * cs_select.cu (which owns the file-scope device scratch and the kernels) and cs_api.cu (the C entry point).
 */
#ifndef CS_SELECT_STATIC_H_
#define CS_SELECT_STATIC_H_

#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/cs.h"

namespace cs {

constexpr uint32_t SELECT_STATIC_MAX_N = CS_SELECT_STATIC_MAX_N;

/* Enqueues on `stream` (current device): load -> one compaction (k_compact) -> emit of the first min(k, unique) entries.
 * No allocation, no synchronisation.  n <= SELECT_STATIC_MAX_N is the caller's to check. */
cudaError_t select_static(const uint64_t* ids, const int32_t* est, uint32_t n, uint32_t k, uint64_t* ids_out, int32_t* est_out,
                          uint32_t* n_out, cudaStream_t stream);

}  // namespace cs
#endif
