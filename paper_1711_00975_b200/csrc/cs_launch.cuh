/*
 * cs_launch.cuh -- host-side launch helpers shared by the particle-pass translation units.
 */
#ifndef CS_LAUNCH_CUH_
#define CS_LAUNCH_CUH_

#include "cs_device.cuh"

namespace cs {

/* Split n particles at xyz into (head, groups of 4, tail) so that the grouped part is 16-byte aligned. */
static inline void split_aligned(const float* xyz, uint64_t n, uint32_t* head, uint64_t* groups) {
    /* xyz is 4-byte aligned (checked by the API), so one of the first four particles starts on a 16-byte line */
    uint32_t h = 0;
    uintptr_t a = reinterpret_cast<uintptr_t>(xyz);
    while (h < 3 && ((a + 12ull * h) & 15u)) ++h;
    if (h > n) h = (uint32_t)n;
    *head = h;
    *groups = (n - h) / 4;
}

template <typename K>
static int blocks_for(K kernel, int sm_count, uint64_t work_items) {
    int per_sm = 0;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, PASS_THREADS, 0);
    if (per_sm < 1) per_sm = 1;
    uint64_t need = (work_items + PASS_THREADS - 1) / PASS_THREADS;
    uint64_t full = (uint64_t)sm_count * per_sm;
    uint64_t b = need < full ? need : full;
    return (int)(b < 1 ? 1 : b);
}

}  // namespace cs
#endif
