/*
 * cs_scan_common.cuh -- device helpers shared by the estimate-side kernels (cs_scan.cu, cs_scan_staged.cu):
 * row value s_j(c)*T[j][h_j(c)], estimate with early exit against tau ("median > theta"),
 * warp-aggregated candidate append, dispatch on the row count.
 */
#ifndef CS_SCAN_COMMON_CUH_
#define CS_SCAN_COMMON_CUH_

#include "cs_device.cuh"
#include "cs_launch.cuh"

namespace cs {

__device__ __forceinline__ int32_t ld_table(const int32_t* p) {
    int32_t v;
    asm volatile("ld.global.relaxed.gpu.s32 %0, [%1];" : "=r"(v) : "l"(p));   // L2 is the point of coherence
    return v;
}

/* s_j(c) * T[j][h_j(c)] for row j of scale s */
template <bool BIG, bool POW2>
__device__ __forceinline__ int32_t row_value(const PassParams& P, const int32_t* T, const RowCoef& rc, int j,
                                             uint32_t c0, uint32_t c1) {
    uint32_t b;
    int32_t sg;
    bucket_sign<BIG, POW2>(rc, c0, c1, P.w, b, sg);
    return mul_sign(ld_table(T + (uint64_t)j * P.w + b), sg);
}

/* Estimate with early exit.  Returns true iff Estimate(c) >= tau; then est holds the estimate. */
template <int D, bool POW2, bool BIG>
__device__ __forceinline__ bool estimate_ge(const PassParams& P, int s, uint64_t c, int32_t tau, int32_t& est) {
    const int d = D ? D : P.d;
    const int max_fail = P.rank;                 // est >= tau  <=>  at most rank row values are < tau (rank = (d-1)/2)
    const uint32_t c0 = cell_c0(c), c1 = cell_c1(c);
    const int32_t* T = P.sc[s].T;
    const RowCoef* rows = &P.rows[s * d];
    int32_t v[D ? D : CS_MAX_ROWS];
    int fail = 0;
#pragma unroll
    for (int j = 0; j < d; ++j) {
        if (fail <= max_fail) {
            v[j] = row_value<BIG, POW2>(P, T, rows[j], j, c0, c1);
            fail += (v[j] < tau);
        }
    }
    if (fail > max_fail) return false;
    if constexpr (D > 0) est = select_of<D>(v, P.rank);
    else                 est = select_rt(v, d, P.rank);
    return true;
}

template <int D, bool POW2, bool BIG>
__device__ __forceinline__ int32_t estimate_full(const PassParams& P, int s, uint64_t c) {
    int32_t est = 0;
    estimate_ge<D, POW2, BIG>(P, s, c, INT32_MIN, est);
    return est;
}

/* Duplicate filter of the re-scan.  The same cell arrives once per particle it holds (tens of times for the heavy cells
 * of a coarse mesh), always with the same estimate: only its first arrival needs the exact estimate and a list entry.
 * The set holds every cell that reached this point since cs_scan_begin -- appended or found below tau, which only rises.
 * Returns true for the first arrival.  A crowded table (more than 32 probes) answers true: a duplicate entry is
 * harmless, the selector removes it.  The host clears the set before it re-runs a chunk whose entries were dropped. */
static __device__ __noinline__ bool seen_first_time(const ScanTarget& tg, uint64_t c) {
    if (tg.seen_mask == 0 || c == ~0ull) return true;
    uint32_t s = (uint32_t)(mix64(c) >> 24) & tg.seen_mask;
    for (int probe = 0; probe < 32; ++probe) {
        const unsigned long long old = atomicCAS(tg.seen + s, ~0ull, (unsigned long long)c);
        if (old == ~0ull) return true;
        if (old == c) return false;
        s = (s + 1) & tg.seen_mask;
    }
    return true;
}

/* Warp-aggregated append of (c, est) to the candidate list of one scale.  Must be reached by all 32 lanes.
 * One global atomic per warp that has something to append; the estimate range of the list (which bounds the radix
 * passes of the selector) is computed when the list is compacted (k_est_range), not here: three atomics per append on
 * the one sector that holds the ScanState serialise at the L2 when many cells qualify (cfg 5: 3e5 appends per launch). */
__device__ __forceinline__ void append_candidate(const ScanTarget& tg, bool emit, uint64_t c, int32_t est) {
    const uint32_t mask = __ballot_sync(0xFFFFFFFFu, emit);
    if (mask == 0) return;
    const uint32_t lane = threadIdx.x & 31u;
    const int leader = __ffs(mask) - 1;
    uint32_t base = 0;
    if ((int)lane == leader) base = atomicAdd(&tg.st->count, (uint32_t)__popc(mask));
    base = __shfl_sync(0xFFFFFFFFu, base, leader);
    if (emit) {
        uint64_t pos = (uint64_t)base + __popc(mask & ((1u << lane) - 1u));
        if (pos < tg.cap) {
            tg.id[pos] = c;
            tg.ek[pos] = est_to_key(est);
        }
    }
}

/* Estimate of an arbitrary caller-supplied 64-bit cell id (any value: ids >= 2^60 take the __umul64hi form). */
template <int D, bool POW2>
__device__ __forceinline__ int32_t estimate_any(const PassParams& P, int s, uint64_t c) {
    if ((c >> 31) == 0) return estimate_full<D, POW2, false>(P, s, c);
    if ((c >> 60) == 0) return estimate_full<D, POW2, true>(P, s, c);
    const int d = D ? D : P.d;
    int32_t v[CS_MAX_ROWS];
    for (int j = 0; j < d; ++j) {
        const RowCoef& rc = P.rows[s * d + j];
        uint64_t r = affine_mod_p_wide(coef_a(rc.h), coef_b(rc.h), c);
        uint64_t r2 = affine_mod_p_wide(coef_a(rc.s), coef_b(rc.s), c);
        uint32_t b = POW2 ? ((uint32_t)r & (uint32_t)(P.w - 1)) : (uint32_t)(r % P.w);
        v[j] = mul_sign(ld_table(P.sc[s].T + (uint64_t)j * P.w + b), 1 - 2 * (int32_t)((uint32_t)r2 & 1u));
    }
    return select_rt(v, d, P.rank);
}

/* ---- helpers of the bitmap prefilters (cs_scan_bitmap.cu, cs_scan_staged.cu) --------------------------------- */

__device__ __forceinline__ uint32_t ld_bits(const uint32_t* p) {
    uint32_t v;
    asm volatile("ld.global.relaxed.gpu.u32 %0, [%1];" : "=r"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ uint32_t lds_u32s(uint32_t addr) {
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr));
    return v;
}

/* bucket hash of row rc (w a power of two); BIG: cell ids of this mesh can exceed 2^31 */
template <bool BIG>
__device__ __forceinline__ uint32_t bucket_of(const RowCoef& rc, uint32_t c0, uint32_t c1, uint32_t wmask) {
    return affine_low32<BIG>(rc.h, c0, c1) & wmask;
}

#define CS_DISPATCH_D(CALL)                                    \
    switch (P.d) {                                             \
        case 1: CALL(1); break;  case 2: CALL(2); break;       \
        case 3: CALL(3); break;  case 4: CALL(4); break;       \
        case 5: CALL(5); break;  case 6: CALL(6); break;       \
        case 7: CALL(7); break;  case 8: CALL(8); break;       \
        default: CALL(0); break;                               \
    }

static inline int blocks_1d(uint64_t m) {
    uint64_t b = (m + PASS_THREADS - 1) / PASS_THREADS;
    if (b > 148 * 8) b = 148 * 8;
    return (int)(b < 1 ? 1 : b);
}

}  // namespace cs
#endif
