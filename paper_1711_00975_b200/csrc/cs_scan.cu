/*
 * cs_scan.cu -- estimate-side particle passes of libcs.so (sm_100a):
 *   k_estimate    one thread per cell id: 2d hashes, d gathers, median of d
 *   k_scan        candidate re-scan: every kept particle of the replayed stream is estimated against the
 *                 finished tables; a cell is appended to the candidate list iff its estimate >= tau.  The
 *                 median test exits as soon as more than (d-1)/2 rows are below tau (PAPER.md:304-306
 *                 "estimate mode" with a threshold, restricted to occupied cells; R10).
 *   k_scan_cells  the same for explicit cell ids (merging candidate lists of stream shards).
 * The paper's Estimate kernel uses one block per cell with t threads and a shared-memory rank count
 * (Alg. 4 l.4-20); here one thread owns a cell, the d values stay in registers and the median is a
 * compare-exchange network.
 */
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
    const int max_fail = (d - 1) / 2;            // est >= tau  <=>  at most (d-1)/2 row values are < tau
    const uint32_t c0 = (uint32_t)c, c1 = (uint32_t)(c >> 32);
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
    if constexpr (D > 0) est = median_of<D>(v);
    else                 est = median_rt(v, d);
    return true;
}

template <int D, bool POW2, bool BIG>
__device__ __forceinline__ int32_t estimate_full(const PassParams& P, int s, uint64_t c) {
    int32_t est = 0;
    estimate_ge<D, POW2, BIG>(P, s, c, INT32_MIN, est);
    return est;
}

/* Warp-aggregated append of (c, est) to the candidate list of one scale.  Must be reached by all 32 lanes. */
__device__ __forceinline__ void append_candidate(const ScanTarget& tg, bool emit, uint64_t c, int32_t est) {
    const uint32_t mask = __ballot_sync(0xFFFFFFFFu, emit);
    if (mask == 0) return;
    const uint32_t lane = threadIdx.x & 31u;
    const int leader = __ffs(mask) - 1;
    int32_t lo = __reduce_min_sync(0xFFFFFFFFu, emit ? est : INT32_MAX);
    int32_t hi = __reduce_max_sync(0xFFFFFFFFu, emit ? est : INT32_MIN);
    uint32_t base = 0;
    if ((int)lane == leader) {
        base = atomicAdd(&tg.st->count, (uint32_t)__popc(mask));
        atomicMin(&tg.st->est_min, lo);
        atomicMax(&tg.st->est_max, hi);
    }
    base = __shfl_sync(0xFFFFFFFFu, base, leader);
    if (emit) {
        uint64_t pos = (uint64_t)base + __popc(mask & ((1u << lane) - 1u));
        if (pos < tg.cap) {
            tg.id[pos] = c;
            tg.ek[pos] = est_to_key(est);
        }
    }
}

template <int D, bool POW2>
__device__ __forceinline__ void scan_particle(const PassParams& P, const ScanParams& S, const int32_t* tau,
                                              bool keep, float x, float y, float z) {
    for (int s = 0; s < P.n_scales; ++s) {
        uint64_t c = 0;
        int32_t est = 0;
        bool emit = false;
        if (keep) {
            c = cell_of(x, y, z, P.sc[s]);
            emit = P.sc[s].big ? estimate_ge<D, POW2, true>(P, s, c, tau[s], est)
                               : estimate_ge<D, POW2, false>(P, s, c, tau[s], est);
        }
        append_candidate(S.tg[s], emit, c, est);
    }
}

template <int D, bool POW2>
__global__ void __launch_bounds__(PASS_THREADS)
k_scan(const __grid_constant__ PassParams P, const __grid_constant__ ScanParams S,
       const float* __restrict__ xyz, uint64_t n, uint32_t head, uint64_t groups) {
    int32_t tau[CS_MAX_SCALES];
#pragma unroll
    for (int s = 0; s < CS_MAX_SCALES; ++s) tau[s] = s < P.n_scales ? S.tg[s].st->tau : 0;

    const uint64_t stride = (uint64_t)gridDim.x * PASS_THREADS;
    const float4* body = reinterpret_cast<const float4*>(xyz + 3 * (uint64_t)head);
    /* warp-uniform trip count: the loop variable is the group index of lane 0 */
    const uint32_t lane = threadIdx.x & 31u;
    for (uint64_t g0 = (uint64_t)blockIdx.x * PASS_THREADS + (threadIdx.x - lane); g0 < groups; g0 += stride) {
        const uint64_t g = g0 + lane;
        const bool in = g < groups;
        float4 q0 = make_float4(0.f, 0.f, 0.f, 0.f), q1 = q0, q2 = q0;
        if (in) {
            q0 = ld_stream16(body + 3 * g);
            q1 = ld_stream16(body + 3 * g + 1);
            q2 = ld_stream16(body + 3 * g + 2);
        }
        const uint64_t i0 = P.index0 + head + 4 * g;
        bool k0 = in, k1 = in, k2 = in, k3 = in;
        if (P.sample && in) {
            k0 = keep_particle(P.K, i0 + 0, P.Tp);
            k1 = keep_particle(P.K, i0 + 1, P.Tp);
            k2 = keep_particle(P.K, i0 + 2, P.Tp);
            k3 = keep_particle(P.K, i0 + 3, P.Tp);
        }
        scan_particle<D, POW2>(P, S, tau, k0, q0.x, q0.y, q0.z);
        scan_particle<D, POW2>(P, S, tau, k1, q0.w, q1.x, q1.y);
        scan_particle<D, POW2>(P, S, tau, k2, q1.z, q1.w, q2.x);
        scan_particle<D, POW2>(P, S, tau, k3, q2.y, q2.z, q2.w);
    }
    if (blockIdx.x == 0 && threadIdx.x < 32) {        // warp 0: the <= 6 edge particles
        const uint64_t tail0 = (uint64_t)head + 4 * groups;
        const uint64_t n_edge = (uint64_t)head + (n - tail0);
        const bool in = threadIdx.x < n_edge;
        uint64_t i = 0;
        float x = 0.f, y = 0.f, z = 0.f;
        bool keep = false;
        if (in) {
            i = threadIdx.x < head ? threadIdx.x : tail0 + (threadIdx.x - head);
            keep = !P.sample || keep_particle(P.K, P.index0 + i, P.Tp);
            const float* p = xyz + 3 * i;
            x = ld_stream4(p); y = ld_stream4(p + 1); z = ld_stream4(p + 2);
        }
        scan_particle<D, POW2>(P, S, tau, keep, x, y, z);
    }
}

/* Estimate of an arbitrary caller-supplied 64-bit cell id (any value: ids >= 2^60 take the __umul64hi form). */
template <int D, bool POW2>
__device__ __forceinline__ int32_t estimate_any(const PassParams& P, int s, uint64_t c) {
    if ((c >> 32) == 0) return estimate_full<D, POW2, false>(P, s, c);
    if ((c >> 60) == 0) return estimate_full<D, POW2, true>(P, s, c);
    const int d = D ? D : P.d;
    int32_t v[CS_MAX_ROWS];
    for (int j = 0; j < d; ++j) {
        const RowCoef& rc = P.rows[s * d + j];
        uint64_t r = affine_mod_p_wide(coef_a(rc.h), rc.h.b, c);
        uint64_t r2 = affine_mod_p_wide(coef_a(rc.s), rc.s.b, c);
        uint32_t b = POW2 ? ((uint32_t)r & (uint32_t)(P.w - 1)) : (uint32_t)(r % P.w);
        v[j] = mul_sign(ld_table(P.sc[s].T + (uint64_t)j * P.w + b), 1 - 2 * (int32_t)((uint32_t)r2 & 1u));
    }
    return median_rt(v, d);
}

template <int D, bool POW2>
__global__ void __launch_bounds__(PASS_THREADS)
k_estimate(const __grid_constant__ PassParams P, int s, const uint64_t* __restrict__ cells, uint64_t m,
           int32_t* __restrict__ est) {
    const uint64_t stride = (uint64_t)gridDim.x * PASS_THREADS;
    for (uint64_t i = (uint64_t)blockIdx.x * PASS_THREADS + threadIdx.x; i < m; i += stride)
        est[i] = estimate_any<D, POW2>(P, s, cells[i]);
}

template <int D, bool POW2>
__global__ void __launch_bounds__(PASS_THREADS)
k_scan_cells(const __grid_constant__ PassParams P, const __grid_constant__ ScanParams S, int s,
             const uint64_t* __restrict__ cells, uint64_t m) {
    const int32_t tau = S.tg[s].st->tau;
    const uint64_t stride = (uint64_t)gridDim.x * PASS_THREADS;
    const uint32_t lane = threadIdx.x & 31u;
    for (uint64_t i0 = (uint64_t)blockIdx.x * PASS_THREADS + (threadIdx.x - lane); i0 < m; i0 += stride) {
        const uint64_t i = i0 + lane;
        uint64_t c = 0;
        int32_t e = 0;
        bool emit = false;
        if (i < m) {
            c = cells[i];
            e = estimate_any<D, POW2>(P, s, c);
            emit = e >= tau;
        }
        append_candidate(S.tg[s], emit, c, e);
    }
}

/* ---- dispatch on (d, w power of two) ------------------------------------------------------------------ */

#define CS_DISPATCH_D(CALL)                                    \
    switch (P.d) {                                             \
        case 1: CALL(1); break;  case 2: CALL(2); break;       \
        case 3: CALL(3); break;  case 4: CALL(4); break;       \
        case 5: CALL(5); break;  case 6: CALL(6); break;       \
        case 7: CALL(7); break;  case 8: CALL(8); break;       \
        default: CALL(0); break;                               \
    }

template <bool POW2>
static cudaError_t launch_scan_p(const PassParams& P, const ScanParams& S, const float* xyz, uint64_t n, int sm,
                                 cudaStream_t st) {
    uint32_t head;
    uint64_t groups;
    split_aligned(xyz, n, &head, &groups);
#define CS_CALL(DD)                                                                           \
    {                                                                                         \
        int blocks = blocks_for(k_scan<DD, POW2>, sm, groups);                                \
        k_scan<DD, POW2><<<blocks, PASS_THREADS, 0, st>>>(P, S, xyz, n, head, groups);        \
    }
    CS_DISPATCH_D(CS_CALL)
#undef CS_CALL
    return cudaGetLastError();
}

cudaError_t launch_scan(const PassParams& P, const ScanParams& S, const float* xyz, uint64_t n, int sm_count,
                        cudaStream_t st) {
    const bool pow2 = (P.w & (P.w - 1)) == 0;
    return pow2 ? launch_scan_p<true>(P, S, xyz, n, sm_count, st) : launch_scan_p<false>(P, S, xyz, n, sm_count, st);
}

static int blocks_1d(uint64_t m) {
    uint64_t b = (m + PASS_THREADS - 1) / PASS_THREADS;
    if (b > 148 * 8) b = 148 * 8;
    return (int)(b < 1 ? 1 : b);
}

template <bool POW2>
static cudaError_t launch_estimate_p(const PassParams& P, int scale, const uint64_t* cells, uint64_t m,
                                     int32_t* est, cudaStream_t st) {
#define CS_CALL(DD) k_estimate<DD, POW2><<<blocks_1d(m), PASS_THREADS, 0, st>>>(P, scale, cells, m, est)
    CS_DISPATCH_D(CS_CALL)
#undef CS_CALL
    return cudaGetLastError();
}

cudaError_t launch_estimate(const PassParams& P, int scale, const uint64_t* cells, uint64_t m, int32_t* est,
                            cudaStream_t st) {
    if (!m) return cudaSuccess;
    const bool pow2 = (P.w & (P.w - 1)) == 0;
    return pow2 ? launch_estimate_p<true>(P, scale, cells, m, est, st)
                : launch_estimate_p<false>(P, scale, cells, m, est, st);
}

template <bool POW2>
static cudaError_t launch_scan_cells_p(const PassParams& P, const ScanParams& S, int scale, const uint64_t* cells,
                                       uint64_t m, cudaStream_t st) {
#define CS_CALL(DD) k_scan_cells<DD, POW2><<<blocks_1d(m), PASS_THREADS, 0, st>>>(P, S, scale, cells, m)
    CS_DISPATCH_D(CS_CALL)
#undef CS_CALL
    return cudaGetLastError();
}

cudaError_t launch_scan_cells(const PassParams& P, const ScanParams& S, int scale, const uint64_t* cells,
                              uint64_t m, cudaStream_t st) {
    if (!m) return cudaSuccess;
    const bool pow2 = (P.w & (P.w - 1)) == 0;
    return pow2 ? launch_scan_cells_p<true>(P, S, scale, cells, m, st)
                : launch_scan_cells_p<false>(P, S, scale, cells, m, st);
}

}  // namespace cs
