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
#include "cs_scan_common.cuh"

namespace cs {

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
            if (emit) emit = seen_first_time(S.tg[s], c);
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
            emit = e >= tau && seen_first_time(S.tg[s], c);
        }
        append_candidate(S.tg[s], emit, c, e);
    }
}

/* Full-dictionary search (Alg. 1 l.7-13: "for all j in [n]: Estimate(M, j)", the paper's "GPU without
 * heap" query, :304-306): cells first .. first + m - 1 of scale s, no positions needed. */
template <int D, bool POW2>
__global__ void __launch_bounds__(PASS_THREADS)
k_scan_range(const __grid_constant__ PassParams P, const __grid_constant__ ScanParams S, int s, uint64_t first,
             uint64_t m) {
    const int32_t tau = S.tg[s].st->tau;
    const uint64_t stride = (uint64_t)gridDim.x * PASS_THREADS;
    const uint32_t lane = threadIdx.x & 31u;
    for (uint64_t i0 = (uint64_t)blockIdx.x * PASS_THREADS + (threadIdx.x - lane); i0 < m; i0 += stride) {
        const uint64_t i = i0 + lane;
        const uint64_t c = first + i;
        int32_t e = 0;
        bool emit = false;
        if (i < m) emit = P.sc[s].big ? estimate_ge<D, POW2, true>(P, s, c, tau, e) : estimate_ge<D, POW2, false>(P, s, c, tau, e);
        append_candidate(S.tg[s], emit, c, e);
    }
}

/* Children of mesh cells on a finer nested mesh (Gc = r * Gp): out[i * r^3 + t] = id on the fine mesh of the t-th
 * sub-cell of parent i.  Used by the positions-free hierarchical query (Alg. 3: search the coarse
 * layer, then only the children of its heavy cells). */
__global__ void __launch_bounds__(256)
k_expand_children(const uint64_t* __restrict__ parents, uint64_t m, uint32_t Gp, uint32_t Gc, uint32_t r,
                  uint64_t* __restrict__ out) {
    const uint64_t r3 = (uint64_t)r * r * r;
    const uint64_t total = m * r3;
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += stride) {
        const uint64_t p = parents[i / r3];
        const uint32_t t = (uint32_t)(i % r3);
        const uint32_t px = (uint32_t)(p % Gp), py = (uint32_t)((p / Gp) % Gp), pz = (uint32_t)(p / ((uint64_t)Gp * Gp));
        const uint32_t cx = px * r + t % r, cy = py * r + (t / r) % r, cz = pz * r + t / (r * r);
        out[i] = (uint64_t)cx + (uint64_t)Gc * ((uint64_t)cy + (uint64_t)Gc * cz);
    }
}

cudaError_t launch_expand_children(const uint64_t* parents, uint64_t m, uint32_t Gp, uint32_t Gc, uint32_t r, uint64_t* out,
                                   cudaStream_t st) {
    if (!m) return cudaSuccess;
    uint64_t blocks = (m * r * r * r + 255) / 256;
    if (blocks > 148 * 8) blocks = 148 * 8;
    k_expand_children<<<(int)blocks, 256, 0, st>>>(parents, m, Gp, Gc, r, out);
    return cudaGetLastError();
}

/* 26-neighbour shell of mesh cells, periodic (Fig. 14: the particles of the heavy cells "and their
 * surroundings" go to the offline halo finder): out[27*i + t], t = (dx+1) + 3*(dy+1) + 9*(dz+1). */
__global__ void __launch_bounds__(256)
k_expand_neighbours(const uint64_t* __restrict__ ids, uint64_t m, uint32_t G, uint64_t* __restrict__ out) {
    const uint64_t total = m * 27;
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += stride) {
        const uint64_t c = ids[i / 27];
        const uint32_t t = (uint32_t)(i % 27);
        const uint32_t x = (uint32_t)(c % G), y = (uint32_t)((c / G) % G), z = (uint32_t)(c / ((uint64_t)G * G));
        const uint32_t nx = (x + G + t % 3 - 1) % G, ny = (y + G + (t / 3) % 3 - 1) % G, nz = (z + G + t / 9 - 1) % G;
        out[i] = (uint64_t)nx + (uint64_t)G * ((uint64_t)ny + (uint64_t)G * nz);
    }
}

cudaError_t launch_expand_neighbours(const uint64_t* ids, uint64_t m, uint32_t G, uint64_t* out, cudaStream_t st) {
    if (!m) return cudaSuccess;
    uint64_t blocks = (m * 27 + 255) / 256;
    if (blocks > 148 * 8) blocks = 148 * 8;
    k_expand_neighbours<<<(int)blocks, 256, 0, st>>>(ids, m, G, out);
    return cudaGetLastError();
}

/* ---- dispatch on (d, w power of two) ------------------------------------------------------------------ */

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

template <bool POW2>
static cudaError_t launch_scan_range_p(const PassParams& P, const ScanParams& S, int scale, uint64_t first, uint64_t m,
                                       cudaStream_t st) {
#define CS_CALL(DD) k_scan_range<DD, POW2><<<blocks_1d(m), PASS_THREADS, 0, st>>>(P, S, scale, first, m)
    CS_DISPATCH_D(CS_CALL)
#undef CS_CALL
    return cudaGetLastError();
}

cudaError_t launch_scan_range(const PassParams& P, const ScanParams& S, int scale, uint64_t first, uint64_t m,
                              cudaStream_t st) {
    if (!m) return cudaSuccess;
    const bool pow2 = (P.w & (P.w - 1)) == 0;
    return pow2 ? launch_scan_range_p<true>(P, S, scale, first, m, st) : launch_scan_range_p<false>(P, S, scale, first, m, st);
}

}  // namespace cs
