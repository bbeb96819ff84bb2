/*
 * cs_kernels.cu -- the particle passes of libcs.so, hand-written for sm_100a:
 *   k_update   quantise + (sample) + 2d hashes + d red.global.add.s32 per kept particle
 *   k_scan     the same front end, d gathers with early exit against tau, median, append   (a5-a6)
 *   k_estimate one thread per cell id: 2d hashes, d gathers, median network                (a5)
 * Paper passages: Add / Estimate PAPER.md:134-139; UPDATE / Estimate thread code PAPER.md:326-373 (prior
 * art: one block per item with t threads on a GTX 1080 -- here one thread owns whole particles, 4 at a time,
 * loaded as three 16-byte vectors, and all hash coefficients sit in the constant bank as kernel parameters).
 */
#include "cs_device.cuh"
#include "cs_launch.cuh"

namespace cs {

/* ------------------------------------------------------------------------------------------------------
 * update
 * ------------------------------------------------------------------------------------------------------ */

template <int D, bool POW2, bool BIG>
__device__ __forceinline__ void add_rows(const PassParams& P, int s, uint64_t c) {
    const int d = D ? D : P.d;
    const uint32_t c0 = cell_c0(c), c1 = cell_c1(c);
    int32_t* T = P.sc[s].T;
    const RowCoef* rows = &P.rows[s * d];
#pragma unroll
    for (int j = 0; j < d; ++j) {
        uint32_t b;
        int32_t sg;
        bucket_sign<BIG, POW2>(rows[j], c0, c1, P.w, b, sg);
        red_add(T + (uint64_t)j * P.w + b, sg);
    }
}

template <int D, bool POW2>
__device__ __forceinline__ void add_particle(const PassParams& P, float x, float y, float z) {
    for (int s = 0; s < P.n_scales; ++s) {
        uint64_t c = cell_of(x, y, z, P.sc[s]);
        if (P.sc[s].big) add_rows<D, POW2, true>(P, s, c);
        else             add_rows<D, POW2, false>(P, s, c);
    }
}

/* Particles [head, head + 4*groups) are read as groups of 4 (3 x 16 B per thread, 16-byte aligned);
 * the <= 3 particles before and the <= 3 after are read with scalar loads by block 0. */
template <int D, bool POW2>
__global__ void __launch_bounds__(PASS_THREADS)
k_update(const __grid_constant__ PassParams P, const float* __restrict__ xyz, uint64_t n, uint32_t head,
         uint64_t groups) {
    const uint64_t stride = (uint64_t)gridDim.x * PASS_THREADS;
    const float4* body = reinterpret_cast<const float4*>(xyz + 3 * (uint64_t)head);
    for (uint64_t g = (uint64_t)blockIdx.x * PASS_THREADS + threadIdx.x; g < groups; g += stride) {
        float4 q0 = ld_stream16(body + 3 * g);
        float4 q1 = ld_stream16(body + 3 * g + 1);
        float4 q2 = ld_stream16(body + 3 * g + 2);
        const uint64_t i0 = P.index0 + head + 4 * g;
        if (!P.sample) {
            add_particle<D, POW2>(P, q0.x, q0.y, q0.z);
            add_particle<D, POW2>(P, q0.w, q1.x, q1.y);
            add_particle<D, POW2>(P, q1.z, q1.w, q2.x);
            add_particle<D, POW2>(P, q2.y, q2.z, q2.w);
        } else {
            if (keep_particle(P.K, i0 + 0, P.Tp)) add_particle<D, POW2>(P, q0.x, q0.y, q0.z);
            if (keep_particle(P.K, i0 + 1, P.Tp)) add_particle<D, POW2>(P, q0.w, q1.x, q1.y);
            if (keep_particle(P.K, i0 + 2, P.Tp)) add_particle<D, POW2>(P, q1.z, q1.w, q2.x);
            if (keep_particle(P.K, i0 + 3, P.Tp)) add_particle<D, POW2>(P, q2.y, q2.z, q2.w);
        }
    }
    if (blockIdx.x == 0) {
        const uint64_t tail0 = (uint64_t)head + 4 * groups;
        const uint64_t n_edge = (uint64_t)head + (n - tail0);          // <= 6
        if (threadIdx.x < n_edge) {
            uint64_t i = threadIdx.x < head ? threadIdx.x : tail0 + (threadIdx.x - head);
            if (!P.sample || keep_particle(P.K, P.index0 + i, P.Tp)) {
                const float* p = xyz + 3 * i;
                add_particle<D, POW2>(P, ld_stream4(p), ld_stream4(p + 1), ld_stream4(p + 2));
            }
        }
    }
}

template <int D, bool POW2>
static cudaError_t launch_update_t(const PassParams& P, const float* xyz, uint64_t n, int sm_count,
                                   cudaStream_t st) {
    uint32_t head;
    uint64_t groups;
    split_aligned(xyz, n, &head, &groups);
    int blocks = blocks_for(k_update<D, POW2>, sm_count, groups);
    k_update<D, POW2><<<blocks, PASS_THREADS, 0, st>>>(P, xyz, n, head, groups);
    return cudaGetLastError();
}

template <bool POW2>
static cudaError_t launch_update_d(const PassParams& P, const float* xyz, uint64_t n, int sm, cudaStream_t st) {
    switch (P.d) {
        case 1: return launch_update_t<1, POW2>(P, xyz, n, sm, st);
        case 2: return launch_update_t<2, POW2>(P, xyz, n, sm, st);
        case 3: return launch_update_t<3, POW2>(P, xyz, n, sm, st);
        case 4: return launch_update_t<4, POW2>(P, xyz, n, sm, st);
        case 5: return launch_update_t<5, POW2>(P, xyz, n, sm, st);
        case 6: return launch_update_t<6, POW2>(P, xyz, n, sm, st);
        case 7: return launch_update_t<7, POW2>(P, xyz, n, sm, st);
        case 8: return launch_update_t<8, POW2>(P, xyz, n, sm, st);
        default: return launch_update_t<0, POW2>(P, xyz, n, sm, st);   // 9..32 rows: runtime loop
    }
}

cudaError_t launch_update(const PassParams& P, const float* xyz, uint64_t n, int sm_count, cudaStream_t st) {
    const bool pow2 = (P.w & (P.w - 1)) == 0;
    return pow2 ? launch_update_d<true>(P, xyz, n, sm_count, st) : launch_update_d<false>(P, xyz, n, sm_count, st);
}

/* ------------------------------------------------------------------------------------------------------
 * sampling prefilter ("sampling hash ... for each element")
 * For sample_p well below 1 the kept particles are first copied to a dense buffer (one pass: 12 B read per
 * particle, the sampling hash, 12 B written per kept particle); every later pass -- row groups, scales, chunks of
 * the binned update, the re-scan -- then runs on the kept particles only, without a sampling hash.  The order of
 * the kept particles in the buffer is arbitrary (Add commutes; candidates are a set).
 * ------------------------------------------------------------------------------------------------------ */

/* One block iteration = 4096 particles (4 groups of 4 per thread): every thread first evaluates its 16 sampling hashes,
 * the block reserves its output range with ONE global atomic (a reservation per warp or per 1024 particles serialises at
 * the L2: same-address atomics), then the groups that hold a kept particle are loaded (3 x 16 B) and the kept particles
 * written at the thread's offset.  The order of the kept particles in the buffer is arbitrary. */
constexpr int CK_U = 4;
__global__ void __launch_bounds__(PASS_THREADS)
k_compact_kept(const float* __restrict__ xyz, uint64_t n, uint32_t head, uint64_t groups, uint64_t index0, uint64_t K,
               uint64_t Tp, float* __restrict__ out, uint32_t* count, uint32_t cap) {
    __shared__ uint32_t s_warp[PASS_THREADS / 32];
    __shared__ uint32_t s_base;
    const uint64_t per_iter = (uint64_t)PASS_THREADS * CK_U;
    const uint64_t stride = (uint64_t)gridDim.x * per_iter;
    const float4* body = reinterpret_cast<const float4*>(xyz + 3 * (uint64_t)head);
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    /* block-uniform trip count; block 0 runs one extra iteration for the <= 6 edge particles (thread = particle) */
    const uint64_t iters = (groups + stride - 1) / stride;
    for (uint64_t it = 0; it < iters + (blockIdx.x == 0 ? 1 : 0); ++it) {
        const bool edge = it == iters;
        const uint64_t g0 = it * stride + (uint64_t)blockIdx.x * per_iter + threadIdx.x;
        uint32_t kbits = 0;                                  // bit 4*u + q: particle q of group g0 + u*PASS_THREADS
        uint64_t edge_i = 0;
        if (!edge) {
#pragma unroll
            for (int u = 0; u < CK_U; ++u) {
                const uint64_t g = g0 + (uint64_t)u * PASS_THREADS;
                if (g < groups) {
                    const uint64_t i0 = index0 + head + 4 * g;
#pragma unroll
                    for (int q = 0; q < 4; ++q) kbits |= (uint32_t)keep_particle(K, i0 + q, Tp) << (4 * u + q);
                }
            }
        } else {
            const uint64_t tail0 = (uint64_t)head + 4 * groups;
            const uint64_t n_edge = (uint64_t)head + (n - tail0);
            if (threadIdx.x < n_edge) {
                edge_i = threadIdx.x < head ? threadIdx.x : tail0 + (threadIdx.x - head);
                kbits = keep_particle(K, index0 + edge_i, Tp) ? 1u : 0u;
            }
        }
        const uint32_t c = __popc(kbits);
        uint32_t incl = c;
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            const uint32_t v = __shfl_up_sync(0xFFFFFFFFu, incl, off);
            if (lane >= off) incl += v;
        }
        if (lane == 31) s_warp[warp] = incl;
        __syncthreads();
        if (threadIdx.x == 0) {
            uint32_t sum = 0;
            for (int w = 0; w < PASS_THREADS / 32; ++w) { const uint32_t x = s_warp[w]; s_warp[w] = sum; sum += x; }
            s_base = sum ? atomicAdd(count, sum) : 0;
        }
        __syncthreads();
        uint64_t pos = (uint64_t)s_base + s_warp[warp] + incl - c;
        if (!edge) {
#pragma unroll
            for (int u = 0; u < CK_U; ++u) {
                const uint32_t kb = (kbits >> (4 * u)) & 15u;
                if (kb) {                                    // 48 B are only fetched where something is kept
                    const uint64_t g = g0 + (uint64_t)u * PASS_THREADS;
                    const float4 q0 = ld_stream16(body + 3 * g), q1 = ld_stream16(body + 3 * g + 1),
                                 q2 = ld_stream16(body + 3 * g + 2);
                    const float px[4] = {q0.x, q0.w, q1.z, q2.y}, py[4] = {q0.y, q1.x, q1.w, q2.z},
                                pz[4] = {q0.z, q1.y, q2.x, q2.w};
#pragma unroll
                    for (int q = 0; q < 4; ++q)
                        if (kb & (1u << q)) {
                            if (pos < cap) { out[3 * pos] = px[q]; out[3 * pos + 1] = py[q]; out[3 * pos + 2] = pz[q]; }
                            ++pos;                           // *count > cap is reported to the host, which then falls back
                        }
                }
            }
        } else if (kbits) {
            const float* p = xyz + 3 * edge_i;
            if (pos < cap) { out[3 * pos] = ld_stream4(p); out[3 * pos + 1] = ld_stream4(p + 1); out[3 * pos + 2] = ld_stream4(p + 2); }
        }
        __syncthreads();                                  // s_warp / s_base are rewritten by the next iteration
    }
}

/* *count (device, zeroed by the caller) = kept particles of xyz[0..n); the first min(*count, cap) are in out. */
cudaError_t launch_compact_kept(const float* xyz, uint64_t n, uint64_t index0, uint64_t K, uint64_t Tp, float* out,
                                uint32_t* count, uint32_t cap, int sm_count, cudaStream_t st) {
    uint32_t head;
    uint64_t groups;
    split_aligned(xyz, n, &head, &groups);
    int blocks = blocks_for(k_compact_kept, sm_count, (groups + CK_U - 1) / CK_U);
    k_compact_kept<<<blocks, PASS_THREADS, 0, st>>>(xyz, n, head, groups, index0, K, Tp, out, count, cap);
    return cudaGetLastError();
}

/* ------------------------------------------------------------------------------------------------------
 * packed 64-bit particle records ("3 coordinates in 64 bits"; R23)
 * rec = qx | qy << 21 | qz << 42 = the particle's cell on the 2^21 mesh; cell on a mesh of G: i = (q*G) >> 21 per axis.
 * k_pack_records    float32 positions -> records (quantise with G = 2^21).
 * k_unpack_centres  records -> float32 positions at the centre of the record's cell on the FINEST mesh Gf of the
 *                   handle.  The float quantisation of that centre gives back exactly i = (q*Gf) >> 21 (the centre is
 *                   0.5 cells from either boundary and float32 rounding moves x*scale by < 0.25 for Gf <= 2^20), and
 *                   for every coarser mesh that divides Gf the nested floors agree, so the ordinary passes run on
 *                   the unpacked buffer unchanged and compute the integer rule bit for bit.
 * ------------------------------------------------------------------------------------------------------ */
__global__ void __launch_bounds__(256)
k_pack_records(const float* __restrict__ xyz, uint64_t n, float qscale21, uint64_t* __restrict__ recs) {
    const float top = (float)((1u << 21) - 1);
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const float* p = xyz + 3 * i;
        const uint64_t qx = quantise_axis(ld_stream4(p), qscale21, top), qy = quantise_axis(ld_stream4(p + 1), qscale21, top),
                       qz = quantise_axis(ld_stream4(p + 2), qscale21, top);
        recs[i] = qx | (qy << 21) | (qz << 42);
    }
}

__global__ void __launch_bounds__(256)
k_unpack_centres(const uint64_t* __restrict__ recs, uint64_t n, uint32_t Gf, float cell_f, float* __restrict__ xyz) {
    const uint64_t M = (1ull << 21) - 1;
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const uint64_t r = recs[i];
        const uint32_t ix = (uint32_t)(((r & M) * Gf) >> 21), iy = (uint32_t)((((r >> 21) & M) * Gf) >> 21),
                       iz = (uint32_t)((((r >> 42) & M) * Gf) >> 21);
        float* p = xyz + 3 * i;
        p[0] = __fmul_rn(__fadd_rn((float)ix, 0.5f), cell_f);
        p[1] = __fmul_rn(__fadd_rn((float)iy, 0.5f), cell_f);
        p[2] = __fmul_rn(__fadd_rn((float)iz, 0.5f), cell_f);
    }
}

cudaError_t launch_pack_records(const float* xyz, uint64_t n, float qscale21, uint64_t* recs, cudaStream_t st) {
    if (!n) return cudaSuccess;
    uint64_t blocks = (n + 255) / 256;
    if (blocks > 148 * 16) blocks = 148 * 16;
    k_pack_records<<<(int)blocks, 256, 0, st>>>(xyz, n, qscale21, recs);
    return cudaGetLastError();
}

cudaError_t launch_unpack_centres(const uint64_t* recs, uint64_t n, uint32_t Gf, float cell_f, float* xyz, cudaStream_t st) {
    if (!n) return cudaSuccess;
    uint64_t blocks = (n + 255) / 256;
    if (blocks > 148 * 16) blocks = 148 * 16;
    k_unpack_centres<<<(int)blocks, 256, 0, st>>>(recs, n, Gf, cell_f, xyz);
    return cudaGetLastError();
}

/* T += in (merge / restore by linearity), wraparound. */
__global__ void __launch_bounds__(256) k_table_add(int32_t* __restrict__ T, const int32_t* __restrict__ in, uint64_t n) {
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride)
        T[i] = (int32_t)((uint32_t)T[i] + (uint32_t)in[i]);
}

cudaError_t launch_table_add(int32_t* T, const int32_t* in, uint64_t n, cudaStream_t st) {
    if (!n) return cudaSuccess;
    uint64_t blocks = (n + 255) / 256;
    if (blocks > 148 * 8) blocks = 148 * 8;
    k_table_add<<<(int)blocks, 256, 0, st>>>(T, in, n);
    return cudaGetLastError();
}

}  // namespace cs
