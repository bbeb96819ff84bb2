/*
 * cs_scan_bitmap.cu -- candidate re-scan through a 1-bit-per-counter prefilter (DESIGN.md
 * section 6).
 *
 * Estimate(c) >= tau needs more than half of the rows with s_j(c)*T[j][h_j(c)] >= tau.  For
 * tau >= 1 a row can only pass if |T[j][h_j(c)]| >= tau, whatever its sign hash says.  So once a collection
 * threshold tau >= 1 is known,
 *   k_build_bitmap   writes B[j][b] = (|T[j][b]| >= tau), one bit per counter (d*w/8 bytes: 3.5 MiB for cfg 3, against
 *                    112 MiB of counters -- it stays L2-resident whatever the sketch size);
 *   k_scan_bitmap    per kept particle: cell id, BUCKET hashes only (no sign hashes), one 4-byte gather per row into
 *                    the bitmap, stop as soon as more than (d-1)/2 rows are clear.  The first (d-1)/2 + 1 rows
 *                    cannot reject on their own and are issued back to back.  A cell that survives (a few per
 *                    10^4 at the thresholds of the BASELINE configs) gets the exact estimate from the int32 tables
 *                    (both hashes, d gathers, median network) and is appended iff Estimate >= the current tau.
 * The filter has no false negatives for any current tau >= the tau the bitmap was built with, so the candidate
 * list is the same as with the plain scan.
 */
#include "cs_scan_common.cuh"

namespace cs {

/* One thread = one 32-bit word of the bitmap = 32 consecutive counters (n = d*w counters, any multiple or not). */
__global__ void __launch_bounds__(256)
k_build_bitmap(const int32_t* __restrict__ T, uint64_t n, int32_t tau, uint32_t* __restrict__ bm) {
    const uint64_t words = (n + 31) / 32;
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t wd = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; wd < words; wd += stride) {
        uint32_t bits = 0;
        const uint64_t i0 = wd * 32;
        if (i0 + 32 <= n) {
            const int4* p = reinterpret_cast<const int4*>(T + i0);          // tables are cudaMalloc'd: 16-byte aligned
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                const int4 v = p[q];
                const int32_t t[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const int64_t a = t[k] < 0 ? -(int64_t)t[k] : (int64_t)t[k];
                    bits |= (uint32_t)(a >= (int64_t)tau) << (q * 4 + k);
                }
            }
        } else {
            for (uint64_t i = i0; i < n; ++i) {
                const int64_t a = T[i] < 0 ? -(int64_t)T[i] : (int64_t)T[i];
                bits |= (uint32_t)(a >= (int64_t)tau) << (i - i0);
            }
        }
        bm[wd] = bits;
    }
}

/* true iff at most (d-1)/2 rows of cell c are clear in the bitmap of scale s */
template <int D, bool BIG>
__device__ __forceinline__ bool bitmap_survives(const PassParams& P, int s, const uint32_t* __restrict__ bm, uint32_t c0,
                                                uint32_t c1) {
    const int d = D ? D : P.d;
    const int max_fail = P.rank;
    const uint32_t wmask = (uint32_t)(P.w - 1);
    const RowCoef* rows = &P.rows[s * d];
    int fails = 0;
    if (D > 0) {
        constexpr int FIRST = (D - 1) / 2 + 1;
        uint32_t wd[FIRST], h[FIRST];
#pragma unroll
        for (int j = 0; j < FIRST; ++j) {
            h[j] = bucket_of<BIG>(rows[j], c0, c1, wmask);
            wd[j] = ld_bits(bm + (((uint64_t)j * P.w + h[j]) >> 5));
        }
#pragma unroll
        for (int j = 0; j < FIRST; ++j) fails += 1 - (int)((wd[j] >> (h[j] & 31u)) & 1u);
#pragma unroll
        for (int j = FIRST; j < D; ++j) {
            if (fails <= max_fail) {
                const uint32_t hj = bucket_of<BIG>(rows[j], c0, c1, wmask);
                const uint32_t w = ld_bits(bm + (((uint64_t)j * P.w + hj) >> 5));
                fails += 1 - (int)((w >> (hj & 31u)) & 1u);
            }
        }
    } else {
        for (int j = 0; j < d && fails <= max_fail; ++j) {
            const uint32_t hj = bucket_of<BIG>(rows[j], c0, c1, wmask);
            const uint32_t w = ld_bits(bm + (((uint64_t)j * P.w + hj) >> 5));
            fails += 1 - (int)((w >> (hj & 31u)) & 1u);
        }
    }
    return fails <= max_fail;
}

struct BitmapParams {
    const uint32_t* bm[CS_MAX_SCALES];
};

template <int D>
__device__ __forceinline__ void scan_particle_bm(const PassParams& P, const ScanParams& S, const BitmapParams& Bm,
                                                 const int32_t* tau, bool keep, float x, float y, float z) {
    for (int s = 0; s < P.n_scales; ++s) {
        uint64_t c = 0;
        int32_t est = 0;
        bool emit = false;
        if (keep) {
            c = cell_of(x, y, z, P.sc[s]);
            const uint32_t c0 = cell_c0(c), c1 = cell_c1(c);
            const bool live = P.sc[s].big ? bitmap_survives<D, true>(P, s, Bm.bm[s], c0, c1)
                                          : bitmap_survives<D, false>(P, s, Bm.bm[s], c0, c1);
            if (live && seen_first_time(S.tg[s], c)) {   // rare: exact estimate from the counters, once per cell
                emit = P.sc[s].big ? estimate_ge<D, true, true>(P, s, c, tau[s], est)
                                   : estimate_ge<D, true, false>(P, s, c, tau[s], est);
            }
        }
        append_candidate(S.tg[s], emit, c, est);
    }
}

template <int D>
__global__ void __launch_bounds__(PASS_THREADS)
k_scan_bitmap(const __grid_constant__ PassParams P, const __grid_constant__ ScanParams S,
              const __grid_constant__ BitmapParams Bm, const float* __restrict__ xyz, uint64_t n, uint32_t head,
              uint64_t groups) {
    int32_t tau[CS_MAX_SCALES];
#pragma unroll
    for (int s = 0; s < CS_MAX_SCALES; ++s) tau[s] = s < P.n_scales ? S.tg[s].st->tau : 0;

    const uint64_t stride = (uint64_t)gridDim.x * PASS_THREADS;
    const float4* body = reinterpret_cast<const float4*>(xyz + 3 * (uint64_t)head);
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
        scan_particle_bm<D>(P, S, Bm, tau, k0, q0.x, q0.y, q0.z);
        scan_particle_bm<D>(P, S, Bm, tau, k1, q0.w, q1.x, q1.y);
        scan_particle_bm<D>(P, S, Bm, tau, k2, q1.z, q1.w, q2.x);
        scan_particle_bm<D>(P, S, Bm, tau, k3, q2.y, q2.z, q2.w);
    }
    if (blockIdx.x == 0 && threadIdx.x < 32) {        // warp 0: the <= 6 edge particles
        const uint64_t tail0 = (uint64_t)head + 4 * groups;
        const uint64_t n_edge = (uint64_t)head + (n - tail0);
        const bool in = threadIdx.x < n_edge;
        float x = 0.f, y = 0.f, z = 0.f;
        bool keep = false;
        if (in) {
            const uint64_t i = threadIdx.x < head ? threadIdx.x : tail0 + (threadIdx.x - head);
            keep = !P.sample || keep_particle(P.K, P.index0 + i, P.Tp);
            const float* p = xyz + 3 * i;
            x = ld_stream4(p); y = ld_stream4(p + 1); z = ld_stream4(p + 2);
        }
        scan_particle_bm<D>(P, S, Bm, tau, keep, x, y, z);
    }
}

/* ---- host side ------------------------------------------------------------------------------------------ */

cudaError_t launch_build_bitmap(const int32_t* T, uint64_t n_counters, int32_t tau, uint32_t* bm, cudaStream_t st) {
    const uint64_t words = (n_counters + 31) / 32;
    uint64_t blocks = (words + 255) / 256;
    if (blocks > 148 * 8) blocks = 148 * 8;
    k_build_bitmap<<<(int)(blocks ? blocks : 1), 256, 0, st>>>(T, n_counters, tau, bm);
    return cudaGetLastError();
}

/* All scales of P in one pass; bm[s] = bitmap of scale s, built for a tau <= the scale's current tau (>= 1).
 * Needs w a power of two. */
cudaError_t launch_scan_bitmap(const PassParams& P, const ScanParams& S, const uint32_t* const* bm, const float* xyz,
                               uint64_t n, int sm_count, cudaStream_t st) {
    BitmapParams Bm = {};
    for (int s = 0; s < P.n_scales; ++s) Bm.bm[s] = bm[s];
    uint32_t head;
    uint64_t groups;
    split_aligned(xyz, n, &head, &groups);
    const size_t smem = 0;
#define CS_CALL(DD)                                                                                               \
    {                                                                                                             \
        int per_sm = 0;                                                                                           \
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_scan_bitmap<DD>, PASS_THREADS, smem);            \
        if (per_sm < 1) per_sm = 1;                                                                               \
        uint64_t need = (groups + PASS_THREADS - 1) / PASS_THREADS, full = (uint64_t)sm_count * per_sm;           \
        int blocks = (int)(need < full ? (need ? need : 1) : full);                                               \
        k_scan_bitmap<DD><<<blocks, PASS_THREADS, smem, st>>>(P, S, Bm, xyz, n, head, groups);                    \
    }
    CS_DISPATCH_D(CS_CALL)
#undef CS_CALL
    return cudaGetLastError();
}

}  // namespace cs
