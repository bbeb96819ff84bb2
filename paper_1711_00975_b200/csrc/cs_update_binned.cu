/*
 * cs_update_binned.cu -- the Add pass (T[j][h_j(c)] += s_j(c)) without one L2 atomic per
 * counter update.
 *
 * Why: red.global.add.s32 at random addresses is bounded by the L2 tag-lookup rate (measured ~194 G/s chip-wide,
 * ncu: lts__t_tag_requests at ~78 % of peak, half of the requests cross the die fabric), i.e. ~39 ms for the
 * 7.5e9 updates of cfg 3, while shared-memory atomics run at ~2250 G/s.  So the updates are first partitioned
 * by table slice and then applied slice by slice in shared memory:
 *
 *   k_bin_scatter   positions -> quantise -> (sample) -> 2R hashes -> one 2-byte record per (particle, row):
 *                   record = (offset within slice) << 1 | (sign bit);  bin = (row, slice).  Each CTA keeps a
 *                   small staging buffer per bin in shared memory; a bin that has collected 32 records is
 *                   written out as one 64-byte unit to the bin's region in HBM (space reserved with one global
 *                   atomic per unit).  Records that do not fit (a staging buffer or a bin region is full:
 *                   heavily duplicated streams) are applied directly with red.global -- int32 adds commute,
 *                   so the table is the same whichever way a record travels.
 *   k_bin_apply     one CTA per bin: zero a slice of counters in shared memory, stream the bin's records
 *                   (16-byte loads, 8 records each), atomicAdd into shared memory, then T[slice] += it
 *                   with plain coalesced loads/stores (the CTA owns the slice during this kernel).
 *
 * HBM traffic per particle and row: 2 B written + 2 B read, plus 12 B per particle per pass for the positions.
 */
#include "cs_device.cuh"
#include "cs_launch.cuh"

namespace cs {

constexpr int BIN_THREADS = 1024;
constexpr uint32_t UNIT = 32;            // records per flush unit (64 bytes)
// pairs of particles a thread bins between two flush phases: BinParams::pairs (the host sizes the staging buffers with it)

__device__ __forceinline__ float2 ld_stream8(const float2* p) {
    float2 v;
    asm volatile("ld.global.cs.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "l"(p));
    return v;
}
__device__ __forceinline__ uint4 ld_stream16u(const uint4* p) {
    uint4 v;
    asm volatile("ld.global.cs.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
    return v;
}

/* records are written once and read once by k_bin_apply: streaming stores, so that they do not push the counters of the
 * direct rows out of L2 */
__device__ __forceinline__ void st_stream16u(uint4* p, const uint4& v) {
    asm volatile("st.global.cs.v4.u32 [%0], {%1, %2, %3, %4};" :: "l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}

/* Shared-memory layout of k_bin_scatter (dynamic):
 *   cnt[NB] | pad | buf[NB*C] (u16) | 64 B pad
 * All accesses of the hot loop use 32-bit shared-space addresses (no generic-to-shared conversion per access). */
__host__ __device__ inline size_t smem_off_buf(uint32_t nb) { return ((size_t)nb * 4 + 15) & ~(size_t)15; }
size_t scatter_smem_bytes(uint32_t nb, uint32_t C) { return smem_off_buf(nb) + (size_t)nb * C * 2 + 64; }

__device__ __forceinline__ uint32_t atoms_inc(uint32_t addr) {
    uint32_t old;
    asm volatile("atom.shared.add.u32 %0, [%1], 1;" : "=r"(old) : "r"(addr) : "memory");
    return old;
}
__device__ __forceinline__ void sts_u16(uint32_t addr, uint32_t v) {
    asm volatile("st.shared.u16 [%0], %1;" :: "r"(addr), "h"((unsigned short)v) : "memory");
}

/* Apply one record directly (fallback path and the partial buffers at the end of the kernel). */
__device__ __forceinline__ void apply_direct(int32_t* T, uint32_t bin, uint32_t log2S, uint32_t rec) {
    red_add(T + (((uint64_t)bin << log2S) | (rec >> 1)), 1 - 2 * (int32_t)(rec & 1u));
}

/* Loop-invariant values of the insert path, kept in registers. */
struct InsertCtx {
    uint32_t cnt_addr;     // shared address of cnt[0]
    uint32_t buf_addr;     // shared address of buf[0]
    uint32_t C, C2;        // staging capacity in records / bytes
    uint32_t log2S, smask; // slice shift, (1 << log2S) - 1
    uint32_t log2w, wmask;
    int32_t rows_direct;
    uint32_t stat_addr;    // shared address of the CTA's 4 route counters (BinParams::stats)
};

/* BIG: cell ids of the mesh can exceed 2^31 (two-limb form of cs_hash.h). */
template <bool BIG>
__device__ __forceinline__ void row_hashes(const RowCoef& rc, uint32_t c0, uint32_t c1, uint32_t& h, uint32_t& sb) {
    h = affine_low32<BIG>(rc.h, c0, c1);
    sb = affine_low32<BIG>(rc.s, c0, c1) & 1u;
}

/* Rare path: rows of one particle whose staging buffer was full are applied with red.global. */
__device__ __noinline__ void apply_rows_direct(const PassParams& P, uint32_t wmask, uint32_t c0, uint32_t c1, uint32_t ovf) {
    while (ovf) {
        const int j = __ffs(ovf) - 1;
        ovf &= ovf - 1;
        const uint32_t h = affine_low32<true>(P.rows[j].h, c0, c1) & wmask;
        const uint32_t sb = affine_low32<true>(P.rows[j].s, c0, c1) & 1u;
        red_add(P.sc[0].T + (uint64_t)j * P.w + h, 1 - 2 * (int32_t)sb);
    }
}

template <int R, bool BIG>
__device__ __forceinline__ void bin_particle(const PassParams& P, const InsertCtx& X, float x, float y, float z) {
    const uint64_t c = cell_of(x, y, z, P.sc[0]);
    const uint32_t c0 = cell_c0(c), c1 = cell_c1(c);
    int32_t* T = P.sc[0].T;
    uint32_t ovf = 0;
#pragma unroll
    for (int j = 0; j < R; ++j) {
        uint32_t h, sb;
        row_hashes<BIG>(P.rows[j], c0, c1, h, sb);
        if (j < X.rows_direct) {
            red_add(T + (((uint32_t)j << X.log2w) | (h & X.wmask)), 1 - 2 * (int32_t)sb);
            continue;
        }
        /* counter index within the binned rows of this pass (bins cover rows rows_direct .. R-1 only) */
        const uint32_t key = ((uint32_t)(j - X.rows_direct) << X.log2w) | (h & X.wmask);
        const uint32_t bin = key >> X.log2S;
        const uint32_t slot = atoms_inc(X.cnt_addr + bin * 4u);
        if (slot < X.C) sts_u16(X.buf_addr + bin * X.C2 + slot * 2u, ((key & X.smask) << 1) + sb);
        else            ovf |= 1u << j;                                 // staging buffer full
    }
    if (ovf) {
        asm volatile("red.shared.add.u32 [%0], %1;" :: "r"(X.stat_addr), "r"((uint32_t)__popc(ovf)) : "memory");
        apply_rows_direct(P, X.wmask, c0, c1, ovf);
    }
}

/* Particles [head, head + 2*pairs) are read as pairs (3 x 8 B per thread, 8-byte aligned); the <= 1 particle
 * before and the <= 1 after are applied directly by block 0.
 * One round = every thread bins B.pairs pairs; then every bin that holds >= 32 records is flushed.  (A
 * queue of the bins that are due, built in a phase of its own between two more barriers, cost 0.26 ms of 20.2 at cfg 3:
 * with ~130 records per bin and round nearly every bin is due.) */
template <int R, bool BIG>
__global__ void __launch_bounds__(BIN_THREADS, 1)
k_bin_scatter(const __grid_constant__ PassParams P, const __grid_constant__ BinParams B,
              const float* __restrict__ xyz, uint64_t n, uint32_t head, uint64_t pairs) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ uint32_t s_stat[4];
    if (threadIdx.x < 4) s_stat[threadIdx.x] = 0;
    const uint32_t NT = blockDim.x;                                  // 512 or 1024
    uint32_t* cnt = reinterpret_cast<uint32_t*>(smem_raw);
    uint16_t* buf = reinterpret_cast<uint16_t*>(smem_raw + smem_off_buf(B.nb));
    for (uint32_t i = threadIdx.x; i < B.nb; i += NT) cnt[i] = 0;
    __syncthreads();

    InsertCtx X;
    X.cnt_addr = (uint32_t)__cvta_generic_to_shared(cnt);
    X.buf_addr = (uint32_t)__cvta_generic_to_shared(buf);
    X.C = B.C; X.C2 = B.C * 2u;
    X.log2S = B.log2S; X.smask = (1u << B.log2S) - 1u;
    X.log2w = B.log2w; X.wmask = (uint32_t)(P.w - 1);
    X.rows_direct = B.rows_direct;
    X.stat_addr = (uint32_t)__cvta_generic_to_shared(s_stat);

    const float2* body = reinterpret_cast<const float2*>(xyz + 3 * (uint64_t)head);
    const uint64_t per_sub = (uint64_t)gridDim.x * NT;                 // pairs of one sub-round over the grid
    const uint64_t per_round = per_sub * B.pairs;
    const uint64_t rounds = (pairs + per_round - 1) / per_round;
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const uint32_t grp = lane >> 2, l4 = lane & 3u;
    int32_t* T = P.sc[0].T + ((uint64_t)B.rows_direct << B.log2w);      // first binned row: bin << log2S indexes from here

    for (uint64_t r = 0; r < rounds; ++r) {
#pragma unroll 1
        for (uint32_t u = 0; u < B.pairs; ++u) {
            const uint64_t g = r * per_round + u * per_sub + (uint64_t)blockIdx.x * NT + threadIdx.x;
            if (g < pairs) {
                const float2 q0 = ld_stream8(body + 3 * g);
                const float2 q1 = ld_stream8(body + 3 * g + 1);
                const float2 q2 = ld_stream8(body + 3 * g + 2);
                const uint64_t i0 = P.index0 + head + 2 * g;
                if (!P.sample || keep_particle(P.K, i0, P.Tp)) bin_particle<R, BIG>(P, X, q0.x, q0.y, q1.x);
                if (!P.sample || keep_particle(P.K, i0 + 1, P.Tp)) bin_particle<R, BIG>(P, X, q1.y, q2.x, q2.y);
            }
        }
        __syncthreads();
        /* flush: groups of 4 lanes, one bin each; two bins per group and trip, so that the two reservations (global
         * atomics that return a value: ~1 us each) are in flight together */
        const uint32_t nq = B.nb, fstride = (NT / 32) * 8;
        auto reserve = [&](uint32_t e, uint32_t& c, uint32_t& units, uint32_t& base) -> bool {
            c = 0; units = 0; base = 0;
            if (e >= nq) return false;
            c = min(cnt[e], B.C);
            units = c / UNIT;
            if (units == 0) return false;
            if (l4 == 0) {
                base = atomicAdd(&B.cursor[e], units * UNIT);
                atomicAdd(&s_stat[3], units * UNIT);
            }
            return true;
        };
        auto drain = [&](uint32_t bin, uint32_t c, uint32_t units, uint32_t base) {
            uint16_t* src = buf + bin * B.C;
            for (uint32_t u = 0; u < units; ++u) {
                const uint4 v = *reinterpret_cast<const uint4*>(src + u * UNIT + l4 * 8);
                const uint32_t at = base + u * UNIT;
                if (at + UNIT <= B.cap) {
                    st_stream16u(reinterpret_cast<uint4*>(B.bins + (uint64_t)bin * B.cap + at + l4 * 8), v);
                } else {                                               // bin region full: apply directly
                    atomicAdd(&s_stat[1], 8u);
                    if (l4 == 0) atomicSub(&s_stat[3], UNIT);
                    const uint32_t wds[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
                    for (int k = 0; k < 4; ++k) {
                        apply_direct(T, bin, B.log2S, wds[k] & 0xFFFFu);
                        apply_direct(T, bin, B.log2S, wds[k] >> 16);
                    }
                }
            }
            /* move the < 32 leftover records to the front, 8 records per lane (source and destination do not
             * overlap; what is copied past `left` is never read: the 64 B pad covers the last bin's over-read) */
            const uint32_t left = c - units * UNIT;
            if (l4 * 8 < left)
                *reinterpret_cast<uint4*>(src + l4 * 8) = *reinterpret_cast<const uint4*>(src + units * UNIT + l4 * 8);
            if (l4 == 0) cnt[bin] = left;
        };
        for (uint32_t e0 = warp * 8; e0 < nq; e0 += 2 * fstride) {
            const uint32_t ea = e0 + grp, eb = ea + fstride;
            uint32_t ca, ua, ba, cb, ub, bb;
            const bool ona = reserve(ea, ca, ua, ba), onb = reserve(eb, cb, ub, bb);
            ba = __shfl_sync(0xFFFFFFFFu, ba, grp * 4);
            bb = __shfl_sync(0xFFFFFFFFu, bb, grp * 4);
            if (ona) drain(ea, ca, ua, ba);
            if (onb) drain(eb, cb, ub, bb);
        }
        __syncthreads();
    }
    /* partial buffers (< 32 records per bin): applied directly */
    for (uint32_t bin = threadIdx.x; bin < B.nb; bin += NT) {
        const uint32_t c = min(cnt[bin], B.C);
        for (uint32_t i = 0; i < c; ++i) apply_direct(T, bin, B.log2S, buf[bin * B.C + i]);
        if (c) atomicAdd(&s_stat[2], c);
    }
    __syncthreads();
    if (threadIdx.x < 4 && B.stats && s_stat[threadIdx.x]) atomicAdd(&B.stats[threadIdx.x], (unsigned long long)s_stat[threadIdx.x]);
    if (blockIdx.x == 0 && threadIdx.x < 2) {
        const uint64_t tail0 = (uint64_t)head + 2 * pairs;
        uint64_t i = ~0ull;
        if (threadIdx.x == 0 && head) i = 0;
        if (threadIdx.x == 1 && tail0 < n) i = tail0;
        if (i != ~0ull && (!P.sample || keep_particle(P.K, P.index0 + i, P.Tp))) {
            const float* p = xyz + 3 * i;
            const uint64_t c = cell_of(ld_stream4(p), ld_stream4(p + 1), ld_stream4(p + 2), P.sc[0]);
            apply_rows_direct(P, X.wmask, cell_c0(c), cell_c1(c), (1u << R) - 1u);
        }
    }
}

/* One CTA per bin. */
__global__ void __launch_bounds__(BIN_THREADS, 1)
k_bin_apply(int32_t* __restrict__ T, const uint16_t* __restrict__ bins, const uint32_t* __restrict__ cursor,
            uint32_t cap, uint32_t log2S) {
    extern __shared__ __align__(16) int32_t acc[];
    const uint32_t S = 1u << log2S;
    const uint32_t bin = blockIdx.x;
    for (uint32_t i = threadIdx.x; i < S; i += BIN_THREADS) acc[i] = 0;
    __syncthreads();
    const uint32_t len = min(cursor[bin], cap);                        // a multiple of UNIT
    const uint4* src = reinterpret_cast<const uint4*>(bins + (uint64_t)bin * cap);
    const uint32_t nvec = len / 8;
    for (uint32_t v = threadIdx.x; v < nvec; v += BIN_THREADS) {
        const uint4 q = ld_stream16u(src + v);
        const uint32_t wds[4] = {q.x, q.y, q.z, q.w};
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const uint32_t lo = wds[k] & 0xFFFFu, hi = wds[k] >> 16;
            atomicAdd(&acc[lo >> 1], 1 - 2 * (int32_t)(lo & 1u));
            atomicAdd(&acc[hi >> 1], 1 - 2 * (int32_t)(hi & 1u));
        }
    }
    __syncthreads();
    int32_t* dst = T + ((uint64_t)bin << log2S);
    for (uint32_t i = threadIdx.x; i < S; i += BIN_THREADS) {
        const int32_t a = acc[i];
        if (a) dst[i] = (int32_t)((uint32_t)dst[i] + (uint32_t)a);
    }
}

/* ---- host side ------------------------------------------------------------------------------------------ */

template <int R>
static cudaError_t launch_scatter_r(const PassParams& P, const BinParams& B, const float* xyz, uint64_t n, int sm_count,
                                    cudaStream_t st) {
    uint32_t head = (reinterpret_cast<uintptr_t>(xyz) & 7u) ? 1u : 0u;   // 12 B per particle: skip one to reach 8-byte alignment
    if (head > n) head = (uint32_t)n;
    const uint64_t pairs = (n - head) / 2;
    const size_t smem = scatter_smem_bytes(B.nb, B.C);
    cudaError_t e;
#define CS_SCATTER(BIG)                                                                                         \
    e = cudaFuncSetAttribute(k_bin_scatter<R, BIG>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);    \
    if (e != cudaSuccess) return e;                                                                             \
    { int per_sm = 0;                                                                                         \
      cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_bin_scatter<R, BIG>, (int)B.threads, smem);      \
      if (per_sm < 1) per_sm = 1;                                                                               \
      k_bin_scatter<R, BIG><<<sm_count * per_sm, B.threads, smem, st>>>(P, B, xyz, n, head, pairs); }
    if (P.sc[0].big) { CS_SCATTER(true) } else { CS_SCATTER(false) }
#undef CS_SCATTER
    return cudaGetLastError();
}

/* P: PassParams of ONE scale restricted to the R = P.d rows of this pass (rows[0..R), sc[0].T = first row).
 * The caller has zeroed B.cursor[0..nb) on the stream.  Launches scatter + apply. */
cudaError_t launch_update_binned(const PassParams& P, const BinParams& B, const float* xyz, uint64_t n, int sm_count,
                                 cudaStream_t st, PhaseTimer* tm) {
    cudaError_t e;
    if (tm) tm->mark(PH_SCATTER, st);
    switch (P.d) {
        case 1: e = launch_scatter_r<1>(P, B, xyz, n, sm_count, st); break;
        case 2: e = launch_scatter_r<2>(P, B, xyz, n, sm_count, st); break;
        case 3: e = launch_scatter_r<3>(P, B, xyz, n, sm_count, st); break;
        case 4: e = launch_scatter_r<4>(P, B, xyz, n, sm_count, st); break;
        case 5: e = launch_scatter_r<5>(P, B, xyz, n, sm_count, st); break;
        case 6: e = launch_scatter_r<6>(P, B, xyz, n, sm_count, st); break;
        case 7: e = launch_scatter_r<7>(P, B, xyz, n, sm_count, st); break;
        case 8: e = launch_scatter_r<8>(P, B, xyz, n, sm_count, st); break;
        default: return cudaErrorInvalidValue;
    }
    if (e != cudaSuccess) return e;
    if (B.nb == 0) return cudaSuccess;                                       // every row of the pass is direct
    if (tm) tm->mark(PH_APPLY, st);
    const size_t smem = (size_t)4 << B.log2S;
    e = cudaFuncSetAttribute(k_bin_apply, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    k_bin_apply<<<B.nb, BIN_THREADS, smem, st>>>(P.sc[0].T + ((uint64_t)B.rows_direct << B.log2w), B.bins, B.cursor, B.cap,
                                                 B.log2S);
    return cudaGetLastError();
}

}  // namespace cs
