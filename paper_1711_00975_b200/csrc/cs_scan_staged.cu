/*
 * cs_scan_staged.cu -- row-partitioned candidate re-scan for sketches larger than the L2-resident budget
 * (DESIGN.md section 6).
 *
 * Random 4-byte gathers run at ~290 G/s while the rows they touch stay L2-resident and at ~130 G/s (112 MiB)
 * to ~50 G/s (448 MiB) when they do not (measured, cs_probe_l2 mode 2).  The d rows of one scale are therefore
 * split into groups that fit the budget and the scan becomes a pipeline of stages, one per group:
 *   stage 0      positions -> cell id c, row values of group 0, fails = #{values < tau};
 *                a cell is dropped once fails > (d-1)/2 (its median is then < tau);
 *                survivors are written as (c | fails << 60) to a list
 *   stage i      list -> rows of group i -> list
 *   final        (k_stage_final) the survivors of the last stage have Estimate(c) >= tau (or may have, after a bitmap
 *                first stage): the exact median over all d rows is computed for them on dense warps and (c, est) is
 *                appended to the candidate list.
 * Lists are segmented per block (block b of every stage owns segment b), so no global atomic is needed for the
 * survivor lists and the result does not depend on scheduling (the candidate list is sorted afterwards).
 */
#include "cs_scan_common.cuh"

namespace cs {

constexpr uint64_t FAIL_SHIFT = 60;
constexpr uint64_t CELL_MASK = (1ULL << FAIL_SHIFT) - 1;

struct StageParams {
    const uint64_t* in;      // survivor list of the previous stage (unused by stage 0)
    uint64_t* out;           // survivor list of this stage (unused by the last stage)
    const uint32_t* cnt_in;  // entries per segment
    uint32_t* cnt_out;
    uint32_t seg_cap;        // entries per segment
    int32_t row0;            // first row of this stage's group
    int32_t d_all;           // rows of the scale (for the final median)
    int32_t pad;
};

/* Row values of rows [row0, row0 + R) of the (single) scale in P; returns the updated fail count. */
template <int R, bool POW2, bool BIG>
__device__ __forceinline__ int stage_rows(const PassParams& P, int row0, uint64_t c, int32_t tau, int fails,
                                          int max_fail) {
    const uint32_t c0 = cell_c0(c), c1 = cell_c1(c);
    const int32_t* T = P.sc[0].T;
#pragma unroll
    for (int j = 0; j < R; ++j) {
        if (fails <= max_fail) {
            int32_t v = row_value<BIG, POW2>(P, T, P.rows[row0 + j], row0 + j, c0, c1);
            fails += (v < tau);
        }
    }
    return fails;
}

/* A cell that is still alive after the rows of a stage goes to the block's segment of the survivor list.  Must be
 * reached by all 32 lanes (one shared-memory reservation per warp). */
__device__ __forceinline__ void stage_finish(bool live, uint64_t c, int fails, uint64_t* seg_out, uint32_t* s_cnt) {
    const uint32_t mask = __ballot_sync(0xFFFFFFFFu, live);
    if (mask) {
        const uint32_t lane = threadIdx.x & 31u;
        const int leader = __ffs(mask) - 1;
        uint32_t base = 0;
        if ((int)lane == leader) base = atomicAdd(s_cnt, (uint32_t)__popc(mask));
        base = __shfl_sync(0xFFFFFFFFu, base, leader);
        if (live) seg_out[base + __popc(mask & ((1u << lane) - 1u))] = c | ((uint64_t)fails << FAIL_SHIFT);
    }
}

/* One cell through one stage: rows, then stage_finish.  Must be reached by all 32 lanes. */
template <int R, bool POW2>
__device__ __forceinline__ void stage_cell(const PassParams& P, const StageParams& Q,
                                           int32_t tau, int max_fail, bool live, uint64_t c, int fails,
                                           uint64_t* seg_out, uint32_t* s_cnt) {
    if (live) {
        fails = P.sc[0].big ? stage_rows<R, POW2, true>(P, Q.row0, c, tau, fails, max_fail)
                            : stage_rows<R, POW2, false>(P, Q.row0, c, tau, fails, max_fail);
        live = fails <= max_fail;
    }
    stage_finish(live, c, fails, seg_out, s_cnt);
}

/* Stage 0: block b owns position groups [b*gpb, (b+1)*gpb); block 0 also takes the <= 6 edge particles. */
template <int R, bool POW2>
__global__ void __launch_bounds__(PASS_THREADS)
k_stage_first(const __grid_constant__ PassParams P, const __grid_constant__ StageParams Q,
              const __grid_constant__ ScanTarget tg, const float* __restrict__ xyz, uint64_t n, uint32_t head,
              uint64_t groups, uint64_t gpb) {
    __shared__ uint32_t s_cnt;
    if (threadIdx.x == 0) s_cnt = 0;
    __syncthreads();
    const int32_t tau = tg.st->tau;
    const int max_fail = P.rank;
    uint64_t* seg = Q.out + (uint64_t)blockIdx.x * Q.seg_cap;
    const float4* body = reinterpret_cast<const float4*>(xyz + 3 * (uint64_t)head);
    const uint64_t g_lo = (uint64_t)blockIdx.x * gpb;
    const uint64_t g_hi = g_lo + gpb < groups ? g_lo + gpb : groups;
    const uint32_t lane = threadIdx.x & 31u;
    for (uint64_t g0 = g_lo + (threadIdx.x - lane); g0 < g_hi; g0 += PASS_THREADS) {
        const uint64_t g = g0 + lane;
        const bool in = g < g_hi;
        float4 q0 = make_float4(0.f, 0.f, 0.f, 0.f), q1 = q0, q2 = q0;
        if (in) {
            q0 = ld_stream16(body + 3 * g);
            q1 = ld_stream16(body + 3 * g + 1);
            q2 = ld_stream16(body + 3 * g + 2);
        }
        bool k0 = in, k1 = in, k2 = in, k3 = in;
        if (P.sample && in) {
            const uint64_t i0 = P.index0 + head + 4 * g;
            k0 = keep_particle(P.K, i0 + 0, P.Tp);
            k1 = keep_particle(P.K, i0 + 1, P.Tp);
            k2 = keep_particle(P.K, i0 + 2, P.Tp);
            k3 = keep_particle(P.K, i0 + 3, P.Tp);
        }
        stage_cell<R, POW2>(P, Q, tau, max_fail, k0, cell_of(q0.x, q0.y, q0.z, P.sc[0]), 0, seg, &s_cnt);
        stage_cell<R, POW2>(P, Q, tau, max_fail, k1, cell_of(q0.w, q1.x, q1.y, P.sc[0]), 0, seg, &s_cnt);
        stage_cell<R, POW2>(P, Q, tau, max_fail, k2, cell_of(q1.z, q1.w, q2.x, P.sc[0]), 0, seg, &s_cnt);
        stage_cell<R, POW2>(P, Q, tau, max_fail, k3, cell_of(q2.y, q2.z, q2.w, P.sc[0]), 0, seg, &s_cnt);
    }
    if (blockIdx.x == 0 && threadIdx.x < 32) {
        const uint64_t tail0 = (uint64_t)head + 4 * groups;
        const uint64_t n_edge = (uint64_t)head + (n - tail0);
        bool keep = false;
        uint64_t c = 0;
        if (threadIdx.x < n_edge) {
            const uint64_t i = threadIdx.x < head ? threadIdx.x : tail0 + (threadIdx.x - head);
            keep = !P.sample || keep_particle(P.K, P.index0 + i, P.Tp);
            const float* p = xyz + 3 * i;
            c = cell_of(ld_stream4(p), ld_stream4(p + 1), ld_stream4(p + 2), P.sc[0]);
        }
        stage_cell<R, POW2>(P, Q, tau, max_fail, keep, c, 0, seg, &s_cnt);
    }
    __syncthreads();
    if (threadIdx.x == 0) Q.cnt_out[blockIdx.x] = s_cnt;
}

/* Stage i > 0: block b reads segment b of the previous stage. */
template <int R, bool POW2>
__global__ void __launch_bounds__(PASS_THREADS)
k_stage_next(const __grid_constant__ PassParams P, const __grid_constant__ StageParams Q,
             const __grid_constant__ ScanTarget tg) {
    __shared__ uint32_t s_cnt;
    if (threadIdx.x == 0) s_cnt = 0;
    __syncthreads();
    const int32_t tau = tg.st->tau;
    const int max_fail = P.rank;
    const uint64_t* seg_in = Q.in + (uint64_t)blockIdx.x * Q.seg_cap;
    uint64_t* seg = Q.out + (uint64_t)blockIdx.x * Q.seg_cap;
    const uint32_t cnt = Q.cnt_in[blockIdx.x];
    for (uint32_t t0 = 0; t0 < cnt; t0 += PASS_THREADS) {
        const uint32_t t = t0 + threadIdx.x;
        const bool live = t < cnt;
        const uint64_t e = live ? seg_in[t] : 0;
        stage_cell<R, POW2>(P, Q, tau, max_fail, live, e & CELL_MASK, (int)(e >> FAIL_SHIFT), seg, &s_cnt);
    }
    __syncthreads();
    if (threadIdx.x == 0) Q.cnt_out[blockIdx.x] = s_cnt;
}

/* After the last stage: the cells still alive (few) get their exact estimate -- all d rows, values in registers, median
 * network -- and are appended to the candidate list iff Estimate >= tau (a bitmap first stage counts fails
 * conservatively) and, when the duplicate filter is on, on their first arrival.  A kernel of its own so that this runs on
 * full warps: inside the last stage one lane in ten took this path and every warp paid for it (cfg 5: 1400 thread
 * instructions per surviving cell). */
template <int D, bool POW2>
__global__ void __launch_bounds__(PASS_THREADS)
k_stage_final(const __grid_constant__ PassParams P, const __grid_constant__ StageParams Q,
              const __grid_constant__ ScanTarget tg) {
    const int32_t tau = tg.st->tau;
    const uint64_t* seg_in = Q.in + (uint64_t)blockIdx.x * Q.seg_cap;
    const uint32_t cnt = Q.cnt_in[blockIdx.x];
    for (uint32_t t0 = 0; t0 < cnt; t0 += PASS_THREADS) {
        const uint32_t t = t0 + threadIdx.x;
        bool emit = false;
        uint64_t c = 0;
        int32_t est = 0;
        if (t < cnt) {
            c = seg_in[t] & CELL_MASK;
            if (seen_first_time(tg, c)) {
                est = P.sc[0].big ? estimate_full<D, POW2, true>(P, 0, c) : estimate_full<D, POW2, false>(P, 0, c);
                emit = est >= tau;
            }
        }
        append_candidate(tg, emit, c, est);
    }
}

/* ------------------------------------------------------------------------------------------------------------
 * Bitmap first stage.  Once tau >= 1, a row can only pass if |T[j][h_j(c)]| >= tau.  The first FIRST = (d-1)/2 + 1
 * rows (which cannot reject on their own) are tested against
 *   - a coarse bitmap in shared memory: bit i of row j = OR over counters [i*2^g, (i+1)*2^g) of (|T| >= tau); a
 *     clear bit certifies the row as failed without any L2 request (about 40 % of the rows at cfg 3, g = 4);
 *   - else the fine bitmap (1 bit per counter, d*w/8 bytes, L2-resident whatever the sketch size), 4-byte gathers.
 * Only bucket hashes are needed (no sign hashes).  All four particles of a thread are taken through the phases
 * together, so that up to 4*FIRST gathers per thread are in flight.  Fail counts are conservative (a set bit may
 * still fail on the sign or the exact value); survivors go to the per-segment lists in the format of k_stage_first
 * and the remaining rows run in k_stage_next on dense warps; k_stage_final then checks Estimate >= tau exactly.
 * One CTA of 512 threads per SM walks the segments blockIdx.x, blockIdx.x + gridDim.x, ...
 * ------------------------------------------------------------------------------------------------------------ */

constexpr int CB_THREADS = 1024;

struct CoarseParams {
    const uint32_t* fine;      // fine bitmap: bit (j*w + b)
    const uint32_t* coarse;    // rows 0 .. FIRST-1, row j at word offset row_off[j]
    uint32_t g_row[5];         // log2 counters per coarse bit of row j
    uint32_t row_off[6];       // row_off[FIRST] = total words (a multiple of 4)
    uint32_t big;              // cell ids of the mesh can exceed 2^31
    uint32_t nseg;             // segments = grid size of the following stages
};

template <int FIRST, bool BIG>
__device__ __forceinline__ void cb_hashes(const PassParams& P, uint32_t wmask, const uint64_t* c, uint32_t (&h)[2][FIRST]) {
#pragma unroll
    for (int q = 0; q < 2; ++q) {
        const uint32_t c0 = cell_c0(c[q]), c1 = cell_c1(c[q]);
#pragma unroll
        for (int j = 0; j < FIRST; ++j) h[q][j] = bucket_of<BIG>(P.rows[j], c0, c1, wmask);
    }
}

template <int FIRST>
__global__ void __launch_bounds__(CB_THREADS, 1)
k_stage_first_cb(const __grid_constant__ PassParams P, const __grid_constant__ StageParams Q,
                 const __grid_constant__ CoarseParams C, const float* __restrict__ xyz, uint64_t n, uint32_t head,
                 uint64_t groups, uint64_t gpb) {
    extern __shared__ __align__(16) uint32_t cb_smem[];
    __shared__ uint32_t s_cnt;
    const uint32_t cwords = C.row_off[FIRST];                                         // a multiple of 4
    {
        const uint4* src = reinterpret_cast<const uint4*>(C.coarse);
        uint4* dst = reinterpret_cast<uint4*>(cb_smem);
        for (uint32_t i = threadIdx.x; i < cwords / 4; i += CB_THREADS) dst[i] = src[i];
    }
    __syncthreads();
    const uint32_t cs_addr = (uint32_t)__cvta_generic_to_shared(cb_smem);
    const uint32_t wmask = (uint32_t)(P.w - 1);
    const float4* body = reinterpret_cast<const float4*>(xyz + 3 * (uint64_t)head);
    const uint32_t lane = threadIdx.x & 31u;
    const uint32_t below = (1u << lane) - 1u;

    for (uint32_t seg = blockIdx.x; seg < C.nseg; seg += gridDim.x) {
        if (threadIdx.x == 0) s_cnt = 0;
        __syncthreads();
        uint64_t* out = Q.out + (uint64_t)seg * Q.seg_cap;
        const uint64_t g_lo = (uint64_t)seg * gpb;
        const uint64_t g_hi = g_lo + gpb < groups ? g_lo + gpb : groups;
        /* the positions of the next iteration are fetched before this one is hashed (a load issued right before its
         * first use stalls the warp for the whole trip to HBM) */
        float4 n0 = make_float4(0.f, 0.f, 0.f, 0.f), n1 = n0, n2 = n0;
        {
            const uint64_t gf = g_lo + threadIdx.x;
            if (gf < g_hi) { n0 = ld_stream16(body + 3 * gf); n1 = ld_stream16(body + 3 * gf + 1); n2 = ld_stream16(body + 3 * gf + 2); }
        }
        for (uint64_t g0 = g_lo + (threadIdx.x - lane); g0 < g_hi; g0 += CB_THREADS) {
            const uint64_t g = g0 + lane;
            const bool in = g < g_hi;
            const float4 q0 = n0, q1 = n1, q2 = n2;
            {
                const uint64_t gn = g + CB_THREADS;
                if (gn < g_hi) { n0 = ld_stream16(body + 3 * gn); n1 = ld_stream16(body + 3 * gn + 1); n2 = ld_stream16(body + 3 * gn + 2); }
            }
            bool keep[4] = {in, in, in, in};
            if (P.sample && in) {
                const uint64_t i0 = P.index0 + head + 4 * g;
#pragma unroll
                for (int q = 0; q < 4; ++q) keep[q] = keep_particle(P.K, i0 + q, P.Tp);
            }
            uint64_t c[4];
            c[0] = cell_of(q0.x, q0.y, q0.z, P.sc[0]);
            c[1] = cell_of(q0.w, q1.x, q1.y, P.sc[0]);
            c[2] = cell_of(q1.z, q1.w, q2.x, P.sc[0]);
            c[3] = cell_of(q2.y, q2.z, q2.w, P.sc[0]);
            uint32_t live4 = 0, fails4 = 0;
            /* two particles at a time (64 registers per thread at 1024 threads): hashes, coarse bits from shared
             * memory, then the fine words of the undecided rows, all in flight together */
#pragma unroll
            for (int half = 0; half < 2; ++half) {
                uint32_t h[2][FIRST];
                if (C.big) cb_hashes<FIRST, true>(P, wmask, c + 2 * half, h);
                else       cb_hashes<FIRST, false>(P, wmask, c + 2 * half, h);
                uint32_t wd[2][FIRST];
#pragma unroll
                for (int q = 0; q < 2; ++q)
#pragma unroll
                    for (int j = 0; j < FIRST; ++j) {
                        const uint32_t i = h[q][j] >> C.g_row[j];
                        wd[q][j] = (lds_u32s(cs_addr + (C.row_off[j] + (i >> 5)) * 4u) >> (i & 31u)) & 1u;
                    }
#pragma unroll
                for (int q = 0; q < 2; ++q)
#pragma unroll
                    for (int j = 0; j < FIRST; ++j) {
                        uint32_t w = 0;
                        if (keep[2 * half + q] && wd[q][j]) w = ld_bits(C.fine + (((uint64_t)j * P.w + h[q][j]) >> 5));
                        wd[q][j] = w;
                    }
#pragma unroll
                for (int q = 0; q < 2; ++q) {
                    uint32_t fails = 0;
#pragma unroll
                    for (int j = 0; j < FIRST; ++j) fails += 1u - ((wd[q][j] >> (h[q][j] & 31u)) & 1u);
                    if (keep[2 * half + q] && fails < (uint32_t)FIRST) {              // FIRST = rank + 1 fails reject
                        live4 |= 1u << (2 * half + q);
                        fails4 |= fails << (8 * (2 * half + q));
                    }
                }
            }
            /* one reservation in the segment for the survivors among this warp's 128 particles */
            uint32_t m[4], tot = 0;
#pragma unroll
            for (int q = 0; q < 4; ++q) { m[q] = __ballot_sync(0xFFFFFFFFu, (live4 >> q) & 1u); tot += __popc(m[q]); }
            if (tot) {
                uint32_t base = 0;
                if (lane == 0) base = atomicAdd(&s_cnt, tot);
                base = __shfl_sync(0xFFFFFFFFu, base, 0);
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    if ((live4 >> q) & 1u)
                        out[base + __popc(m[q] & below)] = c[q] | ((uint64_t)((fails4 >> (8 * q)) & 0xFFu) << FAIL_SHIFT);
                    base += __popc(m[q]);
                }
            }
        }
        if (seg == 0 && threadIdx.x < 32) {           // the <= 6 edge particles: passed on undecided (fails = 0)
            const uint64_t tail0 = (uint64_t)head + 4 * groups;
            const uint64_t n_edge = (uint64_t)head + (n - tail0);
            bool keep = false;
            uint64_t c = 0;
            if (threadIdx.x < n_edge) {
                const uint64_t i = threadIdx.x < head ? threadIdx.x : tail0 + (threadIdx.x - head);
                keep = !P.sample || keep_particle(P.K, P.index0 + i, P.Tp);
                const float* p = xyz + 3 * i;
                c = cell_of(ld_stream4(p), ld_stream4(p + 1), ld_stream4(p + 2), P.sc[0]);
            }
            const uint32_t mask = __ballot_sync(0xFFFFFFFFu, keep);
            if (mask) {
                const int leader = __ffs(mask) - 1;
                uint32_t base = 0;
                if ((int)lane == leader) base = atomicAdd(&s_cnt, (uint32_t)__popc(mask));
                base = __shfl_sync(0xFFFFFFFFu, base, leader);
                if (keep) out[base + __popc(mask & below)] = c;
            }
        }
        __syncthreads();
        if (threadIdx.x == 0) Q.cnt_out[seg] = s_cnt;
        __syncthreads();
    }
}

/* ---- host side ------------------------------------------------------------------------------------------ */

template <int R, bool POW2>
static void launch_stage(bool first, int blocks, const PassParams& P, const StageParams& Q, const ScanTarget& tg,
                         const float* xyz, uint64_t n, uint32_t head, uint64_t groups, uint64_t gpb, cudaStream_t st) {
    if (first) k_stage_first<R, POW2><<<blocks, PASS_THREADS, 0, st>>>(P, Q, tg, xyz, n, head, groups, gpb);
    else       k_stage_next<R, POW2><<<blocks, PASS_THREADS, 0, st>>>(P, Q, tg);
}

/* the survivors of the last stage (list Q.in) -> exact estimates -> candidate list */
template <bool POW2>
static void launch_final(int blocks, const PassParams& P, const StageParams& Q, const ScanTarget& tg, cudaStream_t st) {
#define CS_CALL(DD) k_stage_final<DD, POW2><<<blocks, PASS_THREADS, 0, st>>>(P, Q, tg)
    CS_DISPATCH_D(CS_CALL)
#undef CS_CALL
}

template <bool POW2>
static void launch_stage_r(int R, bool first, int blocks, const PassParams& P, const StageParams& Q,
                           const ScanTarget& tg, const float* xyz, uint64_t n, uint32_t head, uint64_t groups,
                           uint64_t gpb, cudaStream_t st) {
    switch (R) {
        case 1: launch_stage<1, POW2>(first, blocks, P, Q, tg, xyz, n, head, groups, gpb, st); break;
        case 2: launch_stage<2, POW2>(first, blocks, P, Q, tg, xyz, n, head, groups, gpb, st); break;
        case 3: launch_stage<3, POW2>(first, blocks, P, Q, tg, xyz, n, head, groups, gpb, st); break;
        case 4: launch_stage<4, POW2>(first, blocks, P, Q, tg, xyz, n, head, groups, gpb, st); break;
        case 5: launch_stage<5, POW2>(first, blocks, P, Q, tg, xyz, n, head, groups, gpb, st); break;
        case 6: launch_stage<6, POW2>(first, blocks, P, Q, tg, xyz, n, head, groups, gpb, st); break;
        case 7: launch_stage<7, POW2>(first, blocks, P, Q, tg, xyz, n, head, groups, gpb, st); break;
        default: launch_stage<8, POW2>(first, blocks, P, Q, tg, xyz, n, head, groups, gpb, st); break;
    }
}

uint64_t staged_list_entries(uint64_t n, uint32_t blocks) {
    const uint64_t groups = n / 4 + 1;
    const uint64_t gpb = (groups + blocks - 1) / blocks;
    return (uint64_t)blocks * (4 * gpb + 8);
}

/* P: PassParams of ONE scale (n_scales = 1, rows[0..d), d = all its rows).  rows_per_stage in [1, 8]. */
cudaError_t launch_scan_staged(const PassParams& P, const ScanTarget& tg, const StageBuffers& B, int rows_per_stage,
                               const float* xyz, uint64_t n, cudaStream_t st, uint64_t* launches, PhaseTimer* tm) {
    uint32_t head;
    uint64_t groups;
    split_aligned(xyz, n, &head, &groups);
    const int blocks = (int)B.blocks;
    const uint64_t gpb = (groups + blocks - 1) / blocks;
    const uint32_t seg_cap = (uint32_t)(4 * gpb + 8);
    if ((uint64_t)blocks * seg_cap > B.cap_entries) return cudaErrorInvalidValue;
    const bool pow2 = (P.w & (P.w - 1)) == 0;
    if (rows_per_stage > 8) rows_per_stage = 8;
    if (rows_per_stage < 1) rows_per_stage = 1;
    const int stages = (P.d + rows_per_stage - 1) / rows_per_stage;
    const int each = (P.d + stages - 1) / stages;                 /* balanced groups */
    int cur = 0;
    for (int row0 = 0, i = 0; row0 < P.d; row0 += each, ++i) {
        const int R = row0 + each <= P.d ? each : P.d - row0;
        const bool last = row0 + R >= P.d;
        StageParams Q;
        Q.in = B.list[cur];
        Q.cnt_in = B.cnt[cur];
        Q.out = B.list[cur ^ 1];
        Q.cnt_out = B.cnt[cur ^ 1];
        Q.seg_cap = seg_cap;
        Q.row0 = row0;
        Q.d_all = P.d;
        Q.pad = 0;
        if (tm) tm->mark(i == 0 ? PH_SCAN_FIRST : PH_SCAN_NEXT, st);
        if (pow2) launch_stage_r<true>(R, i == 0, blocks, P, Q, tg, xyz, n, head, groups, gpb, st);
        else      launch_stage_r<false>(R, i == 0, blocks, P, Q, tg, xyz, n, head, groups, gpb, st);
        *launches += 1;
        cur ^= 1;
        if (last) {
            StageParams F = Q;
            F.in = B.list[cur];
            F.cnt_in = B.cnt[cur];
            if (pow2) launch_final<true>(blocks, P, F, tg, st);
            else      launch_final<false>(blocks, P, F, tg, st);
            *launches += 1;
        }
    }
    return cudaGetLastError();
}

/* coarse word cw: bit b = OR of the fine bits [(cw*32 + b) << g, +2^g) */
__global__ void __launch_bounds__(256)
k_build_coarse(const uint32_t* __restrict__ fine, uint64_t n_coarse_words, int g, uint32_t* __restrict__ coarse) {
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t cw = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; cw < n_coarse_words; cw += stride) {
        uint32_t bits = 0;
        for (int b = 0; b < 32; ++b) {
            const uint64_t start = (cw * 32 + b) << g;
            uint32_t any = 0;
            if (g >= 5) {
                for (uint64_t k = 0; k < (1ull << (g - 5)); ++k) any |= fine[(start >> 5) + k];
            } else {
                any = (fine[start >> 5] >> (start & 31u)) & (g == 0 ? 1u : ((1u << (1u << g)) - 1u));
            }
            bits |= (uint32_t)(any != 0) << b;
        }
        coarse[cw] = bits;
    }
}

/* Shape of the coarse bitmap: g = the smallest group size 2^g whose FIRST rows fit the shared-memory budget, then as
 * many leading rows as still fit at 2^(g-1).  false: shape not supported by the bitmap first stage (the caller uses the
 * plain stages). */
bool coarse_shape(int d, int rank, uint64_t w, CoarseShape* out) {
    const int first = rank + 1, rest = d - first;
    const uint64_t budget = 190 * 1024;                                       // all rows at 2^g
    /* with leading rows at 2^(g-1).  What is left of the 228 KB is the L1 cache of the position loads and of the fine-bitmap
     * gathers: measured at cfg 3 (g = 4), first stage 13.2 / 12.6 / 12.0 / 17.3 ms with 128 / 160 / 192 / 224 KB of bitmap */
    const uint64_t budget_fine = 192 * 1024;
    if (first > 5 || rest < 1 || rest > 8 || (w & (w - 1)) || w < 4096) return false;
    for (uint32_t g = 0; g <= 8; ++g) {
        if ((w >> g) < 128) break;
        const uint64_t row = (w >> g) / 8;                                    // bytes per row at 2^g
        if ((uint64_t)first * row > budget) continue;
        uint32_t nf = 0;
        if (g >= 1)
            while (nf < (uint32_t)first && (uint64_t)(nf + 1) * 2 * row + (uint64_t)(first - nf - 1) * row <= budget_fine) ++nf;
        out->g = g;
        out->n_fine = nf;
        uint32_t off = 0;
        for (int j = 0; j <= first; ++j) {
            out->row_off[j] = off;
            off += (uint32_t)(((uint32_t)j < nf ? 2 * row : row) / 4);
        }
        return true;
    }
    return false;
}

/* fine: bitmap of the scale (bit j*w + b), already built for the current tau; coarse: scratch of shape.row_off[first] words */
cudaError_t launch_scan_staged_cb(const PassParams& P, const ScanTarget& tg, const StageBuffers& B, const uint32_t* fine,
                                  uint32_t* coarse, const CoarseShape& shape, bool rebuild_coarse, const float* xyz,
                                  uint64_t n, int sm_count, cudaStream_t st, uint64_t* launches, PhaseTimer* tm) {
    const int first = P.rank + 1, rest = P.d - first;
    if (rebuild_coarse) {
        if (tm) tm->mark(PH_BITMAP, st);
        for (int part = 0; part < 2; ++part) {              // rows [0, n_fine) at g-1, rows [n_fine, first) at g
            const uint32_t j0 = part ? shape.n_fine : 0, j1 = part ? (uint32_t)first : shape.n_fine;
            if (j0 == j1) continue;
            const uint64_t words = shape.row_off[j1] - shape.row_off[j0];
            uint64_t blocks = (words + 255) / 256;
            if (blocks > 148 * 8) blocks = 148 * 8;
            k_build_coarse<<<(int)blocks, 256, 0, st>>>(fine + (uint64_t)j0 * P.w / 32, words, (int)(part ? shape.g : shape.g - 1),
                                                        coarse + shape.row_off[j0]);
            *launches += 1;
        }
    }
    uint32_t head;
    uint64_t groups;
    split_aligned(xyz, n, &head, &groups);
    const int blocks = (int)B.blocks;
    const uint64_t gpb = (groups + blocks - 1) / blocks;
    const uint32_t seg_cap = (uint32_t)(4 * gpb + 8);
    if ((uint64_t)blocks * seg_cap > B.cap_entries) return cudaErrorInvalidValue;
    StageParams Q;
    Q.in = nullptr; Q.cnt_in = nullptr;
    Q.out = B.list[0]; Q.cnt_out = B.cnt[0];
    Q.seg_cap = seg_cap; Q.row0 = 0; Q.d_all = P.d; Q.pad = 0;
    CoarseParams C;
    C.fine = fine; C.coarse = coarse; C.nseg = (uint32_t)blocks;
    for (int j = 0; j < 5; ++j) C.g_row[j] = (uint32_t)j < shape.n_fine ? shape.g - 1 : shape.g;
    for (int j = 0; j < 6; ++j) C.row_off[j] = j <= first ? shape.row_off[j] : 0;
    C.big = P.sc[0].big;
    const size_t smem = (size_t)shape.row_off[first] * 4;
    cudaError_t e = cudaSuccess;
    if (tm) tm->mark(PH_SCAN_FIRST, st);
#define CS_CB(F)                                                                                              \
    case F:                                                                                                   \
        e = cudaFuncSetAttribute(k_stage_first_cb<F>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem); \
        if (e != cudaSuccess) return e;                                                                       \
        k_stage_first_cb<F><<<sm_count < blocks ? sm_count : blocks, CB_THREADS, smem, st>>>(P, Q, C, xyz, n, head,   \
                                                                                               groups, gpb);  \
        break;
    switch (first) { CS_CB(1) CS_CB(2) CS_CB(3) CS_CB(4) CS_CB(5) default: return cudaErrorInvalidValue; }
#undef CS_CB
    *launches += 1;
    StageParams Q2 = Q;
    Q2.in = B.list[0]; Q2.cnt_in = B.cnt[0];
    Q2.out = B.list[1]; Q2.cnt_out = B.cnt[1];
    Q2.row0 = first;
    if (tm) tm->mark(PH_SCAN_NEXT, st);
    /* The rows left go in two stages: ONE row first, then the others.  Nearly every survivor of the bitmap stage arrives one
     * fail short of rejection and leaves after the next row; with all rows in one kernel some lane of every warp needs the
     * later rows, so every warp paid their instructions and their dependent gathers. */
    const int r1 = (rest >= 2 && n >= (1ull << 22)) ? 1 : rest;      /* short chunks: the extra launch costs more */
    launch_stage_r<true>(r1, false, blocks, P, Q2, tg, xyz, n, head, groups, gpb, st);
    StageParams F = Q2;
    F.in = B.list[1];
    F.cnt_in = B.cnt[1];
    *launches += 2;
    if (rest > r1) {
        StageParams Q3 = Q2;
        Q3.in = B.list[1]; Q3.cnt_in = B.cnt[1];
        Q3.out = B.list[0]; Q3.cnt_out = B.cnt[0];
        Q3.row0 = first + r1;
        launch_stage_r<true>(rest - r1, false, blocks, P, Q3, tg, xyz, n, head, groups, gpb, st);
        F.in = B.list[0];
        F.cnt_in = B.cnt[0];
        *launches += 1;
    }
    launch_final<true>(blocks, P, F, tg, st);
    return cudaGetLastError();
}

}  // namespace cs
