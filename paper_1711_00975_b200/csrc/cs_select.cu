/*
 * cs_select.cu -- deterministic selection over the candidate list (sm_100a).
 *
 * The paper keeps "a global array of items above a threshold", raises the threshold geometrically and
 * compacts the array when it grows past k, or a heap whose result depends on arrival order
 * (PAPER.md:142-147).  Here the candidate list is put in its one canonical order
 *     (estimate descending, cell id ascending), each cell once            (R9)
 * by a stable LSD radix sort on (key = 0x7FFFFFFF - est, id), duplicates (same id => same estimate, hence
 * adjacent) are dropped, and the list is cut to the entries that can still matter: every entry whose
 * estimate is >= tau_new, with
 *     tau_new = max(tau_old, min(estimate of the k_max-th entry, thr_min))
 * (no cell with a smaller estimate can enter the top k_max or an excursion set with thr >= thr_min).
 * Top-k for any k <= k_max and the excursion set for any thr >= thr_min are then prefixes of the list.
 *
 * One compaction = ONE cooperative launch (k_compact: every CTA resident, grid-wide barriers between its phases), with
 * no host round trip in it -- for the lists of all scales of a handle that are due at once, each on its share of the grid
 * (select_compact_batch, cs_select_batch.h):
 *   histogram      digit histograms of ALL passes in one sweep over the list
 *   plan           every CTA, from the global counts: which passes are needed (a digit that is the same in every entry
 *                  is skipped: the high bytes of the estimate key almost always are), exclusive digit bases, ping-pong plan
 *   radix passes   one sweep per needed digit: every tile ranks its entries (warp match.any + per-warp digit counters,
 *                  stable), publishes its digit counts and obtains its offsets from the tiles before it by decoupled
 *                  look-back (tiles are dealt round-robin to CTAs that are all running, so nothing waits on a tile that
 *                  has not started)
 *   uniq           drops duplicate ids, again with a look-back over tile totals
 *   cut            fixes the new tau and the number of entries kept, records which half of the ping-pong buffers holds
 *                  the list (the host learns it when it next reads the scan states)
 * Separate launches per phase (round 2's first form: 4 + one per digit) cost 8-9 us each on short lists; a barrier costs
 * about 2.
 */
#include "cs_device.cuh"
#include "cs_select_batch.h"
#include "cs_select_static.h"

#include <atomic>
#include <cooperative_groups.h>

namespace cg = cooperative_groups;

namespace cs {

constexpr int SORT_THREADS = 256;
constexpr int SORT_WARPS = SORT_THREADS / 32;
constexpr int SORT_ITEMS = 8;                              // items per lane: long lists (tiles of 2048 entries)
constexpr int SORT_ITEMS_SHORT = 4;                        // lists whose tiles of 1024 all run at once: shorter chains per
                                                           // tile (cfg 3 select 1.00 -> 0.91 ms; long lists lose: cfg 5 1.33 -> 1.52)
constexpr int SORT_TILE = SORT_THREADS * SORT_ITEMS;       // the long tile (sizes the static scratch)
constexpr uint32_t SHORT_TILES_MAX = 148 * 8;              // upper bound of the tiles a short list has (CTA slots of the GPU)
constexpr int LOOKBACK = 8;                                // predecessors a look-back step fetches together
constexpr int MAX_PASSES = 12;                             // 8 id bytes (ids < 2^60 need 8) + 4 estimate-key bytes

/* Device-side state of one compaction; lives at the start of SelectBuffers::scratch.  Zeroed at allocation; the kernel
 * leaves it zeroed again when it ends. */
struct SortPlan {
    uint32_t hist[MAX_PASSES][256];    // digit counts of the whole list, all passes
    uint32_t uniq_total;               // unique entries
    uint32_t pad[3];
};

/* What every CTA derives for itself (identically) from the global digit counts. */
struct LocalPlan {
    uint32_t base[MAX_PASSES][256];    // first the CTA's own counts (histogram sweep), then exclusive digit bases
    uint32_t active[MAX_PASSES];       // 0: every entry has the same digit in this pass -> nothing to do
    uint32_t src_half[MAX_PASSES];     // which half (0/1) pass p reads
    uint32_t sorted_half;              // half that holds the sorted list
};

/* look-back status word: epoch << 34 | flag << 32 | count; a word of another epoch reads as "not published yet" */
constexpr uint64_t FLAG_AGG = 1, FLAG_INC = 2;
__device__ __forceinline__ uint64_t status_word(uint32_t epoch, uint64_t flag, uint32_t count) {
    return ((uint64_t)epoch << 34) | (flag << 32) | count;
}
__device__ __forceinline__ uint64_t ld_status(const uint64_t* p) {
    uint64_t v;
    asm volatile("ld.global.relaxed.gpu.u64 %0, [%1];" : "=l"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ void st_status(uint64_t* p, uint64_t v) {
    asm volatile("st.global.relaxed.gpu.u64 [%0], %1;" :: "l"(p), "l"(v) : "memory");
}

struct HalfPtrs {
    uint64_t* id[2];
    uint32_t* ek[2];
};

__device__ __forceinline__ uint32_t digit_of(uint64_t id, uint32_t ek, int pass, int id_passes) {
    return pass < id_passes ? ((uint32_t)(id >> (8 * pass)) & 255u) : ((ek >> (8 * (pass - id_passes))) & 255u);
}

/* plan->hist[p][digit] += entries of the list with that digit in pass p, for all passes at once (stride = the nct CTAs
 * that work on this list; bid = this CTA's index among them) */
__device__ __forceinline__ void hist_sweep(const uint64_t* __restrict__ id, const uint32_t* __restrict__ ek, uint32_t n,
                                           int id_passes, int passes, LocalPlan& L, SortPlan* plan, uint32_t bid,
                                           uint32_t nct) {
    for (int i = threadIdx.x; i < passes * 256; i += SORT_THREADS) (&L.base[0][0])[i] = 0;
    __syncthreads();
    const uint32_t stride = nct * SORT_THREADS;
    for (uint32_t i = bid * SORT_THREADS + threadIdx.x; i < n; i += stride) {
        const uint64_t c = id[i];
        const uint32_t k = ek[i];
        for (int p = 0; p < passes; ++p) atomicAdd(&L.base[p][digit_of(c, k, p, id_passes)], 1u);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < passes * 256; i += SORT_THREADS) {
        const uint32_t v = (&L.base[0][0])[i];
        if (v) atomicAdd(&plan->hist[0][0] + i, v);
    }
}

/* Thread t = digit t.  Global digit counts -> exclusive bases, which passes are needed (a digit that is the same in every
 * entry is skipped: the high bytes of the estimate key almost always are), ping-pong plan.  Every CTA computes the same. */
__device__ __forceinline__ void make_plan(const SortPlan* plan, uint32_t n, int passes, uint32_t first_half, LocalPlan& L,
                                          uint32_t* wsum) {
    const uint32_t t = threadIdx.x, lane = t & 31u, warp = t >> 5;
    for (int p = 0; p < passes; ++p) {
        const uint32_t c = __ldcg(&plan->hist[p][t]);
        const int trivial = __syncthreads_or(c == n);
        uint32_t incl = c;
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            const uint32_t u = __shfl_up_sync(0xFFFFFFFFu, incl, off);
            if (lane >= off) incl += u;
        }
        if (lane == 31) wsum[warp] = incl;
        __syncthreads();
        uint32_t base = 0;
        for (uint32_t q = 0; q < warp; ++q) base += wsum[q];
        L.base[p][t] = base + incl - c;                        // exclusive base of digit t
        if (t == 0) L.active[p] = trivial ? 0u : 1u;
        __syncthreads();
    }
    if (t == 0) {
        uint32_t half = first_half;
        for (int p = 0; p < passes; ++p) {
            L.src_half[p] = half;
            if (L.active[p]) half ^= 1u;
        }
        L.sorted_half = half;
    }
    __syncthreads();
}

/* One tile of one radix pass, stable.  Warp wq of the tile owns entries [t0 + wq*SORT_SEG, +SORT_SEG) in order; within a
 * round of 32 the rank among equal digits comes from match.any, across rounds from a per-warp counter.  The tile publishes
 * its digit counts and obtains its offsets from the tiles before it by decoupled look-back (status: tiles x 256 words).
 * Tiles are dealt to the (co-resident) CTAs round-robin and each CTA takes its tiles in increasing order, so a tile only
 * ever waits for tiles that are done or running. */
template <int ITEMS>
__device__ __forceinline__ void pass_tile(const HalfPtrs& H, uint32_t n, int pass, int id_passes, uint32_t tile,
                                          const LocalPlan& L, uint32_t (*wcnt)[256], uint64_t* __restrict__ status,
                                          uint32_t epoch) {
    const uint32_t lane = threadIdx.x & 31u, wq = threadIdx.x >> 5;
    for (int i = threadIdx.x; i < SORT_WARPS * 256; i += SORT_THREADS) (&wcnt[0][0])[i] = 0;
    __syncthreads();
    const uint32_t src = L.src_half[pass];
    const uint64_t* __restrict__ sid = H.id[src];
    const uint32_t* __restrict__ sek = H.ek[src];
    uint64_t* __restrict__ did = H.id[src ^ 1u];
    uint32_t* __restrict__ dek = H.ek[src ^ 1u];

    const uint32_t base = tile * (SORT_THREADS * ITEMS) + wq * (32 * ITEMS);
    uint64_t kid[ITEMS];
    uint32_t kek[ITEMS], off[ITEMS];
    uint32_t* mine = wcnt[wq];
#pragma unroll
    for (int r = 0; r < ITEMS; ++r) {
        const uint32_t i = base + r * 32 + lane;
        const bool valid = i < n;
        kid[r] = valid ? __ldcg(sid + i) : 0;                   // written by other CTAs in the pass before: L2, not L1
        kek[r] = valid ? __ldcg(sek + i) : 0;
        const uint32_t dg = valid ? digit_of(kid[r], kek[r], pass, id_passes) : 255u;
        const uint32_t peers = __match_any_sync(0xFFFFFFFFu, dg);
        const uint32_t rank = __popc(peers & ((1u << lane) - 1u));
        const uint32_t before = mine[dg];
        __syncwarp();
        if (rank == 0) mine[dg] = before + __popc(peers);       // invalid lanes inflate digit 255 of the last tile only:
        __syncwarp();                                           // nothing is ranked after them
        off[r] = before + rank;
    }
    __syncthreads();
    {   /* thread t = digit t: tile count -> publish -> look back -> per-warp bases */
        const uint32_t t = threadIdx.x;
        uint32_t cnt = 0;
#pragma unroll
        for (int q = 0; q < SORT_WARPS; ++q) cnt += wcnt[q][t];
        uint64_t* my = status + (uint64_t)tile * 256 + t;
        uint32_t excl = 0;
        if (tile == 0) {
            st_status(my, status_word(epoch, FLAG_INC, cnt));
        } else {
            st_status(my, status_word(epoch, FLAG_AGG, cnt));
            /* LOOKBACK predecessors per step, fetched together: when a whole wave of tiles starts at once nobody has an
             * inclusive word yet and the walk is a chain of L2 round trips; the window divides its length */
            bool done = false;
            for (uint32_t j = tile; j > 0 && !done;) {
                const uint32_t m = j < (uint32_t)LOOKBACK ? j : (uint32_t)LOOKBACK;
                uint64_t w[LOOKBACK];
#pragma unroll
                for (int q = 0; q < LOOKBACK; ++q)
                    if ((uint32_t)q < m) w[q] = ld_status(status + (uint64_t)(j - 1 - q) * 256 + t);
#pragma unroll
                for (int q = 0; q < LOOKBACK; ++q) {
                    if ((uint32_t)q < m && !done) {
                        while ((uint32_t)(w[q] >> 34) != epoch || ((w[q] >> 32) & 3u) == 0)
                            w[q] = ld_status(status + (uint64_t)(j - 1 - q) * 256 + t);
                        excl += (uint32_t)w[q];
                        done = ((w[q] >> 32) & FLAG_INC) != 0;
                    }
                }
                j -= m;
            }
            st_status(my, status_word(epoch, FLAG_INC, excl + cnt));
        }
        uint32_t run = L.base[pass][t] + excl;
#pragma unroll
        for (int q = 0; q < SORT_WARPS; ++q) {
            const uint32_t c = wcnt[q][t];
            wcnt[q][t] = run;
            run += c;
        }
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < ITEMS; ++r) {
        const uint32_t i = base + r * 32 + lane;
        if (i < n) {
            const uint32_t dg = digit_of(kid[r], kek[r], pass, id_passes);
            const uint32_t dst = mine[dg] + off[r];
            did[dst] = kid[r];
            dek[dst] = kek[r];
        }
    }
    __syncthreads();                                            // wcnt is reused by the CTA's next tile
}

/* ---- duplicate removal on the sorted list ------------------------------------------------------------------------ */

/* One tile: each thread owns ITEMS consecutive entries; block scan of the per-thread counts of "first of its id"
 * flags; the tile's offset comes from a look-back over the tile totals (ustatus: one word per tile). */
template <int ITEMS>
__device__ __forceinline__ void uniq_tile(const HalfPtrs& H, uint32_t n, uint32_t tile, uint32_t tiles, const LocalPlan& L,
                                          SortPlan* plan, uint32_t* wsum, uint32_t* s_excl, uint64_t* __restrict__ ustatus,
                                          uint32_t epoch) {
    const uint32_t src = L.sorted_half;
    const uint64_t* __restrict__ sid = H.id[src];
    const uint32_t* __restrict__ sek = H.ek[src];
    uint64_t* __restrict__ did = H.id[src ^ 1u];
    uint32_t* __restrict__ dek = H.ek[src ^ 1u];
    const uint32_t first = tile * (SORT_THREADS * ITEMS) + threadIdx.x * ITEMS;
    uint64_t v[ITEMS];
    uint64_t prev = (first > 0 && first <= n) ? __ldcg(sid + first - 1) : 0;
    uint32_t flags = 0, c = 0;
#pragma unroll
    for (int r = 0; r < ITEMS; ++r) {
        const uint32_t i = first + r;
        v[r] = i < n ? __ldcg(sid + i) : 0;
        if (i < n && (i == 0 || v[r] != prev)) { flags |= 1u << r; ++c; }
        prev = v[r];
    }
    const uint32_t lane = threadIdx.x & 31u, wq = threadIdx.x >> 5;
    uint32_t incl = c;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
        const uint32_t u = __shfl_up_sync(0xFFFFFFFFu, incl, off);
        if (lane >= off) incl += u;
    }
    if (lane == 31) wsum[wq] = incl;
    __syncthreads();
    uint32_t wbase = 0, total = 0;
    for (uint32_t q = 0; q < SORT_WARPS; ++q) { if (q < wq) wbase += wsum[q]; total += wsum[q]; }
    if (threadIdx.x == 0) {
        uint32_t excl = 0;
        if (tile == 0) {
            st_status(ustatus, status_word(epoch, FLAG_INC, total));
        } else {
            st_status(ustatus + tile, status_word(epoch, FLAG_AGG, total));
            bool done = false;
            for (uint32_t j = tile; j > 0 && !done;) {
                const uint32_t m = j < (uint32_t)LOOKBACK ? j : (uint32_t)LOOKBACK;
                uint64_t w[LOOKBACK];
#pragma unroll
                for (int q = 0; q < LOOKBACK; ++q)
                    if ((uint32_t)q < m) w[q] = ld_status(ustatus + (j - 1 - q));
#pragma unroll
                for (int q = 0; q < LOOKBACK; ++q) {
                    if ((uint32_t)q < m && !done) {
                        while ((uint32_t)(w[q] >> 34) != epoch || ((w[q] >> 32) & 3u) == 0) w[q] = ld_status(ustatus + (j - 1 - q));
                        excl += (uint32_t)w[q];
                        done = ((w[q] >> 32) & FLAG_INC) != 0;
                    }
                }
                j -= m;
            }
            st_status(ustatus + tile, status_word(epoch, FLAG_INC, excl + total));
        }
        *s_excl = excl;
        if (tile == tiles - 1) plan->uniq_total = excl + total;
    }
    __syncthreads();
    uint32_t dst = *s_excl + wbase + incl - c;
#pragma unroll
    for (int r = 0; r < ITEMS; ++r) {
        if (flags & (1u << r)) {
            did[dst] = v[r];
            dek[dst] = __ldcg(sek + first + r);
            ++dst;
        }
    }
    __syncthreads();                                            // wsum / s_excl are reused by the CTA's next tile
}

/* One thread.  The m unique sorted entries are in half `half`.  Fixes the new tau and the number of entries kept. */
__device__ __forceinline__ void cut_list(const HalfPtrs& H, uint32_t half, uint32_t m, ScanState* st, uint64_t k_max,
                                         int32_t thr_min) {
    const uint32_t* __restrict__ ek = H.ek[half];
    int32_t tau_k;
    if (k_max == 0) tau_k = INT32_MAX;                       // no top-k asked: only thr_min bounds tau
    else tau_k = (m >= k_max) ? key_to_est(__ldcg(ek + k_max - 1)) : INT32_MIN;
    int32_t tau = min(tau_k, thr_min);
    tau = max(tau, st->tau);
    /* entries are ordered by estimate descending: keep the prefix with est >= tau, i.e. key <= key(tau) */
    const uint32_t key_tau = est_to_key(tau);
    uint32_t lo = 0, hi = m;                                 // first index with key > key_tau
    while (lo < hi) {
        uint32_t mid = lo + (hi - lo) / 2;
        if (__ldcg(ek + mid) <= key_tau) lo = mid + 1; else hi = mid;
    }
    st->uniq = m;
    st->count = lo;
    st->tau = tau;
    st->est_max = lo ? key_to_est(__ldcg(ek)) : INT32_MIN;
    st->est_min = lo ? key_to_est(__ldcg(ek + lo - 1)) : INT32_MAX;
    st->half = half;
}

/* The empty list: nothing to sort, tau = max(tau, min(INT32_MIN or INT32_MAX, thr_min)) as for any other list. */
__global__ void k_cut_empty(const __grid_constant__ HalfPtrs H, uint32_t half, ScanState* st, uint64_t k_max, int32_t thr_min) {
    cut_list(H, half, 0u, st, k_max, thr_min);
}

/* One list of a launch of k_compact and the CTAs [cta0, cta0 + ctas) of the grid that work on it. */
struct CompactList {
    HalfPtrs H;
    uint32_t n, first_half;
    int id_passes, passes;
    SortPlan* plan;
    uint64_t* status;
    uint64_t* ustatus;
    uint32_t epoch0;
    ScanState* st;
    uint32_t cta0, ctas;
};
struct CompactBatch {
    int n_lists, max_passes;
    uint64_t k_max;
    int32_t thr_min;
    CompactList L[CS_MAX_SCALES];
};

/* The compaction of up to CS_MAX_SCALES lists in one cooperative launch (all CTAs co-resident; grid-wide barriers between
 * the phases), each list on its own share of the grid:
 *   digit histograms of all passes | plan | one sweep per needed digit | duplicate removal | cut | plan zeroed again
 * With one list a pass that no entry needs is skipped with its barrier; with several, every CTA takes the barriers of
 * max_passes passes (the lists need different ones). */
template <bool MULTI, int ITEMS>
__global__ void __launch_bounds__(SORT_THREADS, 4)
k_compact(const __grid_constant__ CompactBatch B) {
    __shared__ LocalPlan L;
    __shared__ uint32_t wcnt[SORT_WARPS][256];
    __shared__ uint32_t wsum[SORT_WARPS];
    __shared__ uint32_t s_excl;
    cg::grid_group grid = cg::this_grid();
    int li = 0;
    if (MULTI)
        while (li + 1 < B.n_lists && blockIdx.x >= B.L[li].cta0 + B.L[li].ctas) ++li;
    const CompactList& M = B.L[li];                           // one list: a static index, operands straight from the constant bank
    const uint32_t bid = blockIdx.x - M.cta0, nct = M.ctas;
    const uint32_t n = M.n, tiles = (n + SORT_THREADS * ITEMS - 1) / (SORT_THREADS * ITEMS);

    hist_sweep(M.H.id[M.first_half], M.H.ek[M.first_half], n, M.id_passes, M.passes, L, M.plan, bid, nct);
    grid.sync();
    make_plan(M.plan, n, M.passes, M.first_half, L, wsum);
    for (int p = 0; p < B.max_passes; ++p) {
        const bool mine = p < M.passes && L.active[p];
        if (!MULTI && !mine) continue;
        if (mine)
            for (uint32_t tile = bid; tile < tiles; tile += nct)
                pass_tile<ITEMS>(M.H, n, p, M.id_passes, tile, L, wcnt, M.status, (M.epoch0 + (uint32_t)p) & 0x3FFFFFFFu);
        grid.sync();
    }
    for (uint32_t tile = bid; tile < tiles; tile += nct)
        uniq_tile<ITEMS>(M.H, n, tile, tiles, L, M.plan, wsum, &s_excl, M.ustatus, (M.epoch0 + (uint32_t)M.passes) & 0x3FFFFFFFu);
    grid.sync();
    if (bid == 0) {
        if (threadIdx.x == 0) cut_list(M.H, L.sorted_half ^ 1u, __ldcg(&M.plan->uniq_total), M.st, B.k_max, B.thr_min);
        __syncthreads();
        for (int i = threadIdx.x; i < M.passes * 256; i += SORT_THREADS) (&M.plan->hist[0][0])[i] = 0;   // for the next compaction
        if (threadIdx.x == 0) M.plan->uniq_total = 0;
    }
}

__global__ void __launch_bounds__(256)
k_emit(const uint64_t* __restrict__ id, const uint32_t* __restrict__ ek, uint32_t n, uint64_t* __restrict__ ids_out,
       int32_t* __restrict__ est_out) {
    uint32_t i = blockIdx.x * 256 + threadIdx.x;
    if (i < n) {
        ids_out[i] = id[i];
        est_out[i] = key_to_est(ek[i]);
    }
}

/* *n_out = number of leading entries with estimate >= thr (list sorted by key ascending) */
__global__ void k_count_ge(const uint32_t* __restrict__ ek, uint32_t n, int32_t thr, uint32_t* n_out) {
    const uint32_t key_thr = est_to_key(thr);
    uint32_t lo = 0, hi = n;
    while (lo < hi) {
        uint32_t mid = lo + (hi - lo) / 2;
        if (ek[mid] <= key_thr) lo = mid + 1; else hi = mid;
    }
    *n_out = lo;
}

/* ---- host orchestration ----------------------------------------------------------------------------------- */

static uint32_t tiles_of(uint64_t n, int items = SORT_ITEMS) {
    const uint64_t tile = (uint64_t)SORT_THREADS * items;
    return (uint32_t)((n + tile - 1) / tile);
}

/* scratch layout (uint32 words): SortPlan | status[rows][256] (u64) | ustatus[rows] (u64); rows: the long tiles of a full
 * buffer, or the short tiles of the longest list that is sorted with short tiles */
static uint64_t plan_words() { return (sizeof(SortPlan) + 15) / 16 * 4; }
static uint64_t status_rows(uint64_t cap) {
    const uint64_t t = tiles_of(cap);
    return (t > SHORT_TILES_MAX ? t : SHORT_TILES_MAX) + 1;
}
uint64_t select_scratch_words(uint64_t n) {
    const uint64_t t = status_rows(n);
    return plan_words() + t * 256 * 2 + t * 2 + 16;
}

/* CTAs of k_compact that fit on the current device at once (the bound of a cooperative launch). */
static cudaError_t resident_ctas(uint32_t* out) {
    static std::atomic<uint32_t> cached[64];
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    uint32_t v = dev < 64 ? cached[dev].load(std::memory_order_relaxed) : 0u;
    if (!v) {
        int per_sm = 1 << 30, sms = 0;
        const void* fns[4] = {(const void*)k_compact<false, SORT_ITEMS>, (const void*)k_compact<true, SORT_ITEMS>,
                              (const void*)k_compact<false, SORT_ITEMS_SHORT>, (const void*)k_compact<true, SORT_ITEMS_SHORT>};
        for (int f = 0; f < 4; ++f) {                        /* one bound for all forms of the kernel */
            int x = 0;
            e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&x, fns[f], SORT_THREADS, 0);
            if (e != cudaSuccess) return e;
            if (x < per_sm) per_sm = x;
        }
        e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) return e;
        v = (uint32_t)(per_sm * sms);
        if (!v) return cudaErrorLaunchOutOfResources;
        if (dev < 64) cached[dev].store(v, std::memory_order_relaxed);
    }
    *out = v;
    return cudaSuccess;
}

/* Shares the grid among the lists of a batch (in proportion to their tiles, at least one CTA each, at most `budget` in
 * all) and launches k_compact.  k_compact works with any share that is resident at once (tiles are dealt round-robin).
 * Where fewer CTAs fit than the occupancy calculation says (a context restricted to part of the SMs), the launch is
 * refused: halve the budget and retry. */
static cudaError_t launch_batch(CompactBatch& cb, cudaStream_t stream, bool allow_short) {
    uint32_t budget = 0;
    cudaError_t e = resident_ctas(&budget);
    if (e != cudaSuccess) return e;
    for (;;) {
        /* short tiles when every one of them gets a CTA of its own in this launch */
        uint64_t total_short = 0;
        for (int i = 0; i < cb.n_lists; ++i) total_short += tiles_of(cb.L[i].n, SORT_ITEMS_SHORT);
        const bool use_short = allow_short && total_short <= budget && total_short <= SHORT_TILES_MAX;
        const int items = use_short ? SORT_ITEMS_SHORT : SORT_ITEMS;
        uint64_t total = 0;
        for (int i = 0; i < cb.n_lists; ++i) total += tiles_of(cb.L[i].n, items);
        uint32_t at = 0;
        for (int i = 0; i < cb.n_lists; ++i) {
            const uint32_t t = tiles_of(cb.L[i].n, items);
            uint32_t c = total <= budget ? t : (uint32_t)((uint64_t)budget * t / total);
            if (c > t) c = t;
            if (c < 1) c = 1;
            cb.L[i].cta0 = at;
            cb.L[i].ctas = c;
            at += c;
        }
        void* args[] = {&cb};
        const void* fn = cb.n_lists > 1
            ? (use_short ? (const void*)k_compact<true, SORT_ITEMS_SHORT> : (const void*)k_compact<true, SORT_ITEMS>)
            : (use_short ? (const void*)k_compact<false, SORT_ITEMS_SHORT> : (const void*)k_compact<false, SORT_ITEMS>);
        e = cudaLaunchCooperativeKernel(fn, dim3(at), dim3(SORT_THREADS), args, 0, stream);
        if (e != cudaErrorCooperativeLaunchTooLarge || budget <= (uint32_t)cb.n_lists) return e;
        cudaGetLastError();
        budget /= 2;
    }
}

cudaError_t select_compact_batch(const CompactRequest* req, int count, uint32_t cap, uint64_t k_max, int32_t thr_min,
                                 cudaStream_t stream, uint64_t* launches) {
    if (count < 0 || count > CS_MAX_SCALES) return cudaErrorInvalidValue;
    CompactBatch cb;
    cb.n_lists = 0; cb.max_passes = 0; cb.k_max = k_max; cb.thr_min = thr_min;
    for (int r = 0; r < count; ++r) {
        const CompactRequest& q = req[r];
        HalfPtrs H;
        for (int h = 0; h < 2; ++h) { H.id[h] = q.B->id[h]; H.ek[h] = q.B->ek[h]; }
        if (q.n == 0) {
            k_cut_empty<<<1, 1, 0, stream>>>(H, (uint32_t)q.src, q.st_dev, k_max, thr_min);
            *launches += 1;
            cudaError_t e = cudaGetLastError();
            if (e != cudaSuccess) return e;
            continue;
        }
        if (*q.epoch >= 0x3FFFFFFFu - 2u * MAX_PASSES) {     /* epochs are 30 bits wide: before they repeat, forget every */
            cudaError_t e = cudaMemsetAsync(q.B->scratch, 0, (size_t)select_scratch_words(cap) * sizeof(uint32_t), stream);
            if (e != cudaSuccess) return e;                  /* word written */
            *q.epoch = 0;
        }
        CompactList& M = cb.L[cb.n_lists++];
        M.H = H;
        M.n = q.n;
        M.first_half = (uint32_t)q.src;
        M.id_passes = (q.id_bits + 7) / 8;
        M.passes = M.id_passes + 4;
        M.plan = reinterpret_cast<SortPlan*>(q.B->scratch);
        M.status = reinterpret_cast<uint64_t*>(q.B->scratch + plan_words());
        M.ustatus = M.status + status_rows(cap) * 256;
        M.epoch0 = *q.epoch + 1;
        *q.epoch += (uint32_t)M.passes + 1;                  /* one epoch per look-back sweep: the passes, then uniq's */
        M.st = q.st_dev;
        if (M.passes > cb.max_passes) cb.max_passes = M.passes;
    }
    if (cb.n_lists == 0) return cudaSuccess;
    *launches += 1;
    return launch_batch(cb, stream, true);
}

/* Enqueues one compaction of the first n entries of half `src` (one launch on `stream`, no synchronisation).  Afterwards
 * st_dev->half names the half that holds the list and st_dev->count its length.  *epoch: per-buffer sweep counter. */
cudaError_t select_compact(const SelectBuffers& B, uint32_t cap, int src, uint32_t n, int id_bits, ScanState* st_dev,
                           uint64_t k_max, int32_t thr_min, cudaStream_t stream, uint64_t* launches, uint32_t* epoch) {
    const CompactRequest q = {&B, src, n, id_bits, st_dev, epoch};
    return select_compact_batch(&q, 1, cap, k_max, thr_min, stream, launches);
}

/* ---- allocation-free selection over a caller's candidate list (cs_select_static, include/cs.h) -------------------------
 * Everything a compaction needs -- both halves of the ping-pong list, the plan, the look-back status words, the scan
 * state -- sits in one file-scope device array of fixed size; every GPU that loads the library holds it until exit.
 * In host code `g_static_scratch` is only the symbol's host-side stand-in: its device address comes from
 * cudaGetSymbolAddress, once per device, and that address is what the kernels are given. */
constexpr uint32_t STATIC_TILES = SELECT_STATIC_MAX_N / SORT_TILE;
struct StaticScratch {
    uint64_t id[2][SELECT_STATIC_MAX_N];
    uint32_t ek[2][SELECT_STATIC_MAX_N];
    SortPlan plan;
    uint64_t status[(STATIC_TILES + 1) * 256];
    uint64_t ustatus[STATIC_TILES + 1];
    ScanState st;
};
static_assert(SELECT_STATIC_MAX_N % SORT_TILE == 0, "whole tiles");
static __device__ __align__(256) unsigned char g_static_scratch[sizeof(StaticScratch)];

/* Caller's (id, estimate) pairs -> half 0 as (id, key); what must start at zero is cleared: the array keeps the last
 * call's contents (digit counts if that call was cut short, status words of its epochs, its scan state). */
__global__ void __launch_bounds__(256)
k_static_load(StaticScratch* S, const uint64_t* __restrict__ ids, const int32_t* __restrict__ est, uint32_t n, uint32_t tiles) {
    const uint32_t stride = gridDim.x * 256u, t0 = blockIdx.x * 256u + threadIdx.x;
    for (uint32_t i = t0; i < n; i += stride) {
        S->id[0][i] = ids[i];
        S->ek[0][i] = est_to_key(est[i]);
    }
    for (uint32_t i = t0; i < MAX_PASSES * 256u; i += stride) (&S->plan.hist[0][0])[i] = 0;
    for (uint32_t i = t0; i < (tiles + 1) * 256u; i += stride) S->status[i] = 0;
    for (uint32_t i = t0; i <= tiles; i += stride) S->ustatus[i] = 0;
    if (t0 == 0) {
        S->plan.uniq_total = 0;
        S->st.count = 0; S->st.tau = INT32_MIN; S->st.est_min = INT32_MAX; S->st.est_max = INT32_MIN;
        S->st.uniq = 0; S->st.half = 0;
    }
}

/* First min(k, kept) entries of the list k_compact left -> the caller's arrays. */
__global__ void __launch_bounds__(256)
k_static_emit(const StaticScratch* S, uint32_t k, uint64_t* __restrict__ ids_out, int32_t* __restrict__ est_out,
              uint32_t* __restrict__ n_out) {
    const uint32_t half = S->st.half, kept = S->st.count < k ? S->st.count : k;
    for (uint32_t i = blockIdx.x * 256u + threadIdx.x; i < kept; i += gridDim.x * 256u) {
        ids_out[i] = S->id[half][i];
        est_out[i] = key_to_est(S->ek[half][i]);
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) *n_out = kept;
}

/* Device address of the scratch array on the current device (looked up once per device, with that device current). */
static cudaError_t static_scratch(StaticScratch** out) {
    static std::atomic<StaticScratch*> cached[64];
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    StaticScratch* ptr = (dev >= 0 && dev < 64) ? cached[dev].load(std::memory_order_acquire) : nullptr;
    if (!ptr) {
        e = cudaGetSymbolAddress((void**)&ptr, g_static_scratch);
        if (e != cudaSuccess) return e;
        if (!ptr) return cudaErrorInvalidSymbol;
        if (dev >= 0 && dev < 64) cached[dev].store(ptr, std::memory_order_release);
    }
    *out = ptr;
    return cudaSuccess;
}

cudaError_t select_static(const uint64_t* ids, const int32_t* est, uint32_t n, uint32_t k, uint64_t* ids_out, int32_t* est_out,
                          uint32_t* n_out, cudaStream_t stream) {
    StaticScratch* S = nullptr;
    cudaError_t e = static_scratch(&S);
    if (e != cudaSuccess) return e;
    const uint32_t tiles = tiles_of(n);
    k_static_load<<<tiles ? tiles : 1, 256, 0, stream>>>(S, ids, est, n, tiles);
    if (n) {
        CompactBatch cb;
        cb.n_lists = 1; cb.max_passes = MAX_PASSES; cb.k_max = k; cb.thr_min = INT32_MAX;
        CompactList& M = cb.L[0];
        for (int h = 0; h < 2; ++h) { M.H.id[h] = S->id[h]; M.H.ek[h] = S->ek[h]; }
        M.n = n; M.first_half = 0;
        M.id_passes = 8; M.passes = MAX_PASSES;               /* every id byte; constant digits are skipped on the device */
        M.plan = &S->plan; M.status = S->status; M.ustatus = S->ustatus;
        M.epoch0 = 1;                                         /* the status words were just zeroed: epoch 0 = not published */
        M.st = &S->st;
        e = launch_batch(cb, stream, false);              /* the static status words cover long tiles only */
        if (e != cudaSuccess) return e;
    }
    const uint32_t eb = (k + 255u) / 256u;
    k_static_emit<<<eb ? (eb < 256u ? eb : 256u) : 1, 256, 0, stream>>>(S, k, ids_out, est_out, n_out);
    return cudaGetLastError();
}

cudaError_t launch_emit_prefix(const uint64_t* id, const uint32_t* ek, uint32_t n, uint64_t* ids_out,
                               int32_t* est_out, cudaStream_t st) {
    if (!n) return cudaSuccess;
    k_emit<<<(n + 255) / 256, 256, 0, st>>>(id, ek, n, ids_out, est_out);
    return cudaGetLastError();
}

cudaError_t launch_count_ge(const uint32_t* ek, uint32_t n, int32_t thr, uint32_t* n_out_dev, cudaStream_t st) {
    k_count_ge<<<1, 1, 0, st>>>(ek, n, thr, n_out_dev);
    return cudaGetLastError();
}

}  // namespace cs
