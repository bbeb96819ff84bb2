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
 * One compaction = a fixed sequence of launches, with no host round trip in it:
 *   k_radix_hist   digit histograms of ALL passes in one sweep over the list
 *   k_radix_plan   one block: which passes are needed (a digit that is the same in every entry is skipped on the device:
 *                  the high bytes of the estimate key almost always are), exclusive digit bases, ping-pong plan
 *   k_radix_pass   one launch per digit: every tile ranks its entries (warp match.any + per-warp digit counters, stable),
 *                  publishes its digit counts and obtains its offsets from the tiles before it by decoupled look-back
 *                  (tiles take tickets in order, so a tile only ever waits for tiles that already run)
 *   k_uniq         drops duplicate ids, again with a look-back over tile totals
 *   k_cut          fixes the new tau and the number of entries kept, records which half of the ping-pong buffers holds
 *                  the list (the host learns it when it next reads the scan states)
 */
#include "cs_device.cuh"

namespace cs {

constexpr int SORT_THREADS = 256;
constexpr int SORT_WARPS = SORT_THREADS / 32;
constexpr int SORT_ITEMS = 8;                              // items per lane
constexpr int SORT_TILE = SORT_THREADS * SORT_ITEMS;       // 2048 entries per block
constexpr int SORT_SEG = 32 * SORT_ITEMS;                  // consecutive entries owned by one warp
constexpr int MAX_PASSES = 12;                             // 8 id bytes (ids < 2^60 need 8) + 4 estimate-key bytes

/* Device-side plan of one compaction; lives at the start of SelectBuffers::scratch, zeroed before every compaction. */
struct SortPlan {
    uint32_t hist[MAX_PASSES][256];    // digit counts; k_radix_plan turns them into exclusive bases
    uint32_t active[MAX_PASSES];       // 0: every entry has the same digit in this pass -> nothing to do
    uint32_t src_half[MAX_PASSES];     // which half (0/1) pass p reads
    uint32_t ticket[MAX_PASSES + 1];   // tile tickets per pass, last = k_uniq
    uint32_t sorted_half;              // half that holds the sorted list
    uint32_t uniq_total;               // unique entries
    uint32_t pad[2];
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

/* hist[p][digit] += entries of the list with that digit in pass p, for all passes at once */
__global__ void __launch_bounds__(SORT_THREADS)
k_radix_hist(const uint64_t* __restrict__ id, const uint32_t* __restrict__ ek, uint32_t n, int id_passes, int passes,
             SortPlan* plan) {
    __shared__ uint32_t h[MAX_PASSES][256];
    for (int i = threadIdx.x; i < passes * 256; i += SORT_THREADS) (&h[0][0])[i] = 0;
    __syncthreads();
    const uint32_t stride = gridDim.x * SORT_THREADS;
    for (uint32_t i = blockIdx.x * SORT_THREADS + threadIdx.x; i < n; i += stride) {
        const uint64_t c = id[i];
        const uint32_t k = ek[i];
        for (int p = 0; p < passes; ++p) atomicAdd(&h[p][digit_of(c, k, p, id_passes)], 1u);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < passes * 256; i += SORT_THREADS) {
        const uint32_t v = (&h[0][0])[i];
        if (v) atomicAdd(&plan->hist[0][0] + i, v);
    }
}

/* One block of 256 threads: thread t = digit t. */
__global__ void __launch_bounds__(256) k_radix_plan(SortPlan* plan, uint32_t n, int passes, uint32_t first_half) {
    __shared__ uint32_t wsum[8];
    __shared__ uint32_t s_active[MAX_PASSES];
    const uint32_t t = threadIdx.x, lane = t & 31u, warp = t >> 5;
    for (int p = 0; p < passes; ++p) {
        const uint32_t c = plan->hist[p][t];
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
        plan->hist[p][t] = base + incl - c;                    // exclusive base of digit t
        if (t == 0) s_active[p] = trivial ? 0u : 1u;
        __syncthreads();
    }
    if (t == 0) {
        uint32_t half = first_half;
        for (int p = 0; p < passes; ++p) {
            plan->active[p] = s_active[p];
            plan->src_half[p] = half;
            if (s_active[p]) half ^= 1u;
        }
        plan->sorted_half = half;
    }
}

/* One radix pass, stable.  Warp wq of a tile owns entries [t0 + wq*SORT_SEG, +SORT_SEG) in order; within a round of 32
 * the rank among equal digits comes from match.any, across rounds from a per-warp counter.  status: tiles x 256 words. */
__global__ void __launch_bounds__(SORT_THREADS)
k_radix_pass(const __grid_constant__ HalfPtrs H, uint32_t n, int pass, int id_passes, SortPlan* plan,
             uint64_t* __restrict__ status, uint32_t epoch) {
    if (!plan->active[pass]) return;
    __shared__ uint32_t wcnt[SORT_WARPS][256];
    __shared__ uint32_t s_tile;
    const uint32_t lane = threadIdx.x & 31u, wq = threadIdx.x >> 5;
    if (threadIdx.x == 0) s_tile = atomicAdd(&plan->ticket[pass], 1u);
    for (int i = threadIdx.x; i < SORT_WARPS * 256; i += SORT_THREADS) (&wcnt[0][0])[i] = 0;
    __syncthreads();
    const uint32_t tile = s_tile;
    const uint32_t src = plan->src_half[pass];
    const uint64_t* __restrict__ sid = H.id[src];
    const uint32_t* __restrict__ sek = H.ek[src];
    uint64_t* __restrict__ did = H.id[src ^ 1u];
    uint32_t* __restrict__ dek = H.ek[src ^ 1u];

    const uint32_t base = tile * SORT_TILE + wq * SORT_SEG;
    uint64_t kid[SORT_ITEMS];
    uint32_t kek[SORT_ITEMS], off[SORT_ITEMS];
    uint32_t* mine = wcnt[wq];
#pragma unroll
    for (int r = 0; r < SORT_ITEMS; ++r) {
        const uint32_t i = base + r * 32 + lane;
        const bool valid = i < n;
        kid[r] = valid ? sid[i] : 0;
        kek[r] = valid ? sek[i] : 0;
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
            for (uint32_t j = tile; j-- > 0;) {
                const uint64_t* theirs = status + (uint64_t)j * 256 + t;
                uint64_t w;
                do { w = ld_status(theirs); } while ((uint32_t)(w >> 34) != epoch || ((w >> 32) & 3u) == 0);
                excl += (uint32_t)w;
                if ((w >> 32) & FLAG_INC) break;
            }
            st_status(my, status_word(epoch, FLAG_INC, excl + cnt));
        }
        uint32_t run = plan->hist[pass][t] + excl;
#pragma unroll
        for (int q = 0; q < SORT_WARPS; ++q) {
            const uint32_t c = wcnt[q][t];
            wcnt[q][t] = run;
            run += c;
        }
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < SORT_ITEMS; ++r) {
        const uint32_t i = base + r * 32 + lane;
        if (i < n) {
            const uint32_t dg = digit_of(kid[r], kek[r], pass, id_passes);
            const uint32_t dst = mine[dg] + off[r];
            did[dst] = kid[r];
            dek[dst] = kek[r];
        }
    }
}

/* ---- duplicate removal on the sorted list ------------------------------------------------------------------------ */

/* Each thread owns SORT_ITEMS consecutive entries; block scan of the per-thread counts of "first of its id" flags; the
 * tile's offset comes from a look-back over the tile totals (ustatus: one word per tile). */
__global__ void __launch_bounds__(SORT_THREADS)
k_uniq(const __grid_constant__ HalfPtrs H, uint32_t n, SortPlan* plan, uint64_t* __restrict__ ustatus, uint32_t epoch,
       uint32_t tiles) {
    __shared__ uint32_t wsum[SORT_WARPS];
    __shared__ uint32_t s_tile, s_excl;
    if (threadIdx.x == 0) s_tile = atomicAdd(&plan->ticket[MAX_PASSES], 1u);
    __syncthreads();
    const uint32_t tile = s_tile;
    const uint32_t src = plan->sorted_half;
    const uint64_t* __restrict__ sid = H.id[src];
    const uint32_t* __restrict__ sek = H.ek[src];
    uint64_t* __restrict__ did = H.id[src ^ 1u];
    uint32_t* __restrict__ dek = H.ek[src ^ 1u];
    const uint32_t first = tile * SORT_TILE + threadIdx.x * SORT_ITEMS;
    uint64_t v[SORT_ITEMS];
    uint64_t prev = (first > 0 && first <= n) ? sid[first - 1] : 0;
    uint32_t flags = 0, c = 0;
#pragma unroll
    for (int r = 0; r < SORT_ITEMS; ++r) {
        const uint32_t i = first + r;
        v[r] = i < n ? sid[i] : 0;
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
            for (uint32_t j = tile; j-- > 0;) {
                uint64_t w;
                do { w = ld_status(ustatus + j); } while ((uint32_t)(w >> 34) != epoch || ((w >> 32) & 3u) == 0);
                excl += (uint32_t)w;
                if ((w >> 32) & FLAG_INC) break;
            }
            st_status(ustatus + tile, status_word(epoch, FLAG_INC, excl + total));
        }
        s_excl = excl;
        if (tile == tiles - 1) plan->uniq_total = excl + total;
    }
    __syncthreads();
    uint32_t dst = s_excl + wbase + incl - c;
#pragma unroll
    for (int r = 0; r < SORT_ITEMS; ++r) {
        if (flags & (1u << r)) {
            did[dst] = v[r];
            dek[dst] = sek[first + r];
            ++dst;
        }
    }
}

/* One thread.  The m unique sorted entries are in half `half` (or, with plan != NULL, in the half k_uniq wrote: the one
 * opposite to plan->sorted_half, m = plan->uniq_total).  Fixes the new tau and the number of entries kept. */
__global__ void k_cut(const __grid_constant__ HalfPtrs H, const SortPlan* plan, uint32_t half_const, ScanState* st,
                      uint64_t k_max, int32_t thr_min) {
    const uint32_t half = plan ? (plan->sorted_half ^ 1u) : half_const;
    const uint32_t m = plan ? plan->uniq_total : 0u;
    const uint32_t* __restrict__ ek = H.ek[half];
    int32_t tau_k;
    if (k_max == 0) tau_k = INT32_MAX;                       // no top-k asked: only thr_min bounds tau
    else tau_k = (m >= k_max) ? key_to_est(ek[k_max - 1]) : INT32_MIN;
    int32_t tau = min(tau_k, thr_min);
    tau = max(tau, st->tau);
    /* entries are ordered by estimate descending: keep the prefix with est >= tau, i.e. key <= key(tau) */
    const uint32_t key_tau = est_to_key(tau);
    uint32_t lo = 0, hi = m;                                 // first index with key > key_tau
    while (lo < hi) {
        uint32_t mid = lo + (hi - lo) / 2;
        if (ek[mid] <= key_tau) lo = mid + 1; else hi = mid;
    }
    st->uniq = m;
    st->count = lo;
    st->tau = tau;
    st->est_max = lo ? key_to_est(ek[0]) : INT32_MIN;
    st->est_min = lo ? key_to_est(ek[lo - 1]) : INT32_MAX;
    st->half = half;
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

static uint32_t tiles_of(uint64_t n) { return (uint32_t)((n + SORT_TILE - 1) / SORT_TILE); }

/* scratch layout (uint32 words): SortPlan | status[tiles][256] (u64) | ustatus[tiles] (u64) */
static uint64_t plan_words() { return (sizeof(SortPlan) + 15) / 16 * 4; }
uint64_t select_scratch_words(uint64_t n) {
    const uint64_t t = tiles_of(n) + 1;
    return plan_words() + t * 256 * 2 + t * 2 + 16;
}

/* Enqueues one compaction of the first n entries of half `src` (all on `stream`, no synchronisation).  Afterwards
 * st_dev->half names the half that holds the list and st_dev->count its length.  *epoch: per-buffer launch counter. */
cudaError_t select_compact(const SelectBuffers& B, uint32_t cap, int src, uint32_t n, int id_bits, ScanState* st_dev,
                           uint64_t k_max, int32_t thr_min, cudaStream_t stream, uint64_t* launches, uint32_t* epoch) {
    HalfPtrs H;
    for (int h = 0; h < 2; ++h) { H.id[h] = B.id[h]; H.ek[h] = B.ek[h]; }
    if (n == 0) {
        k_cut<<<1, 1, 0, stream>>>(H, nullptr, (uint32_t)src, st_dev, k_max, thr_min);
        *launches += 1;
        return cudaGetLastError();
    }
    SortPlan* plan = reinterpret_cast<SortPlan*>(B.scratch);
    uint64_t* status = reinterpret_cast<uint64_t*>(B.scratch + plan_words());
    uint64_t* ustatus = status + (uint64_t)(tiles_of(cap) + 1) * 256;
    const uint32_t tiles = tiles_of(n);
    const int id_passes = (id_bits + 7) / 8, passes = id_passes + 4;
    cudaError_t e = cudaMemsetAsync(plan, 0, sizeof(SortPlan), stream);
    if (e != cudaSuccess) return e;
    uint32_t hb = tiles < 148u * 8u ? tiles : 148u * 8u;
    k_radix_hist<<<hb, SORT_THREADS, 0, stream>>>(B.id[src], B.ek[src], n, id_passes, passes, plan);
    k_radix_plan<<<1, 256, 0, stream>>>(plan, n, passes, (uint32_t)src);
    for (int p = 0; p < passes; ++p) {
        *epoch += 1;
        k_radix_pass<<<tiles, SORT_THREADS, 0, stream>>>(H, n, p, id_passes, plan, status, *epoch & 0x3FFFFFFFu);
    }
    *epoch += 1;
    k_uniq<<<tiles, SORT_THREADS, 0, stream>>>(H, n, plan, ustatus, *epoch & 0x3FFFFFFFu, tiles);
    k_cut<<<1, 1, 0, stream>>>(H, plan, 0u, st_dev, k_max, thr_min);
    *launches += 4 + passes;
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
