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
 * Kernels: k_hist (per-tile digit counts), k_exscan (single-block exclusive scan), k_scatter (stable
 * scatter: warp match.any ranks + per-warp digit counters), k_uniq_count / k_uniq_scatter, k_cut, k_emit.
 */
#include "cs_device.cuh"

namespace cs {

constexpr int SORT_THREADS = 256;
constexpr int SORT_WARPS = SORT_THREADS / 32;
constexpr int SORT_ITEMS = 8;                              // items per lane
constexpr int SORT_TILE = SORT_THREADS * SORT_ITEMS;       // 2048 entries per block
constexpr int SORT_SEG = 32 * SORT_ITEMS;                  // consecutive entries owned by one warp

__device__ __forceinline__ uint32_t digit_of(uint64_t id, uint32_t ek, int from_ek, int shift, uint32_t ek_base) {
    return from_ek ? (((ek - ek_base) >> shift) & 255u) : ((uint32_t)(id >> shift) & 255u);
}

/* counts[digit * nblocks + block] = number of entries of this block's tile with that digit */
__global__ void __launch_bounds__(SORT_THREADS)
k_hist(const uint64_t* __restrict__ id, const uint32_t* __restrict__ ek, uint32_t n, int from_ek, int shift,
       uint32_t ek_base, uint32_t* __restrict__ counts, uint32_t nblocks) {
    __shared__ uint32_t h[256];
    h[threadIdx.x] = 0;
    __syncthreads();
    const uint32_t t0 = blockIdx.x * SORT_TILE;
    for (int r = 0; r < SORT_ITEMS; ++r) {
        uint32_t i = t0 + r * SORT_THREADS + threadIdx.x;
        if (i < n) atomicAdd(&h[digit_of(from_ek ? 0 : id[i], from_ek ? ek[i] : 0, from_ek, shift, ek_base)], 1u);
    }
    __syncthreads();
    counts[threadIdx.x * nblocks + blockIdx.x] = h[threadIdx.x];
}

/* In-place exclusive prefix sum of a[0..len) by one block of 1024 threads; *total_out (optional) = sum.
 * Tiles of 16384 words: 16 words per thread (four 16-byte accesses when aligned), warp-shuffle scans, a running carry
 * between tiles. */
constexpr int EX_PER = 16;
__global__ void __launch_bounds__(1024) k_exscan(uint32_t* __restrict__ a, uint32_t len, uint32_t* total_out) {
    __shared__ uint32_t wsum[32];
    __shared__ uint32_t s_carry;
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) s_carry = 0;
    __syncthreads();
    const bool vec = (reinterpret_cast<uintptr_t>(a) & 15u) == 0;
    for (uint32_t t0 = 0; t0 < len; t0 += 1024 * EX_PER) {
        const uint32_t i = t0 + threadIdx.x * EX_PER;
        uint32_t v[EX_PER];
        if (vec && i + EX_PER <= len) {
#pragma unroll
            for (int q = 0; q < EX_PER / 4; ++q) {
                const uint4 u = reinterpret_cast<const uint4*>(a + i)[q];
                v[4 * q] = u.x; v[4 * q + 1] = u.y; v[4 * q + 2] = u.z; v[4 * q + 3] = u.w;
            }
        } else {
#pragma unroll
            for (int k = 0; k < EX_PER; ++k) v[k] = i + k < len ? a[i + k] : 0;
        }
        uint32_t mine = 0;
#pragma unroll
        for (int k = 0; k < EX_PER; ++k) mine += v[k];
        uint32_t incl = mine;
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            const uint32_t u = __shfl_up_sync(0xFFFFFFFFu, incl, off);
            if (lane >= off) incl += u;
        }
        if (lane == 31) wsum[warp] = incl;
        __syncthreads();
        if (warp == 0) {
            uint32_t w = wsum[lane], wi = w;
#pragma unroll
            for (int off = 1; off < 32; off <<= 1) {
                const uint32_t u = __shfl_up_sync(0xFFFFFFFFu, wi, off);
                if (lane >= off) wi += u;
            }
            wsum[lane] = wi - w;                                   // exclusive prefix of the warp totals
        }
        __syncthreads();
        uint32_t run = s_carry + wsum[warp] + incl - mine;
#pragma unroll
        for (int k = 0; k < EX_PER; ++k) {
            const uint32_t x = v[k];
            v[k] = run;
            run += x;
        }
        if (vec && i + EX_PER <= len) {
#pragma unroll
            for (int q = 0; q < EX_PER / 4; ++q)
                reinterpret_cast<uint4*>(a + i)[q] = make_uint4(v[4 * q], v[4 * q + 1], v[4 * q + 2], v[4 * q + 3]);
        } else {
#pragma unroll
            for (int k = 0; k < EX_PER; ++k)
                if (i + k < len) a[i + k] = v[k];
        }
        __syncthreads();
        if (threadIdx.x == 1023) s_carry = run;                    // total up to the end of this tile
        __syncthreads();
    }
    if (total_out && threadIdx.x == 0) *total_out = s_carry;
}

/* Stable scatter of one radix pass.  Warp wq owns entries [t0 + wq*SORT_SEG, +SORT_SEG) in order; within a
 * round of 32 the rank among equal digits comes from match.any, across rounds from a per-warp counter. */
__global__ void __launch_bounds__(SORT_THREADS)
k_scatter(const uint64_t* __restrict__ sid, const uint32_t* __restrict__ sek, uint64_t* __restrict__ did,
          uint32_t* __restrict__ dek, uint32_t n, int from_ek, int shift, uint32_t ek_base,
          const uint32_t* __restrict__ offsets, uint32_t nblocks) {
    __shared__ uint32_t wcnt[SORT_WARPS][256];
    const uint32_t lane = threadIdx.x & 31u, wq = threadIdx.x >> 5;
    for (int i = threadIdx.x; i < SORT_WARPS * 256; i += SORT_THREADS) (&wcnt[0][0])[i] = 0;
    __syncthreads();
    const uint32_t base = blockIdx.x * SORT_TILE + wq * SORT_SEG;
    uint64_t kid[SORT_ITEMS];
    uint32_t kek[SORT_ITEMS], off[SORT_ITEMS];
    uint32_t* mine = wcnt[wq];
#pragma unroll
    for (int r = 0; r < SORT_ITEMS; ++r) {
        const uint32_t i = base + r * 32 + lane;
        const bool valid = i < n;
        kid[r] = valid ? sid[i] : 0;
        kek[r] = valid ? sek[i] : 0;
        const uint32_t dg = valid ? digit_of(kid[r], kek[r], from_ek, shift, ek_base) : 255u;
        const uint32_t peers = __match_any_sync(0xFFFFFFFFu, dg);
        const uint32_t rank = __popc(peers & ((1u << lane) - 1u));
        const uint32_t before = mine[dg];
        __syncwarp();
        if (rank == 0) mine[dg] = before + __popc(peers);
        __syncwarp();
        off[r] = before + rank;
    }
    __syncthreads();
    {   /* thread t = digit t: turn per-warp counts into per-warp bases (global offset of this block first) */
        uint32_t run = offsets[threadIdx.x * nblocks + blockIdx.x];
#pragma unroll
        for (int q = 0; q < SORT_WARPS; ++q) {
            uint32_t c = wcnt[q][threadIdx.x];
            wcnt[q][threadIdx.x] = run;
            run += c;
        }
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < SORT_ITEMS; ++r) {
        const uint32_t i = base + r * 32 + lane;
        if (i < n) {
            const uint32_t dg = digit_of(kid[r], kek[r], from_ek, shift, ek_base);
            const uint32_t dst = mine[dg] + off[r];
            did[dst] = kid[r];
            dek[dst] = kek[r];
        }
    }
}

/* ---- estimate range of an unsorted list (bounds the radix passes over the estimate key) -------------------------- */

__global__ void k_est_range_init(ScanState* st) {
    st->est_min = INT32_MAX;
    st->est_max = INT32_MIN;
}

__global__ void __launch_bounds__(256) k_est_range(const uint32_t* __restrict__ ek, uint32_t n, ScanState* st) {
    uint32_t lo = 0xFFFFFFFFu, hi = 0;                     // keys: ascending key = descending estimate
    const uint32_t stride = gridDim.x * 256;
    for (uint32_t i = blockIdx.x * 256 + threadIdx.x; i < n; i += stride) {
        const uint32_t k = ek[i];
        lo = min(lo, k); hi = max(hi, k);
    }
    lo = __reduce_min_sync(0xFFFFFFFFu, lo);
    hi = __reduce_max_sync(0xFFFFFFFFu, hi);
    if ((threadIdx.x & 31) == 0 && lo <= hi) {
        atomicMax(&st->est_max, key_to_est(lo));
        atomicMin(&st->est_min, key_to_est(hi));
    }
}

cudaError_t launch_est_range(const uint32_t* ek, uint32_t n, ScanState* st_dev, cudaStream_t st) {
    k_est_range_init<<<1, 1, 0, st>>>(st_dev);
    if (n) {
        uint32_t blocks = (n + 255) / 256;
        if (blocks > 148 * 4) blocks = 148 * 4;
        k_est_range<<<blocks, 256, 0, st>>>(ek, n, st_dev);
    }
    return cudaGetLastError();
}

/* ---- duplicate removal on the sorted list --------------------------------------------------------------- */

__device__ __forceinline__ bool is_first(const uint64_t* id, uint32_t i) { return i == 0 || id[i] != id[i - 1]; }

__global__ void __launch_bounds__(SORT_THREADS)
k_uniq_count(const uint64_t* __restrict__ id, uint32_t n, uint32_t* __restrict__ blockcnt) {
    __shared__ uint32_t wsum[SORT_WARPS];
    const uint32_t t0 = blockIdx.x * SORT_TILE;
    uint32_t c = 0;
    for (int r = 0; r < SORT_ITEMS; ++r) {
        uint32_t i = t0 + r * SORT_THREADS + threadIdx.x;
        if (i < n) c += is_first(id, i);
    }
    c = __reduce_add_sync(0xFFFFFFFFu, c);
    if ((threadIdx.x & 31) == 0) wsum[threadIdx.x >> 5] = c;
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t s = 0;
        for (int q = 0; q < SORT_WARPS; ++q) s += wsum[q];
        blockcnt[blockIdx.x] = s;
    }
}

/* Each thread owns SORT_ITEMS consecutive entries; block-exclusive scan of the per-thread flag counts. */
__global__ void __launch_bounds__(SORT_THREADS)
k_uniq_scatter(const uint64_t* __restrict__ sid, const uint32_t* __restrict__ sek, uint64_t* __restrict__ did,
               uint32_t* __restrict__ dek, uint32_t n, const uint32_t* __restrict__ blockoff) {
    __shared__ uint32_t wsum[SORT_WARPS];
    const uint32_t first = blockIdx.x * SORT_TILE + threadIdx.x * SORT_ITEMS;
    uint32_t flags = 0, c = 0;
#pragma unroll
    for (int r = 0; r < SORT_ITEMS; ++r) {
        uint32_t i = first + r;
        if (i < n && is_first(sid, i)) { flags |= 1u << r; ++c; }
    }
    const uint32_t lane = threadIdx.x & 31u, wq = threadIdx.x >> 5;
    uint32_t incl = c;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
        uint32_t v = __shfl_up_sync(0xFFFFFFFFu, incl, off);
        if (lane >= off) incl += v;
    }
    if (lane == 31) wsum[wq] = incl;
    __syncthreads();
    uint32_t wbase = 0;
    for (uint32_t q = 0; q < wq; ++q) wbase += wsum[q];
    uint32_t dst = blockoff[blockIdx.x] + wbase + incl - c;
#pragma unroll
    for (int r = 0; r < SORT_ITEMS; ++r) {
        if (flags & (1u << r)) {
            did[dst] = sid[first + r];
            dek[dst] = sek[first + r];
            ++dst;
        }
    }
}

/* One thread: m unique sorted entries in ek[0..m).  Fixes the new tau and the number of entries kept. */
__global__ void k_cut(const uint32_t* __restrict__ ek, const uint32_t* __restrict__ m_ptr, uint32_t m_const,
                      ScanState* st, uint64_t k_max, int32_t thr_min) {
    const uint32_t m = m_ptr ? *m_ptr : m_const;
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

uint64_t select_scratch_words(uint64_t n) {
    return (uint64_t)tiles_of(n) * 256 + tiles_of(n) + 64;
}

static int bits_of(uint64_t v) {
    int b = 0;
    while (v) { ++b; v >>= 1; }
    return b;
}

int select_compact(const SelectBuffers& B, int src, uint32_t n, int id_bits, int32_t est_min, int32_t est_max,
                   ScanState* st_dev, uint64_t k_max, int32_t thr_min, cudaStream_t stream, uint64_t* launches,
                   cudaError_t* err) {
    *err = cudaSuccess;
    int cur = src;
    if (n == 0) {
        k_cut<<<1, 1, 0, stream>>>(B.ek[cur], nullptr, 0, st_dev, k_max, thr_min);
        *launches += 1;
        *err = cudaGetLastError();
        return cur;
    }
    const uint32_t nb = tiles_of(n);
    uint32_t* counts = B.scratch;                     // 256 * nb words
    uint32_t* blockcnt = B.scratch + (uint64_t)256 * nb;   // nb words
    uint32_t* total = blockcnt + nb;                  // 1 word
    /* LSD passes: id bytes first (least significant key), then the estimate key relative to its minimum */
    const uint32_t ek_base = est_to_key(est_max);                    // smallest key present
    const uint32_t ek_span = est_to_key(est_min) - ek_base;          // largest key - smallest key
    const int id_passes = (id_bits + 7) / 8, ek_passes = (bits_of(ek_span) + 7) / 8;
    for (int p = 0; p < id_passes + ek_passes; ++p) {
        const int from_ek = p >= id_passes;
        const int shift = 8 * (from_ek ? p - id_passes : p);
        k_hist<<<nb, SORT_THREADS, 0, stream>>>(B.id[cur], B.ek[cur], n, from_ek, shift, ek_base, counts, nb);
        k_exscan<<<1, 1024, 0, stream>>>(counts, 256 * nb, nullptr);
        k_scatter<<<nb, SORT_THREADS, 0, stream>>>(B.id[cur], B.ek[cur], B.id[cur ^ 1], B.ek[cur ^ 1], n, from_ek,
                                                   shift, ek_base, counts, nb);
        *launches += 3;
        cur ^= 1;
    }
    k_uniq_count<<<nb, SORT_THREADS, 0, stream>>>(B.id[cur], n, blockcnt);
    k_exscan<<<1, 1024, 0, stream>>>(blockcnt, nb, total);
    k_uniq_scatter<<<nb, SORT_THREADS, 0, stream>>>(B.id[cur], B.ek[cur], B.id[cur ^ 1], B.ek[cur ^ 1], n, blockcnt);
    cur ^= 1;
    k_cut<<<1, 1, 0, stream>>>(B.ek[cur], total, 0, st_dev, k_max, thr_min);
    *launches += 4;
    *err = cudaGetLastError();
    return cur;
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
