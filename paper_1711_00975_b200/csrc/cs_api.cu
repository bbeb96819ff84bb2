/*
 * cs_api.cu -- host runtime and C ABI of libcs.so (include/cs.h): handle, hash-coefficient derivation,
 * launch scheduling of the update / scan passes, candidate-buffer management (chunking, compaction, growth),
 * double-buffered host streaming.  Every step of the path runs in the CUDA kernels of cs_kernels.cu,
 * cs_scan.cu and cs_select.cu; there is no CPU fallback and nothing here touches oracle/.
 */
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

#include "cs_internal.h"
#include "cs_select_batch.h"
#include "cs_select_static.h"

using namespace cs;

namespace {

thread_local char g_err[512] = "";

int fail(int code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

#define CS_CUDA(call)                                                                              \
    do {                                                                                           \
        cudaError_t e_ = (call);                                                                   \
        if (e_ != cudaSuccess)                                                                     \
            return fail(e_ == cudaErrorMemoryAllocation ? CS_ERR_NOMEM : CS_ERR_CUDA, "%s: %s",    \
                        #call, cudaGetErrorString(e_));                                            \
    } while (0)

/* ---- host arithmetic: splitmix64 stream and coefficient derivation (R1-R2) ------------------- */

uint64_t host_mix64(uint64_t z) {
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}

uint64_t stream_at(uint64_t seed, uint64_t n) { return host_mix64(seed + n * GAMMA); }

void derive_coeffs(uint64_t seed, int d, uint64_t* out_4d, uint64_t* K_out) {
    for (int j = 0; j < d; ++j) {
        const uint64_t n0 = 4 * (uint64_t)j;
        out_4d[4 * j + 0] = stream_at(seed, n0 + 1) % (P61 - 1) + 1;   /* a  in [1, p-1] */
        out_4d[4 * j + 1] = stream_at(seed, n0 + 2) % P61;             /* b  in [0, p-1] */
        out_4d[4 * j + 2] = stream_at(seed, n0 + 3) % (P61 - 1) + 1;   /* a' */
        out_4d[4 * j + 3] = stream_at(seed, n0 + 4) % P61;             /* b' */
    }
    if (K_out) *K_out = stream_at(seed, 4 * (uint64_t)d + 1);
}

uint64_t sample_threshold(double p) {
    if (!(p > 0.0) || !(p < 1.0)) return 0;
    return (uint64_t)std::floor(std::ldexp(p, 64));
}

int bit_length(uint64_t v) {
    int b = 0;
    while (v) { ++b; v >>= 1; }
    return b;
}

constexpr int STAGE_SLOTS = 3;
constexpr uint64_t STAGE_PARTICLES = 1ull << 24;      /* default particles per staging slot (192 MiB) */
constexpr uint64_t MAX_CHUNK = 1ull << 27;            /* default particles per scan launch */
constexpr uint32_t MIN_CAP = 1u << 22;                /* candidate entries per scale */
constexpr uint64_t BIN_CHUNK = 1ull << 30;            /* default particles per scatter/apply pair of the binned update: every
                                                       * launch ends with partial staging buffers and a partial wave of bins
                                                       * (cfg 3: 37.6 / 37.0 / 36.7 / 36.5 ms per step at 2^27 / 2^28 / 2^29 / 2^30) */
constexpr uint64_t COMPACT_CHUNK = 1ull << 28;        /* default particles per sampling-compaction launch */

}  // namespace

struct cs_sketch {
    int d = 0, n_scales = 0, device = 0, sm_count = 148;
    uint64_t w = 0, seed = 0, K = 0;
    double L = 0;
    uint32_t G[CS_MAX_SCALES] = {};
    int id_bits[CS_MAX_SCALES] = {};
    uint64_t coef[CS_MAX_SCALES][4 * CS_MAX_ROWS] = {};
    PassParams P = {};
    int32_t* T[CS_MAX_SCALES] = {};
    cudaStream_t stream = nullptr;
    uint64_t upd_index = 0, scan_index = 0, launches = 0;
    uint64_t table_budget = 64ull << 20;   /* bytes of counters one update pass may touch (cs_set_table_budget) */
    /* cs_set_chunk_sizes: how the passes cut a call into launches (the result never depends on them) */
    uint64_t stage_particles = STAGE_PARTICLES, bin_chunk = BIN_CHUNK, scan_chunk = MAX_CHUNK, compact_chunk = COMPACT_CHUNK;

    /* candidate collection */
    bool scanning = false;
    uint64_t k_max = 0;
    int32_t thr_min = INT32_MAX;
    uint32_t cap = 0;
    uint32_t cap_min = MIN_CAP;        /* cs_set_candidate_capacity */
    SelectBuffers sb[CS_MAX_SCALES] = {};
    unsigned long long* seen[CS_MAX_SCALES] = {};   /* duplicate filter of the re-scan (cs_scan_common.cuh), per scale */
    uint64_t seen_slots = 0;
    bool use_seen[CS_MAX_SCALES] = {};    /* switched on per scale once a compaction finds the list heavily duplicated */
    uint32_t compact_n[CS_MAX_SCALES] = {};   /* entries the compaction in flight started from (0: none in flight) */
    int cur[CS_MAX_SCALES] = {};
    bool dirty[CS_MAX_SCALES] = {};
    uint32_t last_compact[CS_MAX_SCALES] = {};
    uint32_t epoch[CS_MAX_SCALES] = {};   /* look-back epochs of the selector (cs_select.cu), one counter per scale */
    uint64_t n_compactions[CS_MAX_SCALES] = {};
    uint64_t n_scan_launches = 0;
    double rate = 1.0;
    bool first_chunk = true;
    uint64_t scanned = 0;              /* particles scanned since cs_scan_begin */
    ScanState* st_dev = nullptr;      /* CS_MAX_SCALES entries */
    ScanState* st_host = nullptr;     /* pinned mirror */
    uint32_t* word_dev = nullptr;     /* 1 scratch word */
    uint32_t* word_host = nullptr;    /* pinned */
    uint64_t* out_ids = nullptr;      /* staging for cs_topk / cs_excursion results */
    int32_t* out_est = nullptr;
    uint64_t out_cap = 0;

    /* binned update (cs_update_binned.cu) */
    int update_mode = 0;               /* cs_set_update_mode: 0 auto, 1 direct red.global, 2 binned */
    int bin_rows_direct = -1;          /* rows of each binned pass that still go through red.global; -1 = auto */
    uint16_t* bins = nullptr;          /* record regions */
    uint64_t bins_records = 0;         /* capacity of `bins` in records */
    uint32_t* cursor = nullptr;        /* BIN_MAX words */
    unsigned long long* bin_stats = nullptr;   /* 4 device counters of the binned route (cs_update_stats) */
    PhaseTimer tm;                     /* cs_set_timing / cs_get_timing */

    /* bitmap prefilter of the scan (cs_scan_bitmap.cu): B[j][b] = |T[j][b]| >= tau_bm, per scale */
    int scan_mode = 0;                 /* cs_set_scan_mode: 0 auto, 1 plain, 2 bitmap, 3 bitmap first stage */
    uint32_t* bm[CS_MAX_SCALES] = {};
    int32_t tau_bm[CS_MAX_SCALES] = {};
    bool bm_valid[CS_MAX_SCALES] = {};
    uint32_t* coarse = nullptr;        /* coarse bitmap of scale 0 (bitmap first stage, single-scale handles) */

    /* dense buffer of kept particles for strongly sampled streams (k_compact_kept) */
    float* kept = nullptr;
    uint64_t kept_cap = 0;             /* particles */

    /* packed records: positions of one batch unpacked to cell centres of the finest mesh */
    float* unpacked = nullptr;
    uint64_t unpacked_alloc = 0;       /* particles */

    /* scratch kept between calls: hash table of cs_recount, id expansion of cs_scan_children / cs_expand_neighbours */
    uint64_t* ht_keys = nullptr;
    uint32_t* ht_vals = nullptr;
    uint64_t ht_size = 0;              /* slots allocated */
    uint64_t* ids_scratch = nullptr;
    uint64_t ids_scratch_cap = 0;      /* ids */

    /* survivor lists of the row-partitioned scan */
    StageBuffers stb = {};

    /* host streaming */
    float* stage[STAGE_SLOTS] = {};
    uint64_t stage_alloc = 0;          /* particles each allocated slot holds */
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t ev_full[STAGE_SLOTS] = {}, ev_free[STAGE_SLOTS] = {};

    /* replay cache (cs_set_replay_cache): what the last update call read, kept for the re-scan of the same buffer */
    uint64_t replay_limit = 0;         /* bytes of device memory the handle may hold for it; 0 = off */
    unsigned char* host_cache = nullptr;   /* raw batches of the last host-streamed update call */
    uint64_t host_cache_bytes = 0;     /* allocated */
    const void* hc_host = nullptr;     /* key: host address, items, bytes per item */
    uint64_t hc_n = 0;
    size_t hc_bpp = 0;
    bool hc_valid = false;
    float* kept_arena = nullptr;       /* kept particles of sampled update calls, segment after segment */
    uint64_t kept_arena_cap = 0, kept_arena_used = 0;   /* particles */
    struct KeptSeg { const float* src; uint64_t n, index0; double p; uint64_t off, cnt; };
    std::vector<KeptSeg> kept_segs;
};

/* Every entry point that takes a handle runs on the handle's device, whatever device is current (and restores it). */
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    cudaError_t err = cudaSuccess;
    explicit DeviceGuard(const cs_sketch* s) {
        err = cudaGetDevice(&prev);
        if (err == cudaSuccess && s && prev != s->device) {
            err = cudaSetDevice(s->device);
            switched = err == cudaSuccess;
        }
    }
    ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
    DeviceGuard(const DeviceGuard&) = delete;
    DeviceGuard& operator=(const DeviceGuard&) = delete;
};
#define CS_ENTER(s)                                                                                    \
    if (!(s)) return fail(CS_ERR_ARG, "null handle");                                                  \
    DeviceGuard guard_(s);                                                                             \
    if (guard_.err != cudaSuccess) return fail(CS_ERR_CUDA, "cannot switch to the handle's device %d: %s", \
                                                (s)->device, cudaGetErrorString(guard_.err))

namespace {

void free_candidates(cs_sketch* s) {
    for (int i = 0; i < CS_MAX_SCALES; ++i) {
        for (int h = 0; h < 2; ++h) {
            if (s->sb[i].id[h]) cudaFree(s->sb[i].id[h]);
            if (s->sb[i].ek[h]) cudaFree(s->sb[i].ek[h]);
            s->sb[i].id[h] = nullptr;
            s->sb[i].ek[h] = nullptr;
        }
        if (s->sb[i].scratch) cudaFree(s->sb[i].scratch);
        s->sb[i].scratch = nullptr;
        if (s->seen[i]) cudaFree(s->seen[i]);
        s->seen[i] = nullptr;
    }
    s->seen_slots = 0;
    s->cap = 0;
}

int alloc_candidates(cs_sketch* s, uint32_t cap) {
    free_candidates(s);
    for (int i = 0; i < s->n_scales; ++i) {
        for (int h = 0; h < 2; ++h) {
            CS_CUDA(cudaMalloc(&s->sb[i].id[h], (size_t)cap * sizeof(uint64_t)));
            CS_CUDA(cudaMalloc(&s->sb[i].ek[h], (size_t)cap * sizeof(uint32_t)));
        }
        CS_CUDA(cudaMalloc(&s->sb[i].scratch, (size_t)select_scratch_words(cap) * sizeof(uint32_t)));
        CS_CUDA(cudaMemsetAsync(s->sb[i].scratch, 0, (size_t)select_scratch_words(cap) * sizeof(uint32_t), s->stream));
        s->cur[i] = 0;
    }
    /* duplicate filter of the re-scan: 2 slots per list entry, at most 2^25 slots (256 MiB) per scale */
    uint64_t slots = 2 * (uint64_t)cap;
    if (slots > (1ull << 25)) slots = 1ull << 25;
    for (int i = 0; i < s->n_scales; ++i) CS_CUDA(cudaMalloc(&s->seen[i], slots * sizeof(unsigned long long)));
    s->seen_slots = slots;
    s->cap = cap;
    return CS_OK;
}

/* Empty the duplicate filters (cs_scan_begin; before a chunk whose entries were dropped is re-run). */
int clear_seen(cs_sketch* s) {
    for (int i = 0; i < s->n_scales; ++i)
        if (s->seen[i]) CS_CUDA(cudaMemsetAsync(s->seen[i], 0xFF, s->seen_slots * sizeof(unsigned long long), s->stream));
    return CS_OK;
}

/* Double the candidate capacity, keeping the entries held (all scales). */
int grow_candidates(cs_sketch* s) {
    if (s->cap >= (1u << 30)) return fail(CS_ERR_NOMEM, "candidate list would exceed 2^30 entries per scale");
    const uint32_t cap = s->cap * 2;
    CS_CUDA(cudaStreamSynchronize(s->stream));
    for (int i = 0; i < s->n_scales; ++i) {
        SelectBuffers nb = {};
        for (int h = 0; h < 2; ++h) {
            CS_CUDA(cudaMalloc(&nb.id[h], (size_t)cap * sizeof(uint64_t)));
            CS_CUDA(cudaMalloc(&nb.ek[h], (size_t)cap * sizeof(uint32_t)));
        }
        CS_CUDA(cudaMalloc(&nb.scratch, (size_t)select_scratch_words(cap) * sizeof(uint32_t)));
        CS_CUDA(cudaMemsetAsync(nb.scratch, 0, (size_t)select_scratch_words(cap) * sizeof(uint32_t), s->stream));
        const uint32_t held = s->st_host[i].count < s->cap ? s->st_host[i].count : s->cap;
        const int c = s->cur[i];                             /* the list stays in the same half: the device names it too */
        CS_CUDA(cudaMemcpyAsync(nb.id[c], s->sb[i].id[c], (size_t)held * 8, cudaMemcpyDeviceToDevice, s->stream));
        CS_CUDA(cudaMemcpyAsync(nb.ek[c], s->sb[i].ek[c], (size_t)held * 4, cudaMemcpyDeviceToDevice, s->stream));
        CS_CUDA(cudaStreamSynchronize(s->stream));
        for (int h = 0; h < 2; ++h) { cudaFree(s->sb[i].id[h]); cudaFree(s->sb[i].ek[h]); }
        cudaFree(s->sb[i].scratch);
        s->sb[i] = nb;
    }
    s->cap = cap;
    return CS_OK;
}

int read_states(cs_sketch* s) {
    CS_CUDA(cudaMemcpyAsync(s->st_host, s->st_dev, sizeof(ScanState) * s->n_scales, cudaMemcpyDeviceToHost, s->stream));
    CS_CUDA(cudaStreamSynchronize(s->stream));
    for (int i = 0; i < s->n_scales; ++i) {
        s->cur[i] = (int)(s->st_host[i].half & 1u);          /* compactions move the list */
        /* The duplicate filter costs one atomicCAS at a random address per cell that passes the last stage: it pays when
         * cells arrive many times (coarse meshes, concentrated streams: measured 2x fewer launches at cfg 1), not when
         * almost every cell holds one particle (cfg 5: +2.4 ms).  Decided from what the last compaction found. */
        if (s->compact_n[i]) {
            if (s->compact_n[i] >= 4096 && 2 * (uint64_t)s->compact_n[i] >= 3 * (uint64_t)s->st_host[i].uniq) s->use_seen[i] = true;
            s->compact_n[i] = 0;
        }
    }
    return CS_OK;
}

/* Sort + dedupe + cut the candidate lists of the scales in `mask`, in one launch: enqueued only, no synchronisation.
 * A list may end up in the other half of its ping-pong buffers: the caller reads the states back (read_states) before it
 * uses s->cur again. */
int compact_scales(cs_sketch* s, uint32_t mask) {
    CompactRequest req[CS_MAX_SCALES];
    int count = 0;
    for (int i = 0; i < s->n_scales; ++i) {
        if (!(mask >> i & 1u)) continue;
        const uint32_t n = s->st_host[i].count < s->cap ? s->st_host[i].count : s->cap;
        req[count++] = CompactRequest{&s->sb[i], s->cur[i], n, s->id_bits[i], s->st_dev + i, &s->epoch[i]};
        s->dirty[i] = false;
        s->n_compactions[i] += 1;
        s->compact_n[i] = n;
    }
    if (!count) return CS_OK;
    s->tm.mark(PH_SELECT, s->stream);
    cudaError_t e = select_compact_batch(req, count, s->cap, s->k_max, s->thr_min, s->stream, &s->launches);
    s->tm.stop(s->stream);
    if (e != cudaSuccess) return fail(CS_ERR_CUDA, "select_compact: %s", cudaGetErrorString(e));
    return CS_OK;
}

int compact_scale(cs_sketch* s, int i) { return compact_scales(s, 1u << i); }

void fill_scan_params(cs_sketch* s, ScanParams* S) {
    memset(S, 0, sizeof(*S));
    for (int i = 0; i < s->n_scales; ++i) {
        S->tg[i].id = s->sb[i].id[s->cur[i]];
        S->tg[i].ek = s->sb[i].ek[s->cur[i]];
        S->tg[i].st = s->st_dev + i;
        S->tg[i].cap = s->cap;
        S->tg[i].seen = s->seen[i];
        S->tg[i].seen_mask = (s->seen[i] && s->use_seen[i]) ? (uint32_t)(s->seen_slots - 1) : 0u;
    }
}

PassParams pass_params(const cs_sketch* s, uint64_t index0, double sample_p) {
    PassParams P = s->P;
    P.index0 = index0;
    P.sample = sample_p < 1.0 ? 1 : 0;
    P.Tp = sample_threshold(sample_p);
    return P;
}

bool bad_p(double p) { return !(p > 0.0) || p > 1.0; }

/* ---- binned update: plan + passes (kernels in cs_update_binned.cu) -------------------- */

constexpr uint32_t BIN_MAX = 4096;                    /* bins per pass (words of `cursor`) */
constexpr uint64_t BIN_MIN_N = 1ull << 22;            /* auto mode: below this the direct kernel is as fast */
constexpr size_t BIN_SMEM = 216 * 1024;               /* shared memory of one scatter CTA (8 pairs per round at cfg 3: 211 KB) */
constexpr uint32_t PAIRS_MIN = 5, PAIRS_MAX = 12;     /* pairs of particles per thread between two flush phases */

struct BinPlan {
    uint32_t log2w, log2S, SL, C, threads, pairs;
    int rows_per_pass, rows_direct;       /* rows of one pass, and how many of them take the direct route */
};

int ilog2(uint64_t v) { return bit_length(v) - 1; }

uint32_t staging_capacity(uint32_t threads, uint32_t SL, uint32_t pairs) {
    const double lambda = 2.0 * pairs * threads / SL;              /* records per bin, round and CTA */
    /* up to 31 records left from the round before + this round's arrivals (Poisson, mean lambda) + 3 sigma: the few
     * records beyond (measured 3e-8 of all at cfg 3) take the red.global route.  Sized at 6 sigma the same shared memory
     * holds 6 pairs per round instead of 8 at cfg 3, and the flush phases between rounds are what the extra pairs save. */
    uint32_t C = (uint32_t)(32.0 + lambda + 3.0 * std::sqrt(lambda) + 8.0);
    C = (C + 7u) & ~7u;
    return C > 384 ? 384 : C;                          /* beyond: staging overflows go through red.global */
}

/* Rows of a pass of r rows that take the direct route.  Hybrid: the scatter kernel is bound by the integer pipes,
 * the direct rows by the L2 tag rate, so both run together; auto = 3/7 of the rows (measured best at d = 7) as long
 * as they stay L2-resident. */
int direct_rows(const cs_sketch* s, int r) {
    int rd = s->bin_rows_direct;
    if (rd < 0) {
        rd = (3 * r + 3) / 7;
        const uint64_t fit = s->table_budget / (s->w * sizeof(int32_t));
        if ((uint64_t)rd > fit) rd = (int)fit;
    }
    return rd < r ? rd : r;
}

/* false: this shape cannot be binned (w not a power of two, too small or too wide): use the direct kernel */
bool bin_plan(const cs_sketch* s, BinPlan* pl) {
    const uint64_t w = s->w;
    if (w & (w - 1)) return false;
    const int lw = ilog2(w);
    if (lw < 8 || lw > 25) return false;
    int lS = lw - 7;                                   /* 128 slices per row ... */
    if (lS < 8) lS = 8;
    if (lS > 15) lS = 15;                              /* ... of at most 2^15 counters (128 KB, 15-bit offsets) */
    const uint32_t SL = (uint32_t)(w >> lS);
    int rows = 0;
    for (int r = 1; r <= 8 && r <= s->d; ++r) {
        const uint32_t nb = (uint32_t)(r - direct_rows(s, r)) * SL;
        if (nb <= BIN_MAX && scatter_smem_bytes(nb, staging_capacity(1024, SL, PAIRS_MIN)) <= BIN_SMEM) rows = r;
    }
    if (!rows) return false;
    const int groups = (s->d + rows - 1) / rows;
    rows = (s->d + groups - 1) / groups;               /* balanced row groups */
    pl->log2w = (uint32_t)lw; pl->log2S = (uint32_t)lS; pl->SL = SL;
    pl->rows_per_pass = rows;
    pl->rows_direct = direct_rows(s, rows);
    /* two CTAs of 512 threads per SM when their staging buffers fit: one CTA's flush phase overlaps the other's hashing */
    const uint32_t nb = (uint32_t)(rows - pl->rows_direct) * SL;
    pl->threads = scatter_smem_bytes(nb, staging_capacity(512, SL, PAIRS_MAX)) <= 110 * 1024 ? 512 : 1024;
    /* as many pairs per round as the staging buffers have room for: the flush phases between rounds are overhead */
    pl->pairs = PAIRS_MIN;
    while (pl->pairs < PAIRS_MAX && scatter_smem_bytes(nb, staging_capacity(pl->threads, SL, pl->pairs + 1)) <=
                                        (pl->threads == 512 ? 110 * 1024 : BIN_SMEM))
        pl->pairs += 1;
    pl->C = staging_capacity(pl->threads, SL, pl->pairs);
    return true;
}

int update_binned(cs_sketch* s, const BinPlan& pl, const float* xyz, uint64_t n, uint64_t index0, double sample_p) {
    const PassParams full = pass_params(s, index0, sample_p);
    const int each = pl.rows_per_pass;
    uint64_t BC = s->bin_chunk;
    const double keep = sample_p < 1.0 ? sample_p : 1.0;
    uint64_t cap = 0, need = 0;
    for (;;) {                                          /* record scratch: 2 B x binned rows per particle of a chunk */
        const uint64_t chunk_max = n < BC ? n : BC;
        cap = (uint64_t)((double)chunk_max * keep / pl.SL * 1.04) + 2048;
        cap = (cap + 31) & ~(uint64_t)31;
        need = cap * each * pl.SL;
        if (s->bins_records >= need || BC <= (1ull << 27)) break;
        size_t free_b = 0, total_b = 0;                 /* a chunk whose scratch would take more than a quarter of what is */
        if (cudaMemGetInfo(&free_b, &total_b) != cudaSuccess) { cudaGetLastError(); break; }   /* free is halved */
        if (need * sizeof(uint16_t) <= free_b / 4) break;
        BC /= 2;
    }
    if (!s->cursor) CS_CUDA(cudaMalloc(&s->cursor, BIN_MAX * sizeof(uint32_t)));
    if (!s->bin_stats) {
        CS_CUDA(cudaMalloc(&s->bin_stats, 4 * sizeof(unsigned long long)));
        CS_CUDA(cudaMemsetAsync(s->bin_stats, 0, 4 * sizeof(unsigned long long), s->stream));
    }
    if (s->bins_records < need) {
        CS_CUDA(cudaStreamSynchronize(s->stream));
        if (s->bins) cudaFree(s->bins);
        s->bins = nullptr; s->bins_records = 0;
        CS_CUDA(cudaMalloc(&s->bins, need * sizeof(uint16_t)));
        s->bins_records = need;
    }
    for (uint64_t off = 0; off < n; off += BC) {
        uint64_t m = n - off < BC ? n - off : BC;
        for (int i = 0; i < s->n_scales; ++i)
            for (int j0 = 0; j0 < s->d; j0 += each) {
                const int nr = j0 + each <= s->d ? each : s->d - j0;
                PassParams P = full;
                P.index0 = index0 + off;
                P.n_scales = 1;
                P.d = nr;
                P.sc[0] = full.sc[i];
                P.sc[0].T = full.sc[i].T + (uint64_t)j0 * s->w;
                for (int j = 0; j < nr; ++j) P.rows[j] = full.rows[i * s->d + j0 + j];
                BinParams B;
                B.bins = s->bins; B.cursor = s->cursor; B.cap = (uint32_t)cap;
                B.rows_direct = pl.rows_direct < nr ? pl.rows_direct : nr;
                B.nb = (uint32_t)(nr - B.rows_direct) * pl.SL;
                B.threads = pl.threads; B.C = pl.C; B.pairs = pl.pairs; B.log2S = pl.log2S; B.log2w = pl.log2w;
                B.stats = s->bin_stats;
                if (B.nb) CS_CUDA(cudaMemsetAsync(s->cursor, 0, B.nb * sizeof(uint32_t), s->stream));
                cudaError_t e = launch_update_binned(P, B, xyz + 3 * off, m, s->sm_count, s->stream, &s->tm);
                s->tm.stop(s->stream);
                if (e != cudaSuccess) return fail(CS_ERR_CUDA, "binned update kernels: %s", cudaGetErrorString(e));
                s->launches += B.nb ? 2 : 1;
            }
    }
    return CS_OK;
}

/* Row-partitioned update: red.global.add runs at its L2 rate only while the counters a
 * pass touches stay L2-resident (measured: ~194 G/s up to ~56 MiB, 107 G/s at 112 MiB, 25 G/s at 448 MiB), so
 * the d rows of each scale are split into groups of at most table_budget bytes and the positions are re-read
 * once per group (12 B/particle at HBM rate, far cheaper than DRAM-backed atomics).  Each group is the same
 * kernel with a PassParams that names only that group's rows and tables. */
int update_passes_raw(cs_sketch* s, const float* xyz, uint64_t n, uint64_t index0, double sample_p) {
    BinPlan pl;
    if (s->update_mode != 1 && (s->update_mode == 2 || n >= BIN_MIN_N) && bin_plan(s, &pl))
        return update_binned(s, pl, xyz, n, index0, sample_p);
    const PassParams full = pass_params(s, index0, sample_p);
    const uint64_t row_bytes = s->w * sizeof(int32_t);
    const uint64_t all_bytes = row_bytes * s->d * s->n_scales;
    if (all_bytes <= s->table_budget) {
        s->tm.mark(PH_SCATTER, s->stream);
        cudaError_t e = launch_update(full, xyz, n, s->sm_count, s->stream);
        s->tm.stop(s->stream);
        if (e != cudaSuccess) return fail(CS_ERR_CUDA, "update kernel: %s", cudaGetErrorString(e));
        s->launches += 1;
        return CS_OK;
    }
    uint64_t fit = s->table_budget / row_bytes;               /* rows of one scale that fit the budget */
    if (fit < 1) fit = 1;
    if (fit >= (uint64_t)s->d) {                               /* whole scales fit: group scales */
        const int per = (int)(fit / s->d);
        const int groups = (s->n_scales + per - 1) / per;
        const int each = (s->n_scales + groups - 1) / groups;
        for (int s0 = 0; s0 < s->n_scales; s0 += each) {
            const int ns = s0 + each <= s->n_scales ? each : s->n_scales - s0;
            PassParams P = full;
            P.n_scales = ns;
            for (int i = 0; i < ns; ++i) {
                P.sc[i] = full.sc[s0 + i];
                for (int j = 0; j < s->d; ++j) P.rows[i * s->d + j] = full.rows[(s0 + i) * s->d + j];
            }
            s->tm.mark(PH_SCATTER, s->stream);
            cudaError_t e = launch_update(P, xyz, n, s->sm_count, s->stream);
            s->tm.stop(s->stream);
            if (e != cudaSuccess) return fail(CS_ERR_CUDA, "update kernel: %s", cudaGetErrorString(e));
            s->launches += 1;
        }
        return CS_OK;
    }
    const int groups = (int)((s->d + fit - 1) / fit);          /* balanced row groups, one scale at a time */
    const int each = (s->d + groups - 1) / groups;
    for (int i = 0; i < s->n_scales; ++i)
        for (int j0 = 0; j0 < s->d; j0 += each) {
            const int nr = j0 + each <= s->d ? each : s->d - j0;
            PassParams P = full;
            P.n_scales = 1;
            P.d = nr;
            P.sc[0] = full.sc[i];
            P.sc[0].T = full.sc[i].T + (uint64_t)j0 * s->w;
            for (int j = 0; j < nr; ++j) P.rows[j] = full.rows[i * s->d + j0 + j];
            s->tm.mark(PH_SCATTER, s->stream);
            cudaError_t e = launch_update(P, xyz, n, s->sm_count, s->stream);
            s->tm.stop(s->stream);
            if (e != cudaSuccess) return fail(CS_ERR_CUDA, "update kernel: %s", cudaGetErrorString(e));
            s->launches += 1;
        }
    return CS_OK;
}

}  // namespace

namespace {

void free_stage_lists(cs_sketch* s) {
    for (int h = 0; h < 2; ++h) {
        if (s->stb.list[h]) cudaFree(s->stb.list[h]);
        if (s->stb.cnt[h]) cudaFree(s->stb.cnt[h]);
        s->stb.list[h] = nullptr;
        s->stb.cnt[h] = nullptr;
    }
    s->stb.cap_entries = 0;
}

int ensure_stage_lists(cs_sketch* s, uint64_t n) {
    const uint32_t blocks = (uint32_t)s->sm_count * 8;
    const uint64_t need = staged_list_entries(n, blocks);
    if (s->stb.cap_entries >= need && s->stb.blocks == blocks) return CS_OK;
    CS_CUDA(cudaStreamSynchronize(s->stream));
    free_stage_lists(s);
    for (int h = 0; h < 2; ++h) {
        CS_CUDA(cudaMalloc(&s->stb.list[h], need * sizeof(uint64_t)));
        CS_CUDA(cudaMalloc(&s->stb.cnt[h], blocks * sizeof(uint32_t)));
    }
    s->stb.blocks = blocks;
    s->stb.cap_entries = need;
    return CS_OK;
}

/* One scan launch over a chunk, shaped by the table budget: everything at once when all
 * tables fit; else scale by scale -- the one-kernel scan when the scale fits, the staged pipeline when not. */
int launch_scan_chunk(cs_sketch* s, const float* xyz, uint64_t n, uint64_t index0, double sample_p) {
    const PassParams full = pass_params(s, index0, sample_p);
    ScanParams S;
    fill_scan_params(s, &S);
    /* bitmap prefilter: valid once every scale collects against a tau >= 1 (|T| >= tau is then necessary for a row
     * to pass); rebuilt (d*w/8 bytes, microseconds) whenever a compaction has raised tau */
    CoarseShape cshape;
    const bool staged_bm = s->n_scales == 1 && coarse_shape(s->d, s->P.rank, s->w, &cshape);
    bool use_bm = (s->scan_mode == 2 || s->scan_mode == 3 || (s->scan_mode == 0 && staged_bm)) && (s->w & (s->w - 1)) == 0;
    for (int i = 0; i < s->n_scales && use_bm; ++i) use_bm = s->st_host[i].tau >= 1;
    if (use_bm) {
        const uint64_t counters = (uint64_t)s->d * s->w;
        bool rebuilt = false;
        for (int i = 0; i < s->n_scales; ++i) {
            if (!s->bm[i]) CS_CUDA(cudaMalloc(&s->bm[i], ((counters + 31) / 32) * sizeof(uint32_t)));
            if (!s->bm_valid[i] || s->tau_bm[i] != s->st_host[i].tau) {
                s->tm.mark(PH_BITMAP, s->stream);
                cudaError_t eb = launch_build_bitmap(s->T[i], counters, s->st_host[i].tau, s->bm[i], s->stream);
                s->tm.stop(s->stream);
                if (eb != cudaSuccess) return fail(CS_ERR_CUDA, "bitmap kernel: %s", cudaGetErrorString(eb));
                s->launches += 1;
                s->tau_bm[i] = s->st_host[i].tau;
                s->bm_valid[i] = true;
                rebuilt = true;
            }
        }
        if (s->scan_mode != 2 && staged_bm) {
            /* bitmap first stage (coarse bitmap in shared memory) + the remaining rows on dense warps */
            int rc = ensure_stage_lists(s, n);
            if (rc) return rc;
            if (!s->coarse) {
                CS_CUDA(cudaMalloc(&s->coarse, (size_t)cshape.row_off[s->P.rank + 1] * sizeof(uint32_t)));
                rebuilt = true;
            }
            cudaError_t ec = launch_scan_staged_cb(full, S.tg[0], s->stb, s->bm[0], s->coarse, cshape, rebuilt, xyz, n,
                                                   s->sm_count, s->stream, &s->launches, &s->tm);
            s->tm.stop(s->stream);
            if (ec != cudaSuccess) return fail(CS_ERR_CUDA, "bitmap stage kernels: %s", cudaGetErrorString(ec));
            s->n_scan_launches += 1;
            return CS_OK;
        }
        s->tm.mark(PH_SCAN_FIRST, s->stream);
        cudaError_t eb = launch_scan_bitmap(full, S, s->bm, xyz, n, s->sm_count, s->stream);
        s->tm.stop(s->stream);
        if (eb != cudaSuccess) return fail(CS_ERR_CUDA, "bitmap scan kernel: %s", cudaGetErrorString(eb));
        s->launches += 1;
        s->n_scan_launches += 1;
        return CS_OK;
    }
    const uint64_t row_bytes = s->w * sizeof(int32_t);
    const uint64_t scale_bytes = row_bytes * s->d;
    cudaError_t e = cudaSuccess;
    if (scale_bytes * s->n_scales <= s->table_budget) {
        s->tm.mark(PH_SCAN_FIRST, s->stream);
        e = launch_scan(full, S, xyz, n, s->sm_count, s->stream);
        s->tm.stop(s->stream);
        s->launches += 1;
    } else {
        for (int i = 0; i < s->n_scales && e == cudaSuccess; ++i) {
            PassParams P = full;
            P.n_scales = 1;
            P.sc[0] = full.sc[i];
            for (int j = 0; j < s->d; ++j) P.rows[j] = full.rows[i * s->d + j];
            if (scale_bytes <= s->table_budget) {
                ScanParams S1 = {};
                S1.tg[0] = S.tg[i];
                s->tm.mark(PH_SCAN_FIRST, s->stream);
                e = launch_scan(P, S1, xyz, n, s->sm_count, s->stream);
                s->tm.stop(s->stream);
                s->launches += 1;
            } else {
                int rc = ensure_stage_lists(s, n);
                if (rc) return rc;
                uint64_t fit = s->table_budget / row_bytes;
                if (fit < 1) fit = 1;
                e = launch_scan_staged(P, S.tg[i], s->stb, (int)(fit > 8 ? 8 : fit), xyz, n, s->stream, &s->launches, &s->tm);
                s->tm.stop(s->stream);
            }
        }
    }
    if (e != cudaSuccess) return fail(CS_ERR_CUDA, "scan kernel: %s", cudaGetErrorString(e));
    s->n_scan_launches += 1;
    return CS_OK;
}

/* After a chunk: which scales must be compacted now (list past half the buffer, or doubled since last time). */
bool wants_compaction(const cs_sketch* s, int i) {
    const uint32_t c = s->st_host[i].count;
    uint64_t base = s->last_compact[i];
    if (base < s->k_max) base = s->k_max;
    if (base < 8192) base = 8192;
    /* compacting raises tau (the k_max-th estimate seen so far), which sharpens every later chunk's filter -- unless tau
     * already sits at the excursion limit thr_min, above which it never goes: then only buffer pressure counts */
    const bool tau_capped = s->thr_min != INT32_MAX && s->st_host[i].tau >= s->thr_min;
    return s->dirty[i] && (c > s->cap / 2 || (!tau_capped && 2 * (uint64_t)c >= 3 * base));
}

/* Replay n device-resident particles against the tables, collecting candidates.
 * Invariant that makes overflow impossible on a retry: a chunk of at most `free` particles cannot append more
 * than `free` entries to any scale. */
int scan_device_raw(cs_sketch* s, const float* xyz, uint64_t n, double sample_p) {
    uint64_t done = 0;
    while (done < n) {
        uint32_t free_min = s->cap;
        for (int i = 0; i < s->n_scales; ++i) {
            uint32_t held = s->st_host[i].count;
            uint32_t fr = held < s->cap ? s->cap - held : 0;
            if (fr < free_min) free_min = fr;
        }
        if (free_min < s->cap / 2) {                     /* lists are legitimately large: make room */
            uint32_t due = 0;
            for (int i = 0; i < s->n_scales; ++i)
                if (s->dirty[i] && s->st_host[i].count > s->cap / 2) due |= 1u << i;
            if (due) {
                int rc = compact_scales(s, due);
                if (rc) return rc;
                rc = read_states(s);
                if (rc) return rc;
                for (int i = 0; i < s->n_scales; ++i) s->last_compact[i] = s->st_host[i].count;
                continue;
            }
            int rc = grow_candidates(s);
            if (rc) return rc;
            continue;
        }
        /* optimistic chunk: expect at most rate * chunk new entries per scale, keep a factor 2 of slack */
        double want = (double)free_min / (2.0 * (s->rate > 1e-9 ? s->rate : 1e-9));
        uint64_t chunk = want >= (double)s->scan_chunk ? s->scan_chunk : (uint64_t)want;
        if (s->first_chunk && s->k_max) {                /* a small first chunk fixes a first tau cheaply */
            uint64_t c0 = 8 * s->k_max > (1u << 18) ? 8 * s->k_max : (1u << 18);
            if (chunk > c0) chunk = c0;
        } else if (s->k_max && chunk > 4 * s->scanned) {  /* tau still rises fast: grow geometrically, not at once ... */
            bool capped = s->thr_min != INT32_MAX;           /* ... unless it already sits at the excursion limit everywhere */
            for (int i = 0; i < s->n_scales && capped; ++i) capped = s->st_host[i].tau >= s->thr_min;
            if (!capped) chunk = 4 * s->scanned;
        }
        if (chunk > n - done) chunk = n - done;
        if (chunk < n - done) chunk &= ~(uint64_t)3;     /* keep the 16-byte phase of the remaining stream */
        if (chunk == 0) chunk = (n - done) < 4 ? (n - done) : 4;

        for (;;) {
            uint32_t before[CS_MAX_SCALES];
            for (int i = 0; i < s->n_scales; ++i) before[i] = s->st_host[i].count;
            int rc = launch_scan_chunk(s, xyz + 3 * done, chunk, s->scan_index + done, sample_p);
            if (rc) return rc;
            rc = read_states(s);
            if (rc) return rc;
            bool overflow = false;
            double r = 0.0;
            for (int i = 0; i < s->n_scales; ++i) {
                if (s->st_host[i].count != before[i]) s->dirty[i] = true;
                if (s->st_host[i].count > s->cap) overflow = true;
                double ri = (double)(s->st_host[i].count - before[i]) / (double)chunk;
                if (ri > r) r = ri;
            }
            s->rate = r;
            if (!overflow) break;
            /* Entries past the capacity were dropped: dedupe / cut every list, then re-run this chunk with a
             * size that cannot overflow.  What the failed run appended is valid and is deduplicated later.  The
             * duplicate filter knows the dropped cells as seen: it is emptied first. */
            rc = clear_seen(s);
            if (rc) return rc;
            rc = compact_scales(s, (1u << s->n_scales) - 1u);
            if (rc) return rc;
            rc = read_states(s);
            if (rc) return rc;
            free_min = s->cap;
            for (int i = 0; i < s->n_scales; ++i) {
                s->last_compact[i] = s->st_host[i].count;
                uint32_t fr = s->cap - s->st_host[i].count;
                if (fr < free_min) free_min = fr;
            }
            while (free_min < s->cap / 2) {
                rc = grow_candidates(s);
                if (rc) return rc;
                free_min = s->cap;
                for (int i = 0; i < s->n_scales; ++i) {
                    uint32_t fr = s->cap - s->st_host[i].count;
                    if (fr < free_min) free_min = fr;
                }
            }
            if (chunk > free_min) chunk = free_min & ~3u;
        }
        done += chunk;
        s->scanned += chunk;
        s->first_chunk = false;
        uint32_t due = 0;
        for (int i = 0; i < s->n_scales; ++i)
            if (wants_compaction(s, i)) due |= 1u << i;
        if (due) {
            int rc = compact_scales(s, due);
            if (rc) return rc;
            rc = read_states(s);
            if (rc) return rc;
            for (int i = 0; i < s->n_scales; ++i)
                if (!s->dirty[i]) s->last_compact[i] = s->st_host[i].count;
        }
    }
    s->scan_index += n;
    return CS_OK;
}

/* ---- strongly sampled streams: compact the kept particles once, then run every pass on them ------------------ */

constexpr double COMPACT_BELOW_P = 0.5;               /* sample_p below which compaction pays */
constexpr uint64_t COMPACT_MIN_N = 1ull << 20;

/* Kept particles of xyz[0..m) (running index index0) -> dst (room for cap particles); *cnt = their number, or
 * UINT64_MAX if they did not fit (the caller then takes another route for this chunk). */
int compact_chunk(cs_sketch* s, const float* xyz, uint64_t m, uint64_t index0, double sample_p, float* dst, uint64_t cap,
                  uint64_t* cnt) {
    CS_CUDA(cudaMemsetAsync(s->word_dev, 0, 4, s->stream));
    s->tm.mark(PH_COMPACT, s->stream);
    cudaError_t e = launch_compact_kept(xyz, m, index0, s->K, sample_threshold(sample_p), dst, s->word_dev,
                                        (uint32_t)(cap < 0xFFFFFFFFull ? cap : 0xFFFFFFFFull), s->sm_count, s->stream);
    s->tm.stop(s->stream);
    if (e != cudaSuccess) return fail(CS_ERR_CUDA, "compaction kernel: %s", cudaGetErrorString(e));
    s->launches += 1;
    CS_CUDA(cudaMemcpyAsync(s->word_host, s->word_dev, 4, cudaMemcpyDeviceToHost, s->stream));
    CS_CUDA(cudaStreamSynchronize(s->stream));
    *cnt = *s->word_host <= cap ? *s->word_host : UINT64_MAX;
    return CS_OK;
}

/* scratch buffer for the kept particles of one chunk (no replay cache, or the cache is full) */
int ensure_kept(cs_sketch* s, uint64_t m, double sample_p) {
    const uint64_t want = (uint64_t)((double)(m < s->compact_chunk ? m : s->compact_chunk) * sample_p * 1.05) + 65536;
    if (s->kept_cap >= want) return CS_OK;
    CS_CUDA(cudaStreamSynchronize(s->stream));
    if (s->kept) cudaFree(s->kept);
    s->kept = nullptr; s->kept_cap = 0;
    CS_CUDA(cudaMalloc(&s->kept, want * 12));
    s->kept_cap = want;
    return CS_OK;
}

bool wants_compaction_of_stream(uint64_t n, double sample_p) { return sample_p < COMPACT_BELOW_P && n >= COMPACT_MIN_N; }

/* Replay cache, sampled streams: reserve room for the kept particles of an update call over (xyz, n, index0, p) in the
 * arena.  Returns the index of the new segment, or -1 (cache off / no room: the caller uses the scratch buffer). */
int kept_seg_begin(cs_sketch* s, const float* xyz, uint64_t n, uint64_t index0, double p) {
    if (!s->replay_limit) return -1;
    for (size_t i = 0; i < s->kept_segs.size(); ++i)       /* the same buffer again: its old copy is stale */
        if (s->kept_segs[i].src == xyz && s->kept_segs[i].index0 == index0) s->kept_segs[i].n = 0;
    const uint64_t want = (uint64_t)((double)n * p * 1.05) + 65536;
    if (s->kept_arena_cap - s->kept_arena_used < want) {       /* grow (geometrically, within the budget), keeping what is held */
        const uint64_t room = s->replay_limit > s->host_cache_bytes ? (s->replay_limit - s->host_cache_bytes) / 12 : 0;
        uint64_t cap = 2 * s->kept_arena_cap > s->kept_arena_used + 2 * want ? 2 * s->kept_arena_cap : s->kept_arena_used + 2 * want;
        if (cap > room) cap = room;
        if (cap < s->kept_arena_used + want) return -1;
        float* grown = nullptr;
        if (cudaMalloc(&grown, cap * 12) != cudaSuccess) { cudaGetLastError(); return -1; }
        if (s->kept_arena) {
            if (cudaMemcpyAsync(grown, s->kept_arena, s->kept_arena_used * 12, cudaMemcpyDeviceToDevice, s->stream) != cudaSuccess ||
                cudaStreamSynchronize(s->stream) != cudaSuccess) { cudaGetLastError(); cudaFree(grown); return -1; }
            cudaFree(s->kept_arena);
        }
        s->kept_arena = grown;
        s->kept_arena_cap = cap;
    }
    if (s->kept_segs.size() >= 4096) return -1;
    cs_sketch::KeptSeg g = {xyz, n, index0, p, s->kept_arena_used, 0};
    s->kept_segs.push_back(g);
    return (int)s->kept_segs.size() - 1;
}

void kept_cache_clear(cs_sketch* s) { s->kept_segs.clear(); s->kept_arena_used = 0; }

int update_passes(cs_sketch* s, const float* xyz, uint64_t n, uint64_t index0, double sample_p) {
    if (!wants_compaction_of_stream(n, sample_p)) return update_passes_raw(s, xyz, n, index0, sample_p);
    int seg = kept_seg_begin(s, xyz, n, index0, sample_p);
    uint64_t pending = 0;                                     /* kept particles of the segment not yet added to the tables */
    for (uint64_t off = 0; off < n; off += s->compact_chunk) {
        const uint64_t m = n - off < s->compact_chunk ? n - off : s->compact_chunk;
        uint64_t cnt = UINT64_MAX;
        int rc = CS_OK;
        if (seg >= 0) {
            /* replay cache: all chunks are compacted into one segment first, the update then runs ONCE over it (fewer,
             * larger scatter launches: cfg 5 takes 4 instead of 16) */
            cs_sketch::KeptSeg& g = s->kept_segs[seg];
            float* dst = s->kept_arena + 3 * (g.off + g.cnt);
            rc = compact_chunk(s, xyz + 3 * off, m, index0 + off, sample_p, dst, s->kept_arena_cap - (g.off + g.cnt), &cnt);
            if (rc) return rc;
            if (cnt != UINT64_MAX) { g.cnt += cnt; pending += cnt; continue; }
            /* does not fit after all: no cache entry; what the segment holds so far is added now */
            if (pending) {
                rc = update_passes_raw(s, s->kept_arena + 3 * (g.off + g.cnt - pending), pending, 0, 1.0);
                if (rc) return rc;
                pending = 0;
            }
            s->kept_segs.pop_back();
            seg = -1;
        }
        rc = ensure_kept(s, m, sample_p);
        if (rc) return rc;
        rc = compact_chunk(s, xyz + 3 * off, m, index0 + off, sample_p, s->kept, s->kept_cap, &cnt);
        if (rc) return rc;
        if (cnt == UINT64_MAX) rc = update_passes_raw(s, xyz + 3 * off, m, index0 + off, sample_p);
        else if (cnt)          rc = update_passes_raw(s, s->kept, cnt, 0, 1.0);
        if (rc) return rc;
    }
    if (seg >= 0) {
        const cs_sketch::KeptSeg& g = s->kept_segs[seg];
        s->kept_arena_used = g.off + g.cnt;
        if (pending) return update_passes_raw(s, s->kept_arena + 3 * g.off, pending, 0, 1.0);
    }
    return CS_OK;
}

int scan_device(cs_sketch* s, const float* xyz, uint64_t n, double sample_p) {
    if (!wants_compaction_of_stream(n, sample_p)) return scan_device_raw(s, xyz, n, sample_p);
    for (size_t i = 0; i < s->kept_segs.size(); ++i) {       /* replay of a buffer whose kept particles are still held */
        const cs_sketch::KeptSeg& g = s->kept_segs[i];
        if (g.src == xyz && g.n == n && g.index0 == s->scan_index && g.p == sample_p) {
            const uint64_t next = s->scan_index + n;
            int rc = g.cnt ? scan_device_raw(s, s->kept_arena + 3 * g.off, g.cnt, 1.0) : CS_OK;
            s->scan_index = next;
            return rc;
        }
    }
    for (uint64_t off = 0; off < n; off += s->compact_chunk) {
        const uint64_t m = n - off < s->compact_chunk ? n - off : s->compact_chunk;
        uint64_t cnt = 0;
        int rc = ensure_kept(s, m, sample_p);
        if (rc) return rc;
        rc = compact_chunk(s, xyz + 3 * off, m, s->scan_index, sample_p, s->kept, s->kept_cap, &cnt);
        if (rc) return rc;
        if (cnt == UINT64_MAX) {
            rc = scan_device_raw(s, xyz + 3 * off, m, sample_p);       /* advances scan_index by m itself */
        } else {
            const uint64_t next = s->scan_index + m;
            if (cnt) rc = scan_device_raw(s, s->kept, cnt, 1.0);       /* p = 1: the index is not used */
            s->scan_index = next;
        }
        if (rc) return rc;
    }
    return CS_OK;
}

/* Bring the list of one scale into its final form (sorted, unique, cut) if anything was appended.  others_too (the
 * result calls cs_topk / cs_excursion): the other scales that wait for the same are compacted in the same launch, and
 * one read-back (a stream synchronisation) serves them all. */
int finalize_scale(cs_sketch* s, int i, bool others_too = false) {
    if (!s->dirty[i]) return CS_OK;
    uint32_t due = 0;
    for (int j = 0; j < s->n_scales; ++j)
        if (s->dirty[j] && (others_too || j == i)) due |= 1u << j;
    int rc = compact_scales(s, due);
    if (rc) return rc;
    rc = read_states(s);
    if (rc) return rc;
    for (int j = 0; j < s->n_scales; ++j)
        if (due >> j & 1u) s->last_compact[j] = s->st_host[j].count;
    return CS_OK;
}

int ensure_out(cs_sketch* s, uint64_t n) {
    if (n <= s->out_cap) return CS_OK;
    if (s->out_ids) cudaFree(s->out_ids);
    if (s->out_est) cudaFree(s->out_est);
    s->out_ids = nullptr; s->out_est = nullptr; s->out_cap = 0;
    CS_CUDA(cudaMalloc(&s->out_ids, n * sizeof(uint64_t)));
    CS_CUDA(cudaMalloc(&s->out_est, n * sizeof(int32_t)));
    s->out_cap = n;
    return CS_OK;
}

/* First n entries of the final list of scale i -> caller's buffers (device or host). */
int emit_prefix(cs_sketch* s, int i, uint32_t n, uint64_t* ids_out, int32_t* est_out) {
    if (!n) return CS_OK;
    int rc = ensure_out(s, n);
    if (rc) return rc;
    cudaError_t e = launch_emit_prefix(s->sb[i].id[s->cur[i]], s->sb[i].ek[s->cur[i]], n, s->out_ids, s->out_est, s->stream);
    if (e != cudaSuccess) return fail(CS_ERR_CUDA, "emit kernel: %s", cudaGetErrorString(e));
    s->launches += 1;
    CS_CUDA(cudaMemcpyAsync(ids_out, s->out_ids, (size_t)n * 8, cudaMemcpyDefault, s->stream));
    CS_CUDA(cudaMemcpyAsync(est_out, s->out_est, (size_t)n * 4, cudaMemcpyDefault, s->stream));
    CS_CUDA(cudaStreamSynchronize(s->stream));
    return CS_OK;
}

int ensure_staging(cs_sketch* s) {
    if (!s->copy_stream) {
        CS_CUDA(cudaStreamCreateWithFlags(&s->copy_stream, cudaStreamNonBlocking));
        for (int k = 0; k < STAGE_SLOTS; ++k) {
            CS_CUDA(cudaEventCreateWithFlags(&s->ev_full[k], cudaEventDisableTiming));
            CS_CUDA(cudaEventCreateWithFlags(&s->ev_free[k], cudaEventDisableTiming));
        }
    }
    return CS_OK;
}

void free_stage_slots(cs_sketch* s) {
    for (int k = 0; k < STAGE_SLOTS; ++k) {
        if (s->stage[k]) cudaFree(s->stage[k]);
        s->stage[k] = nullptr;
    }
    s->stage_alloc = 0;
}

int ensure_stage_slots(cs_sketch* s) {
    if (s->stage[0] && s->stage_alloc == s->stage_particles) return CS_OK;
    CS_CUDA(cudaStreamSynchronize(s->stream));
    free_stage_slots(s);
    for (int k = 0; k < STAGE_SLOTS; ++k) CS_CUDA(cudaMalloc(&s->stage[k], s->stage_particles * 12));
    s->stage_alloc = s->stage_particles;
    return CS_OK;
}

void free_host_cache(cs_sketch* s) {
    if (s->host_cache) cudaFree(s->host_cache);
    s->host_cache = nullptr; s->host_cache_bytes = 0; s->hc_valid = false;
}

/* Host-streamed pass (SURVEY 8.a a8; PAPER.md:295-298 batch flow, :570 I/O overlapped with compute): n items of bpp
 * bytes in host memory are cut into batches of stage_particles items; batch b is copied with cudaMemcpyAsync on the
 * copy stream into ring slot b mod 3 (after the kernels that last read the slot, ev_free) while the kernels of batch
 * b-1 run on the handle's stream; body(dev_ptr, items, first_item) enqueues the work of one batch.
 * Replay cache: when the handle may hold the whole buffer (cs_set_replay_cache), an update call copies the batches
 * into one device buffer instead of the ring (fill), and a following scan call of the same host buffer (replay) finds
 * them there: the stream crosses PCIe once. */
template <class Body>
int stream_host(cs_sketch* s, const void* host, size_t bpp, uint64_t n, bool fill_allowed, bool replay_allowed, Body body) {
    const uint64_t B = s->stage_particles;
    const uint64_t batches = (n + B - 1) / B;
    if (replay_allowed && s->hc_valid && s->hc_host == host && s->hc_n == n && s->hc_bpp == bpp) {
        for (uint64_t b = 0; b < batches; ++b) {
            const uint64_t off = b * B, m = n - off < B ? n - off : B;
            int rc = body(s->host_cache + off * bpp, m, off);
            if (rc) return rc;
        }
        return CS_OK;
    }
    int rc = ensure_staging(s);
    if (rc) return rc;
    bool fill = false;
    if (fill_allowed) {
        s->hc_valid = false;                               /* whatever was cached belongs to an older update call */
        const uint64_t kept_bytes = s->kept_arena_cap * 12;
        if (s->replay_limit >= kept_bytes && s->replay_limit - kept_bytes >= n * bpp) {
            if (s->host_cache_bytes < n * bpp) {
                CS_CUDA(cudaStreamSynchronize(s->stream));
                free_host_cache(s);
                if (cudaMalloc(&s->host_cache, n * bpp) == cudaSuccess) s->host_cache_bytes = n * bpp;
                else { cudaGetLastError(); s->host_cache = nullptr; }
            }
            fill = s->host_cache != nullptr;
        }
    }
    if (!fill) {
        rc = ensure_stage_slots(s);
        if (rc) return rc;
    }
    auto slot_ptr = [&](uint64_t b) -> unsigned char* {
        return fill ? s->host_cache + b * B * bpp : reinterpret_cast<unsigned char*>(s->stage[b % STAGE_SLOTS]);
    };
    auto copy_in = [&](uint64_t b) -> int {
        const int slot = (int)(b % STAGE_SLOTS);
        const uint64_t off = b * B, m = n - off < B ? n - off : B;
        if (!fill) CS_CUDA(cudaStreamWaitEvent(s->copy_stream, s->ev_free[slot], 0));
        CS_CUDA(cudaMemcpyAsync(slot_ptr(b), static_cast<const unsigned char*>(host) + off * bpp, m * bpp,
                                cudaMemcpyHostToDevice, s->copy_stream));
        CS_CUDA(cudaEventRecord(s->ev_full[slot], s->copy_stream));
        return CS_OK;
    };
    rc = copy_in(0);
    if (rc) return rc;
    for (uint64_t b = 0; b < batches; ++b) {
        if (b + 1 < batches) {                               /* the next copy runs while this batch is processed */
            rc = copy_in(b + 1);
            if (rc) return rc;
        }
        const int slot = (int)(b % STAGE_SLOTS);
        const uint64_t off = b * B, m = n - off < B ? n - off : B;
        CS_CUDA(cudaStreamWaitEvent(s->stream, s->ev_full[slot], 0));
        rc = body(slot_ptr(b), m, off);
        if (rc) return rc;
        CS_CUDA(cudaEventRecord(s->ev_free[slot], s->stream));
    }
    CS_CUDA(cudaStreamSynchronize(s->copy_stream));          /* the host buffer may be reused on return */
    if (fill) { s->hc_host = host; s->hc_n = n; s->hc_bpp = bpp; s->hc_valid = true; }
    return CS_OK;
}

int ensure_ids_scratch(cs_sketch* s, uint64_t ids) {
    if (s->ids_scratch_cap >= ids) return CS_OK;
    CS_CUDA(cudaStreamSynchronize(s->stream));
    if (s->ids_scratch) cudaFree(s->ids_scratch);
    s->ids_scratch = nullptr; s->ids_scratch_cap = 0;
    CS_CUDA(cudaMalloc(&s->ids_scratch, ids * sizeof(uint64_t)));
    s->ids_scratch_cap = ids;
    return CS_OK;
}

int check_xyz(const cs_sketch* s, const float* xyz, uint64_t n, double sample_p) {
    if (!s) return fail(CS_ERR_ARG, "null handle");
    if (bad_p(sample_p)) return fail(CS_ERR_ARG, "sample_p must be in (0, 1]");
    if (n && !xyz) return fail(CS_ERR_ARG, "null positions with n > 0");
    if (reinterpret_cast<uintptr_t>(xyz) & 3u) return fail(CS_ERR_ARG, "positions must be 4-byte aligned");
    return CS_OK;
}

}  // namespace

namespace {

/* Finest mesh of the handle if every other mesh divides it (packed records need nested meshes), else 0. */
uint32_t finest_nested_mesh(const cs_sketch* s) {
    uint32_t gf = 0;
    for (int i = 0; i < s->n_scales; ++i) if (s->G[i] > gf) gf = s->G[i];
    for (int i = 0; i < s->n_scales; ++i) if (gf % s->G[i]) return 0;
    return gf;
}

int check_records(const cs_sketch* s, const uint64_t* recs, uint64_t n, double sample_p) {
    if (!s) return fail(CS_ERR_ARG, "null handle");
    if (bad_p(sample_p)) return fail(CS_ERR_ARG, "sample_p must be in (0, 1]");
    if (n && !recs) return fail(CS_ERR_ARG, "null records with n > 0");
    if (reinterpret_cast<uintptr_t>(recs) & 7u) return fail(CS_ERR_ARG, "records must be 8-byte aligned");
    if (!finest_nested_mesh(s)) return fail(CS_ERR_ARG, "packed records need meshes that all divide the finest one");
    return CS_OK;
}

/* m <= stage_particles device records -> s->unpacked -> the ordinary update / scan passes */
int records_batch(cs_sketch* s, const uint64_t* recs_dev, uint64_t m, uint64_t index0, double sample_p, bool scan) {
    if (s->unpacked_alloc < m) {
        CS_CUDA(cudaStreamSynchronize(s->stream));
        if (s->unpacked) cudaFree(s->unpacked);
        s->unpacked = nullptr; s->unpacked_alloc = 0;
        const uint64_t want = m > s->stage_particles ? m : s->stage_particles;
        CS_CUDA(cudaMalloc(&s->unpacked, want * 12));
        s->unpacked_alloc = want;
    }
    const uint32_t gf = finest_nested_mesh(s);
    cudaError_t e = launch_unpack_centres(recs_dev, m, gf, (float)(s->L / (double)gf), s->unpacked, s->stream);
    if (e != cudaSuccess) return fail(CS_ERR_CUDA, "unpack kernel: %s", cudaGetErrorString(e));
    s->launches += 1;
    return scan ? scan_device(s, s->unpacked, m, sample_p) : update_passes(s, s->unpacked, m, index0, sample_p);
}

int records_device(cs_sketch* s, const uint64_t* recs_dev, uint64_t n, double sample_p, bool scan) {
    const uint64_t B = s->stage_particles;
    for (uint64_t off = 0; off < n; off += B) {
        const uint64_t m = n - off < B ? n - off : B;
        int rc = records_batch(s, recs_dev + off, m, s->upd_index + off, sample_p, scan);
        if (rc) return rc;
    }
    if (!scan) s->upd_index += n;
    return CS_OK;
}

/* records in host memory: 8 B per particle over PCIe through the same ring of staging slots */
int records_host(cs_sketch* s, const uint64_t* recs_host, uint64_t n, double sample_p, bool scan) {
    int rc = stream_host(s, recs_host, 8, n, !scan, scan, [&](const void* dev, uint64_t m, uint64_t off) -> int {
        return records_batch(s, static_cast<const uint64_t*>(dev), m, s->upd_index + off, sample_p, scan);
    });
    if (rc) return rc;
    if (!scan) s->upd_index += n;
    return CS_OK;
}

}  // namespace

/* =========================================================================================================
 * C ABI
 * ========================================================================================================= */

extern "C" {

const char* cs_version(void) { return "cs-b200 0.1 (sm_100a)"; }

const char* cs_last_error(void) { return g_err; }

int cs_derive_coeffs(uint64_t seed, int d, uint64_t* out_4d, uint64_t* K_out) {
    if (d < 1 || d > CS_MAX_ROWS || !out_4d) return fail(CS_ERR_ARG, "cs_derive_coeffs: bad d or null output");
    derive_coeffs(seed, d, out_4d, K_out);
    return CS_OK;
}

uint64_t cs_sample_threshold(double sample_p) { return sample_threshold(sample_p); }

int cs_hash_cell(uint64_t a, uint64_t b, uint64_t c, int big, uint64_t* r_out, uint32_t* low32_out) {
    if (!r_out || !low32_out) return fail(CS_ERR_ARG, "cs_hash_cell: null output");
    if (a < 1 || a >= P61 || b >= P61) return fail(CS_ERR_ARG, "cs_hash_cell: a must be in [1, p-1], b in [0, p-1]");
    if (c >= (1ull << 60) || (!big && c >= (1ull << 31)) || (big == 2 && (c >> 31) >= HASH_TB))
        return fail(CS_ERR_ARG, "cs_hash_cell: c out of range for this form");
    const HashCoef k = split_coef(a, b);
    if (big == 2) {
        const uint64_t tb = affine_mod_p<true>(k, 0u, cell_c1(c));      /* the table entry: (A*c1 + b) mod p */
        *low32_out = affine_low32_tb(k, cell_c0(c), tb);
        *r_out = affine_mod_p_tb(k, cell_c0(c), tb);
    } else if (big) {
        *r_out = affine_mod_p<true>(k, cell_c0(c), cell_c1(c));
        *low32_out = affine_low32<true>(k, cell_c0(c), cell_c1(c));
    } else {
        *r_out = affine_mod_p<false>(k, cell_c0(c), 0);
        *low32_out = affine_low32<false>(k, cell_c0(c), 0);
    }
    return CS_OK;
}

int cs_create_multi(cs_sketch** out, int n_scales, int d, uint64_t w, const uint32_t* G, double L, uint64_t seed) {
    if (!out) return fail(CS_ERR_ARG, "null output handle");
    *out = nullptr;
    if (!G) return fail(CS_ERR_ARG, "null grid list");
    if (n_scales < 1 || n_scales > CS_MAX_SCALES) return fail(CS_ERR_ARG, "n_scales must be in [1, %d]", CS_MAX_SCALES);
    if (d < 1 || d > CS_MAX_ROWS) return fail(CS_ERR_ARG, "d must be in [1, %d]", CS_MAX_ROWS);
    if (n_scales * d > CS_MAX_HASH_ROWS) return fail(CS_ERR_ARG, "n_scales * d must be <= %d", CS_MAX_HASH_ROWS);
    if (w < 1 || w > (1ull << 31)) return fail(CS_ERR_ARG, "w must be in [1, 2^31]");
    if (!(L > 0.0) || !std::isfinite(L)) return fail(CS_ERR_ARG, "L must be finite and > 0");
    for (int i = 0; i < n_scales; ++i)
        if (G[i] < 1 || G[i] > (1u << 20)) return fail(CS_ERR_ARG, "G must be in [1, 2^20]");

    int dev = 0;
    CS_CUDA(cudaGetDevice(&dev));
    cs_sketch* s = new (std::nothrow) cs_sketch();
    if (!s) return fail(CS_ERR_NOMEM, "host allocation failed");
    s->d = d; s->n_scales = n_scales; s->w = w; s->L = L; s->seed = seed; s->device = dev;
    /* the selector's 30-bit look-back epochs start three compactions short of where they are rewound (cs_select.cu), so
     * that every handle that lives that long takes the rewind once, early: a path that otherwise runs after ~10^8
     * compactions would never be exercised */
    for (int i = 0; i < n_scales; ++i) s->epoch[i] = 0x3FFFFFFFu - 64u;
    int sm = 0;
    if (cudaDeviceGetAttribute(&sm, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && sm > 0) s->sm_count = sm;

    PassParams& P = s->P;
    P.w = w; P.d = d; P.n_scales = n_scales; P.rank = (d - 1) / 2;
    for (int i = 0; i < n_scales; ++i) {
        uint64_t Ki = 0;
        derive_coeffs(seed + (uint64_t)i, d, s->coef[i], &Ki);
        if (i == 0) s->K = Ki;                                        /* one sampling key: scale 0's */
        for (int j = 0; j < d; ++j) {
            const uint64_t* c = &s->coef[i][4 * j];
            P.rows[i * d + j].h = split_coef(c[0], c[1]);
            P.rows[i * d + j].s = split_coef(c[2], c[3]);
        }
        s->G[i] = G[i];
        const uint64_t cells = (uint64_t)G[i] * G[i] * G[i];
        s->id_bits[i] = bit_length(cells - 1);
        P.sc[i].G = G[i];
        P.sc[i].qscale = (float)((double)G[i] / L);
        P.sc[i].top = (float)(G[i] - 1);
        P.sc[i].big = cells > (1ull << 31) ? 1u : 0u;
    }
    P.K = s->K;

    auto bail = [&](int rc) { cs_destroy(s); return rc; };
    for (int i = 0; i < n_scales; ++i) {
        cudaError_t e = cudaMalloc(&s->T[i], (size_t)d * w * sizeof(int32_t));
        if (e != cudaSuccess) return bail(fail(e == cudaErrorMemoryAllocation ? CS_ERR_NOMEM : CS_ERR_CUDA,
                                               "cudaMalloc(table): %s", cudaGetErrorString(e)));
        e = cudaMemset(s->T[i], 0, (size_t)d * w * sizeof(int32_t));
        if (e != cudaSuccess) return bail(fail(CS_ERR_CUDA, "cudaMemset(table): %s", cudaGetErrorString(e)));
        P.sc[i].T = s->T[i];
    }
    cudaError_t e = cudaMalloc(&s->st_dev, sizeof(ScanState) * CS_MAX_SCALES);
    if (e == cudaSuccess) e = cudaMallocHost(&s->st_host, sizeof(ScanState) * CS_MAX_SCALES);
    if (e == cudaSuccess) e = cudaMalloc(&s->word_dev, 64);
    if (e == cudaSuccess) e = cudaMallocHost(&s->word_host, 64);
    if (e != cudaSuccess) return bail(fail(CS_ERR_CUDA, "state allocation: %s", cudaGetErrorString(e)));
    memset(s->st_host, 0, sizeof(ScanState) * CS_MAX_SCALES);
    *out = s;
    return CS_OK;
}

int cs_create(cs_sketch** out, int d, uint64_t w, uint32_t G, double L, uint64_t seed) {
    return cs_create_multi(out, 1, d, w, &G, L, seed);
}

int cs_destroy(cs_sketch* s) {
    if (!s) return CS_OK;
    DeviceGuard guard_(s);
    if (s->stream || s->T[0]) cudaStreamSynchronize(s->stream);
    if (s->copy_stream) cudaStreamSynchronize(s->copy_stream);
    free_candidates(s);
    free_stage_lists(s);
    if (s->bins) cudaFree(s->bins);
    if (s->cursor) cudaFree(s->cursor);
    if (s->bin_stats) cudaFree(s->bin_stats);
    s->tm.destroy();
    if (s->kept) cudaFree(s->kept);
    if (s->unpacked) cudaFree(s->unpacked);
    for (int i = 0; i < CS_MAX_SCALES; ++i) if (s->bm[i]) cudaFree(s->bm[i]);
    if (s->coarse) cudaFree(s->coarse);
    for (int i = 0; i < CS_MAX_SCALES; ++i) if (s->T[i]) cudaFree(s->T[i]);
    if (s->st_dev) cudaFree(s->st_dev);
    if (s->st_host) cudaFreeHost(s->st_host);
    if (s->word_dev) cudaFree(s->word_dev);
    if (s->word_host) cudaFreeHost(s->word_host);
    if (s->out_ids) cudaFree(s->out_ids);
    if (s->out_est) cudaFree(s->out_est);
    for (int k = 0; k < STAGE_SLOTS; ++k) {
        if (s->stage[k]) cudaFree(s->stage[k]);
        if (s->ev_full[k]) cudaEventDestroy(s->ev_full[k]);
        if (s->ev_free[k]) cudaEventDestroy(s->ev_free[k]);
    }
    if (s->copy_stream) cudaStreamDestroy(s->copy_stream);
    if (s->host_cache) cudaFree(s->host_cache);
    if (s->kept_arena) cudaFree(s->kept_arena);
    if (s->ht_keys) cudaFree(s->ht_keys);
    if (s->ht_vals) cudaFree(s->ht_vals);
    if (s->ids_scratch) cudaFree(s->ids_scratch);
    delete s;
    return CS_OK;
}

int cs_reset(cs_sketch* s) {
    CS_ENTER(s);
    for (int i = 0; i < s->n_scales; ++i)
        CS_CUDA(cudaMemsetAsync(s->T[i], 0, (size_t)s->d * s->w * sizeof(int32_t), s->stream));
    s->upd_index = 0; s->scan_index = 0; s->scanning = false;
    kept_cache_clear(s);
    for (int i = 0; i < CS_MAX_SCALES; ++i) { s->dirty[i] = false; s->last_compact[i] = 0; }
    memset(s->st_host, 0, sizeof(ScanState) * CS_MAX_SCALES);
    return CS_OK;
}

int cs_set_stream(cs_sketch* s, void* cuda_stream) {
    CS_ENTER(s);
    CS_CUDA(cudaStreamSynchronize(s->stream));           /* work already queued finishes on the old stream */
    s->stream = (cudaStream_t)cuda_stream;
    return CS_OK;
}

int cs_set_table_budget(cs_sketch* s, uint64_t bytes) {
    CS_ENTER(s);
    if (bytes < 4) return fail(CS_ERR_ARG, "budget must be at least one counter");
    s->table_budget = bytes;
    return CS_OK;
}

int cs_set_chunk_sizes(cs_sketch* s, uint64_t stage_particles, uint64_t update_chunk, uint64_t scan_chunk,
                       uint64_t compact_chunk) {
    CS_ENTER(s);
    const uint64_t v[4] = {stage_particles, update_chunk, scan_chunk, compact_chunk};
    for (int i = 0; i < 4; ++i)
        if (v[i] && (v[i] < 64 || v[i] > (1ull << 30) || (v[i] & 3u)))
            return fail(CS_ERR_ARG, "chunk sizes must be multiples of 4 in [64, 2^30] (0 = keep)");
    if (stage_particles && stage_particles != s->stage_particles) {
        CS_CUDA(cudaStreamSynchronize(s->stream));
        if (s->copy_stream) CS_CUDA(cudaStreamSynchronize(s->copy_stream));
        free_stage_slots(s);
        kept_cache_clear(s);                               /* segments keyed by addresses inside the old ring */
        s->stage_particles = stage_particles;
    }
    if (update_chunk) s->bin_chunk = update_chunk;
    if (scan_chunk) s->scan_chunk = scan_chunk;
    if (compact_chunk) s->compact_chunk = compact_chunk;
    return CS_OK;
}

int cs_set_replay_cache(cs_sketch* s, uint64_t bytes) {
    CS_ENTER(s);
    CS_CUDA(cudaStreamSynchronize(s->stream));
    if (s->copy_stream) CS_CUDA(cudaStreamSynchronize(s->copy_stream));
    free_host_cache(s);
    if (s->kept_arena) cudaFree(s->kept_arena);
    s->kept_arena = nullptr; s->kept_arena_cap = 0;
    kept_cache_clear(s);
    s->replay_limit = bytes;
    return CS_OK;
}

int cs_set_update_mode(cs_sketch* s, int mode, int rows_direct) {
    CS_ENTER(s);
    if (mode < 0 || mode > 2 || rows_direct < -1 || rows_direct > CS_MAX_ROWS)
        return fail(CS_ERR_ARG, "mode must be 0 (auto), 1 (direct) or 2 (binned); rows_direct in [-1, 32]");
    s->update_mode = mode;
    s->bin_rows_direct = rows_direct;
    return CS_OK;
}

int cs_set_counting_mode(cs_sketch* s, int mode) {
    CS_ENTER(s);
    if (mode < 0 || mode > 1) return fail(CS_ERR_ARG, "mode must be 0 (Count Sketch) or 1 (Count-Min)");
    if (s->upd_index != 0 || s->scanning) return fail(CS_ERR_STATE, "the counting mode can only change on an empty sketch");
    for (int i = 0; i < s->n_scales; ++i)
        for (int j = 0; j < s->d; ++j) {
            const uint64_t* c = &s->coef[i][4 * j];
            /* Count-Min: a sign hash with all-zero limbs evaluates to residue 0, i.e. sign +1, in every form of cs_hash.h */
            s->P.rows[i * s->d + j].s = mode ? HashCoef{0, 0, 0, 0, 0, 0} : split_coef(c[2], c[3]);
        }
    s->P.rank = mode ? 0 : (s->d - 1) / 2;
    if (s->coarse) {                                   /* its shape depends on the rank */
        CS_CUDA(cudaStreamSynchronize(s->stream));
        cudaFree(s->coarse);
        s->coarse = nullptr;
    }
    return CS_OK;
}

int cs_set_scan_mode(cs_sketch* s, int mode) {
    CS_ENTER(s);
    if (mode < 0 || mode > 3) return fail(CS_ERR_ARG, "mode must be 0 (auto), 1 (plain), 2 (bitmap) or 3 (bitmap stages)");
    s->scan_mode = mode;
    return CS_OK;
}

int cs_set_update_index(cs_sketch* s, uint64_t index) {
    CS_ENTER(s);
    s->upd_index = index;
    return CS_OK;
}

int cs_set_scan_index(cs_sketch* s, uint64_t index) {
    CS_ENTER(s);
    s->scan_index = index;
    return CS_OK;
}

int cs_get_update_index(cs_sketch* s, uint64_t* index_out) {
    if (!s || !index_out) return fail(CS_ERR_ARG, "null argument");
    *index_out = s->upd_index;
    return CS_OK;
}

int cs_update(cs_sketch* s, const float* xyz_dev, uint64_t n, double sample_p) {
    int rc = check_xyz(s, xyz_dev, n, sample_p);
    if (rc) return rc;
    if (!n) return CS_OK;
    DeviceGuard guard_(s);
    rc = update_passes(s, xyz_dev, n, s->upd_index, sample_p);
    if (rc) return rc;
    s->upd_index += n;
    return CS_OK;
}

int cs_update_host(cs_sketch* s, const float* xyz_host, uint64_t n, double sample_p) {
    int rc = check_xyz(s, xyz_host, n, sample_p);
    if (rc) return rc;
    if (!n) return CS_OK;
    DeviceGuard guard_(s);
    rc = stream_host(s, xyz_host, 12, n, true, false, [&](const void* dev, uint64_t m, uint64_t off) -> int {
        return update_passes(s, static_cast<const float*>(dev), m, s->upd_index + off, sample_p);
    });
    if (rc) return rc;
    s->upd_index += n;
    return CS_OK;
}

int cs_pack_records(cs_sketch* s, const float* xyz_dev, uint64_t n, uint64_t* recs_dev) {
    CS_ENTER(s);
    if (n && (!xyz_dev || !recs_dev)) return fail(CS_ERR_ARG, "null buffer with n > 0");
    if ((reinterpret_cast<uintptr_t>(xyz_dev) & 3u) || (reinterpret_cast<uintptr_t>(recs_dev) & 7u))
        return fail(CS_ERR_ARG, "positions must be 4-byte aligned, records 8-byte aligned");
    cudaError_t e = launch_pack_records(xyz_dev, n, (float)((double)(1u << 21) / s->L), recs_dev, s->stream);
    if (e != cudaSuccess) return fail(CS_ERR_CUDA, "pack kernel: %s", cudaGetErrorString(e));
    s->launches += n ? 1 : 0;
    return CS_OK;
}

int cs_update_records(cs_sketch* s, const uint64_t* recs_dev, uint64_t n, double sample_p) {
    int rc = check_records(s, recs_dev, n, sample_p);
    if (rc || !n) return rc;
    DeviceGuard guard_(s);
    return records_device(s, recs_dev, n, sample_p, false);
}

int cs_update_records_host(cs_sketch* s, const uint64_t* recs_host, uint64_t n, double sample_p) {
    int rc = check_records(s, recs_host, n, sample_p);
    if (rc || !n) return rc;
    DeviceGuard guard_(s);
    return records_host(s, recs_host, n, sample_p, false);
}

int cs_scan_records(cs_sketch* s, const uint64_t* recs_dev, uint64_t n, double sample_p) {
    int rc = check_records(s, recs_dev, n, sample_p);
    if (rc) return rc;
    if (!s->scanning) return fail(CS_ERR_STATE, "cs_scan_records before cs_scan_begin");
    if (!n) return CS_OK;
    DeviceGuard guard_(s);
    return records_device(s, recs_dev, n, sample_p, true);
}

int cs_scan_records_host(cs_sketch* s, const uint64_t* recs_host, uint64_t n, double sample_p) {
    int rc = check_records(s, recs_host, n, sample_p);
    if (rc) return rc;
    if (!s->scanning) return fail(CS_ERR_STATE, "cs_scan_records_host before cs_scan_begin");
    if (!n) return CS_OK;
    DeviceGuard guard_(s);
    return records_host(s, recs_host, n, sample_p, true);
}

int cs_estimate(cs_sketch* s, int scale, const uint64_t* cells_dev, uint64_t m, int32_t* est_dev) {
    CS_ENTER(s);
    if (scale < 0 || scale >= s->n_scales) return fail(CS_ERR_ARG, "scale out of range");
    if (m && (!cells_dev || !est_dev)) return fail(CS_ERR_ARG, "null buffer with m > 0");
    if (!m) return CS_OK;
    PassParams P = pass_params(s, 0, 1.0);
    cudaError_t e = launch_estimate(P, scale, cells_dev, m, est_dev, s->stream);
    if (e != cudaSuccess) return fail(CS_ERR_CUDA, "estimate kernel: %s", cudaGetErrorString(e));
    s->launches += 1;
    return CS_OK;
}

int cs_scan_begin(cs_sketch* s, uint64_t k_max, int32_t thr_min) {
    CS_ENTER(s);
    if (k_max > (1ull << 26)) return fail(CS_ERR_ARG, "k_max must be <= 2^26");
    uint64_t want = 16 * k_max;                          /* <= 2^30, the limit of the list (grow_candidates) */
    if (want < s->cap_min) want = s->cap_min;
    uint64_t cap = s->cap_min;
    while (cap < want) cap *= 2;
    if (s->cap != cap) {
        int rc = alloc_candidates(s, (uint32_t)cap);
        if (rc) return rc;
    }
    s->k_max = k_max; s->thr_min = thr_min;
    s->scan_index = 0; s->rate = 1.0; s->first_chunk = true; s->n_scan_launches = 0; s->scanned = 0;
    for (int i = 0; i < CS_MAX_SCALES; ++i) s->bm_valid[i] = false;    /* the tables may have changed */
    for (int i = 0; i < s->n_scales; ++i) {
        s->st_host[i].count = 0;
        s->st_host[i].tau = k_max ? INT32_MIN : thr_min;
        s->st_host[i].est_min = INT32_MAX;
        s->st_host[i].est_max = INT32_MIN;
        s->st_host[i].uniq = 0;
        s->st_host[i].half = 0;
        s->cur[i] = 0;
        s->use_seen[i] = false;
        s->compact_n[i] = 0;
        s->dirty[i] = false; s->last_compact[i] = 0; s->n_compactions[i] = 0;
    }
    CS_CUDA(cudaMemcpyAsync(s->st_dev, s->st_host, sizeof(ScanState) * s->n_scales, cudaMemcpyHostToDevice, s->stream));
    CS_CUDA(cudaStreamSynchronize(s->stream));
    int rcs = clear_seen(s);
    if (rcs) return rcs;
    s->scanning = true;
    return CS_OK;
}

int cs_set_candidate_capacity(cs_sketch* s, uint64_t entries) {
    CS_ENTER(s);
    if (entries < 1024 || entries > (1ull << 30) || (entries & (entries - 1)))
        return fail(CS_ERR_ARG, "capacity must be a power of two in [2^10, 2^30]");
    s->cap_min = (uint32_t)entries;
    return CS_OK;
}

int cs_scan(cs_sketch* s, const float* xyz_dev, uint64_t n, double sample_p) {
    int rc = check_xyz(s, xyz_dev, n, sample_p);
    if (rc) return rc;
    if (!s->scanning) return fail(CS_ERR_STATE, "cs_scan before cs_scan_begin");
    if (!n) return CS_OK;
    DeviceGuard guard_(s);
    return scan_device(s, xyz_dev, n, sample_p);
}

int cs_scan_host(cs_sketch* s, const float* xyz_host, uint64_t n, double sample_p) {
    int rc = check_xyz(s, xyz_host, n, sample_p);
    if (rc) return rc;
    if (!s->scanning) return fail(CS_ERR_STATE, "cs_scan_host before cs_scan_begin");
    if (!n) return CS_OK;
    DeviceGuard guard_(s);
    return stream_host(s, xyz_host, 12, n, false, true, [&](const void* dev, uint64_t m, uint64_t) -> int {
        return scan_device(s, static_cast<const float*>(dev), m, sample_p);
    });
}

int cs_scan_cells(cs_sketch* s, int scale, const uint64_t* cells_dev, uint64_t m) {
    CS_ENTER(s);
    if (scale < 0 || scale >= s->n_scales) return fail(CS_ERR_ARG, "scale out of range");
    if (m && !cells_dev) return fail(CS_ERR_ARG, "null cells with m > 0");
    if (!s->scanning) return fail(CS_ERR_STATE, "cs_scan_cells before cs_scan_begin");
    uint64_t done = 0;
    while (done < m) {
        uint32_t held = s->st_host[scale].count;
        uint32_t fr = held < s->cap ? s->cap - held : 0;
        if (fr < s->cap / 2) {
            if (s->dirty[scale]) {
                int rc = finalize_scale(s, scale);
                if (rc) return rc;
                continue;
            }
            int rc = grow_candidates(s);
            if (rc) return rc;
            continue;
        }
        uint64_t chunk = m - done < fr ? m - done : fr;      /* cannot overflow: one entry per cell at most */
        ScanParams S;
        fill_scan_params(s, &S);
        PassParams P = pass_params(s, 0, 1.0);
        cudaError_t e = launch_scan_cells(P, S, scale, cells_dev + done, chunk, s->stream);
        if (e != cudaSuccess) return fail(CS_ERR_CUDA, "scan_cells kernel: %s", cudaGetErrorString(e));
        s->launches += 1;
        int rc = read_states(s);
        if (rc) return rc;
        if (s->st_host[scale].count != held) s->dirty[scale] = true;
        done += chunk;
    }
    return CS_OK;
}

int cs_scan_children(cs_sketch* s, int parent_scale, int child_scale, const uint64_t* parent_ids_dev, uint64_t m) {
    CS_ENTER(s);
    if (parent_scale < 0 || parent_scale >= s->n_scales || child_scale < 0 || child_scale >= s->n_scales)
        return fail(CS_ERR_ARG, "scale out of range");
    if (m && !parent_ids_dev) return fail(CS_ERR_ARG, "null parents with m > 0");
    if (!s->scanning) return fail(CS_ERR_STATE, "cs_scan_children before cs_scan_begin");
    const uint32_t Gp = s->G[parent_scale], Gc = s->G[child_scale];
    if (Gc % Gp || Gc / Gp < 1 || Gc / Gp > 64) return fail(CS_ERR_ARG, "the child mesh must be a 1..64-fold refinement of the parent mesh");
    const uint32_t r = Gc / Gp;
    const uint64_t r3 = (uint64_t)r * r * r;
    const uint64_t per = (1ull << 21) / r3 ? (1ull << 21) / r3 : 1;      /* parents per expansion: <= 2^21 ids (16 MiB) */
    int rc = ensure_ids_scratch(s, per * r3);
    if (rc) return rc;
    for (uint64_t off = 0; off < m && rc == CS_OK; off += per) {
        const uint64_t mm = m - off < per ? m - off : per;
        cudaError_t e = launch_expand_children(parent_ids_dev + off, mm, Gp, Gc, r, s->ids_scratch, s->stream);
        if (e != cudaSuccess) { rc = fail(CS_ERR_CUDA, "expand kernel: %s", cudaGetErrorString(e)); break; }
        s->launches += 1;
        rc = cs_scan_cells(s, child_scale, s->ids_scratch, mm * r3);
    }
    return rc;
}

int cs_scan_all(cs_sketch* s, int scale) {
    CS_ENTER(s);
    if (scale < 0 || scale >= s->n_scales) return fail(CS_ERR_ARG, "scale out of range");
    if (!s->scanning) return fail(CS_ERR_STATE, "cs_scan_all before cs_scan_begin");
    const uint64_t m = (uint64_t)s->G[scale] * s->G[scale] * s->G[scale];
    uint64_t done = 0;
    while (done < m) {
        uint32_t held = s->st_host[scale].count;
        uint32_t fr = held < s->cap ? s->cap - held : 0;
        if (fr < s->cap / 2) {                                   /* make room: compact (raises tau), else grow */
            if (s->dirty[scale]) {
                int rc = finalize_scale(s, scale);
                if (rc) return rc;
                continue;
            }
            int rc = grow_candidates(s);
            if (rc) return rc;
            continue;
        }
        /* optimistic chunk: few cells pass tau once the list is full; an overflow is detected, compacted and re-run */
        uint64_t chunk = s->st_host[scale].tau > INT32_MIN ? (uint64_t)fr * 64 : fr;
        if (chunk > m - done) chunk = m - done;
        for (;;) {
            ScanParams S;
            fill_scan_params(s, &S);
            PassParams P = pass_params(s, 0, 1.0);
            cudaError_t e = launch_scan_range(P, S, scale, done, chunk, s->stream);
            if (e != cudaSuccess) return fail(CS_ERR_CUDA, "scan_range kernel: %s", cudaGetErrorString(e));
            s->launches += 1;
            int rc = read_states(s);
            if (rc) return rc;
            if (s->st_host[scale].count != held) s->dirty[scale] = true;
            if (s->st_host[scale].count <= s->cap) break;
            rc = compact_scale(s, scale);                        /* entries past the capacity were dropped */
            if (rc) return rc;
            rc = read_states(s);
            if (rc) return rc;
            s->last_compact[scale] = s->st_host[scale].count;
            held = s->st_host[scale].count;
            while (s->cap - held < s->cap / 2) {
                rc = grow_candidates(s);
                if (rc) return rc;
            }
            if (chunk > s->cap - held) chunk = s->cap - held;    /* cannot overflow: one entry per cell at most */
        }
        done += chunk;
        if (wants_compaction(s, scale)) {
            int rc = finalize_scale(s, scale);
            if (rc) return rc;
        }
    }
    return CS_OK;
}

int cs_topk(cs_sketch* s, int scale, uint64_t k, uint64_t* ids_out, int32_t* est_out, uint64_t* n_out) {
    if (!s || !n_out) return fail(CS_ERR_ARG, "null argument");
    DeviceGuard guard_(s);
    if (scale < 0 || scale >= s->n_scales) return fail(CS_ERR_ARG, "scale out of range");
    if (k && (!ids_out || !est_out)) return fail(CS_ERR_ARG, "null output with k > 0");
    if (!s->scanning) return fail(CS_ERR_STATE, "cs_topk before cs_scan_begin");
    if (k > s->k_max) return fail(CS_ERR_ARG, "k exceeds the k_max given to cs_scan_begin");
    int rc = finalize_scale(s, scale, true);
    if (rc) return rc;
    const uint32_t held = s->st_host[scale].count;
    const uint32_t n = k < held ? (uint32_t)k : held;
    rc = emit_prefix(s, scale, n, ids_out, est_out);
    if (rc) return rc;
    *n_out = n;
    return CS_OK;
}

int cs_excursion(cs_sketch* s, int scale, int32_t thr, uint64_t cap, uint64_t* ids_out, int32_t* est_out,
                 uint64_t* n_total) {
    if (!s || !n_total) return fail(CS_ERR_ARG, "null argument");
    DeviceGuard guard_(s);
    if (scale < 0 || scale >= s->n_scales) return fail(CS_ERR_ARG, "scale out of range");
    if (cap && (!ids_out || !est_out)) return fail(CS_ERR_ARG, "null output with cap > 0");
    if (!s->scanning) return fail(CS_ERR_STATE, "cs_excursion before cs_scan_begin");
    if (thr < s->thr_min) return fail(CS_ERR_ARG, "thr is below the thr_min given to cs_scan_begin");
    int rc = finalize_scale(s, scale, true);
    if (rc) return rc;
    const uint32_t held = s->st_host[scale].count;
    cudaError_t e = launch_count_ge(s->sb[scale].ek[s->cur[scale]], held, thr, s->word_dev, s->stream);
    if (e != cudaSuccess) return fail(CS_ERR_CUDA, "count kernel: %s", cudaGetErrorString(e));
    s->launches += 1;
    CS_CUDA(cudaMemcpyAsync(s->word_host, s->word_dev, 4, cudaMemcpyDeviceToHost, s->stream));
    CS_CUDA(cudaStreamSynchronize(s->stream));
    const uint32_t total = *s->word_host;
    const uint32_t n = cap < total ? (uint32_t)cap : total;
    rc = emit_prefix(s, scale, n, ids_out, est_out);
    if (rc) return rc;
    *n_total = total;
    return CS_OK;
}

int cs_recount(cs_sketch* s, int scale, const uint64_t* ids_dev, uint64_t m, const float* xyz_dev, uint64_t n,
               uint32_t* counts_dev, float* xyz_out_dev, uint64_t cap, uint64_t* n_out) {
    CS_ENTER(s);
    if (scale < 0 || scale >= s->n_scales) return fail(CS_ERR_ARG, "scale out of range");
    if (m > (1ull << 28)) return fail(CS_ERR_ARG, "at most 2^28 cells");
    if ((m && (!ids_dev || !counts_dev)) || (n && !xyz_dev)) return fail(CS_ERR_ARG, "null buffer with a non-zero size");
    if (reinterpret_cast<uintptr_t>(xyz_dev) & 3u) return fail(CS_ERR_ARG, "positions must be 4-byte aligned");
    if (xyz_out_dev && !n_out) return fail(CS_ERR_ARG, "n_out is required with xyz_out_dev");
    if (n_out) *n_out = 0;
    if (!m || !n) return CS_OK;
    uint64_t size = 1024;
    while (size < 4 * m) size *= 2;                                   /* load factor <= 1/4 */
    if (s->ht_size < size) {
        CS_CUDA(cudaStreamSynchronize(s->stream));
        if (s->ht_keys) cudaFree(s->ht_keys);
        if (s->ht_vals) cudaFree(s->ht_vals);
        s->ht_keys = nullptr; s->ht_vals = nullptr; s->ht_size = 0;
        CS_CUDA(cudaMalloc(&s->ht_keys, size * sizeof(uint64_t)));
        CS_CUDA(cudaMalloc(&s->ht_vals, size * sizeof(uint32_t)));
        s->ht_size = size;
    }
    CS_CUDA(cudaMemsetAsync(s->ht_keys, 0xFF, size * sizeof(uint64_t), s->stream));
    CS_CUDA(cudaMemsetAsync(s->ht_vals, 0xFF, size * sizeof(uint32_t), s->stream));
    CS_CUDA(cudaMemsetAsync(s->word_dev, 0, 4, s->stream));
    cudaError_t e = launch_ht_build(ids_dev, (uint32_t)m, s->ht_keys, s->ht_vals, (uint32_t)(size - 1), s->stream);
    if (e == cudaSuccess)
        e = launch_recount(s->P.sc[scale], xyz_dev, n, s->ht_keys, s->ht_vals, (uint32_t)(size - 1), counts_dev, xyz_out_dev,
                           s->word_dev, cap, s->sm_count, s->stream);
    if (e != cudaSuccess) return fail(CS_ERR_CUDA, "cs_recount: %s", cudaGetErrorString(e));
    s->launches += 2;
    CS_CUDA(cudaMemcpyAsync(s->word_host, s->word_dev, 4, cudaMemcpyDeviceToHost, s->stream));
    CS_CUDA(cudaStreamSynchronize(s->stream));
    if (n_out) *n_out = *s->word_host;
    return CS_OK;
}

/* 26-neighbour shell (Fig. 14: the heavy cells "and their surroundings"): ids_out[27*i + t], t =
 * (dx+1) + 3*(dy+1) + 9*(dz+1), = the cell at offset (dx, dy, dz) from ids_dev[i] on the mesh of `scale`, wrapped
 * periodically (the box is periodic, BASELINE.json configs); t = 13 is the cell itself. */
int cs_expand_neighbours(cs_sketch* s, int scale, const uint64_t* ids_dev, uint64_t m, uint64_t* ids_out_dev) {
    CS_ENTER(s);
    if (scale < 0 || scale >= s->n_scales) return fail(CS_ERR_ARG, "scale out of range");
    if (m && (!ids_dev || !ids_out_dev)) return fail(CS_ERR_ARG, "null buffer with m > 0");
    if (m > (1ull << 32)) return fail(CS_ERR_ARG, "at most 2^32 cells");
    if (!m) return CS_OK;
    cudaError_t e = launch_expand_neighbours(ids_dev, m, s->G[scale], ids_out_dev, s->stream);
    if (e != cudaSuccess) return fail(CS_ERR_CUDA, "neighbour kernel: %s", cudaGetErrorString(e));
    s->launches += 1;
    return CS_OK;
}

int cs_scan_stats(cs_sketch* s, int scale, uint64_t* out4_host) {
    if (!s || !out4_host) return fail(CS_ERR_ARG, "null argument");
    DeviceGuard guard_(s);
    if (scale < 0 || scale >= s->n_scales) return fail(CS_ERR_ARG, "scale out of range");
    if (!s->scanning) return fail(CS_ERR_STATE, "cs_scan_stats before cs_scan_begin");
    int rc = read_states(s);
    if (rc) return rc;
    out4_host[0] = s->st_host[scale].count;
    out4_host[1] = (uint64_t)(int64_t)s->st_host[scale].tau;
    out4_host[2] = s->n_compactions[scale];
    out4_host[3] = s->n_scan_launches;
    return CS_OK;
}

int cs_sketch_read(cs_sketch* s, int scale, int32_t* out_d_by_w) {
    if (!s || !out_d_by_w) return fail(CS_ERR_ARG, "null argument");
    DeviceGuard guard_(s);
    if (scale < 0 || scale >= s->n_scales) return fail(CS_ERR_ARG, "scale out of range");
    CS_CUDA(cudaMemcpyAsync(out_d_by_w, s->T[scale], (size_t)s->d * s->w * sizeof(int32_t), cudaMemcpyDefault, s->stream));
    CS_CUDA(cudaStreamSynchronize(s->stream));
    return CS_OK;
}

int cs_sketch_add(cs_sketch* s, int scale, const int32_t* in_d_by_w) {
    if (!s || !in_d_by_w) return fail(CS_ERR_ARG, "null argument");
    DeviceGuard guard_(s);
    if (scale < 0 || scale >= s->n_scales) return fail(CS_ERR_ARG, "scale out of range");
    const uint64_t n = (uint64_t)s->d * s->w;
    cudaPointerAttributes at;
    const int32_t* src = in_d_by_w;
    int32_t* tmp = nullptr;
    cudaError_t e = cudaPointerGetAttributes(&at, in_d_by_w);
    if (e != cudaSuccess || at.type != cudaMemoryTypeDevice) {        /* host input: stage it on the device */
        cudaGetLastError();
        CS_CUDA(cudaMalloc(&tmp, n * sizeof(int32_t)));
        e = cudaMemcpyAsync(tmp, in_d_by_w, n * sizeof(int32_t), cudaMemcpyHostToDevice, s->stream);
        if (e != cudaSuccess) { cudaFree(tmp); return fail(CS_ERR_CUDA, "cudaMemcpyAsync: %s", cudaGetErrorString(e)); }
        src = tmp;
    }
    e = launch_table_add(s->T[scale], src, n, s->stream);
    s->launches += 1;
    if (tmp) {
        cudaStreamSynchronize(s->stream);
        cudaFree(tmp);
    }
    if (e != cudaSuccess) return fail(CS_ERR_CUDA, "table add kernel: %s", cudaGetErrorString(e));
    return CS_OK;
}

int cs_table_ptr(cs_sketch* s, int scale, int32_t** table_dev_out) {
    if (!s || !table_dev_out) return fail(CS_ERR_ARG, "null argument");
    if (scale < 0 || scale >= s->n_scales) return fail(CS_ERR_ARG, "scale out of range");
    *table_dev_out = s->T[scale];
    return CS_OK;
}

int cs_coeffs(cs_sketch* s, int scale, uint64_t* out_4d_host, uint64_t* K_out_host) {
    if (!s || !out_4d_host) return fail(CS_ERR_ARG, "null argument");
    if (scale < 0 || scale >= s->n_scales) return fail(CS_ERR_ARG, "scale out of range");
    memcpy(out_4d_host, s->coef[scale], sizeof(uint64_t) * 4 * s->d);
    if (K_out_host) *K_out_host = s->K;
    return CS_OK;
}

int cs_set_timing(cs_sketch* s, int on) {
    CS_ENTER(s);
    CS_CUDA(cudaStreamSynchronize(s->stream));
    s->tm.clear();
    s->tm.on = on != 0;
    return CS_OK;
}

int cs_get_timing(cs_sketch* s, double* ms_out, uint64_t* spans_out) {
    CS_ENTER(s);
    if (!ms_out) return fail(CS_ERR_ARG, "null output");
    CS_CUDA(cudaStreamSynchronize(s->stream));
    for (int p = 0; p < CS_N_PHASES; ++p) { ms_out[p] = 0.0; if (spans_out) spans_out[p] = 0; }
    for (const PhaseTimer::Span& sp : s->tm.spans) {
        float ms = 0.f;
        CS_CUDA(cudaEventElapsedTime(&ms, s->tm.pool[sp.a], s->tm.pool[sp.b]));
        ms_out[sp.phase] += ms;
        if (spans_out) spans_out[sp.phase] += 1;
    }
    s->tm.clear();
    return CS_OK;
}

int cs_update_stats(cs_sketch* s, uint64_t* out4_host) {
    CS_ENTER(s);
    if (!out4_host) return fail(CS_ERR_ARG, "null output");
    for (int i = 0; i < 4; ++i) out4_host[i] = 0;
    if (!s->bin_stats) return CS_OK;
    unsigned long long v[4];
    CS_CUDA(cudaMemcpyAsync(v, s->bin_stats, sizeof(v), cudaMemcpyDeviceToHost, s->stream));
    CS_CUDA(cudaStreamSynchronize(s->stream));
    CS_CUDA(cudaMemsetAsync(s->bin_stats, 0, sizeof(v), s->stream));
    for (int i = 0; i < 4; ++i) out4_host[i] = v[i];
    return CS_OK;
}

int cs_launch_count(cs_sketch* s, uint64_t* n_out) {
    if (!s || !n_out) return fail(CS_ERR_ARG, "null argument");
    DeviceGuard guard_(s);
    *n_out = s->launches;
    return CS_OK;
}

int cs_select_static(const uint64_t* ids_dev, const int32_t* est_dev, uint64_t n, uint64_t k, uint64_t* ids_out_dev,
                     int32_t* est_out_dev, uint32_t* n_out_dev, void* cuda_stream) {
    if (n > CS_SELECT_STATIC_MAX_N)
        return fail(CS_ERR_ARG, "cs_select_static: n = %llu candidates exceed the static scratch (CS_SELECT_STATIC_MAX_N = %u)",
                    (unsigned long long)n, (unsigned)CS_SELECT_STATIC_MAX_N);
    if (k > CS_SELECT_STATIC_MAX_N)
        return fail(CS_ERR_ARG, "cs_select_static: k = %llu exceeds CS_SELECT_STATIC_MAX_N = %u", (unsigned long long)k,
                    (unsigned)CS_SELECT_STATIC_MAX_N);
    if (!n_out_dev || (n && (!ids_dev || !est_dev)) || (n && k && (!ids_out_dev || !est_out_dev)))
        return fail(CS_ERR_ARG, "cs_select_static: null pointer with a non-zero size");
    cudaError_t e = select_static(ids_dev, est_dev, (uint32_t)n, (uint32_t)k, ids_out_dev, est_out_dev, n_out_dev,
                                  (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return fail(CS_ERR_CUDA, "cs_select_static: %s", cudaGetErrorString(e));
    return CS_OK;
}

}  /* extern "C" */
