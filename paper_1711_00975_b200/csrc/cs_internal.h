/*
 * cs_internal.h -- structures shared by the host runtime (cs_api.cu) and the kernels (cs_kernels.cu,
 * cs_select.cu) of libcs.so.  Nothing in oracle/ includes this file.
 */
#ifndef CS_INTERNAL_H_
#define CS_INTERNAL_H_

#include <cuda_runtime.h>
#include <stdint.h>

#include <vector>

#include "../../include/cs.h"
#include "cs_hash.h"

namespace cs {

/* Phase timing (cs_set_timing / cs_get_timing): CUDA events recorded on the handle's stream between the launches of
 * the kernel classes below; mark(p) closes the running span and opens one of phase p, stop() closes it.  Off: no-ops. */
enum Phase { PH_SCATTER = 0, PH_APPLY, PH_COMPACT, PH_SCAN_FIRST, PH_SCAN_NEXT, PH_BITMAP, PH_SELECT, PH_OTHER, PH_COUNT };
struct PhaseTimer {
    bool on = false;
    std::vector<cudaEvent_t> pool;
    size_t used = 0;
    struct Span { int phase; size_t a, b; };
    std::vector<Span> spans;
    int open_phase = -1;
    size_t open_ev = 0;
    size_t record(cudaStream_t st) {
        if (used == pool.size()) {
            cudaEvent_t e;
            cudaEventCreate(&e);
            pool.push_back(e);
        }
        cudaEventRecord(pool[used], st);
        return used++;
    }
    void mark(int phase, cudaStream_t st) {
        if (!on) return;
        const size_t e = record(st);
        if (open_phase >= 0) spans.push_back({open_phase, open_ev, e});
        open_phase = phase;
        open_ev = e;
    }
    void stop(cudaStream_t st) {
        if (!on || open_phase < 0) return;
        const size_t e = record(st);
        spans.push_back({open_phase, open_ev, e});
        open_phase = -1;
    }
    void clear() { spans.clear(); used = 0; open_phase = -1; }
    void destroy() { for (cudaEvent_t e : pool) cudaEventDestroy(e); pool.clear(); clear(); }
};

constexpr uint64_t GAMMA = 0x9E3779B97F4A7C15ULL;     // splitmix64 increment

struct RowCoef {
    HashCoef h;   // bucket hash
    HashCoef s;   // sign hash
};

struct ScaleParams {
    int32_t* T;        // d*w counters of this scale, row-major T[j*w + b]
    float qscale;      // (float)((double)G / L)
    float top;         // (float)(G - 1)
    uint32_t G;
    uint32_t big;      // 1 if G^3 > 2^31 (cell ids need the c1 multiplies, cs_hash.h)
};

/* Per-scale candidate collection state, in device memory, mirrored to pinned host memory after each chunk. */
struct ScanState {
    uint32_t count;    // entries appended (may exceed cap: the excess was dropped -> chunk is re-run)
    int32_t tau;       // current collection threshold: only estimates >= tau are collected
    int32_t est_min;   // min / max estimate among the entries held (bounds the radix passes over the estimate)
    int32_t est_max;
    uint32_t uniq;     // number of unique entries after the last compaction, before the cut
    uint32_t half;     // which half of the ping-pong candidate buffers holds the list (set by every compaction)
    uint32_t pad[2];
};

struct ScanTarget {
    uint64_t* id;      // candidate cell ids      (current ping-pong half)
    uint32_t* ek;      // candidate keys: 0x7FFFFFFF - est  (ascending key = descending estimate)
    ScanState* st;
    uint32_t cap;
    uint32_t seen_mask;            // slots - 1 of the seen set (0: no set)
    unsigned long long* seen;      // open-addressing set of the cells that reached the final check of this scan (see
                                   // seen_first_time, cs_scan_common.cuh); all-ones = empty slot
};

/* Everything a pass over particles needs, passed by value as a __grid_constant__ kernel parameter
 * (constant bank -> uniform registers; < 4 KB). */
struct PassParams {
    RowCoef rows[CS_MAX_HASH_ROWS];     // rows[s*d + j]
    ScaleParams sc[CS_MAX_SCALES];
    uint64_t w;                          // counters per row
    uint64_t K;                          // sampling key
    uint64_t Tp;                         // floor(sample_p * 2^64)
    uint64_t index0;                     // running index of particle 0 of this launch
    int32_t d;
    int32_t n_scales;
    int32_t sample;                      // 0: keep everything (sample_p >= 1)
    int32_t rank;                        // Estimate = the rank-th smallest row value: (d-1)/2 (median), 0 for Count-Min
};

struct ScanParams {
    ScanTarget tg[CS_MAX_SCALES];
};

/* Binned update (cs_update_binned.cu): the rows of one pass are cut into slices of 2^log2S counters; bin =
 * (row, slice) = counter index >> log2S; a record is (offset in slice) << 1 | sign bit, 2 bytes. */
struct BinParams {
    uint16_t* bins;       // nb regions of `cap` records each
    uint32_t* cursor;     // records reserved per bin (zeroed before each pass)
    uint32_t cap;         // records per bin region, a multiple of 32
    uint32_t nb;          // bins of this pass = binned rows << (log2w - log2S)
    uint32_t threads;     // CTA size of the scatter kernel (512 or 1024)
    uint32_t C;           // records per shared-memory staging buffer, a multiple of 8
    uint32_t pairs;       // pairs of particles per thread between two flush phases (the host sizes C with it)
    uint32_t log2S;       // <= 15
    uint32_t log2w;
    int32_t rows_direct;  // the first rows_direct rows of the pass use red.global instead of the bins
    unsigned long long* stats;  // 4 counters (may be NULL): records that left the binned route -- [0] staging buffer full,
                                // [1] bin region full, [2] leftovers of partial buffers at kernel end; [3] records binned
};
size_t scatter_smem_bytes(uint32_t nb, uint32_t C);
cudaError_t launch_update_binned(const PassParams& P, const BinParams& B, const float* xyz, uint64_t n, int sm_count,
                                 cudaStream_t st, PhaseTimer* tm);

/* kernel launchers (cs_kernels.cu) */
cudaError_t launch_pack_records(const float* xyz, uint64_t n, float qscale21, uint64_t* recs, cudaStream_t st);
cudaError_t launch_unpack_centres(const uint64_t* recs, uint64_t n, uint32_t Gf, float cell_f, float* xyz, cudaStream_t st);
cudaError_t launch_compact_kept(const float* xyz, uint64_t n, uint64_t index0, uint64_t K, uint64_t Tp, float* out,
                                uint32_t* count, uint32_t cap, int sm_count, cudaStream_t st);
cudaError_t launch_update(const PassParams& P, const float* xyz, uint64_t n, int sm_count, cudaStream_t st);
cudaError_t launch_scan(const PassParams& P, const ScanParams& S, const float* xyz, uint64_t n, int sm_count,
                        cudaStream_t st);
/* bitmap-prefiltered scan (cs_scan_bitmap.cu) */
cudaError_t launch_build_bitmap(const int32_t* T, uint64_t n_counters, int32_t tau, uint32_t* bm, cudaStream_t st);
cudaError_t launch_scan_bitmap(const PassParams& P, const ScanParams& S, const uint32_t* const* bm, const float* xyz,
                               uint64_t n, int sm_count, cudaStream_t st);
/* row-partitioned scan of one scale (cs_scan_staged.cu) */
struct StageBuffers {
    uint64_t* list[2];     // survivor lists (ping-pong), cap_entries each
    uint32_t* cnt[2];      // entries per segment, `blocks` words each
    uint32_t blocks;       // grid size of every stage = number of segments
    uint64_t cap_entries;
};
uint64_t staged_list_entries(uint64_t n, uint32_t blocks);
cudaError_t launch_scan_staged(const PassParams& P, const ScanTarget& tg, const StageBuffers& B, int rows_per_stage,
                               const float* xyz, uint64_t n, cudaStream_t st, uint64_t* launches, PhaseTimer* tm);
/* Coarse bitmap of the first rank+1 rows held in shared memory by the first scan stage: the first n_fine rows at one bit
 * per 2^(g-1) counters, the others at one bit per 2^g counters (as fine as 224 KB of shared memory allow). */
struct CoarseShape {
    uint32_t g, n_fine;
    uint32_t row_off[6];       // word offset of row j; row_off[first] = total words
};
bool coarse_shape(int d, int rank, uint64_t w, CoarseShape* out);
cudaError_t launch_scan_staged_cb(const PassParams& P, const ScanTarget& tg, const StageBuffers& B, const uint32_t* fine,
                                  uint32_t* coarse, const CoarseShape& shape, bool rebuild_coarse, const float* xyz,
                                  uint64_t n, int sm_count, cudaStream_t st, uint64_t* launches, PhaseTimer* tm);
cudaError_t launch_scan_cells(const PassParams& P, const ScanParams& S, int scale, const uint64_t* cells,
                              uint64_t m, cudaStream_t st);
cudaError_t launch_scan_range(const PassParams& P, const ScanParams& S, int scale, uint64_t first, uint64_t m,
                              cudaStream_t st);
cudaError_t launch_expand_children(const uint64_t* parents, uint64_t m, uint32_t Gp, uint32_t Gc, uint32_t r, uint64_t* out,
                                   cudaStream_t st);
cudaError_t launch_expand_neighbours(const uint64_t* ids, uint64_t m, uint32_t G, uint64_t* out, cudaStream_t st);
cudaError_t launch_estimate(const PassParams& P, int scale, const uint64_t* cells, uint64_t m, int32_t* est,
                            cudaStream_t st);
cudaError_t launch_table_add(int32_t* T, const int32_t* in, uint64_t n, cudaStream_t st);

/* second pass restricted to output cells (cs_recount.cu) */
cudaError_t launch_ht_build(const uint64_t* ids, uint32_t m, uint64_t* keys, uint32_t* vals, uint32_t mask, cudaStream_t st);
cudaError_t launch_recount(const ScaleParams& sp, const float* xyz, uint64_t n, const uint64_t* keys, const uint32_t* vals,
                           uint32_t mask, uint32_t* counts, float* out, uint32_t* out_count, uint64_t cap, int sm_count,
                           cudaStream_t st);

/* selection (cs_select.cu): sort the first n candidates of one half by (ek ascending, id ascending), drop
 * duplicate ids, cut to the entries that can still matter and update *st (count, tau, est_min, est_max, half).
 * scratch: at least select_scratch_words(cap) uint32 words. */
struct SelectBuffers {
    uint64_t* id[2];
    uint32_t* ek[2];
    uint32_t* scratch;
};
uint64_t select_scratch_words(uint64_t cap);      /* scratch must be zeroed once after allocation */
/* Enqueues one compaction of the first n entries of half `src` of buffers with room for `cap` entries: no host round
 * trip inside; st_dev->half / count / tau describe the result.  *launches += kernels launched; *epoch: per-buffer counter. */
cudaError_t select_compact(const SelectBuffers& B, uint32_t cap, int src, uint32_t n, int id_bits, ScanState* st_dev,
                           uint64_t k_max, int32_t thr_min, cudaStream_t stream, uint64_t* launches, uint32_t* epoch);
cudaError_t launch_emit_prefix(const uint64_t* id, const uint32_t* ek, uint32_t n, uint64_t* ids_out,
                               int32_t* est_out, cudaStream_t st);
/* number of leading entries (sorted by ek ascending) with estimate >= thr, written to *n_out_dev */
cudaError_t launch_count_ge(const uint32_t* ek, uint32_t n, int32_t thr, uint32_t* n_out_dev, cudaStream_t st);

}  // namespace cs
#endif
