/*
 * cs.h -- C ABI of libcs.so: the Count-Sketch heavy-hitter pass of arXiv 1711.00975 on one B200 (sm_100a).
 *
 * Problem statement this boundary follows (PAPER.md = the paper's text; DESIGN.md section 3 = readings):
 *   given N-body particles in a box and a regular G^3 mesh, return the k cells holding the most particles
 *   with an estimate of each count, and the excursion set = all cells whose estimated
 *   count is at least a limit, in ONE streaming pass over the particles into a
 *   Count Sketch plus one replay of the stream against the finished sketch
 *   (estimate mode, restricted to the cells that occur in the stream).
 *
 * Conventions for every call
 *   - extern "C", returns an int status: CS_OK (0) or a negative CS_ERR_* code.  Nothing throws, aborts or
 *     prints.  cs_last_error() returns a thread-local, NUL-terminated message for the last failing call.
 *   - "dev" pointers are CUDA device memory on the handle's device (the device that was current at cs_create; every
 *     call switches to it for its duration and restores the caller's current device); "host" pointers are host memory (pinned
 *     memory makes the host-streamed calls asynchronous, pageable memory is accepted and slower); "any"
 *     pointers may be either (the library copies with cudaMemcpyDefault).
 *   - The caller owns every input / output buffer.  The handle owns the counter tables, the candidate buffers,
 *     the staging ring and all scratch; cs_destroy frees them.
 *   - All device work is enqueued on the handle's stream (cs_set_stream; default: the legacy default stream).
 *     cs_estimate / cs_sketch_add / cs_reset do not synchronise.  cs_update is asynchronous except that it waits for
 *     the stream when it (re)allocates its record scratch (first large call) and, for sample_p < 0.5, once per 2^28
 *     particles to read back the number of kept particles.  cs_update_host returns after the last host->device copy
 *     has been issued and waited for (the host buffer may then be reused); cs_scan*, cs_topk, cs_excursion,
 *     cs_recount, cs_sketch_read, cs_scan_stats synchronise the stream because they hand host-visible results or
 *     sizes back.
 *   - Positions are an array of structures: float32 x,y,z per particle, 12 bytes per particle, at least
 *     4-byte aligned (16-byte aligned input takes the fully vectorised path from its first particle).
 *   - There is no CPU fallback: every step below runs in CUDA kernels of this library; without a usable
 *     CUDA device cs_create fails with CS_ERR_CUDA.
 *
 * Arithmetic (bit-exact contract; the paper fixes only "2-independent hashes",
 * PAPER.md:105, and "4-byte integer counters"):
 *   p = 2^61 - 1.  splitmix64 stream of seed: x_n = mix64(seed + n*0x9E3779B97F4A7C15), n = 1, 2, ...
 *   Row j of a scale takes x_{4j+1..4j+4} as a_j, b_j, a'_j, b'_j with a = (x mod (p-1)) + 1, b = x mod p;
 *   sampling key K = x_{4d+1} of scale 0; scale s draws from the stream of seed + s.
 *   quantise: per axis i = (uint32) min(max(floorf(x * (float)((double)G / L)), 0), G-1)  (one IEEE binary32
 *   multiply, no FMA; NaN -> 0);  cell id c = ix + G*(iy + G*iz)  (uint64).
 *   bucket h_j(c) = ((a_j*c + b_j) mod p) mod w;  sign s_j(c) = 1 - 2*(((a'_j*c + b'_j) mod p) & 1).
 *   Add(c): T[j][h_j(c)] += s_j(c) for every row j (int32, wraparound)
 *   Estimate(c) = the floor((d-1)/2)-th smallest (0-based) of s_j(c)*T[j][h_j(c)]
 *   sampling (sample_p < 1): the particle with running index i (0-based, counted over every particle passed
 *   in, kept or not) is kept iff mix64(K + (i+1)*0x9E3779B97F4A7C15) < floor(sample_p * 2^64).
 */
#ifndef CS_H_
#define CS_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define CS_OK          0
#define CS_ERR_ARG    -1   /* invalid argument (ranges below), null pointer with a non-zero size */
#define CS_ERR_NOMEM  -2   /* host or device allocation failed */
#define CS_ERR_CUDA   -3   /* a CUDA runtime call or kernel failed; text in cs_last_error() */
#define CS_ERR_STATE  -4   /* call out of order (cs_scan / cs_topk / cs_excursion before cs_scan_begin) */

#define CS_MAX_ROWS    32  /* d */
#define CS_MAX_SCALES  8   /* grids sketched in one pass */
#define CS_MAX_HASH_ROWS 64 /* n_scales * d: all hash coefficients travel as kernel parameters */

typedef struct cs_sketch cs_sketch;   /* opaque */

/* ---- host-only helpers (no CUDA device needed) --------------------------------------------------------- */

/* Library version string, e.g. "cs-b200 0.1 (sm_100a)". */
const char* cs_version(void);

/* Message of the last failing call on this thread ("" if none). */
const char* cs_last_error(void);

/* Hash coefficients of one scale, as the library derives them on the host (R1-R2):
 * out_4d[4*j + 0..3] = a_j, b_j, a'_j, b'_j for j < d; *K_out (may be NULL) = sampling key x_{4d+1}.
 * 1 <= d <= CS_MAX_ROWS.  Pure host arithmetic. */
int cs_derive_coeffs(uint64_t seed, int d, uint64_t* out_4d, uint64_t* K_out);

/* floor(sample_p * 2^64) as the sampler compares against (R13); 0 for p outside (0, 1). */
uint64_t cs_sample_threshold(double sample_p);

/* Host evaluation of the library's limb-split hash arithmetic -- the same inline functions the kernels compile
 * (csrc/cs_hash.h) -- so that it can be checked against big-integer arithmetic without a GPU:
 * *r_out = (a*c + b) mod (2^61-1), canonical, through the full-residue form; *low32_out = its low 32 bits through
 * the short form the kernels use for power-of-two w and for the sign.  big = 0 selects the form compiled for
 * meshes with G^3 <= 2^31 (needs c < 2^31), big = 1 the general one (c < 2^60), big = 2 the table form used when
 * the high limb of every cell id is < 64 (needs c < 2^37).  1 <= a < p, b < p. */
int cs_hash_cell(uint64_t a, uint64_t b, uint64_t c, int big, uint64_t* r_out, uint32_t* low32_out);

/* ---- life cycle --------------------------------------------------------------------------------------- */

/* cs_create: one sketch of d rows x w int32 counters over a G^3 mesh on a box of side L.
 * cs_create_multi: n_scales sketches (same d, w; grid G[s], coefficients from seed + s) updated and scanned
 * together in one pass over the particles with one sampling decision per particle.
 * Ranges: 1 <= d <= 32, 1 <= w <= 2^31, 1 <= G <= 2^20 (so G^3 <= 2^60 < p), L finite and > 0,
 * 1 <= n_scales <= 8, n_scales*d <= 64.  Allocates d*w*4 bytes per scale, zeroed.  *out receives the handle. */
int cs_create(cs_sketch** out, int d, uint64_t w, uint32_t G, double L, uint64_t seed);
int cs_create_multi(cs_sketch** out, int n_scales, int d, uint64_t w, const uint32_t* G_host, double L,
                    uint64_t seed);
int cs_destroy(cs_sketch* s);                       /* NULL is accepted */

/* Zero the tables, the running particle indices and the candidates; leaves scan mode. */
int cs_reset(cs_sketch* s);

/* Use `cuda_stream` (a cudaStream_t, e.g. torch.cuda.current_stream().cuda_stream) for all later work. */
int cs_set_stream(cs_sketch* s, void* cuda_stream);

/* Bytes of counters one update pass may touch (default 64 MiB).  When d*w*4*n_scales exceeds it, cs_update
 * splits the rows (or scales) into groups of at most this size and re-reads the positions once per group, so
 * that the red.global.add traffic of each pass stays L2-resident.  The result does not depend on it. */
int cs_set_table_budget(cs_sketch* s, uint64_t bytes);

/* How the passes cut one call into launches (0 = keep the current value); the result never depends on it.
 *   stage_particles  particles per batch of the host-streamed calls = size of one slot of the device staging ring
 *                    (default 2^24: 3 slots x 192 MiB); changing it frees the ring, which is re-allocated on use
 *   update_chunk     particles per scatter/apply pair of the binned update (default 2^30, halved down to 2^27 while the
 *                    record scratch -- 2 B x binned rows per particle, 8.6 GB for 2^30 particles at d = 7 -- would take
 *                    more than a quarter of the free device memory)
 *   scan_chunk       most particles one re-scan launch covers (default 2^27)
 *   compact_chunk    particles per sampling-compaction launch when sample_p < 0.5 (default 2^28)
 * Each a multiple of 4 in [64, 2^30].  Small values make short streams take the multi-batch paths (tests do). */
int cs_set_chunk_sizes(cs_sketch* s, uint64_t stage_particles, uint64_t update_chunk, uint64_t scan_chunk,
                       uint64_t compact_chunk);

/* Replay cache (default 0 = off).  With bytes > 0 the handle may hold up to that much device memory with what the last
 * cs_update* calls read, so that the re-scan of the SAME buffer does not fetch it again:
 *   - cs_update_host / cs_update_records_host of a buffer of at most `bytes` copy it into one device buffer instead of
 *     the staging ring; a following cs_scan_host / cs_scan_records_host with the same host address and length reads
 *     that copy: the stream crosses PCIe once per update + re-scan instead of twice;
 *   - for sample_p < 0.5 the kept particles that cs_update* compacted stay on the device (12 B each); a cs_scan* call
 *     with the same address, length, sample_p and running index re-scans them without a second sampling pass.
 * The caller promises that such a buffer still holds the same particles when it is passed to cs_scan*.  Every
 * cs_update* call refreshes what is held for its buffer; cs_reset drops the kept particles.  Synchronises; frees what
 * was held. */
int cs_set_replay_cache(cs_sketch* s, uint64_t bytes);

/* How cs_update applies the counter updates.  The result never depends on it.
 *   mode 1 "direct": one red.global.add.s32 per (particle, row) into L2-resident row groups (table budget above).
 *   mode 2 "binned": updates are first written as 2-byte records partitioned by table slice, then applied slice by
 *           slice in shared memory (csrc/cs_update_binned.cu); needs w a power of two in [2^8, 2^25], else falls
 *           back to direct.  rows_direct rows of every binned pass still take the direct route, concurrently
 *           (0 = none, -1 = automatic, the default: about 4/7 of the rows while they fit the table budget).
 *   mode 0 "auto" (default): binned for calls of at least 2^22 particles when the shape allows it. */
int cs_set_update_mode(cs_sketch* s, int mode, int rows_direct);

/* Counting mode.  0 (default): Count Sketch as described at the top.  1: the Count-Min variant the paper compares with
 * (Fig. 10): Add increments every row's counter by +1 (no sign hash), Estimate is the MINIMUM
 * over the rows; everything else (hashes h_j, sampling, re-scan, top-k, excursion sets) is unchanged.  Only allowed
 * on an empty sketch (after cs_create / cs_reset, before the first cs_update), else CS_ERR_STATE. */
int cs_set_counting_mode(cs_sketch* s, int mode);

/* How cs_scan evaluates cells.  The result never depends on it.
 *   mode 1 "plain": every cell gets the early-exit estimate from the int32 tables.
 *   mode 2 "bitmap": once the collection threshold tau is >= 1 (and w is a power of two), a 1-bit-per-counter
 *           bitmap |T| >= tau is built and every cell is first tested against it with the bucket hashes alone
 *           (csrc/cs_scan_bitmap.cu); survivors get the exact estimate.
 *   mode 3 "bitmap stages": the same bitmap plus a coarse copy of its first (d-1)/2 + 1 rows in shared memory decide
 *           the first rows; survivors run the remaining rows on dense warps (csrc/cs_scan_staged.cu).  Single-scale
 *           handles, 2 <= d <= 10, w a power of two >= 4096; else as mode 2.
 *   mode 0 "auto" (default): mode 3 where it applies, else mode 1. */
int cs_set_scan_mode(cs_sketch* s, int mode);

/* Running particle index of the update stream / of the current scan (sampling, R13, R17).
 * Setting it lets a stream shard (multi-GPU) reproduce the single-stream sampling decisions. */
int cs_set_update_index(cs_sketch* s, uint64_t index);
int cs_set_scan_index(cs_sketch* s, uint64_t index);
int cs_get_update_index(cs_sketch* s, uint64_t* index_out);

/* ---- stream processing: Alg. 1 l.3-5, Add(M, cell) per kept particle ------ */

/* n particles at xyz_dev (device, AoS float32).  sample_p in (0, 1]; 1 keeps everything and computes no
 * sampling hash.  n = 0 is a no-op.  Asynchronous on the handle's stream. */
int cs_update(cs_sketch* s, const float* xyz_dev, uint64_t n, double sample_p);

/* Same for particles in HOST memory: copied in batches through a ring of device staging buffers with
 * cudaMemcpyAsync on a copy stream, overlapped with the update kernel of the previous batch
 * (PAPER.md:295-298 batch flow, :570 I/O overlapped with compute). */
int cs_update_host(cs_sketch* s, const float* xyz_host, uint64_t n, double sample_p);

/* ---- packed 64-bit particle records ("3 coordinates in 64 bits"; R23) --------------------
 * A record is the particle's cell on the 2^21 mesh: rec = qx | qy << 21 | qz << 42 with q = the quantisation above for
 * G = 2^21.  Its cell on a mesh of G <= 2^20 cells per axis is, per axis, i = (q * G) >> 21 (exact integer rule; it can
 * differ from the float32 rule by one cell for positions within 2^-21 L of a cell boundary).  8 bytes instead of 12
 * cross PCIe in the host-streamed calls.  All meshes of the handle must divide its finest mesh, else CS_ERR_ARG.
 * cs_pack_records converts device positions to records (asynchronous on the handle's stream); the other four calls
 * mirror cs_update / cs_update_host / cs_scan / cs_scan_host, running index and sampling included. */
int cs_pack_records(cs_sketch* s, const float* xyz_dev, uint64_t n, uint64_t* recs_dev);
int cs_update_records(cs_sketch* s, const uint64_t* recs_dev, uint64_t n, double sample_p);
int cs_update_records_host(cs_sketch* s, const uint64_t* recs_host, uint64_t n, double sample_p);
int cs_scan_records(cs_sketch* s, const uint64_t* recs_dev, uint64_t n, double sample_p);
int cs_scan_records_host(cs_sketch* s, const uint64_t* recs_host, uint64_t n, double sample_p);

/* ---- queries ------------------------------------------------------------------------------------------ */

/* est_dev[i] = Estimate(cells_dev[i]) against scale `scale`.  m = 0 is a no-op.
 * Any 64-bit id is accepted and hashed as (a*c + b) mod p; ids of this mesh are < G^3. */
int cs_estimate(cs_sketch* s, int scale, const uint64_t* cells_dev, uint64_t m, int32_t* est_dev);

/* Candidate re-scan (estimate mode restricted to the cells that occur in the replayed stream; R10).
 * cs_scan_begin clears the candidates and the scan index and fixes what may be asked afterwards:
 *   top-k for any k <= k_max, excursion sets for any threshold >= thr_min
 *   (k_max = 0: no top-k; thr_min = INT32_MAX: no excursion set).
 * cs_scan / cs_scan_host replay particles (normally the same stream with the same sample_p, after the last
 * cs_update): every kept particle's cell is estimated against the CURRENT tables; cells whose estimate can
 * still matter are collected, deduplicated and kept ordered by (estimate descending, cell id ascending).
 * The tables must not change between cs_scan_begin and the last cs_topk / cs_excursion. */
int cs_scan_begin(cs_sketch* s, uint64_t k_max, int32_t thr_min);   /* k_max <= 2^26, else CS_ERR_ARG */
/* Initial capacity (entries per scale, a power of two in [2^10, 2^30]; default 2^22) of the candidate list the
 * next cs_scan_begin allocates: max(entries, 16*k_max rounded up to a power of two) <= 2^30.  The list still grows by
 * doubling when the cells that must be kept do not fit; a small value only costs more compactions. */
int cs_set_candidate_capacity(cs_sketch* s, uint64_t entries);
int cs_scan(cs_sketch* s, const float* xyz_dev, uint64_t n, double sample_p);
int cs_scan_host(cs_sketch* s, const float* xyz_host, uint64_t n, double sample_p);

/* Feed cell ids directly as candidates of `scale` (estimated against the current tables, deduplicated with the
 * scanned ones).  Used to merge the candidate lists of several stream shards. */
int cs_scan_cells(cs_sketch* s, int scale, const uint64_t* cells_dev, uint64_t m);

/* Full-dictionary search (Alg. 1 l.7-13; the paper's "GPU without heap" query, :304-306): every cell
 * id 0 .. G^3 - 1 of `scale` becomes a candidate, no positions needed.  Cost grows with G^3 (d gathers per cell until
 * tau rejects early): meant for small meshes and as a cross-check of the re-scan; combine with cs_topk / cs_excursion. */
int cs_scan_all(cs_sketch* s, int scale);

/* Hierarchical, positions-free query (Alg. 3 CSHi: search the coarse layer in full, then
 * only the children of its heavy cells).  With nested meshes (cs_create_multi, G[child] = r * G[parent], r <= 64) the
 * r^3 sub-cells of each given parent cell become candidates of `child_scale`.  Typical use: cs_scan_all(coarse) ->
 * cs_topk(coarse, c*k) -> cs_scan_children(coarse, fine, ids) -> cs_topk(fine, k).  parent_ids_dev: device. */
int cs_scan_children(cs_sketch* s, int parent_scale, int child_scale, const uint64_t* parent_ids_dev, uint64_t m);

/* Top-k (made deterministic, R9): the first min(k, #candidates)
 * candidates in (estimate descending, cell id ascending) order.  ids_out / est_out: any pointer, room for k
 * entries; *n_out (host) = number written.  k <= k_max.  The first result call (cs_topk / cs_excursion) after a scan puts
 * the candidate lists of ALL scales that still wait into their final order, in one launch behind one synchronisation;
 * later result calls on any scale only copy. */
int cs_topk(cs_sketch* s, int scale, uint64_t k, uint64_t* ids_out, int32_t* est_out, uint64_t* n_out);

/* Excursion set (R8): every candidate with estimate >= thr, same order.  Writes the
 * first min(cap, total) entries; *n_total (host) = total.  thr >= thr_min.  Raw estimates, no 1/p rescale. */
int cs_excursion(cs_sketch* s, int scale, int32_t thr, uint64_t cap, uint64_t* ids_out, int32_t* est_out,
                 uint64_t* n_total);

/* Second pass over the stream restricted to m given cells of `scale` (normally the output of cs_topk / cs_excursion;
 * PAPER.md:502-506 keep the particles of the heavy cells for an offline halo finder, :548, :556 exact number of
 * particles in the output cells).  For the n particles at xyz_dev (device, no sampling):
 *   counts_dev[i] += number of particles whose cell is ids_dev[i]   (device, m words, NOT zeroed by the call, so that
 *                    batches accumulate; duplicate ids: the first occurrence counts);
 *   if xyz_out_dev != NULL: those particles are copied there in arbitrary order, at most `cap` of them (device);
 *   *n_out (host) = how many particles of this call belong to the cells (may exceed cap).
 * Synchronises the stream.  m <= 2^28. */
int cs_recount(cs_sketch* s, int scale, const uint64_t* ids_dev, uint64_t m, const float* xyz_dev, uint64_t n,
               uint32_t* counts_dev, float* xyz_out_dev, uint64_t cap, uint64_t* n_out);

/* 26-neighbour shell of m cells of `scale` on the periodic mesh (Fig. 14: keep the particles of the
 * heavy cells AND THEIR SURROUNDINGS for an offline halo finder): ids_out_dev[27*i + t], t = (dx+1) + 3*(dy+1) + 9*(dz+1)
 * with dx, dy, dz in {-1, 0, 1}, = the cell at that offset from ids_dev[i], coordinates wrapped modulo G (t = 13 is the
 * cell itself).  Feed the result to cs_recount (duplicates are harmless there).  Device pointers; ids < G^3;
 * m <= 2^32; asynchronous on the handle's stream. */
int cs_expand_neighbours(cs_sketch* s, int scale, const uint64_t* ids_dev, uint64_t m, uint64_t* ids_out_dev);

/* out4[0] = candidates currently held, out4[1] = current collection threshold tau as (uint64)(int64)tau,
 * out4[2] = compactions run since cs_scan_begin, out4[3] = scan kernel launches since cs_scan_begin. */
int cs_scan_stats(cs_sketch* s, int scale, uint64_t* out4_host);

/* ---- table access: save / restore / merge by linearity ----------------------------------- */

int cs_sketch_read(cs_sketch* s, int scale, int32_t* out_d_by_w);       /* any pointer; row-major T[j*w + b] */
int cs_sketch_add(cs_sketch* s, int scale, const int32_t* in_d_by_w);   /* any pointer; T += in, wraparound  */
int cs_coeffs(cs_sketch* s, int scale, uint64_t* out_4d_host, uint64_t* K_out_host);

/* Device address of the d*w int32 counters of `scale` (row-major, owned by the handle, valid until cs_destroy), so that
 * a collective can sum the tables of several GPUs IN PLACE (ncclAllReduce(int32, sum) on this buffer: PAPER.md:578,
 * SURVEY 8.e) instead of copying them out and adding them back.  The caller orders its accesses after the handle's
 * stream (cs_set_stream) and must not touch the buffer while a cs_update* / cs_scan* call is in flight. */
int cs_table_ptr(cs_sketch* s, int scale, int32_t** table_dev_out);

/* Phase timing.  cs_set_timing(s, 1) makes the handle record CUDA events on its stream between the launches of its
 * kernel classes (one event per class change: no synchronisation, microseconds of host time); cs_get_timing synchronises
 * the stream, writes ms_out[p] = device time spent in phase p since the last call and spans_out[p] (may be NULL) = number
 * of launch groups it was measured over, and forgets them.  Phases: 0 update scatter (k_bin_scatter, or k_update in
 * direct mode), 1 update apply (k_bin_apply), 2 sampling compaction (k_compact_kept), 3 first scan stage / one-kernel
 * scans, 4 later scan stages, 5 bitmap builds, 6 selection (sort + unique + cut), 7 unused. */
#define CS_N_PHASES 8
int cs_set_timing(cs_sketch* s, int on);
int cs_get_timing(cs_sketch* s, double* ms_out, uint64_t* spans_out);

/* Routes the counter updates of the binned cs_update took since the last call (then zeroed): out4[0] = applied with
 * red.global because a shared-memory staging buffer was full, out4[1] = because a bin region was full (both only on
 * heavily duplicated streams), out4[2] = leftovers of partial staging buffers at kernel end, out4[3] = written as
 * binned records.  Synchronises. */
int cs_update_stats(cs_sketch* s, uint64_t* out4_host);

/* Number of kernels this handle has launched since create (bench.py's gpu_launches). */
int cs_launch_count(cs_sketch* s, uint64_t* n_out);

/* ---- measurement probes (the roofline denominators are measured, not assumed) -------------
 * NOT part of the product path: no other call of this library uses them; bench.py calls them to measure the peaks
 * its roofline fractions are quoted against.  They take no handle and run on the current device. */

/* Issues n_ops red.global.add.s32 (mode 0), returning atom.global.add.s32 (mode 1) or 4-byte ld.global
 * gathers (mode 2) to addresses generated in registers, uniform over a table of table_bytes, from all SMs,
 * `reps` times, on `cuda_stream`; *ms_out = average device time of one repetition (CUDA events). */
int cs_probe_l2(int mode, uint64_t table_bytes, uint64_t n_ops, int reps, void* cuda_stream, double* ms_out);

/* Same stream-read shape as cs_update (16-byte loads of n particles) with no hashing or atomics:
 * the position-stream term of the roofline.  *ms_out = average device time of one pass. */
int cs_probe_stream(const float* xyz_dev, uint64_t n, int reps, void* cuda_stream, double* ms_out);

/* ---- selection without any allocation ------------------------------------------------------------------------------
 * For callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid it).  The deterministic selection of PAPER.md:142-147 / :306 (R9) over a candidate list the caller
 * already holds on the device: n pairs (cell id, estimate), e.g. ids of its own and their cs_estimate values.  Output: the
 * distinct ids in the order (estimate descending, id ascending), cut to the first k -- what cs_scan_cells + cs_topk
 * return for the same cells.  Pairs with equal ids must carry equal estimates (as estimates of one sketch do).
 *
 * It takes no handle and runs on the CURRENT device, on `cuda_stream` (a cudaStream_t; NULL = the legacy default
 * stream); all pointers are device pointers on that device: ids_dev[n], est_dev[n] in; ids_out_dev[k], est_out_dev[k]
 * and *n_out_dev (= min(k, number of distinct ids)) out.  Nothing is copied to the host and nothing synchronises: the
 * results are valid once the stream has passed the call.  Inputs are not modified; outputs must not overlap inputs.
 *
 * Its scratch (both halves of the sorting buffer, digit counts, look-back status words: 24 bytes per candidate + 85 KB,
 * 1.6 MB in all) is a file-scope device array inside the library: every GPU that loads the library holds it from load to
 * exit, and the call makes no cudaMalloc / cudaFree / allocating library call.  The first call on each device looks the
 * array's device address up (cudaGetSymbolAddress); make that call outside stream capture.
 *   n > CS_SELECT_STATIC_MAX_N or k > CS_SELECT_STATIC_MAX_N  ->  CS_ERR_ARG, nothing is launched.
 * Every call on a device shares the one array, which keeps the last call's contents (each call re-initialises what must
 * start at zero): calls that overlap on the GPU -- two streams, two host threads -- race.  Calls on one stream, or
 * otherwise ordered, are safe.  Launches 3 kernels (load, one cooperative compaction, emit). */
#define CS_SELECT_STATIC_MAX_N 65536u
int cs_select_static(const uint64_t* ids_dev, const int32_t* est_dev, uint64_t n, uint64_t k, uint64_t* ids_out_dev,
                     int32_t* est_out_dev, uint32_t* n_out_dev, void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* CS_H_ */
