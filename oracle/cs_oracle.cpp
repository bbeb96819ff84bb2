/*
 * cs_oracle.cpp -- CPU ORACLE for the Count-Sketch heavy-hitter pass of arXiv 1711.00975.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may build, load or call it.  It shares no code,
 * header, table or constant generator with paper_1711_00975_b200/ (the CUDA path) and must never be
 * imported by it.  It is deliberately plain: single-threaded, one particle at a time, the paper's
 * operations written out in the paper's order, 128-bit integers and the `%` operator for the modular
 * hashes, std::sort / std::set for selection.  No blocking, fusion, early exit or reordering.
 *
 * What each function follows (PAPER.md = /root/reference/PAPER.md; readings = DESIGN.md section 3):
 *   ora_splitmix64 / ora_coeffs   DESIGN.md R1-R2 (the paper only asks for 2-independent hashes)
 *   ora_affine_mod_p              h(c) = (a*c + b) mod (2^61-1), canonical residue; R1
 *   ora_quantise                  stage 1 "compute cell ID from XYZ"; R7, R11
 *   ora_keep                      "sampling hash" per element; R13
 *   ora_update                    Add(M, s): for all i in [t]: M[i][h_{i,b}(s)] += h_{i,s}(s)
 *   ora_estimate                  Estimate(M, j): median_i M[i][h_{i,b}(j)] * h_{i,s}(j)
 *   ora_scan / ora_topk / ora_excursion
 *                                 estimate mode restricted to the cells seen in the replayed stream
 *                                 (R10), selection made deterministic
 *                                 (R9), excursion set = all cells with
 *                                 estimate >= threshold (R8)
 *   ora_select_streaming          the same selection over one shard of the stream in O(k) memory (full-size
 *                                 parity by shards; mergeability PAPER.md:578)
 *   ora_full_search_topk          Alg. 1 l.7-13 (CSFS query: Estimate every j in [n])
 *   ora_exact_counts              exact counting, PAPER.md:398-402 (the brute-force pin)
 *   ora_update_records / ora_scan_records / ora_cells_of_records
 *                                 the same passes over packed 64-bit records; R23
 *   ora_set_mode(1)               Count-Min variant: Add +1, Estimate = min over the rows
 *
 * Parity pins: tests/test_oracle_pins.py (run with -m "not gpu").  Every function above is pinned there;
 * nothing here is "parity unpinned" except the statistical quality on the paper's real data (out of scope).
 */
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <map>
#include <new>
#include <set>
#include <utility>
#include <vector>

typedef unsigned __int128 u128;

static const uint64_t P61 = (((uint64_t)1) << 61) - 1;       /* the Mersenne prime 2^61 - 1 */
static const uint64_t GAMMA = 0x9E3779B97F4A7C15ULL;          /* splitmix64 increment */

/* splitmix64 output function (public-domain algorithm by S. Vigna, restated). */
static uint64_t mix64(uint64_t z) {
    z ^= z >> 30;
    z *= 0xBF58476D1CE4E5B9ULL;
    z ^= z >> 27;
    z *= 0x94D049BB133111EBULL;
    z ^= z >> 31;
    return z;
}

/* n-th output (n = 1, 2, ...) of the splitmix64 stream started at `seed`: x_n = mix(seed + n*gamma). */
static uint64_t splitmix_nth(uint64_t seed, uint64_t n) { return mix64(seed + n * GAMMA); }

struct RowCoef {
    uint64_t a, b;   /* bucket hash  h(c) = ((a*c + b) mod p) mod w */
    uint64_t a2, b2; /* sign hash    s(c) = 1 - 2*(((a2*c + b2) mod p) & 1) */
};

struct Scale {
    uint32_t G;
    float scale;                 /* (float)((double)G / L), R11 */
    std::vector<RowCoef> rows;   /* d rows */
    std::vector<int32_t> T;      /* d*w counters, row-major T[j*w + b] */
    std::set<uint64_t> cand;     /* candidate cells C of the current scan, R10 */
};

struct Oracle {
    int d;
    uint64_t w;
    double L;
    uint64_t seed;
    uint64_t K;                  /* sampling key */
    std::vector<Scale> sc;
    uint64_t upd_index;          /* particles passed to ora_update since create/reset */
    uint64_t scan_index;         /* particles passed to ora_scan since ora_scan_begin */
    bool scanning;
    int mode;                    /* 0 Count Sketch; 1 Count-Min: Add +1, Estimate = min */
};

static uint64_t affine_mod_p(uint64_t a, uint64_t c, uint64_t b) {
    u128 x = (u128)a * (u128)c + (u128)b;
    return (uint64_t)(x % (u128)P61);      /* canonical residue in [0, p-1] */
}

static uint64_t bucket_of(const RowCoef& r, uint64_t c, uint64_t w) { return affine_mod_p(r.a, c, r.b) % w; }
static int32_t sign_of(const RowCoef& r, uint64_t c) { return (affine_mod_p(r.a2, c, r.b2) & 1) ? -1 : +1; }

/* int32 add / multiply-by-sign with two's-complement wraparound (R16). */
static int32_t wrap_add(int32_t t, int32_t s) { return (int32_t)((uint32_t)t + (uint32_t)s); }
static int32_t wrap_mul_sign(int32_t t, int32_t s) { return s > 0 ? t : (int32_t)(0u - (uint32_t)t); }

static uint32_t quantise_axis(float x, float scale, uint32_t G) {
    volatile float t = x * scale;          /* one IEEE binary32 multiply, round-to-nearest-even, no FMA */
    float f = std::floor((float)t);
    if (!(f >= 0.0f)) f = 0.0f;            /* negative and NaN -> 0 */
    float top = (float)(G - 1);
    if (f > top) f = top;                  /* saturate (covers x == L and +inf) */
    return (uint32_t)f;
}

static uint64_t cell_of(const float* p, float scale, uint32_t G) {
    uint64_t ix = quantise_axis(p[0], scale, G);
    uint64_t iy = quantise_axis(p[1], scale, G);
    uint64_t iz = quantise_axis(p[2], scale, G);
    return ix + (uint64_t)G * (iy + (uint64_t)G * iz);
}

static uint64_t sample_threshold(double p) { return (uint64_t)std::floor(std::ldexp(p, 64)); }

static bool keep_particle(uint64_t K, uint64_t index, double p) {
    if (p >= 1.0) return true;
    return mix64(K + (index + 1) * GAMMA) < sample_threshold(p);
}

static int32_t estimate_cell(const Oracle* o, const Scale& s, uint64_t c) {
    std::vector<int32_t> v((size_t)o->d);
    for (int j = 0; j < o->d; ++j) {
        uint64_t h = bucket_of(s.rows[j], c, o->w);
        int32_t sg = o->mode == 1 ? +1 : sign_of(s.rows[j], c);       /* Count-Min has no sign hash */
        v[j] = wrap_mul_sign(s.T[(size_t)j * o->w + h], sg);
    }
    std::sort(v.begin(), v.end());
    if (o->mode == 1) return v[0];         /* Count-Min: the minimum over the rows */
    return v[(size_t)((o->d - 1) / 2)];    /* median for odd d, lower median for even d (R4) */
}

/* (est descending, id ascending) strict weak order used by every selection below (R9). */
struct Better {
    bool operator()(const std::pair<int32_t, uint64_t>& x, const std::pair<int32_t, uint64_t>& y) const {
        if (x.first != y.first) return x.first > y.first;
        return x.second < y.second;
    }
};

extern "C" {

enum { ORA_OK = 0, ORA_ERR_ARG = -1, ORA_ERR_NOMEM = -2, ORA_ERR_STATE = -4 };

void ora_splitmix64(uint64_t seed, uint64_t n, uint64_t* out) {
    for (uint64_t i = 0; i < n; ++i) out[i] = splitmix_nth(seed, i + 1);
}

uint64_t ora_mix64(uint64_t z) { return mix64(z); }

uint64_t ora_affine_mod_p(uint64_t a, uint64_t c, uint64_t b) { return affine_mod_p(a, c, b); }

/* Coefficients of one scale: out[4*j + 0..3] = a_j, b_j, a'_j, b'_j; *K_out = sampling key x_{4d+1}. */
void ora_coeffs(uint64_t seed, int d, uint64_t* out_4d, uint64_t* K_out) {
    for (int j = 0; j < d; ++j) {
        uint64_t x1 = splitmix_nth(seed, 4 * (uint64_t)j + 1);
        uint64_t x2 = splitmix_nth(seed, 4 * (uint64_t)j + 2);
        uint64_t x3 = splitmix_nth(seed, 4 * (uint64_t)j + 3);
        uint64_t x4 = splitmix_nth(seed, 4 * (uint64_t)j + 4);
        out_4d[4 * j + 0] = (x1 % (P61 - 1)) + 1;   /* a  in [1, p-1] */
        out_4d[4 * j + 1] = x2 % P61;               /* b  in [0, p-1] */
        out_4d[4 * j + 2] = (x3 % (P61 - 1)) + 1;   /* a' in [1, p-1] */
        out_4d[4 * j + 3] = x4 % P61;               /* b' in [0, p-1] */
    }
    if (K_out) *K_out = splitmix_nth(seed, 4 * (uint64_t)d + 1);
}

float ora_scale(uint32_t G, double L) { return (float)((double)G / L); }

void ora_quantise(const float* xyz, uint64_t n, uint32_t G, double L, uint64_t* cells_out) {
    float scale = ora_scale(G, L);
    for (uint64_t i = 0; i < n; ++i) cells_out[i] = cell_of(xyz + 3 * i, scale, G);
}

uint64_t ora_sample_threshold(double p) { return sample_threshold(p); }

/* keep_out[i] = 1 iff the particle with running index index0 + i is kept at rate p under key K. */
void ora_keep(uint64_t K, uint64_t index0, uint64_t n, double p, uint8_t* keep_out) {
    for (uint64_t i = 0; i < n; ++i) keep_out[i] = keep_particle(K, index0 + i, p) ? 1 : 0;
}

int ora_create_multi(Oracle** out, int n_scales, int d, uint64_t w, const uint32_t* G, double L, uint64_t seed) {
    if (!out || !G || n_scales < 1 || n_scales > 8 || d < 1 || d > 32 || w < 1 || w > (((uint64_t)1) << 31) ||
        !(L > 0.0) || !std::isfinite(L))
        return ORA_ERR_ARG;
    for (int s = 0; s < n_scales; ++s)
        if (G[s] < 1 || G[s] > (1u << 20)) return ORA_ERR_ARG;
    Oracle* o = new (std::nothrow) Oracle();
    if (!o) return ORA_ERR_NOMEM;
    o->d = d; o->w = w; o->L = L; o->seed = seed;
    o->upd_index = 0; o->scan_index = 0; o->scanning = false; o->mode = 0;
    try {
        o->sc.resize((size_t)n_scales);
        std::vector<uint64_t> co((size_t)4 * d);
        for (int s = 0; s < n_scales; ++s) {
            uint64_t Ks;
            ora_coeffs(seed + (uint64_t)s, d, co.data(), &Ks);   /* scale s draws from the stream of seed + s */
            if (s == 0) o->K = Ks;                                /* one sampling key: that of scale 0 */
            Scale& S = o->sc[(size_t)s];
            S.G = G[s];
            S.scale = ora_scale(G[s], L);
            S.rows.resize((size_t)d);
            for (int j = 0; j < d; ++j) {
                S.rows[j].a = co[4 * j]; S.rows[j].b = co[4 * j + 1];
                S.rows[j].a2 = co[4 * j + 2]; S.rows[j].b2 = co[4 * j + 3];
            }
            S.T.assign((size_t)d * w, 0);
        }
    } catch (...) { delete o; return ORA_ERR_NOMEM; }
    *out = o;
    return ORA_OK;
}

int ora_create(Oracle** out, int d, uint64_t w, uint32_t G, double L, uint64_t seed) {
    return ora_create_multi(out, 1, d, w, &G, L, seed);
}

int ora_destroy(Oracle* o) { delete o; return ORA_OK; }

/* 0: Count Sketch (default).  1: Count-Min variant (Fig. 10): Add increments by +1, Estimate is
 * the minimum over the rows.  Set it before the first particle is added. */
int ora_set_mode(Oracle* o, int mode) {
    if (!o || mode < 0 || mode > 1) return ORA_ERR_ARG;
    o->mode = mode;
    return ORA_OK;
}

int ora_reset(Oracle* o) {
    if (!o) return ORA_ERR_ARG;
    for (Scale& S : o->sc) { std::fill(S.T.begin(), S.T.end(), 0); S.cand.clear(); }
    o->upd_index = 0; o->scan_index = 0; o->scanning = false;
    return ORA_OK;
}

/* Overrides the running particle index of the update stream (used by tests that shard a stream). */
int ora_set_update_index(Oracle* o, uint64_t index) { if (!o) return ORA_ERR_ARG; o->upd_index = index; return ORA_OK; }
int ora_set_scan_index(Oracle* o, uint64_t index) { if (!o) return ORA_ERR_ARG; o->scan_index = index; return ORA_OK; }

static bool bad_p(double p) { return !(p > 0.0) || p > 1.0; }

/* Stream processing, Alg. 1 l.3-5: for each (kept) particle, for each scale, Add(M, cell). */
int ora_update(Oracle* o, const float* xyz, uint64_t n, double sample_p) {
    if (!o || bad_p(sample_p) || (!xyz && n)) return ORA_ERR_ARG;
    for (uint64_t i = 0; i < n; ++i) {
        uint64_t index = o->upd_index + i;
        if (!keep_particle(o->K, index, sample_p)) continue;
        for (Scale& S : o->sc) {
            uint64_t c = cell_of(xyz + 3 * i, S.scale, S.G);
            for (int j = 0; j < o->d; ++j) {
                uint64_t h = bucket_of(S.rows[j], c, o->w);
                int32_t s = o->mode == 1 ? +1 : sign_of(S.rows[j], c);   /* Add(M, s); Count-Min adds +1 */
                int32_t& ctr = S.T[(size_t)j * o->w + h];
                ctr = wrap_add(ctr, s);
            }
        }
    }
    o->upd_index += n;
    return ORA_OK;
}

int ora_estimate(Oracle* o, int scale, const uint64_t* cells, uint64_t m, int32_t* est_out) {
    if (!o || scale < 0 || scale >= (int)o->sc.size() || ((!cells || !est_out) && m)) return ORA_ERR_ARG;
    const Scale& S = o->sc[(size_t)scale];
    for (uint64_t i = 0; i < m; ++i) est_out[i] = estimate_cell(o, S, cells[i]);
    return ORA_OK;
}

int ora_scan_begin(Oracle* o) {
    if (!o) return ORA_ERR_ARG;
    for (Scale& S : o->sc) S.cand.clear();
    o->scan_index = 0; o->scanning = true;
    return ORA_OK;
}

/* Candidate set C of each scale = cells of the kept particles of the replayed stream (a set). */
int ora_scan(Oracle* o, const float* xyz, uint64_t n, double sample_p) {
    if (!o || bad_p(sample_p) || (!xyz && n)) return ORA_ERR_ARG;
    if (!o->scanning) return ORA_ERR_STATE;
    for (uint64_t i = 0; i < n; ++i) {
        uint64_t index = o->scan_index + i;
        if (!keep_particle(o->K, index, sample_p)) continue;
        for (Scale& S : o->sc) S.cand.insert(cell_of(xyz + 3 * i, S.scale, S.G));
    }
    o->scan_index += n;
    return ORA_OK;
}

/* ---- packed 64-bit particle records ("3 coordinates in 64 bits"; R23) -----------------------
 * A record holds the particle's cell on the 2^21 mesh: rec = qx | qy << 21 | qz << 42, q < 2^21 (= the id that
 * ora_quantise gives for G = 2^21).  Its cell on a mesh of G <= 2^20 cells per axis is, per axis, i = (q * G) >> 21
 * (exact integers), c = ix + G*(iy + G*iz). */
static uint64_t cell_of_record(uint64_t rec, uint32_t G) {
    const uint64_t M = (((uint64_t)1) << 21) - 1;
    uint64_t ix = ((rec & M) * G) >> 21, iy = (((rec >> 21) & M) * G) >> 21, iz = (((rec >> 42) & M) * G) >> 21;
    return ix + (uint64_t)G * (iy + (uint64_t)G * iz);
}

void ora_cells_of_records(const uint64_t* recs, uint64_t n, uint32_t G, uint64_t* cells_out) {
    for (uint64_t i = 0; i < n; ++i) cells_out[i] = cell_of_record(recs[i], G);
}

int ora_update_records(Oracle* o, const uint64_t* recs, uint64_t n, double sample_p) {
    if (!o || bad_p(sample_p) || (!recs && n)) return ORA_ERR_ARG;
    for (uint64_t i = 0; i < n; ++i) {
        if (!keep_particle(o->K, o->upd_index + i, sample_p)) continue;
        for (Scale& S : o->sc) {
            uint64_t c = cell_of_record(recs[i], S.G);
            for (int j = 0; j < o->d; ++j) {
                uint64_t h = bucket_of(S.rows[j], c, o->w);
                int32_t s = o->mode == 1 ? +1 : sign_of(S.rows[j], c);
                int32_t& ctr = S.T[(size_t)j * o->w + h];
                ctr = wrap_add(ctr, s);
            }
        }
    }
    o->upd_index += n;
    return ORA_OK;
}

int ora_scan_records(Oracle* o, const uint64_t* recs, uint64_t n, double sample_p) {
    if (!o || bad_p(sample_p) || (!recs && n)) return ORA_ERR_ARG;
    if (!o->scanning) return ORA_ERR_STATE;
    for (uint64_t i = 0; i < n; ++i) {
        if (!keep_particle(o->K, o->scan_index + i, sample_p)) continue;
        for (Scale& S : o->sc) S.cand.insert(cell_of_record(recs[i], S.G));
    }
    o->scan_index += n;
    return ORA_OK;
}

int ora_candidate_count(Oracle* o, int scale, uint64_t* n_out) {
    if (!o || scale < 0 || scale >= (int)o->sc.size() || !n_out) return ORA_ERR_ARG;
    *n_out = o->sc[(size_t)scale].cand.size();
    return ORA_OK;
}

/* Sorted (est desc, id asc) list of every candidate with est >= thr (thr = INT32_MIN: all of them). */
static void ranked_candidates(const Oracle* o, const Scale& S, int32_t thr, std::vector<std::pair<int32_t, uint64_t>>& out) {
    out.clear();
    for (uint64_t c : S.cand) {
        int32_t e = estimate_cell(o, S, c);
        if (e >= thr) out.push_back(std::make_pair(e, c));
    }
    std::sort(out.begin(), out.end(), Better());
}

int ora_topk(Oracle* o, int scale, uint64_t k, uint64_t* ids_out, int32_t* est_out, uint64_t* n_out) {
    if (!o || scale < 0 || scale >= (int)o->sc.size() || !n_out || ((!ids_out || !est_out) && k)) return ORA_ERR_ARG;
    if (!o->scanning) return ORA_ERR_STATE;
    std::vector<std::pair<int32_t, uint64_t>> r;
    ranked_candidates(o, o->sc[(size_t)scale], INT32_MIN, r);
    uint64_t m = std::min<uint64_t>(k, r.size());
    for (uint64_t i = 0; i < m; ++i) { ids_out[i] = r[i].second; est_out[i] = r[i].first; }
    *n_out = m;
    return ORA_OK;
}

int ora_excursion(Oracle* o, int scale, int32_t thr, uint64_t cap, uint64_t* ids_out, int32_t* est_out, uint64_t* n_total) {
    if (!o || scale < 0 || scale >= (int)o->sc.size() || !n_total || ((!ids_out || !est_out) && cap)) return ORA_ERR_ARG;
    if (!o->scanning) return ORA_ERR_STATE;
    std::vector<std::pair<int32_t, uint64_t>> r;
    ranked_candidates(o, o->sc[(size_t)scale], thr, r);
    uint64_t m = std::min<uint64_t>(cap, r.size());
    for (uint64_t i = 0; i < m; ++i) { ids_out[i] = r[i].second; est_out[i] = r[i].first; }
    *n_total = r.size();
    return ORA_OK;
}

/* Second, structurally different top-k used as a cross-check: a size-k std::set of (est, id) fed one
 * replayed particle at a time (O(k) memory), as SURVEY 8.c.1 describes.  Needs no candidate set. */
int ora_topk_streaming(Oracle* o, int scale, const float* xyz, uint64_t n, double sample_p, uint64_t k,
                       uint64_t* ids_out, int32_t* est_out, uint64_t* n_out) {
    if (!o || scale < 0 || scale >= (int)o->sc.size() || bad_p(sample_p) || !n_out) return ORA_ERR_ARG;
    const Scale& S = o->sc[(size_t)scale];
    std::set<std::pair<int32_t, uint64_t>, Better> best;
    for (uint64_t i = 0; i < n; ++i) {
        if (!keep_particle(o->K, i, sample_p)) continue;
        uint64_t c = cell_of(xyz + 3 * i, S.scale, S.G);
        best.insert(std::make_pair(estimate_cell(o, S, c), c));
        if (best.size() > k) best.erase(std::prev(best.end()));
    }
    uint64_t m = 0;
    for (const auto& e : best) { ids_out[m] = e.second; est_out[m] = e.first; ++m; }
    *n_out = m;
    return ORA_OK;
}

/* Streaming selection over ONE SHARD of a replayed stream (full-size parity runs the oracle over disjoint
 * index ranges and merges the results with the same rule): the particles xyz[0..n) carry the running indices
 * index0 .. index0 + n - 1.  One replayed particle at a time, against the tables as they stand (a shard run first sums
 * the tables of all shards with ora_sketch_add), it keeps
 *   (a) the k best distinct cells seen, in (est desc, id asc) order -- what ora_scan + ora_topk give on this shard;
 *   (b) every distinct cell with estimate >= thr, same order       -- what ora_scan + ora_excursion give on this shard;
 * in O(k + |b|) memory instead of the set of all scanned cells.  thr = INT32_MAX asks for no excursion set. */
int ora_select_streaming(Oracle* o, int scale, const float* xyz, uint64_t n, uint64_t index0, double sample_p, uint64_t k,
                         int32_t thr, uint64_t cap_x, uint64_t* ids_k, int32_t* est_k, uint64_t* n_k, uint64_t* ids_x,
                         int32_t* est_x, uint64_t* n_x) {
    if (!o || scale < 0 || scale >= (int)o->sc.size() || bad_p(sample_p) || !n_k || !n_x || (!xyz && n)) return ORA_ERR_ARG;
    const Scale& S = o->sc[(size_t)scale];
    std::set<std::pair<int32_t, uint64_t>, Better> best, above;
    for (uint64_t i = 0; i < n; ++i) {
        if (!keep_particle(o->K, index0 + i, sample_p)) continue;
        uint64_t c = cell_of(xyz + 3 * i, S.scale, S.G);
        int32_t e = estimate_cell(o, S, c);
        if (k) {
            best.insert(std::make_pair(e, c));
            if (best.size() > k) best.erase(std::prev(best.end()));
        }
        if (thr != INT32_MAX && e >= thr) above.insert(std::make_pair(e, c));
    }
    uint64_t m = 0;
    for (const auto& e : best) { ids_k[m] = e.second; est_k[m] = e.first; ++m; }
    *n_k = m;
    m = 0;
    for (const auto& e : above) {
        if (m < cap_x) { ids_x[m] = e.second; est_x[m] = e.first; }
        ++m;
    }
    *n_x = m;
    return ORA_OK;
}

/* Alg. 1 l.7-13 (CSFS query): Estimate every cell j of the dictionary [G^3], keep the k best. Tiny G only. */
int ora_full_search_topk(Oracle* o, int scale, uint64_t k, uint64_t* ids_out, int32_t* est_out, uint64_t* n_out) {
    if (!o || scale < 0 || scale >= (int)o->sc.size() || !n_out) return ORA_ERR_ARG;
    const Scale& S = o->sc[(size_t)scale];
    uint64_t n = (uint64_t)S.G * S.G * S.G;
    if (n > (((uint64_t)1) << 26)) return ORA_ERR_ARG;
    std::vector<std::pair<int32_t, uint64_t>> r;
    r.reserve((size_t)n);
    for (uint64_t j = 0; j < n; ++j) r.push_back(std::make_pair(estimate_cell(o, S, j), j));
    std::sort(r.begin(), r.end(), Better());
    uint64_t m = std::min<uint64_t>(k, r.size());
    for (uint64_t i = 0; i < m; ++i) { ids_out[i] = r[i].second; est_out[i] = r[i].first; }
    *n_out = m;
    return ORA_OK;
}

int ora_sketch_read(Oracle* o, int scale, int32_t* out_d_by_w) {
    if (!o || scale < 0 || scale >= (int)o->sc.size() || !out_d_by_w) return ORA_ERR_ARG;
    const Scale& S = o->sc[(size_t)scale];
    std::memcpy(out_d_by_w, S.T.data(), S.T.size() * sizeof(int32_t));
    return ORA_OK;
}

/* Merge / restore by linearity: T += in, elementwise with wraparound. */
int ora_sketch_add(Oracle* o, int scale, const int32_t* in_d_by_w) {
    if (!o || scale < 0 || scale >= (int)o->sc.size() || !in_d_by_w) return ORA_ERR_ARG;
    Scale& S = o->sc[(size_t)scale];
    for (size_t i = 0; i < S.T.size(); ++i) S.T[i] = wrap_add(S.T[i], in_d_by_w[i]);
    return ORA_OK;
}

int ora_get_coeffs(Oracle* o, int scale, uint64_t* out_4d, uint64_t* K_out) {
    if (!o || scale < 0 || scale >= (int)o->sc.size() || !out_4d) return ORA_ERR_ARG;
    const Scale& S = o->sc[(size_t)scale];
    for (int j = 0; j < o->d; ++j) {
        out_4d[4 * j] = S.rows[j].a; out_4d[4 * j + 1] = S.rows[j].b;
        out_4d[4 * j + 2] = S.rows[j].a2; out_4d[4 * j + 3] = S.rows[j].b2;
    }
    if (K_out) *K_out = o->K;
    return ORA_OK;
}

/* Per-row (bucket, sign) of a list of cells: hs_out[(i*d + j)*2 + {0,1}] = h_j(c_i), s_j(c_i). */
int ora_hashes(Oracle* o, int scale, const uint64_t* cells, uint64_t m, int64_t* hs_out) {
    if (!o || scale < 0 || scale >= (int)o->sc.size() || ((!cells || !hs_out) && m)) return ORA_ERR_ARG;
    const Scale& S = o->sc[(size_t)scale];
    for (uint64_t i = 0; i < m; ++i)
        for (int j = 0; j < o->d; ++j) {
            hs_out[(i * o->d + j) * 2 + 0] = (int64_t)bucket_of(S.rows[j], cells[i], o->w);
            hs_out[(i * o->d + j) * 2 + 1] = (int64_t)sign_of(S.rows[j], cells[i]);
        }
    return ORA_OK;
}

/* Exact counting: one counter per occupied cell, single pass; sorted by cell id.
 * Returns the number of distinct cells; writes at most cap (id, count) pairs. */
uint64_t ora_exact_counts(const float* xyz, uint64_t n, uint32_t G, double L, uint64_t cap, uint64_t* ids_out,
                          uint64_t* counts_out) {
    std::map<uint64_t, uint64_t> cnt;
    float scale = ora_scale(G, L);
    for (uint64_t i = 0; i < n; ++i) cnt[cell_of(xyz + 3 * i, scale, G)] += 1;
    uint64_t m = 0;
    for (const auto& kv : cnt) {
        if (m < cap) { ids_out[m] = kv.first; counts_out[m] = kv.second; }
        ++m;
    }
    return m;
}

} /* extern "C" */
