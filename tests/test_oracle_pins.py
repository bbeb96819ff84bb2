"""Pins for the CPU oracle (oracle/cs_oracle.cpp) against what the paper and the mathematics fix.

None of these compares the oracle with itself or with the CUDA path.  Sources: tests/golden/pins.json
(public splitmix64 vector + SURVEY.md 8.c.4 values computed before the oracle existed), Python big-integer
arithmetic (the *definition* of the modular hashes), numpy float32 / sort / median library routines, brute-force
exact counting, and the algebraic properties the paper states: linearity / mergeability
(PAPER.md:578), arbitrary stream order, unbiasedness E[c*h(i)] = f_i,
Add / Estimate definitions.
"""
import math

import numpy as np
import pytest

from oracle import cs_oracle as ora

P = 2 ** 61 - 1
GAMMA = 0x9E3779B97F4A7C15
M64 = 2 ** 64 - 1


def _ev(expr: str) -> int:
    return int(eval(expr, {"p": P}))


def _centres(cells, G, L):
    """float32 positions at the centres of the given cells (x fastest), box side L."""
    cells = np.asarray(cells, dtype=np.int64)
    h = L / G
    ix, iy, iz = cells % G, (cells // G) % G, cells // (G * G)
    return np.stack([(ix + 0.5) * h, (iy + 0.5) * h, (iz + 0.5) * h], axis=1).astype(np.float32)


def _py_mix(z):
    z &= M64
    z ^= z >> 30
    z = (z * 0xBF58476D1CE4E5B9) & M64
    z ^= z >> 27
    z = (z * 0x94D049BB133111EB) & M64
    z ^= z >> 31
    return z


# ---- splitmix64, coefficients ---------------------------------------------------------------------------

def test_splitmix64_public_vector(golden):
    g = golden["splitmix64"]
    assert [int(x) for x in ora.splitmix64(1234567, 5)] == [int(s) for s in g["seed_1234567"]]
    assert [int(x) for x in ora.splitmix64(0, 3)] == [int(s, 16) for s in g["seed_0_hex"]]


def test_coefficients_seed1(golden):
    g = golden["coeffs_seed1"]
    co5, K5 = ora.coeffs(1, 5)
    co3, K3 = ora.coeffs(1, 3)
    want = [[int(v) for v in row] for row in g["rows"]]
    assert co5[:3].tolist() == want and co3.tolist() == want
    assert K5 == int(g["K_d5"]) and K3 == int(g["K_d3"])
    # ranges the reading fixes: a in [1, p-1], b in [0, p-1]; derivation from the pinned splitmix stream
    x = [int(v) for v in ora.splitmix64(1, 21)]
    for j in range(5):
        a, b, a2, b2 = (int(v) for v in co5[j])
        assert (a, b, a2, b2) == (x[4 * j] % (P - 1) + 1, x[4 * j + 1] % P, x[4 * j + 2] % (P - 1) + 1, x[4 * j + 3] % P)
        assert 1 <= a < P and 0 <= b < P and 1 <= a2 < P and 0 <= b2 < P
    assert K5 == x[20]


def test_multiscale_seeds_and_single_sampling_key():
    o = ora.OracleSketch(4, 64, (8, 16, 32), 10.0, seed=77)
    _, K0 = ora.coeffs(77, 4)
    for s in range(3):
        co, K = o.coeffs(s)
        want, _ = ora.coeffs(77 + s, 4)
        assert co.tolist() == want.tolist() and K == K0


# ---- Mersenne arithmetic --------------------------------------------------------------------------------

def test_mersenne_closed_forms(golden):
    for c in golden["mersenne"]["cases"]:
        assert ora.affine_mod_p(_ev(c["a"]), _ev(c["c"]), _ev(c["b"])) == _ev(c["r"]), c


def test_affine_mod_p_against_python_bigints():
    rng = np.random.default_rng(7)
    edge = [0, 1, 2, P - 1, P - 2, 2 ** 60, 2 ** 60 - 1, 2 ** 36, 2 ** 37 - 1, 2 ** 32, 2 ** 32 - 1]
    cases = [(a, c, b) for a in edge[1:7] for c in edge for b in (0, 1, P - 1, P - 5)]
    for _ in range(3000):
        cases.append((int(rng.integers(1, P)), int(rng.integers(0, 2 ** 60)), int(rng.integers(0, P))))
    for a, c, b in cases:
        r = ora.affine_mod_p(a, c, b)
        assert r == (a * c + b) % P and 0 <= r < P


# ---- quantisation ---------------------------------------------------------------------------------------

def test_quantise_cases(golden):
    g = golden["quantise_G256_L500"]
    assert float(ora.scale_f32(256, 500.0)) == float.fromhex(g["scale_hex"])
    env = {"nan": float("nan"), "inf": float("inf"), "nextafter": lambda a, b: np.nextafter(np.float32(a), np.float32(b))}
    for c in g["cases"]:
        x = np.float32(eval(c["x"], env))
        cell = int(ora.quantise(np.array([[x, 0.0, 0.0]], dtype=np.float32), 256, 500.0)[0])
        assert cell == c["i"], c
        cell = int(ora.quantise(np.array([[0.0, x, 0.0]], dtype=np.float32), 256, 500.0)[0])
        assert cell == 256 * c["i"], c
        cell = int(ora.quantise(np.array([[0.0, 0.0, x]], dtype=np.float32), 256, 500.0)[0])
        assert cell == 256 * 256 * c["i"], c
    below = np.nextafter(np.float32(500.0), np.float32(0.0))
    for G in g["rounds_up_to_G_at"]:
        s = np.float32(np.float64(G) / np.float64(500.0))
        assert float(below * s) == float(G)                      # the product rounds up to G: the clamp is mandatory
        assert int(ora.quantise(np.array([[below, below, below]], dtype=np.float32), G, 500.0)[0]) == G ** 3 - 1


def test_quantise_against_numpy_float32():
    rng = np.random.default_rng(3)
    for G, L in [(256, 500.0), (4642, 500.0), (1000, 1.0), (1, 7.0), (2 ** 20, 123.25), (37, 1e6)]:
        x = (rng.random((20000, 3)) * 1.2 - 0.1).astype(np.float32) * np.float32(L)
        s = np.float32(np.float64(G) / np.float64(L))
        t = np.floor(x * s)                                                  # numpy float32 multiply + floor
        i = np.clip(t, np.float32(0), np.float32(G - 1)).astype(np.uint64)
        want = i[:, 0] + np.uint64(G) * (i[:, 1] + np.uint64(G) * i[:, 2])
        assert np.array_equal(ora.quantise(x, G, L), want)


def test_cell_id_layout_x_fastest():
    G, L = 5, 5.0
    cells = np.arange(G ** 3)
    assert np.array_equal(ora.quantise(_centres(cells, G, L), G, L), cells.astype(np.uint64))


# ---- worked examples ------------------------------------------------------------------------------------

def test_hand_worked_hash_example(golden):
    g = golden["hash_example"]
    xyz = np.array([[123.456, 250.0, 499.99]], dtype=np.float32)
    c = int(ora.quantise(xyz, 256, 500.0)[0])
    assert c == int(g["cell"]) == 63 + 256 * (128 + 256 * 255)
    co, _ = ora.coeffs(1, 5)
    res = [ora.affine_mod_p(int(co[j, 0]), c, int(co[j, 1])) for j in range(5)]
    assert res == [int(v) for v in g["bucket_residues"]]
    assert res == [(int(co[j, 0]) * c + int(co[j, 1])) % P for j in range(5)]
    o = ora.OracleSketch(5, 2 ** 16, 256, 500.0, 1)
    h, s = o.hashes([c])
    assert h[0].tolist() == g["h"] == [r % 2 ** 16 for r in res]
    assert s[0].tolist() == g["s"]
    assert s[0].tolist() == [1 - 2 * (((int(co[j, 2]) * c + int(co[j, 3])) % P) & 1) for j in range(5)]
    o.update(xyz)
    T = o.sketch()
    want = np.zeros_like(T)
    for j in range(5):
        want[j, g["h"][j]] = g["s"][j]
    assert np.array_equal(T, want)


def test_mini_pipeline(golden):
    g = golden["mini_pipeline"]
    xyz = _centres(g["stream_cells"], 4, 4.0)
    o = ora.OracleSketch(3, 8, 4, 4.0, 1)
    assert np.array_equal(ora.quantise(xyz, 4, 4.0), np.array(g["stream_cells"], dtype=np.uint64))
    o.update(xyz)
    assert o.sketch().tolist() == g["T"]
    for c, hs in g["hs"].items():
        h, s = o.hashes([int(c)])
        assert [[int(a), int(b)] for a, b in zip(h[0], s[0])] == hs
    cells = [int(c) for c in g["est"]]
    assert o.estimate(cells).tolist() == [g["est"][str(c)] for c in cells]
    o.scan_begin()
    o.scan(xyz)
    ids, est = o.topk(2)
    assert [[int(a), int(b)] for a, b in zip(ids, est)] == g["top2"]        # 18 beats 57 on the id tie-break
    ids, est, n = o.excursion(2)
    assert n == 3 and [[int(a), int(b)] for a, b in zip(ids, est)] == g["excursion_thr2"]
    # a table rebuilt by hand from Add's definition and the pinned (h, s)
    T = np.zeros((3, 8), dtype=np.int64)
    for c in g["stream_cells"]:
        for j, (h, s) in enumerate(g["hs"][str(c)]):
            T[j, h] += s
    assert T.tolist() == g["T"]


def test_count_min_mini_pipeline_and_one_sided_error(golden):
    """Count-Min mode: hand-worked tables / estimates of the mini pipeline; on a random stream
    the estimate never undercounts (every row holds the cell's own count plus non-negative collisions) and is exact
    when w is far larger than the number of cells; the Count-Sketch default is untouched by the switch."""
    g, gm = golden["mini_pipeline_count_min"], golden["mini_pipeline"]
    xyz = _centres(gm["stream_cells"], 4, 4.0)
    o = ora.OracleSketch(3, 8, 4, 4.0, 1)
    o.set_mode(1)
    o.update(xyz)
    assert o.sketch().tolist() == g["T"]
    cells = [int(c) for c in g["est"]]
    assert o.estimate(cells).tolist() == [g["est"][str(c)] for c in cells]
    o.scan_begin(); o.scan(xyz)
    ids, est = o.topk(2)
    assert [[int(a), int(b)] for a, b in zip(ids, est)] == g["top2"]
    o.set_mode(0); o.reset(); o.update(xyz)
    assert o.sketch().tolist() == gm["T"]
    rng = np.random.default_rng(11)
    pts = (rng.random((20000, 3)) ** 3 * 50.0).astype(np.float32)           # skewed: heavy cells near the origin
    eid, ecnt = ora.exact_counts(pts, 40, 50.0)
    for w, exact in ((64, False), (1 << 22, True)):
        o = ora.OracleSketch(4, w, 40, 50.0, 9)
        o.set_mode(1)
        o.update(pts)
        assert int(o.sketch().min()) >= 0 and o.sketch().sum(axis=1).tolist() == [len(pts)] * 4
        est = o.estimate(eid)
        assert bool((est.astype(np.int64) >= ecnt.astype(np.int64)).all())
        if exact:
            hb, _ = o.hashes(eid)
            if all(len(set(hb[:, j].tolist())) == len(eid) for j in range(4)):    # collision-free rows
                assert np.array_equal(est.astype(np.uint64), ecnt)
        else:
            assert bool((est.astype(np.int64) > ecnt.astype(np.int64)).any())       # collisions do overcount


def test_packed_records():
    """Packed 64-bit records (R23): the per-axis rule i = (q*G) >> 21 against Python integers,
    nested meshes are consistent (coarse cell = fine cell // r per axis), and the record passes equal the float passes
    on the centres of the 2^20-mesh cells the records fall in (where both quantisations agree by construction)."""
    rng = np.random.default_rng(5)
    q = rng.integers(0, 1 << 21, size=(5000, 3), dtype=np.uint64)
    q[:8] = [[0, 0, 0], [2 ** 21 - 1] * 3, [1, 2 ** 20, 2 ** 21 - 1], [2 ** 20 - 1, 2 ** 20, 2 ** 20 + 1], [511, 512, 513],
             [4095, 4096, 4097], [2 ** 21 - 2, 0, 7], [3, 3, 3]]
    recs = q[:, 0] | (q[:, 1] << np.uint64(21)) | (q[:, 2] << np.uint64(42))
    for G in (1, 2, 3, 256, 1000, 4096, 4642, 1 << 20):
        got = ora.cells_of_records(recs, G)
        ix, iy, iz = [[(int(v) * G) >> 21 for v in q[:, a]] for a in range(3)]
        want = [x + G * (y + G * z) for x, y, z in zip(ix, iy, iz)]
        assert got.tolist() == want
        assert max(max(ix), max(iy), max(iz)) <= G - 1
    c512, c4096 = ora.cells_of_records(recs, 512), ora.cells_of_records(recs, 4096)
    f = [c4096 % 4096, (c4096 // 4096) % 4096, c4096 // 4096 ** 2]
    assert np.array_equal(c512, f[0] // 8 + 512 * (f[1] // 8 + 512 * (f[2] // 8)))
    # pack = quantise on the 2^21 mesh
    L = 500.0
    pts = (rng.random((3000, 3)) * L).astype(np.float32)
    rp = ora.pack_records(pts, L)
    sc = np.float32((1 << 21) / L)
    qq = np.clip(np.floor(pts * sc), 0, (1 << 21) - 1).astype(np.uint64)
    assert np.array_equal(rp, qq[:, 0] | (qq[:, 1] << np.uint64(21)) | (qq[:, 2] << np.uint64(42)))
    # record passes == float passes on cell centres of the finest mesh
    Gs = (64, 256)
    cf = ora.cells_of_records(rp, 256)
    centres = _centres(cf.tolist(), 256, L)
    a, b = ora.OracleSketch(3, 1 << 10, Gs, L, 3), ora.OracleSketch(3, 1 << 10, Gs, L, 3)
    a.update_records(rp, 0.6); b.update(centres, 0.6)
    a.scan_begin(); b.scan_begin()
    a.scan_records(rp, 0.6); b.scan(centres, 0.6)
    for s_ in range(2):
        assert np.array_equal(a.sketch(s_), b.sketch(s_))
        ia, ea = a.topk(50, s_); ib, eb = b.topk(50, s_)
        assert np.array_equal(ia, ib) and np.array_equal(ea, eb)


# ---- sampler --------------------------------------------------------------------------------------------

def test_sampler_pins(golden):
    g = golden["sampler_seed1_d5_p0.1"]
    _, K = ora.coeffs(1, 5)
    assert ora.sample_threshold(0.1) == int(g["T_p_hex"], 16) == math.floor(0.1 * 2 ** 64)
    assert ora.mix64(K + GAMMA) == int(g["u0"]) == _py_mix(K + GAMMA)
    assert ora.mix64(K + 3 * GAMMA) == int(g["u2"])
    keep = ora.keep_mask(K, 0, 10 ** 6, 0.1)
    assert keep[:8].tolist() == g["first8_kept"]
    assert int(keep.sum()) == g["kept_of_first_million"]
    # definition, element by element, on a window that does not start at 0
    win = ora.keep_mask(K, 12345, 200, 0.1)
    assert win.tolist() == [_py_mix(K + (12345 + i + 1) * GAMMA) < int(g["T_p_hex"], 16) for i in range(200)]
    assert ora.keep_mask(K, 0, 1000, 1.0).all()                            # p = 1 keeps everything
    for p in (0.5, 0.25, 1 / 16):
        assert ora.sample_threshold(p) == int(p * 2 ** 64)
        frac = ora.keep_mask(K, 0, 400000, p).mean()
        assert abs(frac - p) < 4 * math.sqrt(p * (1 - p) / 400000)


def test_sampled_update_equals_update_of_kept_particles():
    rng = np.random.default_rng(11)
    xyz = (rng.random((5000, 3)) * 10).astype(np.float32)
    a = ora.OracleSketch(5, 1024, 16, 10.0, 9)
    _, K = a.coeffs()
    a.update(xyz[:3000], 0.3)
    a.update(xyz[3000:], 0.3)                                               # running index continues
    keep = ora.keep_mask(K, 0, 5000, 0.3)
    b = ora.OracleSketch(5, 1024, 16, 10.0, 9)
    b.update(xyz[keep], 1.0)
    assert np.array_equal(a.sketch(), b.sketch())
    a.scan_begin(); a.scan(xyz, 0.3)
    assert a.candidate_count() == len(np.unique(ora.quantise(xyz[keep], 16, 10.0)))


# ---- exact counts, row invariants -----------------------------------------------------------------------

def test_exact_counts_brute_force_no_collisions():
    """w >> #distinct cells: once the occupied cells' buckets are verified distinct in a row, every row value
    s_j(c) * T[j][h_j(c)] must equal the exact count f_c."""
    rng = np.random.default_rng(5)
    G, L, d, w = 64, 64.0, 5, 2 ** 20
    cells = rng.choice(G ** 3, size=40, replace=False)
    freq = rng.integers(1, 30, size=40)
    stream = np.repeat(cells, freq)
    rng.shuffle(stream)
    xyz = _centres(stream, G, L)
    ids, cnt = ora.exact_counts(xyz, G, L)
    order = np.argsort(cells)
    assert np.array_equal(ids, cells[order].astype(np.uint64)) and np.array_equal(cnt, freq[order].astype(np.uint64))
    # independent brute force with numpy
    uq, uc = np.unique(ora.quantise(xyz, G, L), return_counts=True)
    assert np.array_equal(uq, ids) and np.array_equal(uc.astype(np.uint64), cnt)
    checked = 0
    for seed in range(1, 6):
        o = ora.OracleSketch(d, w, G, L, seed)
        o.update(xyz)
        T = o.sketch()
        h, s = o.hashes(ids)
        for j in range(d):
            if len(set(h[:, j].tolist())) != len(ids):
                continue                                                    # a collision in this row: skip it
            checked += 1
            assert np.array_equal(s[:, j] * T[j, h[:, j]], cnt.astype(np.int64))
            assert np.count_nonzero(T[j]) == len(ids)
        if all(len(set(h[:, j].tolist())) == len(ids) for j in range(d)):
            assert np.array_equal(o.estimate(ids), cnt.astype(np.int32))
        # a probe cell none of whose buckets was touched estimates exactly 0
        for probe in range(G ** 3):
            hp, _ = o.hashes([probe])
            if probe not in set(ids.tolist()) and all(T[j, hp[0, j]] == 0 for j in range(d)):
                assert int(o.estimate([probe])[0]) == 0
                break
    assert checked >= 20


def test_row_invariants_and_single_cell_stream():
    rng = np.random.default_rng(1)
    xyz = (rng.random((20001, 3)) * 50).astype(np.float32)
    for d, w in [(5, 997), (4, 256), (7, 1), (1, 64)]:
        o = ora.OracleSketch(d, w, 32, 50.0, 3)
        o.update(xyz)
        T = o.sketch().astype(np.int64)
        assert ((T.sum(axis=1) - 20001) % 2 == 0).all()
        assert (np.abs(T).sum(axis=1) <= 20001).all()
    o = ora.OracleSketch(6, 128, 8, 8.0, 5)
    one = _centres([77] * 13, 8, 8.0)
    o.update(one)
    T = o.sketch()
    h, s = o.hashes([77])
    for j in range(6):
        assert np.count_nonzero(T[j]) == 1 and T[j, h[0, j]] == 13 * s[0, j]
    assert int(o.estimate([77])[0]) == 13


def test_degenerate_grid_and_empty_stream():
    o = ora.OracleSketch(3, 16, 1, 2.0, 4)                                  # G = 1: every particle is cell 0
    o.update(np.zeros((0, 3), dtype=np.float32))
    assert not o.sketch().any()
    xyz = np.array([[0.1, 1.9, 1.0], [5.0, -2.0, float("nan")]], dtype=np.float32)
    assert ora.quantise(xyz, 1, 2.0).tolist() == [0, 0]
    o.update(xyz)
    assert int(o.estimate([0])[0]) == 2
    o.scan_begin(); o.scan(xyz)
    ids, est = o.topk(5)
    assert ids.tolist() == [0] and est.tolist() == [2]
    o.scan_begin()
    ids, est = o.topk(5)
    assert len(ids) == 0
    o.reset()
    assert not o.sketch().any()


# ---- linearity, order, batch split ----------------------------------------------------------------------

def _stream(n, seed, L=100.0):
    rng = np.random.default_rng(seed)
    hot = rng.random((30, 3)) * L
    pick = rng.integers(0, 30, size=n)
    xyz = hot[pick] + rng.normal(0, 0.8, size=(n, 3))
    bg = rng.random(n) < 0.3
    xyz[bg] = rng.random((int(bg.sum()), 3)) * L
    return np.mod(xyz, L).astype(np.float32)


def test_linearity_and_merge():
    A, B = _stream(7000, 1), _stream(5000, 2)
    mk = lambda: ora.OracleSketch(5, 1000, 64, 100.0, 21)                  # non-power-of-two w
    a, b, ab = mk(), mk(), mk()
    a.update(A); b.update(B); ab.update(np.concatenate([A, B]))
    assert np.array_equal(a.sketch() + b.sketch(), ab.sketch())
    a.sketch_add(b.sketch())
    assert np.array_equal(a.sketch(), ab.sketch())
    # p < 1: linear when B's running indices continue A's
    a2, b2, ab2 = mk(), mk(), mk()
    a2.update(A, 0.4); b2.set_update_index(len(A)); b2.update(B, 0.4); ab2.update(np.concatenate([A, B]), 0.4)
    assert np.array_equal(a2.sketch() + b2.sketch(), ab2.sketch())


def test_order_invariance():
    X = _stream(9000, 3)
    perm = np.random.default_rng(0).permutation(len(X))
    a = ora.OracleSketch(7, 4096, 64, 100.0, 2)
    b = ora.OracleSketch(7, 4096, 64, 100.0, 2)
    a.update(X); b.update(X[perm])
    assert np.array_equal(a.sketch(), b.sketch())
    a.scan_begin(); a.scan(X); b.scan_begin(); b.scan(X[perm])
    ia, ea = a.topk(50); ib, eb = b.topk(50)
    assert np.array_equal(ia, ib) and np.array_equal(ea, eb)


@pytest.mark.parametrize("p", [1.0, 0.37])
def test_batch_split_invariance(p):
    X = _stream(6001, 4)
    whole = ora.OracleSketch(5, 2048, 64, 100.0, 8)
    whole.update(X, p)
    parts = ora.OracleSketch(5, 2048, 64, 100.0, 8)
    for lo, hi in [(0, 1), (1, 6), (6, 6), (6, 1031), (1031, 6001)]:
        parts.update(X[lo:hi], p)
    assert np.array_equal(whole.sketch(), parts.sketch())
    whole.scan_begin(); whole.scan(X, p)
    parts.scan_begin()
    for lo, hi in [(0, 3), (3, 4000), (4000, 6001)]:
        parts.scan(X[lo:hi], p)
    assert whole.candidate_count() == parts.candidate_count()
    assert all(np.array_equal(u, v) for u, v in zip(whole.topk(40), parts.topk(40)))


# ---- statistics -----------------------------------------------------------------------------------------

def test_unbiasedness_fixes_the_sign_convention():
    """E[s_j(c) * T[j][h_j(c)]] = f_c: a flipped sign or a dropped sign factor fails this."""
    X = _stream(3000, 9, L=40.0)
    G, L, w = 16, 40.0, 64
    ids, cnt = ora.exact_counts(X, G, L)
    target = int(np.argmax(cnt))
    c, f = int(ids[target]), int(cnt[target])
    vals = []
    for seed in range(1000):
        o = ora.OracleSketch(1, w, G, L, seed)
        o.update(X)
        vals.append(int(o.estimate([c])[0]))                                # d = 1: the estimate is the row value
    vals = np.array(vals, dtype=np.float64)
    se = vals.std(ddof=1) / math.sqrt(len(vals))
    assert abs(vals.mean() - f) < 4 * se
    F2_others = float((cnt.astype(np.float64) ** 2).sum() - f * f)
    assert 0.7 < vals.var() / (F2_others / w) < 1.4                         # per-row variance = F2(others)/w


def test_accuracy_sanity_cfg1_shape():
    """Additive error roughly constant across ranks and of the order of sqrt(F2/w) (Fig. 8)."""
    import torch
    from paper_1711_00975_b200 import synth
    wl = synth.CONFIGS["cfg1"]                                            # full size: the Gaussian regime
    X = synth.generate(wl).numpy()
    o = ora.OracleSketch(wl.d, wl.w, wl.G[0], wl.L, wl.seed)
    o.update(X)
    ids, cnt = ora.exact_counts(X, wl.G[0], wl.L)
    order = np.argsort(-cnt.astype(np.int64), kind="stable")[:2000]
    err = np.abs(o.estimate(ids[order]).astype(np.int64) - cnt[order].astype(np.int64))
    sigma_row = math.sqrt(float((cnt.astype(np.float64) ** 2).sum()) / wl.w)
    # The collision noise is heavy-tailed (a few ~80-particle cells carry most of F2), so only the scale is
    # checked: the median-of-d error sits well below one row's sigma = sqrt(F2/w) and does not grow with rank.
    assert 0.05 * sigma_row < err.mean() < sigma_row
    assert abs(err[:1000].mean() - err[1000:].mean()) < 0.25 * sigma_row


# ---- median ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("d", [1, 2, 3, 4, 5, 7, 8, 16, 31, 32])
def test_median_against_numpy(d):
    """With w = 1 every cell reads T[j][0]; inject row values through sketch_add and compare the estimate with
    numpy's sort / median of s_j * v_j (lower median for even d, R4)."""
    rng = np.random.default_rng(d)
    o = ora.OracleSketch(d, 1, 4, 4.0, 13)
    cells = np.arange(64, dtype=np.uint64)
    _, s = o.hashes(cells)
    lo, hi = -(2 ** 31) + 1, 2 ** 31 - 1
    patterns = [rng.integers(-50, 50, size=d), np.full(d, 7), np.arange(d), np.arange(d)[::-1],
                rng.integers(0, 3, size=d), rng.choice([lo, hi, 0, -1, 1], size=d)]
    patterns += [rng.integers(lo, hi, size=d) for _ in range(10)]
    for v in patterns:
        v = np.asarray(v, dtype=np.int64)
        o.reset()
        o.sketch_add(v.astype(np.int32).reshape(d, 1))
        est = o.estimate(cells)
        vals = s * v[None, :]
        want = np.sort(vals, axis=1)[:, (d - 1) // 2]
        assert np.array_equal(est.astype(np.int64), want)
        if d % 2 == 1:
            assert np.array_equal(est.astype(np.float64), np.median(vals, axis=1))


# ---- selection ------------------------------------------------------------------------------------------

def test_topk_and_excursion_against_full_sort():
    X = _stream(20000, 12, L=64.0)
    G, L = 32, 64.0
    o = ora.OracleSketch(5, 512, G, L, 6)
    o.update(X)
    o.scan_begin(); o.scan(X[:9000]); o.scan(X[9000:])
    occ = np.unique(ora.quantise(X, G, L))
    assert o.candidate_count() == len(occ)
    est = o.estimate(occ).astype(np.int64)
    order = np.lexsort((occ, -est))                                         # est descending, id ascending
    for k in (0, 1, 17, len(occ), len(occ) + 5):
        ids, e = o.topk(k)
        m = min(k, len(occ))
        assert np.array_equal(ids, occ[order[:m]]) and np.array_equal(e.astype(np.int64), est[order[:m]])
    si, se = o.topk_streaming(X, 300)                                       # O(k)-memory streaming set == sort-unique
    assert np.array_equal(si, occ[order[:300]]) and np.array_equal(se.astype(np.int64), est[order[:300]])
    for thr in (-5, 0, 3, int(est.max()), int(est.max()) + 1):
        ids, e, n = o.excursion(thr)
        sel = order[est[order] >= thr]
        assert n == len(sel) and np.array_equal(ids, occ[sel]) and np.array_equal(e.astype(np.int64), est[sel])
        ids2, _, n2 = o.excursion(thr, cap=4)
        assert n2 == n and np.array_equal(ids2, occ[sel][:4])
    # ties exist and are resolved by ascending id
    top_e = est[order[:400]]
    assert (np.diff(top_e) <= 0).all()
    tied = np.flatnonzero(np.diff(top_e) == 0)
    assert len(tied) > 0 and (np.diff(occ[order[:400]].astype(np.int64))[tied] > 0).all()


def test_full_dictionary_search_restricted_to_occupied_cells():
    """Alg. 1 l.7-13 estimates every j in [n]; restricted to the occupied cells it must give the re-scan's answer
    (R10), and every cell it ranks above the re-scan's k-th is either occupied or a fake heavy hitter."""
    X = _stream(4000, 15, L=16.0)
    G, L = 16, 16.0
    o = ora.OracleSketch(5, 256, G, L, 2)
    o.update(X)
    o.scan_begin(); o.scan(X)
    occ = set(np.unique(ora.quantise(X, G, L)).tolist())
    fi, fe = o.full_search_topk(G ** 3)
    assert len(fi) == G ** 3 and sorted(fi.tolist()) == list(range(G ** 3))
    mask = np.array([c in occ for c in fi.tolist()])
    ids, est = o.topk(len(occ))
    assert np.array_equal(fi[mask], ids) and np.array_equal(fe[mask], est)
    assert np.array_equal(fe, o.estimate(fi))


def test_negative_estimates_rank_below_zero():
    o = ora.OracleSketch(3, 8, 4, 4.0, 1)
    g_stream = _centres([0, 0, 0, 57, 57, 63, 18, 18], 4, 4.0)
    o.update(g_stream)
    o.scan_begin(); o.scan(g_stream)
    ids, est = o.topk(10)
    assert ids.tolist() == [0, 18, 57, 63] and est.tolist() == [3, 2, 2, -1]


def test_argument_errors():
    with pytest.raises(RuntimeError):
        ora.OracleSketch(0, 8, 4, 4.0, 1)
    with pytest.raises(RuntimeError):
        ora.OracleSketch(33, 8, 4, 4.0, 1)
    with pytest.raises(RuntimeError):
        ora.OracleSketch(3, 0, 4, 4.0, 1)
    with pytest.raises(RuntimeError):
        ora.OracleSketch(3, 8, 2 ** 20 + 1, 4.0, 1)
    with pytest.raises(RuntimeError):
        ora.OracleSketch(3, 8, 4, float("nan"), 1)
    o = ora.OracleSketch(3, 8, 4, 4.0, 1)
    for p in (0.0, -0.1, 1.5, float("nan")):
        with pytest.raises(RuntimeError):
            o.update(np.zeros((1, 3), dtype=np.float32), p)
    with pytest.raises(RuntimeError):
        o.topk(3)                                                           # before scan_begin


# ---- full-size parity device: the oracle over disjoint index ranges --------------------

@pytest.mark.parametrize("p,G,parts", [(1.0, (32,), 3), (0.6, (16, 32, 64), 4), (0.3, (48,), 7)])
def test_sharded_oracle_equals_single_oracle(p, G, parts):
    """ora_select_streaming over P shards (each with the running index of its first particle), tables summed, lists
    merged by (est desc, id asc, unique), against the plain single-stream oracle: tables, top-k, excursion sets."""
    from sharded_oracle import ShardedOracle
    X = _stream(30001, 21, L=64.0)
    L = 64.0
    o = ora.OracleSketch(5, 1024, G, L, 9)
    o.update(X[:12345], p); o.update(X[12345:], p)
    o.scan_begin(); o.scan(X, p)
    so = ShardedOracle(5, 1024, G, L, 9, parts)
    so.update(X[:12345], p, 0)
    so.update(X[12345:], p, 12345)                         # a second batch continues the running index
    for k, thr in ((50, 3), (100000, -100)):
        sel = so.select(X, k, thr, p, 0)
        for s in range(len(G)):
            assert np.array_equal(so.sketch(s), o.sketch(s))
            (ti, te), (xi, xe) = sel[s]
            oi, oe = o.topk(k, s)
            assert np.array_equal(ti, oi) and np.array_equal(te, oe)
            yi, ye, yn = o.excursion(thr, s)
            assert yn == len(xi) and np.array_equal(xi, yi) and np.array_equal(xe, ye)
    # one shard alone, no excursion set asked: the streaming selection is ora_scan + ora_topk of that shard
    (ti, te), (xi, xe) = so.o[0].select_streaming(X[100:9000], 100, 40, sample_p=p)
    o.scan_begin(); o.set_scan_index(100); o.scan(X[100:9000], p)
    oi, oe = o.topk(40)
    assert np.array_equal(ti, oi) and np.array_equal(te, oe) and len(xi) == 0
    so.close(); o.close()
