"""GPU parity tests of the host-streamed calls (SURVEY 8.a row a8; PAPER.md:295-298 batch flow, :570 I/O overlapped with
compute): cs_update_host / cs_scan_host (float32 positions) and cs_update_records_host / cs_scan_records_host against the
CPU oracle, with the staging batch made small (cs_set_chunk_sizes) so that the stream takes >= 5 batches and every slot of
the 3-slot device ring is reused; pinned and pageable host memory, p = 1 and p = 0.1 (the compaction path, which reads
a count back per chunk), a ragged last batch, a split into two host calls, the replay cache on and off.  Also: the
multi-chunk forms of the device-resident passes (binned update chunks, scan chunks, compaction chunks) at sizes the
oracle replays in seconds.  Bar: bit-exact tables, estimates, top-k and excursion ids and values.
"""
import numpy as np
import pytest
import torch

from oracle import cs_oracle as ora

pytestmark = pytest.mark.gpu

INT32_MAX = 2 ** 31 - 1


@pytest.fixture(scope="module")
def cs():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1711_00975_b200 import build, binding
    build.build_libcs()
    binding.lib()
    return binding


def _gen(name, n, **kw):
    from paper_1711_00975_b200 import synth
    wl = synth.CONFIGS[name].scaled(n, **kw)
    return wl, synth.generate(wl, device="cuda")


def _ids(t):
    return t.cpu().numpy().view(np.uint64)


def _host_copy(t: torch.Tensor, pinned: bool) -> torch.Tensor:
    h = torch.empty(t.shape, dtype=t.dtype, pin_memory=pinned)
    h.copy_(t)
    return h


def _compare(g, o, wl, k, thresholds, host_np=None):
    for s in range(len(wl.G)):
        assert np.array_equal(g.sketch(s).cpu().numpy(), o.sketch(s)), f"sketch differs at scale {s}"
        if host_np is not None:
            cells = ora.quantise(host_np[:2048], wl.G[s], wl.L)
            ge = g.estimate(torch.from_numpy(cells.view(np.int64)).cuda(), s).cpu().numpy()
            assert np.array_equal(ge, o.estimate(cells, s)), f"estimates differ at scale {s}"
        gi, gv = g.topk(k, s, device="cpu")
        oi, ov = o.topk(k, s)
        assert np.array_equal(_ids(gi), oi) and np.array_equal(gv.numpy(), ov), f"top-k differs at scale {s}"
        for thr in thresholds:
            xi, xv, xt = g.excursion(thr, s)
            yi, yv, yt = o.excursion(thr, s)
            assert xt == yt and np.array_equal(_ids(xi), yi) and np.array_equal(xv.cpu().numpy(), yv), (s, thr)


def _check_host_float(cs, wl, xyz, sample_p, stage, pinned, split=None, k=None, thresholds=(), cache=0, compact_chunk=0,
                      update_chunk=0, scan_chunk=0, mode=None):
    """cs_update_host + cs_scan_host over batches of `stage` particles against the oracle fed the same float32 buffer."""
    k = wl.k if k is None else k
    host = _host_copy(xyz, pinned)
    host_np = host.numpy()
    n = host_np.shape[0]
    assert n > 5 * stage, "the ring must wrap: at least 6 batches"
    o = ora.OracleSketch(wl.d, wl.w, wl.G, wl.L, wl.seed)
    g = cs.CountSketch(wl.d, wl.w, list(wl.G), wl.L, wl.seed)
    g.set_chunk_sizes(stage, update_chunk, scan_chunk, compact_chunk)
    if cache:
        g.set_replay_cache(cache)
    if mode is not None:
        g.set_update_mode(*mode)
    cuts = [0, n] if not split else [0] + sorted(split) + [n]
    for a, b in zip(cuts[:-1], cuts[1:]):
        o.update(host_np[a:b], sample_p)
        g.update_host(host[a:b], sample_p)
    thr_min = min(thresholds) if thresholds else INT32_MAX
    o.scan_begin()
    g.scan_begin(k, thr_min)
    for a, b in zip(cuts[:-1], cuts[1:]):
        o.scan(host_np[a:b], sample_p)
        g.scan_host(host[a:b], sample_p)
    _compare(g, o, wl, k, thresholds, host_np)
    launches = g.launch_count()
    g.close(); o.close()
    return launches


@pytest.mark.parametrize("pinned", [True, False])
def test_float_host_stream_ring_wraps_p1(cs, pinned):
    """cfg 3 shape (d = 7, G = 4096), 7 full batches of 2^16 particles + a ragged one: slots 0, 1, 2 are each reused."""
    wl, xyz = _gen("cfg3", 7 * (1 << 16) + 12345)
    _check_host_float(cs, wl, xyz, 1.0, 1 << 16, pinned, k=2000, thresholds=(5,))


def test_float_host_stream_split_calls_and_unaligned_tail(cs):
    """Two host calls whose boundary is neither a batch nor a 4-particle boundary (cfg 4 shape: G = 4642, w = 2^24 scaled
    down to 2^18), 5 + 4 batches."""
    wl, xyz = _gen("cfg4", 9 * (1 << 15) - 77, w=1 << 18)
    _check_host_float(cs, wl, xyz, 1.0, 1 << 15, True, split=[5 * (1 << 15) + 3], k=3000)


@pytest.mark.parametrize("pinned", [True, False])
def test_float_host_stream_sampled_compaction_path(cs, pinned):
    """p = 0.1 with batches of 2^20 particles (>= the compaction threshold), cut into compaction chunks of 2^18: every
    batch reads kept-particle counts back (the host sync inside cs_update_host) while the next copy is in flight.
    cfg 5 shape: 4 nested grids, thresholds and top-k per scale; 6 batches + a ragged one."""
    wl, xyz = _gen("cfg5", 6 * (1 << 20) + 4321)
    _check_host_float(cs, wl, xyz, wl.sample_p, 1 << 20, pinned, k=1000, thresholds=(3, 5), compact_chunk=1 << 18,
                      split=[4 * (1 << 20) + 10001])


def test_float_host_stream_binned_update_per_batch(cs):
    """The binned update (forced) per batch of 2^19 particles, two binned chunks per batch, two scan chunks per batch."""
    wl, xyz = _gen("cfg3", 5 * (1 << 19) + 1001, w=1 << 20)
    _check_host_float(cs, wl, xyz, 1.0, 1 << 19, True, k=3000, update_chunk=1 << 18, scan_chunk=1 << 18, mode=(2, -1))


def test_replay_cache_float_host_and_sampled(cs):
    """cs_set_replay_cache: the scan of the same host buffer reads the device copy (fewer launches is not required, the
    same result is); sampled streams re-scan the kept particles held from the update."""
    wl, xyz = _gen("cfg3", 6 * (1 << 16) + 999)
    a = _check_host_float(cs, wl, xyz, 1.0, 1 << 16, True, k=2000, thresholds=(5,), cache=1 << 30)
    b = _check_host_float(cs, wl, xyz, 1.0, 1 << 16, True, k=2000, thresholds=(5,), cache=1 << 20)   # too small: ring
    assert a > 0 and b > 0
    wl, xyz = _gen("cfg5", 6 * (1 << 20) + 4321)
    with_cache = _check_host_float(cs, wl, xyz, wl.sample_p, 1 << 20, True, k=1000, thresholds=(3,), cache=1 << 30,
                                   compact_chunk=1 << 18)
    without = _check_host_float(cs, wl, xyz, wl.sample_p, 1 << 20, True, k=1000, thresholds=(3,), compact_chunk=1 << 18)
    assert with_cache < without, "the cached re-scan must skip the compaction launches"
    # the cache holds the LAST host call only: a stream split into two calls still gives the same answer
    _check_host_float(cs, wl, xyz, wl.sample_p, 1 << 20, True, k=1000, thresholds=(3,), cache=1 << 30, compact_chunk=1 << 18,
                      split=[3 * (1 << 20) + 5])


def test_replay_cache_device_sampled_stream(cs):
    """Device-resident sampled stream (cfg 5 shape): cs_scan of the buffer cs_update compacted re-uses the kept particles;
    a different buffer, length, p or running index does not hit."""
    wl, xyz = _gen("cfg5", (1 << 22) + 5)
    host_np = xyz.cpu().numpy()
    p = wl.sample_p
    o = ora.OracleSketch(wl.d, wl.w, wl.G, wl.L, wl.seed)
    g = cs.CountSketch(wl.d, wl.w, list(wl.G), wl.L, wl.seed)
    g.set_replay_cache(1 << 28)
    g.set_chunk_sizes(0, 0, 0, 1 << 20)
    for rep in range(2):                                    # the second round goes through cs_reset
        o.reset(); g.reset()
        o.update(host_np, p); g.update(xyz, p)
        o.scan_begin(); g.scan_begin(500, 3)
        l0 = g.launch_count()
        o.scan(host_np, p); g.scan(xyz, p)
        hit = g.launch_count() - l0
        _compare(g, o, wl, 500, (3,), host_np)
    # same stream scanned in two halves: no hit (different length), same answer
    o.scan_begin(); g.scan_begin(500, 3)
    l0 = g.launch_count()
    half = (1 << 21) + 4
    o.scan(host_np[:half], p); o.scan(host_np[half:], p)
    g.scan(xyz[:half], p); g.scan(xyz[half:], p)
    miss = g.launch_count() - l0
    _compare(g, o, wl, 500, (3,), host_np)
    assert hit < miss
    g.close(); o.close()


def _check_host_records(cs, wl, xyz, sample_p, stage, pinned, split=None, k=None, cache=0):
    k = wl.k if k is None else k
    g = cs.CountSketch(wl.d, wl.w, list(wl.G), wl.L, wl.seed)
    o = ora.OracleSketch(wl.d, wl.w, wl.G, wl.L, wl.seed)
    g.set_chunk_sizes(stage, 0, 0, 0)
    if cache:
        g.set_replay_cache(cache)
    recs = _host_copy(g.pack_records(xyz), pinned)
    want = ora.pack_records(xyz.cpu().numpy(), wl.L)
    assert np.array_equal(recs.numpy().view(np.uint64), want)
    n = recs.numel()
    assert n > 5 * stage
    cuts = [0, n] if not split else [0] + sorted(split) + [n]
    for a, b in zip(cuts[:-1], cuts[1:]):
        o.update_records(want[a:b], sample_p)
        g.update_records_host(recs[a:b], sample_p)
    o.scan_begin()
    g.scan_begin(k)
    for a, b in zip(cuts[:-1], cuts[1:]):
        o.scan_records(want[a:b], sample_p)
        g.scan_records_host(recs[a:b], sample_p)
    _compare(g, o, wl, k, ())
    g.close(); o.close()


@pytest.mark.parametrize("pinned,cache", [(True, 0), (False, 0), (True, 1 << 30)])
def test_records_host_stream_ring_wraps(cs, pinned, cache):
    wl, xyz = _gen("cfg4", 7 * (1 << 16) + 4099, w=1 << 18)
    _check_host_records(cs, wl, xyz, 1.0, 1 << 16, pinned, split=[3 * (1 << 16) + 1], k=3000, cache=cache)


def test_records_host_stream_sampled_multiscale(cs):
    wl, xyz = _gen("cfg5", 6 * (1 << 20) + 77)
    _check_host_records(cs, wl, xyz, 0.1, 1 << 20, True, k=500)


# ---- multi-chunk forms of the device-resident passes ---------------------------------------------------------------

@pytest.mark.parametrize("rows_direct", [-1, 0])
def test_binned_update_many_chunks_against_oracle(cs, rows_direct):
    """The binned update cut into 5 scatter/apply chunks (bench.py's cfg 3 run uses 8 of 2^27): chunk offsets, the
    running index under sampling, the ragged last chunk; against the oracle, not against another CUDA path."""
    wl, xyz = _gen("cfg3", 4 * (1 << 20) + 333333)
    host_np = xyz.cpu().numpy()
    for p in (1.0, 0.6):
        o = ora.OracleSketch(wl.d, wl.w, wl.G, wl.L, wl.seed)
        g = cs.CountSketch(wl.d, wl.w, list(wl.G), wl.L, wl.seed)
        g.set_chunk_sizes(0, 1 << 20, 1 << 19, 0)
        g.set_update_mode(2, rows_direct)
        o.update(host_np, p); g.update(xyz, p)
        o.scan_begin(); g.scan_begin(3000, 6)
        o.scan(host_np, p); g.scan(xyz, p)
        _compare(g, o, wl, 3000, (6,), host_np)
        assert g.scan_stats()["scan_launches"] >= 8
        g.close(); o.close()


def test_neighbour_shell_and_recount(cs):
    """cs_expand_neighbours (heavy cells and their surroundings) against a numpy restatement of the
    periodic 27-cell stencil, then cs_recount over the shell against exact counting (oracle pin)."""
    wl, xyz = _gen("cfg1", (1 << 18) + 7)
    host_np = xyz.cpu().numpy()
    G = wl.G[0]
    g = cs.CountSketch(wl.d, wl.w, list(wl.G), wl.L, wl.seed)
    g.update(xyz)
    g.scan_begin(50)
    g.scan(xyz)
    ids, _ = g.topk(50)
    edge = torch.tensor([0, G - 1, G * G * G - 1, (G - 1) * G, 5 + G * (G - 1) + G * G * 0], dtype=torch.int64, device="cuda")
    ids = torch.cat([ids, edge])
    shell = g.expand_neighbours(ids)
    c = _ids(ids).astype(np.int64)
    x, y, z = c % G, (c // G) % G, c // (G * G)
    t = np.arange(27)
    dx, dy, dz = t % 3 - 1, (t // 3) % 3 - 1, t // 9 - 1
    want = ((x[:, None] + dx) % G) + G * (((y[:, None] + dy) % G) + G * ((z[:, None] + dz) % G))
    assert np.array_equal(shell.cpu().numpy(), want)
    assert np.array_equal(shell[:, 13].cpu().numpy(), c)
    counts, _, n_members = g.recount(shell.reshape(-1).contiguous(), xyz)
    eid, ecnt = ora.exact_counts(host_np, G, wl.L)
    exact = dict(zip(eid.tolist(), ecnt.tolist()))
    flat = want.reshape(-1).tolist()
    seen, exp = set(), []
    for cid in flat:                                         # duplicate ids: the first occurrence counts
        exp.append(0 if cid in seen else exact.get(cid, 0))
        seen.add(cid)
    assert counts.cpu().numpy().tolist() == exp
    assert n_members == sum(exp)
    g.close()


def test_handle_stays_on_its_device_when_current_device_changes(cs):
    """Every entry point runs on the handle's device.  With one GPU only the bookkeeping can be checked: calls succeed
    and the caller's current device is unchanged afterwards."""
    wl, xyz = _gen("cfg1", 1 << 16)
    g = cs.CountSketch(wl.d, wl.w, list(wl.G), wl.L, wl.seed)
    before = torch.cuda.current_device()
    g.update(xyz)
    g.scan_begin(10)
    g.scan(xyz)
    g.topk(10)
    assert torch.cuda.current_device() == before
    g.close()


def test_scan_begin_rejects_oversized_k(cs):
    g = cs.CountSketch(3, 64, [8], 1.0, 1)
    with pytest.raises(cs.CsError) as e:
        g.scan_begin((1 << 26) + 1)
    assert e.value.code == cs.CS_ERR_ARG
    g.close()


def test_one_crossing_hierarchical_query_cfg4_shape(cs):
    """bench.py --workload cfg4 --query hierarchical at reduced size: ONE host-streamed update feeds a coarse and the fine
    mesh (G = 4642 = 11 * 422), the query is positions-free (Alg. 3): full search of the coarse
    mesh, then the children of its c*k heaviest cells.  Expected values: the oracle's own full search of the coarse mesh and
    its estimates of exactly those children.  The candidate set differs from the re-scan's on purpose (full dictionary)."""
    from paper_1711_00975_b200 import synth
    Gf, r = 4642, 11
    wl = synth.CONFIGS["cfg4"].scaled(6 * (1 << 16) + 77, w=1 << 16, G=(Gf // r, Gf))
    xyz = synth.generate(wl, device="cuda")
    host = _host_copy(xyz, True)
    k, c = 300, 4
    o = ora.OracleSketch(wl.d, wl.w, wl.G, wl.L, wl.seed)
    o.update(host.numpy())
    g = cs.CountSketch(wl.d, wl.w, list(wl.G), wl.L, wl.seed)
    g.set_chunk_sizes(1 << 16, 0, 0, 0)
    g.update_host(host)
    g.scan_begin(c * k)
    g.scan_all(0)
    parents, pest = g.topk(c * k, 0)
    cells0 = np.arange((Gf // r) ** 3, dtype=np.uint64)
    e0 = o.estimate(cells0, 0)
    order = np.lexsort((cells0, -e0.astype(np.int64)))[: c * k]
    assert np.array_equal(_ids(parents), cells0[order]) and np.array_equal(pest.cpu().numpy(), e0[order])
    g.scan_children(parents, 0, 1)
    kids, kest = g.topk(k, 1, device="cpu")
    p = cells0[order]
    Gp = np.uint64(Gf // r)
    px, py, pz = p % Gp, (p // Gp) % Gp, p // (Gp * Gp)
    t = np.arange(r ** 3, dtype=np.uint64)
    R, G64 = np.uint64(r), np.uint64(Gf)
    cx = (px[:, None] * R + t % R).ravel()
    cy = (py[:, None] * R + (t // R) % R).ravel()
    cz = (pz[:, None] * R + t // (R * R)).ravel()
    kid = np.unique(cx + G64 * (cy + G64 * cz))
    ek = o.estimate(kid, 1)
    ordk = np.lexsort((kid, -ek.astype(np.int64)))[:k]
    assert np.array_equal(_ids(kids), kid[ordk]) and np.array_equal(kest.numpy(), ek[ordk])
    g.close(); o.close()


def test_phase_timing_and_route_counters(cs):
    """cs_set_timing / cs_get_timing / cs_update_stats: the counters of the binned route account for every record
    (particles x binned rows), a single-cell stream pushes almost all of them through the overflow routes, and the phase
    timer reports the kernel classes that ran."""
    from paper_1711_00975_b200 import synth
    wl, xyz = _gen("cfg3", (1 << 22) + 2)
    g = cs.CountSketch(wl.d, wl.w, list(wl.G), wl.L, wl.seed)
    g.set_update_mode(2, 3)                                   # binned, 3 of 7 rows direct -> 4 binned rows
    g.set_timing(True)
    g.update(xyz)
    st = g.update_stats()
    # torch allocations are 256-byte aligned and n is even: no head / tail particle outside the pairs
    assert st["staging_overflow"] + st["region_overflow"] + st["leftover"] + st["binned"] == 4 * ((1 << 22) + 2), st
    assert st["staging_overflow"] == 0 and st["region_overflow"] == 0          # clustered but spread stream: nothing overflows
    g.scan_begin(1000)
    g.scan(xyz)
    g.topk(1000)
    tm = g.get_timing()
    assert tm["update_scatter"][0] > 0 and tm["update_apply"][0] > 0 and tm["scan_first"][0] > 0 and tm["select"][0] > 0
    assert tm["update_scatter"][1] == 1 and tm["compact_kept"] == (0.0, 0)
    assert g.get_timing()["update_scatter"] == (0.0, 0)       # read and forgotten
    g.set_timing(False)
    g.reset()
    one = torch.full((1 << 21, 3), 3.3, dtype=torch.float32, device="cuda")
    g.update(one)
    st = g.update_stats()
    assert st["staging_overflow"] + st["region_overflow"] > 0.9 * 4 * (1 << 21), st
    assert st["staging_overflow"] + st["region_overflow"] + st["leftover"] + st["binned"] == 4 * (1 << 21)
    g.close()
