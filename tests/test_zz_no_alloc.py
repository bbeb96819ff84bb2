"""cs_select_static (include/cs.h): the selection entry point that allocates nothing -- its scratch is a file-scope device
array of the library (CS_SELECT_STATIC_MAX_N candidates).  Checked against the existing path (cs_scan_begin + cs_scan_cells +
cs_topk on a handle: the growable, cudaMalloc'ed candidate buffers) on calls in a row that share the scratch: the second
is smaller than the first, the third larger again, so anything a call leaves behind would show.  Integer work: bit-exact.

This file is named to be collected last: the suite runs with pytest -x, a failure here must not hide other tests.
"""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def cs():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1711_00975_b200 import build, binding
    build.build_libcs()
    binding.lib()
    return binding


@pytest.fixture(scope="module")
def sketch(cs):
    from paper_1711_00975_b200 import synth
    wl = synth.CONFIGS["cfg2"].scaled(400_003)
    xyz = synth.generate(wl, device="cuda")
    g = cs.CountSketch(wl.d, wl.w, list(wl.G), wl.L, wl.seed)
    g.update(xyz)
    yield g, wl, xyz
    g.close()


def _candidates(g, wl, xyz, n, seed):
    """n cell ids: cells of particles (heavy ones repeat), random cells of the mesh, and deliberate duplicates."""
    gen = torch.Generator(device="cuda").manual_seed(seed)
    G = wl.G[0]
    take = torch.randint(0, xyz.shape[0], (n // 2,), device="cuda", generator=gen)
    q = torch.clamp(torch.floor(xyz[take] * np.float32(G / wl.L)), 0, G - 1).to(torch.int64)
    occupied = q[:, 0] + G * (q[:, 1] + G * q[:, 2])
    rand = torch.randint(0, G ** 3, (n - n // 2 - n // 8,), device="cuda", generator=gen)
    cells = torch.cat([occupied, rand])
    dup = cells[torch.randint(0, cells.numel(), (n // 8,), device="cuda", generator=gen)]
    cells = torch.cat([cells, dup])
    cells = cells[torch.randperm(cells.numel(), device="cuda", generator=gen)].contiguous()
    assert cells.numel() == n
    return cells


def _existing_path(g, cells, k):
    g.scan_begin(k)
    g.scan_cells(cells)
    ids, est = g.topk(k)
    return ids.cpu().numpy(), est.cpu().numpy()


def _by_definition(cells, est, k):
    c, first = np.unique(cells.cpu().numpy(), return_index=True)
    e = est.cpu().numpy()[first]
    order = np.lexsort((c, -e.astype(np.int64)))[:k]
    return c[order], e[order]


def test_static_scratch_selection_equals_the_handle_path_on_calls_in_a_row(cs, sketch):
    g, wl, xyz = sketch
    M = cs.SELECT_STATIC_MAX_N
    ids_out = torch.empty(M, dtype=torch.int64, device="cuda")
    est_out = torch.empty(M, dtype=torch.int32, device="cuda")
    n_out = torch.zeros(1, dtype=torch.int32, device="cuda")
    cases = [(60_001, 5_000, 1), (3_001, 700, 2), (M, 20_000, 3), (3_001, 700, 2), (257, 4_000, 4)]
    prepared = []
    for n, k, seed in cases:
        cells = _candidates(g, wl, xyz, n, seed)
        prepared.append((cells, g.estimate(cells), k, _existing_path(g, cells, k)))
    torch.cuda.synchronize()
    for i, (cells, est, k, (want_ids, want_est)) in enumerate(prepared):
        ids_out.fill_(-1); est_out.fill_(-1); n_out.fill_(-1)
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info()[0]
        cs.select_static(cells, est, k, ids_out, est_out, n_out)
        torch.cuda.synchronize()
        if i > 0:                                              # the first call may load its kernels lazily
            assert torch.cuda.mem_get_info()[0] == free_before, f"call {i}: device memory in use changed across the call"
        m = int(n_out.item())
        assert m == len(want_ids), f"call {i}: {m} entries, the handle path returns {len(want_ids)}"
        assert np.array_equal(ids_out[:m].cpu().numpy(), want_ids), f"call {i}: ids differ from the handle path"
        assert np.array_equal(est_out[:m].cpu().numpy(), want_est), f"call {i}: estimates differ from the handle path"
        def_ids, def_est = _by_definition(cells, est, k)
        assert np.array_equal(want_ids, def_ids) and np.array_equal(want_est, def_est)
        assert int(ids_out[m:].max().item() if m < M else -1) == -1, "wrote past the entries it reports"


def test_static_scratch_selection_edges(cs, sketch):
    g, wl, xyz = sketch
    ids_out = torch.full((64,), -1, dtype=torch.int64, device="cuda")
    est_out = torch.full((64,), -1, dtype=torch.int32, device="cuda")
    n_out = torch.full((1,), -1, dtype=torch.int32, device="cuda")
    none = torch.empty(0, dtype=torch.int64, device="cuda")
    cs.select_static(none, none.to(torch.int32), 10, ids_out, est_out, n_out)       # empty list
    assert int(n_out.item()) == 0 and int(ids_out.max().item()) == -1
    one = torch.tensor([7, 7, 7], dtype=torch.int64, device="cuda")                 # one distinct id, k larger than that
    e = torch.tensor([-5, -5, -5], dtype=torch.int32, device="cuda")
    cs.select_static(one, e, 10, ids_out, est_out, n_out)
    assert int(n_out.item()) == 1 and int(ids_out[0].item()) == 7 and int(est_out[0].item()) == -5
    tie = torch.tensor([9, 3, 1 << 59, 5], dtype=torch.int64, device="cuda")        # equal estimates: id ascending
    e = torch.tensor([4, 4, 2 ** 31 - 1, -(2 ** 31)], dtype=torch.int32, device="cuda")
    cs.select_static(tie, e, 4, ids_out, est_out, n_out)
    assert int(n_out.item()) == 4
    assert ids_out[:4].tolist() == [1 << 59, 3, 9, 5] and est_out[:4].tolist() == [2 ** 31 - 1, 4, 4, -(2 ** 31)]
    cs.select_static(tie, e, 0, ids_out, est_out, n_out)                            # k = 0
    assert int(n_out.item()) == 0


def test_static_scratch_selection_rejects_sizes_beyond_its_scratch(cs):
    M = cs.SELECT_STATIC_MAX_N
    ids = torch.zeros(M + 1, dtype=torch.int64, device="cuda")
    est = torch.zeros(M + 1, dtype=torch.int32, device="cuda")
    ids_out = torch.full((M + 1,), -1, dtype=torch.int64, device="cuda")
    est_out = torch.empty(M + 1, dtype=torch.int32, device="cuda")
    n_out = torch.full((1,), -1, dtype=torch.int32, device="cuda")
    with pytest.raises(cs.CsError) as err:
        cs.select_static(ids, est, 10, ids_out, est_out, n_out)
    assert err.value.code == -1 and "CS_SELECT_STATIC_MAX_N" in str(err.value)
    with pytest.raises(cs.CsError) as err:
        cs.select_static(ids[:100], est[:100], M + 1, ids_out, est_out, n_out)
    assert err.value.code == -1 and "CS_SELECT_STATIC_MAX_N" in str(err.value)
    torch.cuda.synchronize()
    assert int(n_out.item()) == -1 and int(ids_out.max().item()) == -1, "a rejected call must launch nothing"
