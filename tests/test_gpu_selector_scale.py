"""The selector (cs_select.cu, one cooperative launch per compaction) on lists longer than the GPU holds tiles at once:
more than 4 x 148 tiles of 2048 entries, so that CTAs take several tiles per sweep and the look-back runs across them.
The ordinary parity cases stay below that size; the full-size runs (tests/test_full_size_parity.py) reach it but are
opt-in.  Expected values: estimates from the oracle, ordered by the definition (R9):
distinct ids, estimate descending, id ascending, first k.
"""
import numpy as np
import pytest
import torch

from oracle import cs_oracle as ora

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def cs():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1711_00975_b200 import build, binding
    build.build_libcs()
    binding.lib()
    return binding


def _by_definition(cells, est, k):
    c, first = np.unique(cells, return_index=True)
    e = est[first]
    order = np.lexsort((c, -e.astype(np.int64)))[:k]
    return c[order], e[order]


@pytest.mark.parametrize("n_cells,k,pieces", [(2_700_001, 1_500_000, 2), (1_300_003, 1_300_003, 1), (4_200_000, 40_000, 3)])
def test_long_candidate_lists(cs, n_cells, k, pieces):
    from paper_1711_00975_b200 import synth
    wl = synth.CONFIGS["cfg3"].scaled(400_001)
    xyz = synth.generate(wl, device="cuda")
    host = xyz.cpu().numpy()
    o = ora.OracleSketch(wl.d, wl.w, wl.G, wl.L, wl.seed)
    o.update(host)
    g = cs.CountSketch(wl.d, wl.w, list(wl.G), wl.L, wl.seed)
    g.update(xyz)
    assert np.array_equal(g.sketch().cpu().numpy(), o.sketch())

    rng = np.random.default_rng(n_cells)
    G = wl.G[0]
    occupied = ora.quantise(host[rng.integers(0, host.shape[0], size=n_cells // 4)], G, wl.L)
    fresh = rng.integers(0, G ** 3, size=n_cells - n_cells // 4 - n_cells // 5, dtype=np.uint64)
    cells = np.concatenate([occupied, fresh])
    cells = np.concatenate([cells, cells[rng.integers(0, len(cells), size=n_cells // 5)]])      # duplicates
    rng.shuffle(cells)
    assert len(cells) == n_cells
    want_ids, want_est = _by_definition(cells, o.estimate(cells), k)

    dev = torch.from_numpy(cells.view(np.int64)).cuda()
    g.scan_begin(k)
    cuts = np.linspace(0, n_cells, pieces + 1).astype(np.int64)
    for lo, hi in zip(cuts[:-1], cuts[1:]):
        g.scan_cells(dev[lo:hi].contiguous())
    ids, est = g.topk(k)
    stats = g.scan_stats()
    assert stats["compactions"] >= 1
    got_ids = ids.cpu().numpy().view(np.uint64)
    assert len(got_ids) == len(want_ids)
    assert np.array_equal(got_ids, want_ids), "ids differ from the definition"
    assert np.array_equal(est.cpu().numpy(), want_est), "estimates differ from the oracle's"
    g.close(); o.close()
