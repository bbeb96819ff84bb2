"""World-size-2 `gloo` test of the stream-sharded pass (paper_1711_00975_b200/sharded.py).

No GPU here, so the engine behind the orchestration is a test-side adapter over the CPU oracle with the
CountSketch method names; what is under test is the HOST logic of the N > 1 path: shard bounds, running-index
offsets (sampling decisions), the int32 table all-reduce, the all-gather + candidate merge.  Expected value:
one oracle over the whole stream (sketch mergeability).
"""
import os
import socket
import sys
from pathlib import Path

import numpy as np
import pytest
import torch
import torch.multiprocessing as mp

ROOT = Path(__file__).resolve().parent.parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

INT32_MAX = 2 ** 31 - 1


class OracleEngine:
    """CountSketch-shaped adapter over oracle.OracleSketch (torch CPU tensors in and out)."""

    def __init__(self, d, w, G, L, seed):
        from oracle import cs_oracle as ora
        self.o = ora.OracleSketch(d, w, G, L, seed)
        self.n_scales = self.o.n_scales
        self.extra = [dict() for _ in range(self.n_scales)]      # cells fed through scan_cells: id -> est

    def reset(self):
        self.o.reset()

    def set_update_index(self, i):
        self.o.set_update_index(i)

    def set_scan_index(self, i):
        self.o.set_scan_index(i)

    def update(self, xyz, p=1.0):
        self.o.update(xyz.numpy(), p)

    def sketch(self, s=0):
        return torch.from_numpy(self.o.sketch(s))

    def sketch_add(self, t, s=0):
        self.o.sketch_add(t.numpy(), s)

    def scan_begin(self, k_max, thr_min=INT32_MAX):
        self.o.scan_begin()
        self.extra = [dict() for _ in range(self.n_scales)]

    def scan(self, xyz, p=1.0):
        self.o.scan(xyz.numpy(), p)

    def scan_cells(self, cells, s=0):
        c = cells.numpy().view(np.uint64)
        for cid, e in zip(c.tolist(), self.o.estimate(c, s).tolist()):
            self.extra[s][cid] = e

    def topk(self, k, s=0):
        n = self.o.candidate_count(s)
        ids, est = self.o.topk(n, s) if n else (np.empty(0, np.uint64), np.empty(0, np.int32))
        merged = dict(zip(ids.tolist(), est.tolist()))
        merged.update(self.extra[s])
        order = sorted(merged.items(), key=lambda t: (-t[1], t[0]))[:k]
        ids = np.array([t[0] for t in order], dtype=np.uint64)
        est = np.array([t[1] for t in order], dtype=np.int32)
        return torch.from_numpy(ids.view(np.int64).copy()), torch.from_numpy(est)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, cfg, ret):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    import torch.distributed as dist
    from paper_1711_00975_b200 import sharded, synth
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        wl = synth.CONFIGS[cfg["name"]].scaled(cfg["n"])
        xyz = synth.generate(wl, device="cpu")
        lo, hi = sharded.shard_bounds(wl.N, rank, world)
        eng = OracleEngine(wl.d, wl.w, list(wl.G), wl.L, wl.seed)
        res = sharded.sharded_pass(eng, xyz[lo:hi].contiguous(), lo, cfg["p"], cfg["k"], INT32_MAX, dist, world)
        tables = [eng.sketch(s).numpy() for s in range(eng.n_scales)]
        ret[rank] = ([(i.numpy().view(np.uint64).copy(), e.numpy().copy()) for i, e in res], tables, (lo, hi))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("cfg", [
    {"name": "cfg1", "n": 40001, "p": 1.0, "k": 50},
    {"name": "cfg5", "n": 30000, "p": 0.37, "k": 40},      # 4 scales, sampled: index offsets matter
])
def test_two_rank_sharded_pass_equals_single_stream(cfg):
    from oracle import cs_oracle as ora
    from paper_1711_00975_b200 import synth
    world = 2
    mgr = mp.Manager()
    ret = mgr.dict()
    mp.spawn(_worker, args=(world, _free_port(), cfg, ret), nprocs=world, join=True)

    wl = synth.CONFIGS[cfg["name"]].scaled(cfg["n"])
    host = synth.generate(wl, device="cpu").numpy()
    o = ora.OracleSketch(wl.d, wl.w, list(wl.G), wl.L, wl.seed)
    o.update(host, cfg["p"])
    o.scan_begin()
    o.scan(host, cfg["p"])
    assert ret[0][2][1] == ret[1][2][0] and ret[0][2][0] == 0 and ret[1][2][1] == wl.N
    for s in range(len(wl.G)):
        want_ids, want_est = o.topk(cfg["k"], s)
        for r in range(world):
            res, tables, _ = ret[r]
            assert np.array_equal(tables[s], o.sketch(s)), f"rank {r}: merged table differs at scale {s}"
            assert np.array_equal(res[s][0], want_ids) and np.array_equal(res[s][1], want_est), \
                f"rank {r}: merged top-k differs at scale {s}"


def test_shard_bounds_cover_the_stream():
    from paper_1711_00975_b200 import sharded
    for n in (0, 1, 7, 1000, (1 << 20) + 3):
        for world in (1, 2, 3, 8):
            spans = [sharded.shard_bounds(n, r, world) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == n
            for a, b in zip(spans[:-1], spans[1:]):
                assert a[1] == b[0] and a[0] % 4 == 0
