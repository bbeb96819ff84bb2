"""The multi-GPU path (PAPER.md:578 sketches of stream shards sum) executed ON a GPU through libcs.so:

  * with a real NCCL process group of one rank: paper_1711_00975_b200.sharded.sharded_pass with the exchange steps
    forced (in-place all-reduce of the handle's own table through cs_table_ptr, all-gather of the top-k ids, merge through
    cs_scan_cells) -- every collective and every merge kernel runs on CUDA tensors, the result must equal the oracle's;
  * with two handles on one GPU standing in for two ranks (two host threads, each its own stream and handle, lock-step
    collectives over their CUDA tensors): shards with running-index offsets, p < 1, several scales; bit-identical to the
    single-stream oracle.  (Kernels of different "ranks" never wait on one another: the lock step is on the host.)
One GPU cannot measure scaling; this checks that the device code path of N > 1 is correct.
"""
import socket
import threading

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


def _ids(t):
    return t.cpu().numpy().view(np.uint64)


def _oracle(wl, host_np, p, k):
    o = ora.OracleSketch(wl.d, wl.w, wl.G, wl.L, wl.seed)
    o.update(host_np, p)
    o.scan_begin()
    o.scan(host_np, p)
    out = [(o.sketch(s), *o.topk(k, s)) for s in range(len(wl.G))]
    o.close()
    return out


def test_table_view_aliases_the_counters(cs):
    from paper_1711_00975_b200 import synth
    wl = synth.CONFIGS["cfg1"].scaled(50001)
    xyz = synth.generate(wl, device="cuda")
    g = cs.CountSketch(wl.d, wl.w, list(wl.G), wl.L, wl.seed)
    g.update(xyz)
    v = g.table_view()
    assert v.shape == (wl.d, wl.w) and v.dtype == torch.int32 and v.is_cuda
    assert torch.equal(v, g.sketch())
    v += 1                                                   # writes through to the handle's table
    assert torch.equal(g.sketch(), v)
    g.close()


def test_sharded_pass_over_a_one_rank_nccl_group(cs):
    import torch.distributed as dist
    from paper_1711_00975_b200 import sharded, synth
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    dist.init_process_group("nccl", init_method=f"tcp://127.0.0.1:{port}", world_size=1, rank=0,
                            device_id=torch.device("cuda", torch.cuda.current_device()))
    try:
        for name, n, p, k in (("cfg3", (1 << 21) + 3, 1.0, 2000), ("cfg5", 1 << 21, 0.3, 500)):
            wl = synth.CONFIGS[name].scaled(n)
            xyz = synth.generate(wl, device="cuda")
            want = _oracle(wl, xyz.cpu().numpy(), p, k)
            g = cs.CountSketch(wl.d, wl.w, list(wl.G), wl.L, wl.seed)
            res = sharded.sharded_pass(g, xyz, 0, p, k, cs.INT32_MAX, dist, 1, force_merge=True)
            for s, (T, oi, ov) in enumerate(want):
                assert np.array_equal(g.sketch(s).cpu().numpy(), T)
                assert np.array_equal(_ids(res[s][0]), oi) and np.array_equal(res[s][1].cpu().numpy(), ov)
            g.close()
    finally:
        dist.destroy_process_group()


class _LockStepGroup:
    """torch.distributed look-alike for `world` host threads of one process sharing one GPU."""

    class ReduceOp:
        SUM = "sum"

    def __init__(self, world):
        self.world = world
        self.bar = threading.Barrier(world)
        self.slots = [None] * world
        self.tls = threading.local()

    def rank(self):
        return self.tls.rank

    def all_reduce(self, t, op=None):
        torch.cuda.current_stream().synchronize()
        self.slots[self.rank()] = t
        self.bar.wait()
        total = torch.zeros_like(t)
        for x in self.slots:
            total += x
        torch.cuda.current_stream().synchronize()
        self.bar.wait()
        t.copy_(total)
        torch.cuda.current_stream().synchronize()
        self.bar.wait()

    def all_gather_into_tensor(self, out, t):
        torch.cuda.current_stream().synchronize()
        self.slots[self.rank()] = t
        self.bar.wait()
        out.copy_(torch.cat([x.reshape(-1) for x in self.slots]))
        torch.cuda.current_stream().synchronize()
        self.bar.wait()


@pytest.mark.parametrize("name,n,p,k", [("cfg3", (1 << 21) + 7, 1.0, 2000), ("cfg5", (1 << 21) + 5, 0.3, 500),
                                        ("cfg1", 300001, 0.6, 100)])
def test_two_handles_stand_in_for_two_ranks(cs, name, n, p, k):
    from paper_1711_00975_b200 import sharded, synth
    wl = synth.CONFIGS[name].scaled(n)
    xyz = synth.generate(wl, device="cuda")
    want = _oracle(wl, xyz.cpu().numpy(), p, k)
    world = 2
    grp = _LockStepGroup(world)
    results, errors = [None] * world, []
    dev = torch.cuda.current_device()

    def run(rank):
        try:
            torch.cuda.set_device(dev)
            grp.tls.rank = rank
            with torch.cuda.stream(torch.cuda.Stream()):
                lo, hi = sharded.shard_bounds(n, rank, world)
                g = cs.CountSketch(wl.d, wl.w, list(wl.G), wl.L, wl.seed)
                res = sharded.sharded_pass(g, xyz[lo:hi], lo, p, k, cs.INT32_MAX, grp, world)
                results[rank] = ([g.sketch(s).cpu().numpy() for s in range(len(wl.G))],
                                 [(_ids(r[0]), r[1].cpu().numpy()) for r in res])
                g.close()
        except Exception as e:                               # noqa: BLE001
            errors.append(e)
            grp.bar.abort()

    th = [threading.Thread(target=run, args=(r,)) for r in range(world)]
    for t in th:
        t.start()
    for t in th:
        t.join()
    assert not errors, errors
    for rank in range(world):
        tables, tops = results[rank]
        for s, (T, oi, ov) in enumerate(want):
            assert np.array_equal(tables[s], T), f"rank {rank}: merged table differs at scale {s}"
            assert np.array_equal(tops[s][0], oi) and np.array_equal(tops[s][1], ov), f"rank {rank}: top-k differs"
