"""Stream-sharded pass over several ranks (sketch mergeability).

Host-side orchestration only: every arithmetic step runs in the engine (binding.CountSketch, i.e. libcs.so);
`torch.distributed` carries the one real exchange, the sum of the int32 tables, plus the all-gather of the
per-rank top-k ids.  The result is bit-identical to a single stream over the concatenated shards:

  * rank r owns the contiguous particle range [index0, index0 + n_r) and offsets its running particle index,
    so the sampling decisions (R13) equal the single-stream ones;
  * int32 adds commute and wrap, so the all-reduced table equals the single-stream table;
  * a cell of the global top-k is in the local top-k of every rank whose shard contains it (the estimate is a
    function of the cell and the global table only), so the union of the local lists contains the global one;
    the merge dedupes by id and keeps the (estimate descending, id ascending) order.

The engine interface used: reset, set_update_index, update, sketch, sketch_add, scan_begin, set_scan_index,
scan, topk, scan_cells, n_scales.  Tests drive this module on CPU (gloo, world size 2) with an engine adapter
of their own.
"""
from __future__ import annotations

import torch


def shard_bounds(n_total: int, rank: int, world: int, align: int = 4):
    """Contiguous range [lo, hi) of rank `rank`: equal parts rounded to `align` particles, last rank takes the rest."""
    per = (n_total // world) // align * align
    lo = rank * per
    hi = n_total if rank == world - 1 else lo + per
    return lo, hi


def merge_tables(engine, dist) -> None:
    """T <- sum over ranks of T: one all-reduce per scale, IN PLACE on the engine's own table when it exposes it
    (binding.CountSketch.table_view: no table-sized temporaries); engines without a view (the CPU test adapter) fall
    back to read + all-reduce + add of the difference."""
    for s in range(engine.n_scales):
        view = engine.table_view(s) if hasattr(engine, "table_view") else None
        if view is not None:
            dist.all_reduce(view, op=dist.ReduceOp.SUM)
            continue
        own = engine.sketch(s)
        total = own.clone()
        dist.all_reduce(total, op=dist.ReduceOp.SUM)
        total -= own
        engine.sketch_add(total, s)


def merge_topk(engine, k: int, dist, world: int):
    """All-gather the local top-k ids of every scale, feed them back as candidates, return the merged top-k."""
    out = []
    for s in range(engine.n_scales):
        ids, _ = engine.topk(k, s)
        pad = torch.full((k,), -1, dtype=torch.int64, device=ids.device)
        pad[: ids.numel()] = ids
        allids = torch.empty(world * k, dtype=torch.int64, device=ids.device)
        dist.all_gather_into_tensor(allids, pad)
        engine.scan_cells(allids[allids >= 0].contiguous(), s)
        out.append(engine.topk(k, s))
    return out


def sharded_pass(engine, xyz_shard, index0: int, sample_p: float, k: int, thr_min: int, dist=None, world: int = 1,
                 update=None, scan=None, topk_device=None, force_merge: bool = False):
    """reset -> update(shard) -> [all-reduce tables] -> re-scan(shard) -> [merge top-k]; returns per-scale (ids, est).

    `update` / `scan` override the engine methods used for the two passes (the host-streamed variants);
    `topk_device` ("cpu") makes the single-rank result land in host memory."""
    engine.reset()
    engine.set_update_index(index0)
    (update or engine.update)(xyz_shard, sample_p)
    merge = world > 1 or (force_merge and dist is not None)     # force_merge: run the exchange steps on a 1-rank group
    if merge:
        merge_tables(engine, dist)
    engine.scan_begin(k, thr_min)
    engine.set_scan_index(index0)
    (scan or engine.scan)(xyz_shard, sample_p)
    if merge:
        return merge_topk(engine, k, dist, world)
    if topk_device is not None:
        return [engine.topk(k, s, device=topk_device) for s in range(engine.n_scales)]
    return [engine.topk(k, s) for s in range(engine.n_scales)]
