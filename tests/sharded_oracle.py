"""Full-size parity device (SURVEY section 4 tier T3, 8.d.4): the CPU oracle run over P disjoint index ranges of one stream.

Valid by the mergeability of the sketch ("sketches from different nodes sum"; itself an oracle pin):
  * update: shard r = particles [lo_r, hi_r) with running index lo_r (ora_set_update_index), each into its own tables;
    the tables are summed elementwise (int32 wraparound);
  * selection: every shard, holding the SUMMED tables, replays its own particles through ora_select_streaming (top-k of
    the shard in O(k) memory + every cell of the shard with estimate >= thr); the lists are merged by the oracle's rule:
    unique by id, (estimate descending, id ascending), first k.  A cell of the global top-k is among the k best of
    every shard that contains it, because its estimate depends on the cell and the summed tables only.

Each shard runs the plain single-threaded oracle (oracle/cs_oracle.cpp) as it stands; the shards run in P Python
threads (ctypes releases the GIL; the oracle has no global state).  This is a parity device, not the timed baseline.
Test infrastructure: imports oracle/, never the CUDA package.
"""
from __future__ import annotations

from concurrent.futures import ThreadPoolExecutor

import numpy as np

from oracle import cs_oracle as ora


def shard_ranges(n: int, parts: int):
    """parts contiguous ranges covering [0, n); boundaries deliberately not multiples of 4."""
    cuts = [0]
    for r in range(1, parts):
        c = (n * r) // parts
        cuts.append(min(n, c + (r % 3)))
    cuts.append(n)
    return [(a, b) for a, b in zip(cuts[:-1], cuts[1:])]


def _merge(lists, k=None):
    """[(ids, est)] -> unique by id, ordered (est desc, id asc), cut to k."""
    ids = np.concatenate([l[0] for l in lists]) if lists else np.empty(0, np.uint64)
    est = np.concatenate([l[1] for l in lists]) if lists else np.empty(0, np.int32)
    ids, first = np.unique(ids, return_index=True)
    est = est[first]
    order = np.lexsort((ids, -est.astype(np.int64)))
    if k is not None:
        order = order[:k]
    return ids[order], est[order]


class ShardedOracle:
    """P oracle handles over disjoint ranges of one stream."""

    def __init__(self, d, w, G, L, seed, parts: int, counting: int = 0):
        self.parts = parts
        self.counting = counting
        self.o = [ora.OracleSketch(d, w, G, L, seed) for _ in range(parts)]
        if counting:
            for o in self.o:
                o.set_mode(counting)
        self.n_scales = self.o[0].n_scales
        self.ranges = None
        self.index0 = 0
        self.pool = ThreadPoolExecutor(max_workers=parts)

    def close(self):
        self.pool.shutdown()
        for o in self.o:
            o.close()

    def update(self, xyz: np.ndarray, sample_p: float = 1.0, index0: int = 0):
        """Adds the stream xyz (running indices index0 ..) to the tables of ALL handles (each ends up holding the sum)."""
        n = xyz.shape[0]
        ranges = shard_ranges(n, self.parts)

        def work(r):
            lo, hi = ranges[r]
            fresh = ora.OracleSketch(self.o[0].d, self.o[0].w, self.o[0].G, self.o[0].L, self.o[0].seed)
            if self.counting:
                fresh.set_mode(self.counting)
            fresh.set_update_index(index0 + lo)
            fresh.update(xyz[lo:hi], sample_p)
            t = [fresh.sketch(s) for s in range(self.n_scales)]
            fresh.close()
            return t

        parts = list(self.pool.map(work, range(self.parts)))
        for s in range(self.n_scales):
            tot = np.zeros_like(parts[0][s], dtype=np.uint32)
            for t in parts:
                tot += t[s].view(np.uint32)                      # two's-complement wraparound
            tot = tot.view(np.int32)
            for o in self.o:
                o.sketch_add(tot, s)

    def sketch(self, scale: int = 0) -> np.ndarray:
        return self.o[0].sketch(scale)

    def estimate(self, cells, scale: int = 0) -> np.ndarray:
        return self.o[0].estimate(cells, scale)

    def select(self, xyz: np.ndarray, k: int, thr: int = ora.INT32_MAX, sample_p: float = 1.0, index0: int = 0):
        """Per scale: (top-k ids, est), (excursion ids, est with estimate >= thr) of the whole replayed stream."""
        n = xyz.shape[0]
        ranges = shard_ranges(n, self.parts)

        def work(r):
            lo, hi = ranges[r]
            return [self.o[r].select_streaming(xyz[lo:hi], index0 + lo, k, thr, sample_p, s) for s in range(self.n_scales)]

        res = list(self.pool.map(work, range(self.parts)))
        out = []
        for s in range(self.n_scales):
            top = _merge([res[r][s][0] for r in range(self.parts)], k)
            exc = _merge([res[r][s][1] for r in range(self.parts)])
            out.append((top, exc))
        return out
