"""Thin ctypes binding over libcs.so (include/cs.h).  Argument marshalling only: every step of the path runs
in the library's CUDA kernels.  torch is used for device memory and streams.  There is no CPU fallback: if the
library is missing or fails to load, importing succeeds but the first use raises.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import torch

_PKG = Path(__file__).resolve().parent
LIB_PATH = _PKG / "libcs.so"

CS_OK, CS_ERR_ARG, CS_ERR_NOMEM, CS_ERR_CUDA, CS_ERR_STATE = 0, -1, -2, -3, -4
INT32_MIN, INT32_MAX = -(2 ** 31), 2 ** 31 - 1

u64, i32, u32, dbl, vp, ci = C.c_uint64, C.c_int32, C.c_uint32, C.c_double, C.c_void_p, C.c_int

# name -> (restype, argtypes); every symbol include/cs.h declares
SIGNATURES = {
    "cs_version": (C.c_char_p, []),
    "cs_last_error": (C.c_char_p, []),
    "cs_derive_coeffs": (ci, [u64, ci, vp, vp]),
    "cs_sample_threshold": (u64, [dbl]),
    "cs_hash_cell": (ci, [u64, u64, u64, ci, vp, vp]),
    "cs_create": (ci, [vp, ci, u64, u32, dbl, u64]),
    "cs_create_multi": (ci, [vp, ci, ci, u64, vp, dbl, u64]),
    "cs_destroy": (ci, [vp]),
    "cs_reset": (ci, [vp]),
    "cs_set_stream": (ci, [vp, vp]),
    "cs_set_table_budget": (ci, [vp, u64]),
    "cs_set_chunk_sizes": (ci, [vp, u64, u64, u64, u64]),
    "cs_set_replay_cache": (ci, [vp, u64]),
    "cs_set_update_mode": (ci, [vp, ci, ci]),
    "cs_set_counting_mode": (ci, [vp, ci]),
    "cs_set_scan_mode": (ci, [vp, ci]),
    "cs_set_update_index": (ci, [vp, u64]),
    "cs_set_scan_index": (ci, [vp, u64]),
    "cs_get_update_index": (ci, [vp, vp]),
    "cs_update": (ci, [vp, vp, u64, dbl]),
    "cs_update_host": (ci, [vp, vp, u64, dbl]),
    "cs_pack_records": (ci, [vp, vp, u64, vp]),
    "cs_update_records": (ci, [vp, vp, u64, dbl]),
    "cs_update_records_host": (ci, [vp, vp, u64, dbl]),
    "cs_scan_records": (ci, [vp, vp, u64, dbl]),
    "cs_scan_records_host": (ci, [vp, vp, u64, dbl]),
    "cs_estimate": (ci, [vp, ci, vp, u64, vp]),
    "cs_scan_begin": (ci, [vp, u64, i32]),
    "cs_set_candidate_capacity": (ci, [vp, u64]),
    "cs_scan": (ci, [vp, vp, u64, dbl]),
    "cs_scan_host": (ci, [vp, vp, u64, dbl]),
    "cs_scan_cells": (ci, [vp, ci, vp, u64]),
    "cs_scan_all": (ci, [vp, ci]),
    "cs_scan_children": (ci, [vp, ci, ci, vp, u64]),
    "cs_topk": (ci, [vp, ci, u64, vp, vp, vp]),
    "cs_excursion": (ci, [vp, ci, i32, u64, vp, vp, vp]),
    "cs_recount": (ci, [vp, ci, vp, u64, vp, u64, vp, vp, u64, vp]),
    "cs_expand_neighbours": (ci, [vp, ci, vp, u64, vp]),
    "cs_scan_stats": (ci, [vp, ci, vp]),
    "cs_sketch_read": (ci, [vp, ci, vp]),
    "cs_sketch_add": (ci, [vp, ci, vp]),
    "cs_coeffs": (ci, [vp, ci, vp, vp]),
    "cs_table_ptr": (ci, [vp, ci, vp]),
    "cs_set_timing": (ci, [vp, ci]),
    "cs_get_timing": (ci, [vp, vp, vp]),
    "cs_update_stats": (ci, [vp, vp]),
    "cs_launch_count": (ci, [vp, vp]),
    "cs_probe_l2": (ci, [ci, u64, u64, ci, vp, vp]),
    "cs_select_static": (ci, [vp, vp, u64, u64, vp, vp, vp, vp]),
    "cs_probe_stream": (ci, [vp, u64, ci, vp, vp]),
}

_lib = None


class CsError(RuntimeError):
    def __init__(self, code: int, what: str, msg: str):
        super().__init__(f"{what} failed with status {code}: {msg}")
        self.code = code


def lib():
    """Loads libcs.so (built by paper_1711_00975_b200.build).  Raises if it is missing: no fallback."""
    global _lib
    if _lib is None:
        if not LIB_PATH.exists():
            raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_1711_00975_b200.build` "
                               "(the CUDA library is the only implementation; there is no CPU fallback)")
        L = C.CDLL(str(LIB_PATH))
        for name, (res, args) in SIGNATURES.items():
            f = getattr(L, name)
            f.restype = res
            f.argtypes = args
        _lib = L
    return _lib


def _chk(rc: int, what: str):
    if rc != 0:
        raise CsError(rc, what, lib().cs_last_error().decode())


def version() -> str:
    return lib().cs_version().decode()


def derive_coeffs(seed: int, d: int):
    """Host-only: (d x 4 array of a, b, a', b'; sampling key K) as the library derives them."""
    import numpy as np
    out = np.empty(4 * d, dtype=np.uint64)
    K = u64(0)
    _chk(lib().cs_derive_coeffs(seed, d, out.ctypes.data_as(vp), C.byref(K)), "cs_derive_coeffs")
    return out.reshape(d, 4), int(K.value)


def hash_cell(a: int, b: int, c: int, big=True):
    """Host-only: ((a*c + b) mod (2^61-1), its low 32 bits) through the library's limb arithmetic (csrc/cs_hash.h)."""
    r, lo = u64(0), u32(0)
    _chk(lib().cs_hash_cell(a, b, c, int(big), C.byref(r), C.byref(lo)), "cs_hash_cell")
    return int(r.value), int(lo.value)


def sample_threshold(p: float) -> int:
    return int(lib().cs_sample_threshold(p))


def _dev_xyz(xyz: torch.Tensor):
    if not xyz.is_cuda or xyz.dtype != torch.float32 or not xyz.is_contiguous() or xyz.numel() % 3:
        raise ValueError("positions must be a contiguous CUDA float32 tensor with 3 floats per particle")
    return xyz.data_ptr(), xyz.numel() // 3


def _host_xyz(xyz: torch.Tensor):
    if xyz.is_cuda or xyz.dtype != torch.float32 or not xyz.is_contiguous() or xyz.numel() % 3:
        raise ValueError("positions must be a contiguous CPU float32 tensor with 3 floats per particle")
    return xyz.data_ptr(), xyz.numel() // 3


class CountSketch:
    """cs_sketch handle.  Methods mirror the C calls of include/cs.h one to one."""

    def __init__(self, d: int, w: int, G, L: float, seed: int, stream: torch.cuda.Stream | None = None):
        Gs = [int(G)] if isinstance(G, int) else [int(g) for g in G]
        self.d, self.w, self.G, self.L, self.seed = int(d), int(w), Gs, float(L), int(seed)
        self.n_scales = len(Gs)
        self._h = vp(None)
        arr = (u32 * len(Gs))(*Gs)
        _chk(lib().cs_create_multi(C.byref(self._h), self.n_scales, self.d, self.w, arr, self.L, self.seed),
             "cs_create_multi")
        self.device = torch.device("cuda", torch.cuda.current_device())
        self.set_stream(stream if stream is not None else torch.cuda.current_stream())

    # -- life cycle
    def close(self):
        if self._h:
            lib().cs_destroy(self._h)
            self._h = vp(None)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def reset(self):
        _chk(lib().cs_reset(self._h), "cs_reset")

    def set_stream(self, stream: torch.cuda.Stream):
        self._stream = stream
        _chk(lib().cs_set_stream(self._h, vp(stream.cuda_stream)), "cs_set_stream")

    def set_table_budget(self, nbytes: int):
        _chk(lib().cs_set_table_budget(self._h, nbytes), "cs_set_table_budget")

    def set_chunk_sizes(self, stage_particles: int = 0, update_chunk: int = 0, scan_chunk: int = 0, compact_chunk: int = 0):
        _chk(lib().cs_set_chunk_sizes(self._h, stage_particles, update_chunk, scan_chunk, compact_chunk), "cs_set_chunk_sizes")

    def set_replay_cache(self, nbytes: int):
        _chk(lib().cs_set_replay_cache(self._h, nbytes), "cs_set_replay_cache")

    def set_update_mode(self, mode: int, rows_direct: int = -1):
        _chk(lib().cs_set_update_mode(self._h, mode, rows_direct), "cs_set_update_mode")

    def set_counting_mode(self, mode: int):
        _chk(lib().cs_set_counting_mode(self._h, mode), "cs_set_counting_mode")

    def set_scan_mode(self, mode: int):
        _chk(lib().cs_set_scan_mode(self._h, mode), "cs_set_scan_mode")

    def set_update_index(self, index: int):
        _chk(lib().cs_set_update_index(self._h, index), "cs_set_update_index")

    def set_scan_index(self, index: int):
        _chk(lib().cs_set_scan_index(self._h, index), "cs_set_scan_index")

    def update_index(self) -> int:
        v = u64(0)
        _chk(lib().cs_get_update_index(self._h, C.byref(v)), "cs_get_update_index")
        return int(v.value)

    # -- stream processing
    def update(self, xyz: torch.Tensor, sample_p: float = 1.0):
        p, n = _dev_xyz(xyz)
        _chk(lib().cs_update(self._h, vp(p), n, sample_p), "cs_update")

    def update_host(self, xyz: torch.Tensor, sample_p: float = 1.0):
        p, n = _host_xyz(xyz)
        _chk(lib().cs_update_host(self._h, vp(p), n, sample_p), "cs_update_host")

    # -- packed 64-bit records
    def pack_records(self, xyz: torch.Tensor) -> torch.Tensor:
        p, n = _dev_xyz(xyz)
        out = torch.empty(n, dtype=torch.int64, device=xyz.device)
        _chk(lib().cs_pack_records(self._h, vp(p), n, vp(out.data_ptr())), "cs_pack_records")
        return out

    def _records(self, fn: str, recs: torch.Tensor, sample_p: float, cuda: bool):
        if recs.is_cuda != cuda or recs.dtype not in (torch.int64, torch.uint64) or not recs.is_contiguous():
            raise ValueError("records must be a contiguous int64/uint64 tensor on the %s" % ("device" if cuda else "host"))
        _chk(getattr(lib(), fn)(self._h, vp(recs.data_ptr()), recs.numel(), sample_p), fn)

    def update_records(self, recs: torch.Tensor, sample_p: float = 1.0):
        self._records("cs_update_records", recs, sample_p, True)

    def update_records_host(self, recs: torch.Tensor, sample_p: float = 1.0):
        self._records("cs_update_records_host", recs, sample_p, False)

    def scan_records(self, recs: torch.Tensor, sample_p: float = 1.0):
        self._records("cs_scan_records", recs, sample_p, True)

    def scan_records_host(self, recs: torch.Tensor, sample_p: float = 1.0):
        self._records("cs_scan_records_host", recs, sample_p, False)

    # -- queries
    def estimate(self, cells: torch.Tensor, scale: int = 0) -> torch.Tensor:
        if not cells.is_cuda or cells.dtype not in (torch.int64, torch.uint64) or not cells.is_contiguous():
            raise ValueError("cells must be a contiguous CUDA int64/uint64 tensor")
        out = torch.empty(cells.numel(), dtype=torch.int32, device=cells.device)
        _chk(lib().cs_estimate(self._h, scale, vp(cells.data_ptr()), cells.numel(), vp(out.data_ptr())), "cs_estimate")
        return out

    def scan_begin(self, k_max: int, thr_min: int = INT32_MAX):
        _chk(lib().cs_scan_begin(self._h, k_max, thr_min), "cs_scan_begin")

    def set_candidate_capacity(self, entries: int):
        _chk(lib().cs_set_candidate_capacity(self._h, entries), "cs_set_candidate_capacity")

    def scan(self, xyz: torch.Tensor, sample_p: float = 1.0):
        p, n = _dev_xyz(xyz)
        _chk(lib().cs_scan(self._h, vp(p), n, sample_p), "cs_scan")

    def scan_host(self, xyz: torch.Tensor, sample_p: float = 1.0):
        p, n = _host_xyz(xyz)
        _chk(lib().cs_scan_host(self._h, vp(p), n, sample_p), "cs_scan_host")

    def scan_cells(self, cells: torch.Tensor, scale: int = 0):
        if not cells.is_cuda or cells.dtype not in (torch.int64, torch.uint64) or not cells.is_contiguous():
            raise ValueError("cells must be a contiguous CUDA int64/uint64 tensor")
        _chk(lib().cs_scan_cells(self._h, scale, vp(cells.data_ptr()), cells.numel()), "cs_scan_cells")

    def scan_all(self, scale: int = 0):
        _chk(lib().cs_scan_all(self._h, scale), "cs_scan_all")

    def scan_children(self, parents: torch.Tensor, parent_scale: int, child_scale: int):
        if not parents.is_cuda or parents.dtype not in (torch.int64, torch.uint64) or not parents.is_contiguous():
            raise ValueError("parents must be a contiguous CUDA int64/uint64 tensor")
        _chk(lib().cs_scan_children(self._h, parent_scale, child_scale, vp(parents.data_ptr()), parents.numel()),
             "cs_scan_children")

    def topk(self, k: int, scale: int = 0, device=None):
        """(ids int64 tensor holding the uint64 cell ids, est int32 tensor), on `device` (default: the GPU)."""
        device = self.device if device is None else torch.device(device)
        ids = torch.empty(max(k, 1), dtype=torch.int64, device=device)
        est = torch.empty(max(k, 1), dtype=torch.int32, device=device)
        n = u64(0)
        _chk(lib().cs_topk(self._h, scale, k, vp(ids.data_ptr()), vp(est.data_ptr()), C.byref(n)), "cs_topk")
        return ids[: n.value], est[: n.value]

    def excursion(self, thr: int, scale: int = 0, cap: int | None = None, device=None):
        """(ids, est, total): all candidates with estimate >= thr (the first `cap` of them if cap is given)."""
        device = self.device if device is None else torch.device(device)
        n = u64(0)
        if cap is None:      # size query first, then fetch everything
            _chk(lib().cs_excursion(self._h, scale, thr, 0, None, None, C.byref(n)), "cs_excursion")
            cap = int(n.value)
        ids = torch.empty(max(cap, 1), dtype=torch.int64, device=device)
        est = torch.empty(max(cap, 1), dtype=torch.int32, device=device)
        _chk(lib().cs_excursion(self._h, scale, thr, cap, vp(ids.data_ptr()), vp(est.data_ptr()), C.byref(n)),
             "cs_excursion")
        m = min(int(n.value), cap)
        return ids[:m], est[:m], int(n.value)

    def recount(self, ids: torch.Tensor, xyz: torch.Tensor, counts: torch.Tensor | None = None, scale: int = 0,
                extract_cap: int = 0):
        """Exact recount of the cells `ids` over `xyz` (counts accumulate into `counts` if given) and, with
        extract_cap > 0, the particles of those cells.  Returns (counts int32 tensor, particles or None, n_members)."""
        p, n = _dev_xyz(xyz)
        if not ids.is_cuda or ids.dtype not in (torch.int64, torch.uint64) or not ids.is_contiguous():
            raise ValueError("ids must be a contiguous CUDA int64/uint64 tensor")
        m = ids.numel()
        if counts is None:
            counts = torch.zeros(max(m, 1), dtype=torch.int32, device=ids.device)
        out = torch.empty((max(extract_cap, 1), 3), dtype=torch.float32, device=ids.device) if extract_cap else None
        nm = u64(0)
        _chk(lib().cs_recount(self._h, scale, vp(ids.data_ptr()), m, vp(p), n, vp(counts.data_ptr()),
                              vp(out.data_ptr()) if out is not None else None, extract_cap, C.byref(nm)), "cs_recount")
        k = min(int(nm.value), extract_cap)
        return counts[:m], (out[:k] if out is not None else None), int(nm.value)

    def expand_neighbours(self, ids: torch.Tensor, scale: int = 0) -> torch.Tensor:
        """(m, 27) tensor: the 26-neighbour shell (periodic) of each cell, column 13 = the cell itself."""
        if not ids.is_cuda or ids.dtype not in (torch.int64, torch.uint64) or not ids.is_contiguous():
            raise ValueError("ids must be a contiguous CUDA int64/uint64 tensor")
        out = torch.empty((ids.numel(), 27), dtype=torch.int64, device=ids.device)
        _chk(lib().cs_expand_neighbours(self._h, scale, vp(ids.data_ptr()), ids.numel(), vp(out.data_ptr())),
             "cs_expand_neighbours")
        return out

    def scan_stats(self, scale: int = 0) -> dict:
        out = (u64 * 4)()
        _chk(lib().cs_scan_stats(self._h, scale, out), "cs_scan_stats")
        tau = out[1] - (1 << 64) if out[1] >= (1 << 63) else out[1]
        return {"candidates": int(out[0]), "tau": int(tau), "compactions": int(out[2]), "scan_launches": int(out[3])}

    # -- table access
    def sketch(self, scale: int = 0, device=None) -> torch.Tensor:
        device = self.device if device is None else torch.device(device)
        out = torch.empty((self.d, self.w), dtype=torch.int32, device=device)
        _chk(lib().cs_sketch_read(self._h, scale, vp(out.data_ptr())), "cs_sketch_read")
        return out

    def sketch_add(self, table: torch.Tensor, scale: int = 0):
        if table.dtype != torch.int32 or not table.is_contiguous() or table.numel() != self.d * self.w:
            raise ValueError("table must be a contiguous int32 tensor with d*w entries")
        _chk(lib().cs_sketch_add(self._h, scale, vp(table.data_ptr())), "cs_sketch_add")

    def table_view(self, scale: int = 0) -> torch.Tensor:
        """(d, w) int32 tensor ALIASING the handle's counters (no copy): for in-place collectives over the table."""
        ptr = vp(None)
        _chk(lib().cs_table_ptr(self._h, scale, C.byref(ptr)), "cs_table_ptr")

        class _Alias:
            __cuda_array_interface__ = {"shape": (self.d, self.w), "typestr": "<i4", "data": (int(ptr.value), False),
                                        "version": 3, "strides": None}
        return torch.as_tensor(_Alias(), device=self.device)

    def coeffs(self, scale: int = 0):
        import numpy as np
        out = np.empty(4 * self.d, dtype=np.uint64)
        K = u64(0)
        _chk(lib().cs_coeffs(self._h, scale, out.ctypes.data_as(vp), C.byref(K)), "cs_coeffs")
        return out.reshape(self.d, 4), int(K.value)

    PHASES = ("update_scatter", "update_apply", "compact_kept", "scan_first", "scan_next", "bitmap", "select", "other")

    def set_timing(self, on: bool):
        _chk(lib().cs_set_timing(self._h, int(on)), "cs_set_timing")

    def get_timing(self) -> dict:
        """{phase: (ms, launch groups)} since the last call."""
        ms = (dbl * 8)()
        sp = (u64 * 8)()
        _chk(lib().cs_get_timing(self._h, ms, sp), "cs_get_timing")
        return {n: (float(ms[i]), int(sp[i])) for i, n in enumerate(self.PHASES)}

    def update_stats(self) -> dict:
        out = (u64 * 4)()
        _chk(lib().cs_update_stats(self._h, out), "cs_update_stats")
        return {"staging_overflow": int(out[0]), "region_overflow": int(out[1]), "leftover": int(out[2]), "binned": int(out[3])}

    def launch_count(self) -> int:
        v = u64(0)
        _chk(lib().cs_launch_count(self._h, C.byref(v)), "cs_launch_count")
        return int(v.value)


def probe_l2(mode: int, table_bytes: int, n_ops: int, reps: int = 3, stream: torch.cuda.Stream | None = None) -> float:
    """Average ms of one repetition of n_ops red (0) / atom (1) / gather (2) operations over a table."""
    st = stream if stream is not None else torch.cuda.current_stream()
    ms = dbl(0.0)
    _chk(lib().cs_probe_l2(mode, table_bytes, n_ops, reps, vp(st.cuda_stream), C.byref(ms)), "cs_probe_l2")
    return float(ms.value)


def probe_stream(xyz: torch.Tensor, reps: int = 3, stream: torch.cuda.Stream | None = None) -> float:
    p, n = _dev_xyz(xyz)
    st = stream if stream is not None else torch.cuda.current_stream()
    ms = dbl(0.0)
    _chk(lib().cs_probe_stream(vp(p), n, reps, vp(st.cuda_stream), C.byref(ms)), "cs_probe_stream")
    return float(ms.value)


SELECT_STATIC_MAX_N = 65536          # CS_SELECT_STATIC_MAX_N of include/cs.h


def select_static(ids: torch.Tensor, est: torch.Tensor, k: int, ids_out: torch.Tensor, est_out: torch.Tensor,
                  n_out: torch.Tensor, stream: torch.cuda.Stream | None = None) -> None:
    """cs_select_static: the first k distinct ids of (ids, est) in the order (est descending, id ascending) -> ids_out[:k],
    est_out[:k], n_out[0] (a CUDA int32/uint32 tensor of one element), asynchronously on `stream`.  The library call
    allocates nothing (its scratch is a fixed device array of the library: n, k <= SELECT_STATIC_MAX_N) and every
    tensor is the caller's, so this wrapper allocates nothing either.  Calls that overlap on the GPU race."""
    for t, name, kinds in ((ids, "ids", (torch.int64, torch.uint64)), (est, "est", (torch.int32,)),
                           (ids_out, "ids_out", (torch.int64, torch.uint64)), (est_out, "est_out", (torch.int32,)),
                           (n_out, "n_out", (torch.int32, torch.uint32))):
        if not t.is_cuda or t.dtype not in kinds or not t.is_contiguous():
            raise ValueError(f"{name} must be a contiguous CUDA tensor of dtype {kinds}")
    if est.numel() != ids.numel() or ids_out.numel() < k or est_out.numel() < k or n_out.numel() < 1:
        raise ValueError("est must match ids; ids_out / est_out need k entries, n_out one")
    st = stream if stream is not None else torch.cuda.current_stream()
    _chk(lib().cs_select_static(vp(ids.data_ptr()), vp(est.data_ptr()), ids.numel(), k, vp(ids_out.data_ptr()),
                                vp(est_out.data_ptr()), vp(n_out.data_ptr()), vp(st.cuda_stream)), "cs_select_static")
