"""ctypes wrapper around oracle/cs_oracle.cpp -- the CPU ORACLE (test infrastructure, not the product).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this
module.  It never imports paper_1711_00975_b200 and shares nothing with it.  All arithmetic is in the C++
file; this wrapper only builds it (g++ -O2 -ffp-contract=off), marshals numpy arrays and raises on errors.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "cs_oracle.cpp"
_LIB = _HERE / "libcs_oracle.so"

INT32_MIN = -(2 ** 31)
INT32_MAX = 2 ** 31 - 1


def build(force: bool = False) -> Path:
    """Compile the oracle shared library in-tree if it is missing or older than its source."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".so.tmp{os.getpid()}")
        cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-Wall", "-Wextra",
               "-o", str(tmp), str(_SRC)]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(str(_LIB))
        u64, i32, u32, dbl, vp, ci = C.c_uint64, C.c_int32, C.c_uint32, C.c_double, C.c_void_p, C.c_int
        sig = {
            "ora_splitmix64": (None, [u64, u64, vp]),
            "ora_mix64": (u64, [u64]),
            "ora_affine_mod_p": (u64, [u64, u64, u64]),
            "ora_coeffs": (None, [u64, ci, vp, vp]),
            "ora_scale": (C.c_float, [u32, dbl]),
            "ora_quantise": (None, [vp, u64, u32, dbl, vp]),
            "ora_sample_threshold": (u64, [dbl]),
            "ora_keep": (None, [u64, u64, u64, dbl, vp]),
            "ora_create": (ci, [vp, ci, u64, u32, dbl, u64]),
            "ora_create_multi": (ci, [vp, ci, ci, u64, vp, dbl, u64]),
            "ora_destroy": (ci, [vp]),
            "ora_set_mode": (ci, [vp, ci]),
            "ora_reset": (ci, [vp]),
            "ora_set_update_index": (ci, [vp, u64]),
            "ora_set_scan_index": (ci, [vp, u64]),
            "ora_update": (ci, [vp, vp, u64, dbl]),
            "ora_estimate": (ci, [vp, ci, vp, u64, vp]),
            "ora_scan_begin": (ci, [vp]),
            "ora_scan": (ci, [vp, vp, u64, dbl]),
            "ora_update_records": (ci, [vp, vp, u64, dbl]),
            "ora_scan_records": (ci, [vp, vp, u64, dbl]),
            "ora_cells_of_records": (None, [vp, u64, u32, vp]),
            "ora_candidate_count": (ci, [vp, ci, vp]),
            "ora_topk": (ci, [vp, ci, u64, vp, vp, vp]),
            "ora_excursion": (ci, [vp, ci, i32, u64, vp, vp, vp]),
            "ora_topk_streaming": (ci, [vp, ci, vp, u64, dbl, u64, vp, vp, vp]),
            "ora_select_streaming": (ci, [vp, ci, vp, u64, u64, dbl, u64, i32, u64, vp, vp, vp, vp, vp, vp]),
            "ora_full_search_topk": (ci, [vp, ci, u64, vp, vp, vp]),
            "ora_sketch_read": (ci, [vp, ci, vp]),
            "ora_sketch_add": (ci, [vp, ci, vp]),
            "ora_get_coeffs": (ci, [vp, ci, vp, vp]),
            "ora_hashes": (ci, [vp, ci, vp, u64, vp]),
            "ora_exact_counts": (u64, [vp, u64, u32, dbl, u64, vp, vp]),
        }
        for name, (res, args) in sig.items():
            f = getattr(L, name)
            f.restype = res
            f.argtypes = args
        _lib = L
    return _lib


def _ptr(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


def _xyz(a) -> np.ndarray:
    a = np.ascontiguousarray(np.asarray(a, dtype=np.float32))
    if a.size % 3:
        raise ValueError("positions must hold 3 floats per particle")
    return a.reshape(-1, 3)


def _chk(rc: int, what: str):
    if rc != 0:
        raise RuntimeError(f"oracle {what} failed with status {rc}")


# ---- free functions -------------------------------------------------------------------------------------

def splitmix64(seed: int, n: int) -> np.ndarray:
    out = np.empty(n, dtype=np.uint64)
    lib().ora_splitmix64(seed, n, _ptr(out))
    return out


def mix64(z: int) -> int:
    return int(lib().ora_mix64(z & (2 ** 64 - 1)))


def affine_mod_p(a: int, c: int, b: int) -> int:
    return int(lib().ora_affine_mod_p(a, c, b))


def coeffs(seed: int, d: int):
    out = np.empty(4 * d, dtype=np.uint64)
    K = C.c_uint64(0)
    lib().ora_coeffs(seed, d, _ptr(out), C.byref(K))
    return out.reshape(d, 4), int(K.value)


def scale_f32(G: int, L: float) -> np.float32:
    return np.float32(lib().ora_scale(G, L))


def quantise(xyz, G: int, L: float) -> np.ndarray:
    p = _xyz(xyz)
    out = np.empty(p.shape[0], dtype=np.uint64)
    lib().ora_quantise(_ptr(p), p.shape[0], G, L, _ptr(out))
    return out


def cells_of_records(recs, G: int) -> np.ndarray:
    """Cell ids on the G mesh of packed 64-bit records (qx | qy << 21 | qz << 42)."""
    r = np.ascontiguousarray(np.asarray(recs, dtype=np.uint64))
    out = np.empty(r.shape[0], dtype=np.uint64)
    lib().ora_cells_of_records(_ptr(r), r.shape[0], G, _ptr(out))
    return out


def pack_records(xyz, L: float) -> np.ndarray:
    """Packed record of each particle = its cell id on the 2^21 mesh (quantise with G = 2^21)."""
    return quantise(xyz, 1 << 21, L)


def sample_threshold(p: float) -> int:
    return int(lib().ora_sample_threshold(p))


def keep_mask(K: int, index0: int, n: int, p: float) -> np.ndarray:
    out = np.empty(n, dtype=np.uint8)
    lib().ora_keep(K, index0, n, p, _ptr(out))
    return out.astype(bool)


def exact_counts(xyz, G: int, L: float):
    p = _xyz(xyz)
    n = p.shape[0]
    ids = np.empty(max(n, 1), dtype=np.uint64)
    cnt = np.empty(max(n, 1), dtype=np.uint64)
    m = int(lib().ora_exact_counts(_ptr(p), n, G, L, n, _ptr(ids), _ptr(cnt)))
    return ids[:m].copy(), cnt[:m].copy()


# ---- handle ---------------------------------------------------------------------------------------------

class OracleSketch:
    """Plain CPU Count Sketch over one or several grids (see cs_oracle.cpp for the passages followed)."""

    def __init__(self, d: int, w: int, G, L: float, seed: int):
        Gs = [int(G)] if np.isscalar(G) else [int(g) for g in G]
        self.d, self.w, self.G, self.L, self.seed = int(d), int(w), Gs, float(L), int(seed)
        self.n_scales = len(Gs)
        arr = np.asarray(Gs, dtype=np.uint32)
        h = C.c_void_p(None)
        _chk(lib().ora_create_multi(C.byref(h), self.n_scales, self.d, self.w, _ptr(arr), self.L, self.seed),
             "create")
        self._h = h

    def close(self):
        if self._h:
            lib().ora_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def reset(self):
        _chk(lib().ora_reset(self._h), "reset")

    def set_mode(self, mode: int):
        """0 Count Sketch (default), 1 Count-Min (Add +1, Estimate = min); before the first update."""
        _chk(lib().ora_set_mode(self._h, mode), "set_mode")

    def set_update_index(self, index: int):
        _chk(lib().ora_set_update_index(self._h, index), "set_update_index")

    def set_scan_index(self, index: int):
        _chk(lib().ora_set_scan_index(self._h, index), "set_scan_index")

    def update(self, xyz, sample_p: float = 1.0):
        p = _xyz(xyz)
        _chk(lib().ora_update(self._h, _ptr(p), p.shape[0], sample_p), "update")

    def estimate(self, cells, scale: int = 0) -> np.ndarray:
        c = np.ascontiguousarray(np.asarray(cells, dtype=np.uint64))
        out = np.empty(c.shape[0], dtype=np.int32)
        _chk(lib().ora_estimate(self._h, scale, _ptr(c), c.shape[0], _ptr(out)), "estimate")
        return out

    def scan_begin(self):
        _chk(lib().ora_scan_begin(self._h), "scan_begin")

    def scan(self, xyz, sample_p: float = 1.0):
        p = _xyz(xyz)
        _chk(lib().ora_scan(self._h, _ptr(p), p.shape[0], sample_p), "scan")

    def update_records(self, recs, sample_p: float = 1.0):
        r = np.ascontiguousarray(np.asarray(recs, dtype=np.uint64))
        _chk(lib().ora_update_records(self._h, _ptr(r), r.shape[0], sample_p), "update_records")

    def scan_records(self, recs, sample_p: float = 1.0):
        r = np.ascontiguousarray(np.asarray(recs, dtype=np.uint64))
        _chk(lib().ora_scan_records(self._h, _ptr(r), r.shape[0], sample_p), "scan_records")

    def candidate_count(self, scale: int = 0) -> int:
        n = C.c_uint64(0)
        _chk(lib().ora_candidate_count(self._h, scale, C.byref(n)), "candidate_count")
        return int(n.value)

    def topk(self, k: int, scale: int = 0):
        ids = np.empty(max(k, 1), dtype=np.uint64)
        est = np.empty(max(k, 1), dtype=np.int32)
        n = C.c_uint64(0)
        _chk(lib().ora_topk(self._h, scale, k, _ptr(ids), _ptr(est), C.byref(n)), "topk")
        return ids[: n.value].copy(), est[: n.value].copy()

    def excursion(self, thr: int, scale: int = 0, cap: int | None = None):
        if cap is None:
            cap = self.candidate_count(scale)
        ids = np.empty(max(cap, 1), dtype=np.uint64)
        est = np.empty(max(cap, 1), dtype=np.int32)
        n = C.c_uint64(0)
        _chk(lib().ora_excursion(self._h, scale, thr, cap, _ptr(ids), _ptr(est), C.byref(n)), "excursion")
        m = min(int(n.value), cap)
        return ids[:m].copy(), est[:m].copy(), int(n.value)

    def topk_streaming(self, xyz, k: int, sample_p: float = 1.0, scale: int = 0):
        p = _xyz(xyz)
        ids = np.empty(max(k, 1), dtype=np.uint64)
        est = np.empty(max(k, 1), dtype=np.int32)
        n = C.c_uint64(0)
        _chk(lib().ora_topk_streaming(self._h, scale, _ptr(p), p.shape[0], sample_p, k, _ptr(ids), _ptr(est),
                                      C.byref(n)), "topk_streaming")
        return ids[: n.value].copy(), est[: n.value].copy()

    def select_streaming(self, xyz, index0: int, k: int, thr: int = INT32_MAX, sample_p: float = 1.0, scale: int = 0):
        """One shard of a replayed stream (running indices index0 ..): (top-k ids, est), (excursion ids, est) of the
        shard against the tables as they stand, in O(k + excursion) memory."""
        p = _xyz(xyz)
        ids = np.empty(max(k, 1), dtype=np.uint64)
        est = np.empty(max(k, 1), dtype=np.int32)
        nk, nx = C.c_uint64(0), C.c_uint64(0)
        cap = 1 << 16
        while True:
            xi = np.empty(cap, dtype=np.uint64)
            xe = np.empty(cap, dtype=np.int32)
            _chk(lib().ora_select_streaming(self._h, scale, _ptr(p), p.shape[0], index0, sample_p, k, thr, cap, _ptr(ids),
                                            _ptr(est), C.byref(nk), _ptr(xi), _ptr(xe), C.byref(nx)), "select_streaming")
            if nx.value <= cap:
                break
            cap = int(nx.value)
        return (ids[: nk.value].copy(), est[: nk.value].copy()), (xi[: nx.value].copy(), xe[: nx.value].copy())

    def full_search_topk(self, k: int, scale: int = 0):
        ids = np.empty(max(k, 1), dtype=np.uint64)
        est = np.empty(max(k, 1), dtype=np.int32)
        n = C.c_uint64(0)
        _chk(lib().ora_full_search_topk(self._h, scale, k, _ptr(ids), _ptr(est), C.byref(n)), "full_search_topk")
        return ids[: n.value].copy(), est[: n.value].copy()

    def sketch(self, scale: int = 0) -> np.ndarray:
        out = np.empty((self.d, self.w), dtype=np.int32)
        _chk(lib().ora_sketch_read(self._h, scale, _ptr(out)), "sketch_read")
        return out

    def sketch_add(self, table, scale: int = 0):
        t = np.ascontiguousarray(np.asarray(table, dtype=np.int32))
        if t.size != self.d * self.w:
            raise ValueError("table must have d*w entries")
        _chk(lib().ora_sketch_add(self._h, scale, _ptr(t)), "sketch_add")

    def coeffs(self, scale: int = 0):
        out = np.empty(4 * self.d, dtype=np.uint64)
        K = C.c_uint64(0)
        _chk(lib().ora_get_coeffs(self._h, scale, _ptr(out), C.byref(K)), "get_coeffs")
        return out.reshape(self.d, 4), int(K.value)

    def hashes(self, cells, scale: int = 0):
        c = np.ascontiguousarray(np.asarray(cells, dtype=np.uint64))
        out = np.empty((c.shape[0], self.d, 2), dtype=np.int64)
        _chk(lib().ora_hashes(self._h, scale, _ptr(c), c.shape[0], _ptr(out)), "hashes")
        return out[:, :, 0].copy(), out[:, :, 1].copy()
