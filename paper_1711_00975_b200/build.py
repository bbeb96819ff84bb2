"""Builds libcs.so (the C-ABI CUDA library, include/cs.h) in-tree for sm_100a with nvcc.

    python -m paper_1711_00975_b200.build [--force]

nvcc cross-compiles without a GPU.  Objects go to paper_1711_00975_b200/csrc/build/ (git-ignored), the
library to paper_1711_00975_b200/libcs.so (git-ignored, but it travels to the GPU box with the snapshot).
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor
from pathlib import Path

PKG = Path(__file__).resolve().parent
CSRC = PKG / "csrc"
OBJ = CSRC / "build"
LIB = PKG / "libcs.so"
SOURCES = ["cs_api.cu", "cs_kernels.cu", "cs_update_binned.cu", "cs_scan.cu", "cs_scan_staged.cu", "cs_scan_bitmap.cu", "cs_select.cu", "cs_recount.cu", "cs_probe.cu"]
HEADERS = ["cs_internal.h", "cs_hash.h", "cs_device.cuh", "cs_launch.cuh", "cs_scan_common.cuh", "../../include/cs.h"]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-std=c++17", "-O3", "-lineinfo",
    "-fmad=false",                      # bit-exact quantisation: no FMA contraction (include/cs.h)
    "-Xcompiler", "-fPIC,-O2,-Wall,-ffp-contract=off",
    "-Xptxas", "-v",
]


def nvcc() -> str:
    exe = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not Path(exe).exists():
        raise RuntimeError("nvcc not found: libcs.so cannot be built (there is no CPU fallback)")
    return exe


def _stale(target: Path, deps) -> bool:
    if not target.exists():
        return True
    t = target.stat().st_mtime
    return any(Path(d).stat().st_mtime > t for d in deps)


def _compile(src: str, force: bool) -> Path:
    obj = OBJ / (src + ".o")
    deps = [CSRC / src] + [CSRC / h for h in HEADERS] + [Path(__file__)]
    if force or _stale(obj, deps):
        cmd = [nvcc(), *NVCC_FLAGS, "-c", str(CSRC / src), "-o", str(obj)]
        r = subprocess.run(cmd, capture_output=True, text=True)
        (OBJ / (src + ".ptxas.log")).write_text(r.stdout + r.stderr)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed on {src}:\n{r.stdout}\n{r.stderr}")
    return obj


def build_libcs(force: bool = False) -> Path:
    OBJ.mkdir(parents=True, exist_ok=True)
    with ThreadPoolExecutor(max_workers=min(len(SOURCES), os.cpu_count() or 1)) as ex:
        objs = list(ex.map(lambda s: _compile(s, force), SOURCES))
    if force or _stale(LIB, objs):
        tmp = LIB.with_suffix(f".so.tmp{os.getpid()}")
        cmd = [nvcc(), "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", str(tmp), *map(str, objs)]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"link failed:\n{r.stdout}\n{r.stderr}")
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build_libcs(force="--force" in sys.argv))
