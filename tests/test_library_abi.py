"""CPU-side checks of the C-ABI library (no GPU, no compute calls): it builds, loads, exports every symbol
include/cs.h declares, its host-only arithmetic reproduces the pinned values (tests/golden/pins.json: values
computed before either implementation existed), and argument validation fails before any CUDA work.
"""
import ctypes as C
import re
from pathlib import Path

import numpy as np
import pytest

ROOT = Path(__file__).resolve().parent.parent
P61 = 2 ** 61 - 1


@pytest.fixture(scope="module")
def cslib():
    from paper_1711_00975_b200 import build, binding
    build.build_libcs()
    return binding.lib()


def _declared_symbols():
    text = (ROOT / "include" / "cs.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(cs_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_are_exported_and_bound(cslib):
    from paper_1711_00975_b200 import binding
    names = _declared_symbols()
    assert len(names) >= 25
    for n in names:
        assert hasattr(cslib, n), f"libcs.so does not export {n}"
        assert n in binding.SIGNATURES, f"binding has no signature for {n}"
    assert sorted(binding.SIGNATURES) == names


def test_version_and_error_string(cslib):
    from paper_1711_00975_b200 import binding
    assert "sm_100a" in binding.version()
    assert isinstance(cslib.cs_last_error(), bytes)


def test_host_coefficients_match_pins(cslib, golden):
    from paper_1711_00975_b200 import binding
    g = golden["coeffs_seed1"]
    co5, K5 = binding.derive_coeffs(1, 5)
    co3, K3 = binding.derive_coeffs(1, 3)
    want = [[int(v) for v in row] for row in g["rows"]]
    assert co5[:3].tolist() == want and co3.tolist() == want
    assert K5 == int(g["K_d5"]) and K3 == int(g["K_d3"])
    for row in co5.tolist():
        a, b, a2, b2 = row
        assert 1 <= a < P61 and 0 <= b < P61 and 1 <= a2 < P61 and 0 <= b2 < P61


def test_host_coefficients_follow_the_splitmix_stream(cslib, golden):
    """Derivation rule (R2) re-derived with Python integers from the public splitmix64 definition."""
    from paper_1711_00975_b200 import binding
    M = 2 ** 64 - 1

    def mix(z):
        z &= M
        z ^= z >> 30
        z = (z * 0xBF58476D1CE4E5B9) & M
        z ^= z >> 27
        z = (z * 0x94D049BB133111EB) & M
        return z ^ (z >> 31)

    for seed, d in [(0, 1), (1234567, 7), (2 ** 64 - 5, 32)]:
        x = [mix(seed + n * 0x9E3779B97F4A7C15) for n in range(1, 4 * d + 2)]
        co, K = binding.derive_coeffs(seed, d)
        for j in range(d):
            assert co[j].tolist() == [x[4 * j] % (P61 - 1) + 1, x[4 * j + 1] % P61,
                                      x[4 * j + 2] % (P61 - 1) + 1, x[4 * j + 3] % P61]
        assert K == x[4 * d]
    assert [int(v) for v in golden["splitmix64"]["seed_1234567"]][:1] == [mix(1234567 + 0x9E3779B97F4A7C15)]


def test_sample_threshold(cslib, golden):
    from paper_1711_00975_b200 import binding
    assert binding.sample_threshold(0.1) == int(golden["sampler_seed1_d5_p0.1"]["T_p_hex"], 16)
    assert binding.sample_threshold(0.5) == 2 ** 63
    assert binding.sample_threshold(1.0) == 0 and binding.sample_threshold(0.0) == 0
    assert binding.sample_threshold(float("nan")) == 0


def test_argument_validation_needs_no_gpu(cslib):
    from paper_1711_00975_b200 import binding
    h = C.c_void_p(None)
    G = (C.c_uint32 * 1)(16)
    bad = [
        dict(n_scales=1, d=0, w=16, L=1.0),
        dict(n_scales=1, d=33, w=16, L=1.0),
        dict(n_scales=0, d=3, w=16, L=1.0),
        dict(n_scales=9, d=3, w=16, L=1.0),
        dict(n_scales=1, d=3, w=0, L=1.0),
        dict(n_scales=1, d=3, w=2 ** 31 + 1, L=1.0),
        dict(n_scales=1, d=3, w=16, L=0.0),
        dict(n_scales=1, d=3, w=16, L=float("inf")),
        dict(n_scales=1, d=3, w=16, L=float("nan")),
    ]
    for kw in bad:
        Gs = (C.c_uint32 * max(kw["n_scales"], 1))(*([16] * max(kw["n_scales"], 1)))
        rc = cslib.cs_create_multi(C.byref(h), kw["n_scales"], kw["d"], kw["w"], Gs, kw["L"], 1)
        assert rc == binding.CS_ERR_ARG, kw
        assert h.value is None
        assert cslib.cs_last_error() != b""
    for g in (0, 2 ** 20 + 1):
        G[0] = g
        assert cslib.cs_create_multi(C.byref(h), 1, 3, 16, G, 1.0, 1) == binding.CS_ERR_ARG
    G8 = (C.c_uint32 * 8)(*([16] * 8))
    assert cslib.cs_create_multi(C.byref(h), 8, 9, 16, G8, 1.0, 1) == binding.CS_ERR_ARG     # 72 hash rows > 64
    assert cslib.cs_create_multi(None, 1, 3, 16, G, 1.0, 1) == binding.CS_ERR_ARG
    assert cslib.cs_derive_coeffs(1, 0, None, None) == binding.CS_ERR_ARG
    assert cslib.cs_destroy(None) == binding.CS_OK
    assert cslib.cs_update(None, None, 0, 1.0) == binding.CS_ERR_ARG


def test_binding_fails_loudly_without_library(monkeypatch, tmp_path):
    from paper_1711_00975_b200 import binding
    monkeypatch.setattr(binding, "_lib", None)
    monkeypatch.setattr(binding, "LIB_PATH", tmp_path / "libcs.so")
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        binding.lib()


def test_limb_hash_arithmetic_against_big_integers(cslib, golden):
    """csrc/cs_hash.h (the inline functions the kernels compile), evaluated on the host through cs_hash_cell,
    against Python big integers: closed forms, residues that land on 0 / p-1 / the fold carries, random values."""
    from paper_1711_00975_b200 import binding
    rng = np.random.default_rng(20260)
    cases = []
    # closed forms of tests/golden (2^61 == 1): (a, c, b) -> r
    for case in golden["mersenne"]["cases"]:
        a, c, b, want = (int(eval(case[key], {"p": P61})) for key in ("a", "c", "b", "r"))
        assert binding.hash_cell(a, b, c, big=True) == (want, want & 0xFFFFFFFF), case
        cases.append((a, b, c))
    edge_a = [1, 2, P61 - 1, P61 - 2, 2 ** 32 - 1, 2 ** 32, 2 ** 32 + 1, 2 ** 60, 2 ** 60 + 1, 2 ** 61 - 2 ** 32 - 1,
              (2 ** 29 - 1) << 32 | 0xFFFFFFFE]
    edge_b = [0, 1, P61 - 1, P61 - 5, 2 ** 32 - 1, 2 ** 32, 2 ** 60]
    edge_c = [0, 1, 5, 2 ** 31 - 1, 2 ** 31, 2 ** 31 + 1, 2 ** 32 - 1, 2 ** 32, 2 ** 36 - 1, 2 ** 37, 2 ** 60 - 1,
              4095 + 4096 * (4095 + 4096 * 4095), 4641 + 4642 * (4641 + 4642 * 4641)]
    for a in edge_a:
        for b in edge_b:
            for c in edge_c:
                cases.append((a, b, c))
    # residues forced to 0, p-1, 1: choose b = (target - a*c) mod p
    for _ in range(300):
        a = int(rng.integers(1, P61)); c = int(rng.integers(0, 2 ** 60))
        for target in (0, P61 - 1, 1, 2 ** 32 - 1, 2 ** 32):
            cases.append((a, (target - a * c) % P61, c))
    for _ in range(20000):
        bits = int(rng.integers(1, 61))
        cases.append((int(rng.integers(1, P61)), int(rng.integers(0, P61)), int(rng.integers(0, 2 ** bits))))
    for a, b, c in cases:
        want = (a * c + b) % P61
        r, lo = binding.hash_cell(a, b, c, big=True)
        assert r == want and lo == want & 0xFFFFFFFF, (a, b, c)
        if c < 2 ** 31:
            r, lo = binding.hash_cell(a, b, c, big=False)
            assert r == want and lo == want & 0xFFFFFFFF, (a, b, c, "small form")
        if c < 2 ** 37:
            r, lo = binding.hash_cell(a, b, c, big=2)
            assert r == want and lo == want & 0xFFFFFFFF, (a, b, c, "table form")
    assert cslib.cs_hash_cell(0, 0, 0, 1, None, None) == binding.CS_ERR_ARG
    r, lo = C.c_uint64(0), C.c_uint32(0)
    assert cslib.cs_hash_cell(1, 0, 2 ** 31, 0, C.byref(r), C.byref(lo)) == binding.CS_ERR_ARG
    assert cslib.cs_hash_cell(P61, 0, 1, 1, C.byref(r), C.byref(lo)) == binding.CS_ERR_ARG
