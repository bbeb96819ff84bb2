"""Seeded synthetic N-body streams (harness code: inputs only, none of the method's arithmetic).

Stand-in for the Millennium / Millennium-XXL snapshots the paper measures on, which are
not available: clustered halos plus a uniform background in a periodic box, with the sizes, grids and sketch
shapes BASELINE.json `configs` fixes.  Recipe:

  * halo catalogue from `gen_seed`: H centres uniform in [0, L)^3, Pareto(alpha = 1.9) weights W = U^(-1/1.9),
    expected size m_h = m_min + (N_halo - H*m_min) * W_h / sum(W) with N_halo = round((1 - f_bg) * N),
    per-axis spread sigma_h = 2 * (m_h / 1000)^(1/3);
  * particle i, independently of every other particle (counter-based draws keyed by (gen_seed, batch, i)):
    with probability f_bg uniform in the box, else halo h with probability m_h / N_halo (inverse CDF, so the
    realised sizes are multinomial) at centre_h + N(0, sigma_h^2) per axis, wrapped x - L*floor(x/L) in float32;
  * order: i.i.d., i.e. not grouped by halo ("arbitrary order").

The same float32 buffer is handed to the oracle and to the CUDA path; nothing here is imported by either.
The counter hash below is a 64-bit finaliser of its own (not the method's splitmix64 stream).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace

import torch

_M64 = (1 << 64) - 1


def _s64(x: int) -> int:
    """Python int -> the int64 with the same 64-bit pattern."""
    x &= _M64
    return x - (1 << 64) if x >= (1 << 63) else x


_C1 = _s64(0xFF51AFD7ED558CCD)
_C2 = _s64(0xC4CEB9FE1A85EC53)
_ODD = _s64(0xD6E8FEB86659FD93)


def _lsr(x: torch.Tensor, s: int) -> torch.Tensor:
    return (x >> s) & ((1 << (64 - s)) - 1)


def _fmix(x: torch.Tensor) -> torch.Tensor:
    x = x ^ _lsr(x, 33)
    x = x * _C1
    x = x ^ _lsr(x, 33)
    x = x * _C2
    x = x ^ _lsr(x, 33)
    return x


def _fmix_int(x: int) -> int:
    x &= _M64
    x ^= x >> 33
    x = (x * 0xFF51AFD7ED558CCD) & _M64
    x ^= x >> 33
    x = (x * 0xC4CEB9FE1A85EC53) & _M64
    x ^= x >> 33
    return x


def _draw_bits(key: int, idx: torch.Tensor, k: int) -> torch.Tensor:
    """64 pseudo-random bits for (key, idx, k): k-th draw of item idx under stream key."""
    ctr = idx * 16 + k
    return _fmix(_fmix(ctr * _ODD + _s64(key)) + _s64(key >> 1))


def _u32f(bits: torch.Tensor) -> torch.Tensor:
    """Uniform float32 in (0, 1) from the top 24 bits."""
    return (_lsr(bits, 40).to(torch.float32) + 0.5) * (1.0 / (1 << 24))


def _u64f(bits: torch.Tensor) -> torch.Tensor:
    """Uniform float64 in (0, 1) from the top 53 bits."""
    return (_lsr(bits, 11).to(torch.float64) + 0.5) * (1.0 / (1 << 53))


@dataclass(frozen=True)
class Workload:
    """One BASELINE.json config: stream shape + the sketch parameters it is run with."""
    name: str
    N: int
    G: tuple          # one grid size per scale
    d: int
    w: int
    k: int
    H: int
    f_bg: float
    m_min: int
    L: float = 500.0
    sample_p: float = 1.0
    seed: int = 1                 # cs_create seed
    gen_seed: int = 1000          # generator seed
    batch: int = 0                # particles per generated batch (0 = one batch)
    thresholds: tuple = ()        # excursion thresholds (cfg 5)
    sigma_mult: float = 1.0       # < 1: the optional concentrated stress variant
    extra: dict = field(default_factory=dict, compare=False)

    def scaled(self, N: int, **kw) -> "Workload":
        """Same recipe at a reduced particle count (parity tests at sizes the oracle finishes quickly)."""
        return replace(self, N=int(N), **kw)


CONFIGS = {
    "cfg1": Workload("cfg1", N=1 << 20, G=(256,), d=5, w=1 << 16, k=100, H=64, f_bg=0.2, m_min=0, gen_seed=1001),
    "cfg2": Workload("cfg2", N=1 << 26, G=(1024,), d=5, w=1 << 20, k=1000, H=10 ** 4, f_bg=0.3, m_min=20,
                     gen_seed=1002),
    "cfg3": Workload("cfg3", N=1 << 30, G=(4096,), d=7, w=1 << 22, k=30000, H=10 ** 6, f_bg=0.3, m_min=20,
                     gen_seed=1003),
    "cfg4": Workload("cfg4", N=10 ** 10, G=(4642,), d=7, w=1 << 24, k=300000, H=10 ** 7, f_bg=0.3, m_min=20,
                     gen_seed=1004, batch=1 << 28),
    "cfg5": Workload("cfg5", N=1 << 30, G=(512, 1024, 2048, 4096), d=5, w=1 << 22, k=10000, H=10 ** 4, f_bg=0.3,
                     m_min=20, sample_p=0.1, gen_seed=1005, thresholds=(8, 32, 128)),
}


class Catalogue:
    """Halo catalogue of a workload on a device (centres, spreads, cumulative selection probabilities)."""

    def __init__(self, wl: Workload, device="cpu"):
        self.wl = wl
        self.device = torch.device(device)
        H = wl.H
        key = _fmix_int(wl.gen_seed * 0x9E3779B1 + 0x5851F42D4C957F2D)
        h = torch.arange(H, dtype=torch.int64, device=self.device)
        L = wl.L
        self.centres = torch.stack([_u32f(_draw_bits(key, h, k)) * L for k in range(3)], dim=1).contiguous()
        u = _u64f(_draw_bits(key, h, 3))
        W = u.pow(-1.0 / 1.9)
        n_halo = round((1.0 - wl.f_bg) * wl.N)
        spare = max(n_halo - H * wl.m_min, 0)
        m = wl.m_min + spare * W / W.sum()
        self.m = m
        self.sigma = (2.0 * wl.sigma_mult * (m / 1000.0).pow(1.0 / 3.0)).to(torch.float32)
        cdf = torch.cumsum(m / m.sum(), dim=0)
        cdf[-1] = 1.0
        self.cdf = cdf

    def positions(self, i0: int, n: int, batch: int = 0, out: torch.Tensor | None = None) -> torch.Tensor:
        """Particles i0 .. i0+n-1 of batch `batch` as an (n, 3) float32 tensor on the catalogue's device."""
        wl = self.wl
        dev = self.device
        key = _fmix_int(_fmix_int(wl.gen_seed * 0x9E3779B1 + 0x2545F4914F6CDD1D) + batch * 0x9E3779B97F4A7C15)
        idx = torch.arange(i0, i0 + n, dtype=torch.int64, device=dev)
        L = wl.L
        is_bg = _u64f(_draw_bits(key, idx, 0)) < wl.f_bg
        hsel = torch.searchsorted(self.cdf, _u64f(_draw_bits(key, idx, 1))).clamp_(max=wl.H - 1)
        u = [_u32f(_draw_bits(key, idx, 2 + k)) for k in range(4)]
        r0 = torch.sqrt(-2.0 * torch.log(u[0]))
        r1 = torch.sqrt(-2.0 * torch.log(u[2]))
        t0 = (2.0 * math.pi) * u[1]
        t1 = (2.0 * math.pi) * u[3]
        z = torch.stack([r0 * torch.cos(t0), r0 * torch.sin(t0), r1 * torch.cos(t1)], dim=1)
        halo_pos = self.centres[hsel] + self.sigma[hsel].unsqueeze(1) * z
        bg_pos = torch.stack([_u32f(_draw_bits(key, idx, 6 + k)) * L for k in range(3)], dim=1)
        pos = torch.where(is_bg.unsqueeze(1), bg_pos, halo_pos).to(torch.float32)
        pos = pos - L * torch.floor(pos / L)          # periodic wrap in float32; a result equal to L is left as is
        if out is not None:
            out.copy_(pos)
            return out
        return pos.contiguous()


def generate(wl: Workload, device="cpu", chunk: int = 1 << 22, batch: int = 0, n: int | None = None,
             catalogue: Catalogue | None = None) -> torch.Tensor:
    """Whole batch `batch` of a workload (n particles, default wl.N) as one (n, 3) float32 tensor."""
    cat = catalogue or Catalogue(wl, device)
    n = wl.N if n is None else int(n)
    out = torch.empty((n, 3), dtype=torch.float32, device=cat.device)
    for i0 in range(0, n, chunk):
        m = min(chunk, n - i0)
        cat.positions(i0, m, batch=batch, out=out[i0:i0 + m])
    return out


def checksum(xyz: torch.Tensor) -> int:
    """Sum of the float32 bit patterns mod 2^64 (recorded beside bench numbers)."""
    bits = xyz.contiguous().view(torch.int32).to(torch.int64) & 0xFFFFFFFF
    return int(bits.sum().item()) & _M64
