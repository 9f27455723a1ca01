"""Seeded synthetic workloads (inputs only -- none of the method's arithmetic lives here).

This module serves BOTH the oracle-side tests and the CUDA-side tests/bench, and imports neither.
It knows the five BASELINE.json configurations (grid, domain, stencil degree, time step, fields)
and how to fill the initial distribution function

    f(x, v) = fx(x) * fv(v) + amp * u(seed + lin)          (one multiply, one add, per point)

where fx / fv are small tables computed once on the host in numpy fp64 (so exp/cos are evaluated
in exactly one place) and u is white noise from a counter-based generator on the C-order linear
index `lin` (stands in for eq (12)'s rand(x)).  The
per-point combination is written with torch elementwise ops that are IEEE-exact, so the CPU and
the CUDA device produce bit-identical arrays (checked in tests).

The noise generator is the published splitmix64 finaliser (Steele/Lea/Flood; Vigna's public-domain
variant) applied to (seed + lin); u = top 53 bits * 2^-53, uniform in [0,1).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace
from typing import List, Optional, Sequence, Tuple

import numpy as np
import torch

_M64 = (1 << 64) - 1


def _s64(x: int) -> int:
    """Reinterpret an unsigned 64-bit constant as signed (torch has no uint64 arithmetic)."""
    x &= _M64
    return x - (1 << 64) if x >= (1 << 63) else x


_GAMMA = 0x9E3779B97F4A7C15
_MUL1 = 0xBF58476D1CE4E5B9
_MUL2 = 0x94D049BB133111EB


def splitmix64_py(x: int) -> int:
    """Pure-python reference of the mixer (used by tests to pin the torch version)."""
    z = (x + _GAMMA) & _M64
    z = ((z ^ (z >> 30)) * _MUL1) & _M64
    z = ((z ^ (z >> 27)) * _MUL2) & _M64
    return z ^ (z >> 31)


def uniform_py(seed: int, lin: int) -> float:
    return (splitmix64_py((seed + lin) & _M64) >> 11) * 2.0 ** -53


def _lsr(z: torch.Tensor, s: int) -> torch.Tensor:
    """Logical shift right on int64 bit patterns."""
    return (z >> s) & ((1 << (64 - s)) - 1)


def uniform_torch(seed: int, lin: torch.Tensor) -> torch.Tensor:
    """u(seed + lin) in [0,1) as float64; lin is an int64 tensor on any device."""
    z = lin + _s64(seed + _GAMMA)
    z = (z ^ _lsr(z, 30)) * _s64(_MUL1)
    z = (z ^ _lsr(z, 27)) * _s64(_MUL2)
    z = z ^ _lsr(z, 31)
    return _lsr(z, 11).to(torch.float64) * (2.0 ** -53)


@dataclass(frozen=True)
class Workload:
    name: str
    n: Tuple[int, int, int, int, int, int]
    lo: Tuple[float, ...]
    dx: Tuple[float, ...]
    degree: int                      # Lagrange degree (odd); stencil width q = degree+1
    dt: float
    seed: int
    noise_amp: float
    kind: str                        # which initial condition / field recipe
    B: Tuple[float, float, float] = (0.0, 0.0, 0.0)   # (q/m) B0
    e_amp: float = 0.05              # E_d(x) = e_amp * sin(x_d/2)

    # ---- geometry -------------------------------------------------------------------------
    @property
    def q(self) -> int:
        return self.degree + 1

    @property
    def npts(self) -> int:
        return int(np.prod(self.n, dtype=np.int64))

    def nodes(self, d: int) -> np.ndarray:
        return np.array([self.lo[d] + float(i) * self.dx[d] for i in range(self.n[d])], dtype=np.float64)

    # ---- small host tables ----------------------------------------------------------------
    def fx(self) -> np.ndarray:
        """Spatial factor on the (nx1,nx2,nx3) grid."""
        x1, x2, x3 = np.meshgrid(self.nodes(0), self.nodes(1), self.nodes(2), indexing="ij")
        if self.kind in ("maxwell_x1", ):
            return 1.0 + 0.01 * np.cos(0.5 * x1)
        if self.kind == "two_stream":
            return 1.0 + 0.02 * np.cos(x1)
        if self.kind == "aniso_x2":
            return 1.0 + 0.01 * np.cos(0.5 * x2)
        if self.kind == "maxwell_xyz":
            return 1.0 + 0.01 * (np.cos(0.5 * x1) + np.cos(0.5 * x2) + np.cos(0.5 * x3))
        raise ValueError(self.kind)

    def fv(self) -> np.ndarray:
        """Velocity factor on the (nv1,nv2,nv3) grid."""
        v1, v2, v3 = np.meshgrid(self.nodes(3), self.nodes(4), self.nodes(5), indexing="ij")
        norm = (2.0 * math.pi) ** -1.5
        if self.kind in ("maxwell_x1", "maxwell_xyz"):
            return norm * np.exp(-0.5 * (v1 * v1 + v2 * v2 + v3 * v3))
        if self.kind == "two_stream":
            m = lambda a: norm * np.exp(-0.5 * (a * a + v2 * v2 + v3 * v3))
            return 0.5 * (m(v1 - 2.0) + m(v1 + 2.0))
        if self.kind == "aniso_x2":
            return np.exp(-0.5 * v1 * v1 - v2 * v2 / 0.5 - 0.5 * v3 * v3)
        raise ValueError(self.kind)

    def E(self) -> List[np.ndarray]:
        """(q/m) E_d(x) = e_amp*sin(x_d/2) on the x grid, d = 0,1,2 (BASELINE.json configs[1])."""
        xs = np.meshgrid(self.nodes(0), self.nodes(1), self.nodes(2), indexing="ij")
        return [np.ascontiguousarray(self.e_amp * np.sin(0.5 * x)) for x in xs]

    # ---- the distribution function ----------------------------------------------------------
    def fill(self, out: torch.Tensor, noise: bool = True, slab_bytes: int = 1 << 29) -> torch.Tensor:
        """Write f into `out` (shape n, float64, any device), x1-slab by x1-slab."""
        assert tuple(out.shape) == tuple(self.n) and out.dtype == torch.float64 and out.is_contiguous()
        dev = out.device
        fx = torch.from_numpy(np.ascontiguousarray(self.fx())).to(dev)
        fv = torch.from_numpy(np.ascontiguousarray(self.fv())).to(dev)
        per_x1 = self.npts // self.n[0]
        step = max(1, slab_bytes // (8 * per_x1))
        for i0 in range(0, self.n[0], step):
            i1 = min(self.n[0], i0 + step)
            slab = out[i0:i1]
            torch.mul(fx[i0:i1, :, :, None, None, None], fv[None, None, None], out=slab)
            if noise and self.noise_amp != 0.0:
                lin = torch.arange(i0 * per_x1, i1 * per_x1, dtype=torch.int64, device=dev)
                u = uniform_torch(self.seed, lin)
                del lin
                u *= self.noise_amp
                slab += u.view(slab.shape)
                del u
        return out

    def make_f(self, device="cpu", noise: bool = True) -> torch.Tensor:
        return self.fill(torch.empty(self.n, dtype=torch.float64, device=device), noise=noise)

    # ---- variants ------------------------------------------------------------------------------
    def reduced(self, n: Sequence[int], name: Optional[str] = None) -> "Workload":
        """Same domain, fields and recipe on a coarser grid (parity-test copies of the big configs)."""
        n = tuple(int(v) for v in n)
        L = [self.dx[d] * self.n[d] for d in range(6)]
        dx = tuple(L[d] / n[d] for d in range(6))
        return replace(self, n=n, dx=dx, name=name or f"{self.name}_r{'x'.join(map(str, n))}")


def _grid(n: Sequence[int], Lx: float, vmax: float):
    n = tuple(int(v) for v in n)
    lo = (0.0, 0.0, 0.0, -vmax, -vmax, -vmax)
    dx = tuple([Lx / n[d] for d in range(3)] + [2.0 * vmax / n[d] for d in range(3, 6)])
    return n, lo, dx


def _mk(name, n, Lx, vmax, **kw) -> Workload:
    n, lo, dx = _grid(n, Lx, vmax)
    return Workload(name=name, n=n, lo=lo, dx=dx, **kw)


FOUR_PI = 4.0 * math.pi
TWO_PI = 2.0 * math.pi

#: BASELINE.json configs[0..4]
C1 = _mk("C1", (8,) * 6, FOUR_PI, 6.0, degree=7, dt=0.1, seed=1001, noise_amp=1e-3, kind="maxwell_x1")
C2 = _mk("C2", (32,) * 6, FOUR_PI, 6.0, degree=7, dt=0.05, seed=1002, noise_amp=1e-3, kind="maxwell_x1")
C3 = _mk("C3", (16, 16, 16, 64, 64, 64), TWO_PI, 8.0, degree=5, dt=0.05, seed=1003, noise_amp=1e-4,
         kind="two_stream")
C4 = _mk("C4", (32,) * 6, FOUR_PI, 6.0, degree=7, dt=0.1, seed=1004, noise_amp=1e-4, kind="aniso_x2",
         B=(0.0, 0.0, 1.0))
C5 = _mk("C5", (48, 48, 48, 32, 32, 32), FOUR_PI, 6.0, degree=9, dt=0.05, seed=1005, noise_amp=1e-4,
         kind="maxwell_xyz", B=(0.0, 0.0, 1.0))

#: The paper's own section-5 benchmark grid: 37 points per dim, odd stencil widths 3/5/7/9, random
#: per-point displacements alpha/dx in [-1, 1] (see random_shifts).  degree here is only the default even-q context.
P37 = _mk("P37", (37,) * 6, FOUR_PI, 6.0, degree=7, dt=0.05, seed=1037, noise_amp=1e-3, kind="maxwell_x1")

#: An extent without specialised sweep kernels (36 is not in {8,16,32,37,48,64}): every sweep of this workload runs the
#: run-time-extent fallback kernels, so that their throughput can be timed and profiled (bench.py --workload G36).
G36 = _mk("G36", (36,) * 6, FOUR_PI, 6.0, degree=7, dt=0.05, seed=1036, noise_amp=1e-3, kind="maxwell_x1")

CONFIGS = {w.name: w for w in (C1, C2, C3, C4, C5, P37, G36)}


def random_shifts(shape: Sequence[int], seed: int, device="cpu", whole_cells: bool = False,
                  slab_bytes: int = 1 << 29) -> torch.Tensor:
    """Per-point displacements in cells for the paper's benchmark: alpha = 2 u(seed + lin) - 1 in [-1, 1) with the
    same counter-based generator as the noise (bit-identical on CPU and CUDA); whole_cells=True rounds them to
    {-1, 0, 1} (the exact-permutation test)."""
    shape = tuple(int(v) for v in shape)
    out = torch.empty(shape, dtype=torch.float64, device=device)
    flat = out.view(-1)
    total = flat.numel()
    step = max(1, slab_bytes // 8)
    for i0 in range(0, total, step):
        i1 = min(total, i0 + step)
        lin = torch.arange(i0, i1, dtype=torch.int64, device=device)
        a = uniform_torch(seed, lin) * 2.0 - 1.0
        if whole_cells:
            a = torch.round(a)
        flat[i0:i1] = a
    return out


def sample_pencils(npencil: int, count: int, seed: int) -> np.ndarray:
    """`count` distinct pencil ids in [0, npencil), seeded (full-size sampled parity)."""
    rng = np.random.default_rng(seed)
    count = min(count, npencil)
    return np.sort(rng.choice(npencil, size=count, replace=False)).astype(np.int64)
