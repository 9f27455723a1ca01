"""ORACLE -- test infrastructure, not the product.

ctypes front-end of ``oracle/bsl6d_oracle.cpp`` (plain CPU C++ written from the paper, see that
file's header).  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` leg may import this package.  It imports nothing from the CUDA package
``paper_2303_05994_b200`` and the CUDA package imports nothing from here.

All arrays are numpy float64, C-contiguous, shape ``(nx1,nx2,nx3,nv1,nv2,nv3)`` unless stated.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "bsl6d_oracle.cpp")
_LIB = os.path.join(_HERE, "libbsl6d_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc.  -ffp-contract=off: no fused multiply-add anywhere."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
               "-o", _LIB + ".tmp", _SRC]
        subprocess.run(cmd, check=True)
        os.replace(_LIB + ".tmp", _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = C.CDLL(_LIB)
        dp, ip = C.POINTER(C.c_double), C.POINTER(C.c_int32)
        lib.oracle_num_threads.restype = C.c_int
        lib.oracle_lagrange_weights.argtypes = [C.c_int, C.c_double, dp]
        lib.oracle_sweep_pencils.argtypes = [C.c_int, C.c_int, C.c_int, C.c_longlong, dp, dp, C.c_double, dp]
        lib.oracle_sweep.argtypes = [ip, dp, dp, C.c_int, dp, C.c_uint, C.c_double, C.c_int]
        lib.oracle_advect.argtypes = [ip, dp, dp, C.c_int, dp, dp, C.c_int, dp, C.c_double]
        lib.oracle_rotate.argtypes = [ip, dp, dp, C.c_int, dp, dp, dp, C.c_double]
        lib.oracle_density.argtypes = [ip, dp, dp, dp]
        lib.oracle_strang_step.argtypes = [ip, dp, dp, C.c_int, dp, dp, dp, dp, dp, C.c_double]
        lib.oracle_rotation_plan.argtypes = [dp, C.c_double, C.POINTER(C.c_int), dp]
        lib.oracle_lagrange_weights_odd.argtypes = [C.c_int, C.c_double, dp]
        lib.oracle_sweep_pointwise.argtypes = [ip, dp, dp, C.c_int, dp, C.c_int]
        _lib = lib
    return _lib


def _dp(a: Optional[np.ndarray]):
    if a is None:
        return None
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"], "oracle wants C-contiguous float64"
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _check(rc: int, what: str):
    if rc != 0:
        raise ValueError(f"oracle.{what} failed with code {rc}")


@dataclass(frozen=True)
class Grid:
    """Node i of dim d sits at lo[d] + i*dx[d]; dims 0-2 periodic (period n*dx), 3-5 zero-extended."""
    n: Sequence[int]
    lo: Sequence[float]
    dx: Sequence[float]

    def _c(self):
        n = (C.c_int32 * 6)(*[int(v) for v in self.n])
        lo = (C.c_double * 6)(*[float(v) for v in self.lo])
        dx = (C.c_double * 6)(*[float(v) for v in self.dx])
        return n, lo, dx

    def nodes(self, d: int) -> np.ndarray:
        return np.array([self.lo[d] + float(i) * self.dx[d] for i in range(self.n[d])], dtype=np.float64)


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def lagrange_weights(q: int, theta: float) -> np.ndarray:
    """l_m(theta) for m = -q/2+1 .. q/2  (eq (7))."""
    w = np.empty(q, dtype=np.float64)
    _check(_load().oracle_lagrange_weights(q, float(theta), _dp(w)), "lagrange_weights")
    return w


def sweep_pencils(g_in: np.ndarray, a: np.ndarray, scale: float, q: int, periodic: bool) -> np.ndarray:
    """P independent pencils g_in[P, n]; pencil p is shifted by alpha_cells = -(a[p]*scale)."""
    g_in = np.ascontiguousarray(g_in, dtype=np.float64)
    a = np.ascontiguousarray(a, dtype=np.float64)
    P, n = g_in.shape
    assert a.shape == (P,)
    out = np.empty_like(g_in)
    _check(_load().oracle_sweep_pencils(n, q, int(bool(periodic)), P, _dp(g_in), _dp(a), float(scale), _dp(out)),
           "sweep_pencils")
    return out


def sweep(f_in: np.ndarray, dim: int, src: np.ndarray, src_mask: int, scale: float, q: int,
          out: Optional[np.ndarray] = None) -> np.ndarray:
    """General sweep along `dim`: alpha_cells = -(src[p]*scale); src dense C-order over dims in src_mask."""
    assert f_in.ndim == 6
    n = (C.c_int32 * 6)(*f_in.shape)
    src = np.ascontiguousarray(src, dtype=np.float64)
    want = int(np.prod([f_in.shape[d] for d in range(6) if src_mask >> d & 1], dtype=np.int64))
    assert src.size == want, (src.size, want)
    if out is None:
        out = np.empty_like(f_in)
    _check(_load().oracle_sweep(n, _dp(f_in), _dp(out), dim, _dp(src), src_mask, float(scale), q), "sweep")
    return out


def lagrange_weights_odd(q: int, alpha: float) -> np.ndarray:
    """l_m(alpha) on the nodes m = -(q-1)/2 .. (q-1)/2, odd q  (eq (6))."""
    w = np.empty(q, dtype=np.float64)
    _check(_load().oracle_lagrange_weights_odd(q, float(alpha), _dp(w)), "lagrange_weights_odd")
    return w


def sweep_pointwise(f_in: np.ndarray, dim: int, alpha_cells: np.ndarray, q: int,
                    out: Optional[np.ndarray] = None) -> np.ndarray:
    """Odd-q sweep along `dim` with one displacement per point (alpha_cells has f's shape), eq (6)."""
    assert f_in.ndim == 6 and alpha_cells.shape == f_in.shape
    n = (C.c_int32 * 6)(*f_in.shape)
    alpha_cells = np.ascontiguousarray(alpha_cells, dtype=np.float64)
    if out is None:
        out = np.empty_like(f_in)
    _check(_load().oracle_sweep_pointwise(n, _dp(f_in), _dp(out), dim, _dp(alpha_cells), q), "sweep_pointwise")
    return out


def advect(grid: Grid, degree: int, f_in: np.ndarray, dim: int, shift_source: Optional[np.ndarray], dt: float,
           out: Optional[np.ndarray] = None) -> np.ndarray:
    n, lo, dx = grid._c()
    assert tuple(f_in.shape) == tuple(grid.n)
    if shift_source is not None:
        shift_source = np.ascontiguousarray(shift_source, dtype=np.float64)
        want = grid.n[dim + 3] if dim < 3 else grid.n[0] * grid.n[1] * grid.n[2]
        assert shift_source.size == want
    if out is None:
        out = np.empty_like(f_in)
    _check(_load().oracle_advect(n, lo, dx, degree, _dp(f_in), _dp(out), dim, _dp(shift_source), float(dt)), "advect")
    return out


def rotate(grid: Grid, degree: int, f_in: np.ndarray, B: Sequence[float], dt: float,
           out: Optional[np.ndarray] = None) -> np.ndarray:
    n, lo, dx = grid._c()
    if out is None:
        out = np.empty_like(f_in)
    Bc = (C.c_double * 3)(*[float(b) for b in B])
    _check(_load().oracle_rotate(n, lo, dx, degree, _dp(f_in), _dp(out), Bc, float(dt)), "rotate")
    return out


def rotation_plan(B: Sequence[float], dt: float):
    """[(axis, angle)] -- the coordinate-axis rotations rotate() applies, in order, for an oblique B (reading R1)."""
    Bc = (C.c_double * 3)(*[float(b) for b in B])
    axes = (C.c_int * 16)()
    ang = (C.c_double * 16)()
    cnt = _load().oracle_rotation_plan(Bc, float(dt), axes, ang)
    if cnt < 0:
        raise ValueError("rotation_plan wants B with at least two non-zero components")
    return [(int(axes[i]), float(ang[i])) for i in range(cnt)]


def density(grid: Grid, f: np.ndarray) -> np.ndarray:
    n, _, dx = grid._c()
    rho = np.empty(tuple(grid.n[:3]), dtype=np.float64)
    _check(_load().oracle_density(n, dx, _dp(f), _dp(rho)), "density")
    return rho


def strang_step(grid: Grid, degree: int, f: np.ndarray, E: Sequence[Optional[np.ndarray]],
                B: Optional[Sequence[float]], dt: float) -> np.ndarray:
    """One Strang step IN PLACE on f (returns f)."""
    n, lo, dx = grid._c()
    Es = [None if e is None else np.ascontiguousarray(e, dtype=np.float64) for e in E]
    Bc = None if B is None else (C.c_double * 3)(*[float(b) for b in B])
    _check(_load().oracle_strang_step(n, lo, dx, degree, _dp(f), _dp(Es[0]), _dp(Es[1]), _dp(Es[2]), Bc, float(dt)),
           "strang_step")
    return f


# ---- field step: plain numpy, see oracle/fields.py ------------------------------------------
from . import fields as _fields  # noqa: E402
import sys as _sys  # noqa: E402

poisson_E = _fields.poisson_E
adiabatic_E = _fields.adiabatic_E


def vp_step(grid, degree, f, B, dt, closure="poisson", c1=1.0, e_fac=1.0):
    """Self-consistent Strang step (oracle/fields.py::vp_step) using this module's sweeps and density."""
    return _fields.vp_step(_sys.modules[__name__], grid, degree, f, B, dt, closure, c1, e_fac)
