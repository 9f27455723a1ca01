"""Full-size parity (-m gpu): the BASELINE.json configs at their real extents, in the launch configuration
bench.py times, checked against the oracle on sampled outputs the oracle can compute one by one.

A sweep is independent per pencil, a rotation about x3 per (x, v3) plane, the density per x-point -- so running
the oracle on a seeded sample of pencils / planes / v-blocks gathered from the GPU's *input* buffer and comparing
with the same pencils of the GPU's output is exact for the sampled elements, not statistical (SURVEY.md 8(c)
"Full-size parity").  Tolerance: 1e-12 * max|reference| (north_star), bit-exact for whole-cell shifts.
"""
from __future__ import annotations

import math

import numpy as np
import pytest
import torch

import bsl6d_workloads as wl
import oracle
import paper_2303_05994_b200 as bsl

pytestmark = pytest.mark.gpu

P_SAMPLES = 2048
TOL = 1e-12


def _need(gb: float):
    from conftest import need_gpu
    need_gpu(gb)


def _split(w, dim):
    n = w.n
    outer = int(np.prod(n[:dim], dtype=np.int64))
    inner = int(np.prod(n[dim + 1:], dtype=np.int64))
    return outer, n[dim], inner


class PencilSample:
    """A seeded set of pencils along `dim`: (o, i) pairs plus the 6-D index of each (swept index = 0)."""

    def __init__(self, w, dim, seed, P=P_SAMPLES):
        rng = np.random.default_rng(seed)
        outer, N, inner = _split(w, dim)
        o = rng.integers(0, outer, P)
        i = rng.integers(0, inner, P)
        o[0], i[0] = 0, 0                                   # the corners of the pencil index space
        o[1], i[1] = outer - 1, inner - 1
        self.dim, self.N, self.outer, self.inner = dim, N, outer, inner
        self.idx = [None] * 6
        rem = o.copy()
        for d in range(dim - 1, -1, -1):
            self.idx[d] = rem % w.n[d]
            rem //= w.n[d]
        rem = i.copy()
        for d in range(5, dim, -1):
            self.idx[d] = rem % w.n[d]
            rem //= w.n[d]
        self.o = torch.from_numpy(o).cuda()
        self.i = torch.from_numpy(i).cuda()

    def gather(self, f: torch.Tensor) -> np.ndarray:
        v = f.view(self.outer, self.N, self.inner)
        return v[self.o, :, self.i].cpu().numpy()           # (P, N)


def check_sweep(ctx, w, og, src_in, dst, dim, kind, dt, seed, E=None, what=""):
    """One named GPU sweep src_in -> dst (may alias) + oracle on sampled pencils.  kind: 'x' or 'E'."""
    s = PencilSample(w, dim, seed)
    g_in = s.gather(src_in)                                 # before the launch: the sweep may run in place
    if kind == "x":
        a = og.nodes(dim + 3)[s.idx[dim + 3]]
        ctx.advect(src_in, dst, dim, None, dt)
    else:
        a = E[dim - 3][s.idx[0], s.idx[1], s.idx[2]]
        ctx.advect(src_in, dst, dim, torch.from_numpy(E[dim - 3]).cuda(), dt)
    got = s.gather(dst)
    ref = oracle.sweep_pencils(g_in, a, dt / w.dx[dim], w.degree + 1, periodic=dim < 3)
    err = np.max(np.abs(got - ref)) / np.max(np.abs(ref))
    assert err <= TOL, f"{w.name} {what} dim {dim}: rel err {err:.3e}"
    return err


class PlaneSample:
    """Seeded (x, v3) planes for a rotation about x3: the (v1, v2) planes f[x1,x2,x3,:,:,j3]."""

    def __init__(self, w, seed, S=48):
        rng = np.random.default_rng(seed)
        self.ix = [torch.from_numpy(rng.integers(0, w.n[d], S)).cuda() for d in range(3)]
        self.j3 = torch.from_numpy(rng.integers(0, w.n[5], S)).cuda()
        self.S = S
        self.grid = oracle.Grid((S, 1, 1, w.n[3], w.n[4], 1), tuple(w.lo), tuple(w.dx))

    def gather(self, f: torch.Tensor) -> np.ndarray:
        p = f[self.ix[0], self.ix[1], self.ix[2], :, :, self.j3]       # (S, nv1, nv2)
        return np.ascontiguousarray(p.cpu().numpy()).reshape(self.grid.n)


def check_density(ctx, w, og, f, seed, S=32):
    rng = np.random.default_rng(seed)
    ix = [rng.integers(0, w.n[d], S) for d in range(3)]
    rho = torch.empty(w.n[:3], dtype=torch.float64, device="cuda")
    ctx.density(f, rho)
    blocks = f[torch.from_numpy(ix[0]).cuda(), torch.from_numpy(ix[1]).cuda(), torch.from_numpy(ix[2]).cuda()]
    mg = oracle.Grid((S, 1, 1) + tuple(w.n[3:]), tuple(w.lo), tuple(w.dx))
    ref = oracle.density(mg, np.ascontiguousarray(blocks.cpu().numpy()).reshape(mg.n)).reshape(S)
    got = rho.cpu().numpy()[ix[0], ix[1], ix[2]]
    assert np.max(np.abs(got - ref)) <= 1e-13 * np.max(np.abs(ref))
    assert torch.isfinite(rho).all()


def _ogrid(w):
    return oracle.Grid(tuple(w.n), tuple(w.lo), tuple(w.dx))


# ------------------------------------------------------------------------------------------------------------
# C2 / C3 (BASELINE configs[1], [2]): the six sweeps in sequence at 32^6 and 16^3 x 64^3, ping-pong buffers
# ------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name", ["C2", "C3"])
def test_six_sweeps_full_size(name):
    _need(20)
    w = wl.CONFIGS[name]
    og = _ogrid(w)
    E = w.E()
    cur = w.make_f("cuda")
    oth = torch.empty_like(cur)
    with bsl.create(w.n, w.lo, w.dx, w.degree) as ctx:
        for d in range(6):
            check_sweep(ctx, w, og, cur, oth, d, "x" if d < 3 else "E", w.dt, 2000 + 10 * d, E=E, what="six sweeps")
            cur, oth = oth, cur
        check_density(ctx, w, og, cur, 2099)
        assert ctx.launch_count() >= 7


def test_C2_full_size_whole_cell_shift_bit_exact():
    """dt = 8*dx1 makes every x1 displacement a whole number of cells (reading S10(ii) on the C2 grid: v nodes
    are -6 + 0.375 j, alpha = -8*v = 48 - 3j, up to 48 cells > n): the GPU output must equal the rolled input bit for bit -- checked on
    the WHOLE array with torch.roll per v1 index, no oracle needed for the expected value."""
    _need(28)
    w = wl.C2
    f = w.make_f("cuda")
    out = torch.empty_like(f)
    with bsl.create(w.n, w.lo, w.dx, w.degree) as ctx:
        ctx.advect(f, out, 0, None, 8.0 * w.dx[0])
    v = _ogrid(w).nodes(3)
    for j1 in range(w.n[3]):
        k = -8.0 * v[j1]
        assert k == int(k)
        # out[i] = in[i + k]  <=>  out = roll(in, -k) along x1
        assert torch.equal(out[:, :, :, j1], torch.roll(f[:, :, :, j1], shifts=-int(k), dims=0)), j1
    # and the oracle agrees on sampled pencils
    s = PencilSample(w, 0, 2100, P=256)
    ref = oracle.sweep_pencils(s.gather(f), v[s.idx[3]], (8.0 * w.dx[0]) / w.dx[0], w.degree + 1, True)
    assert np.array_equal(s.gather(out), ref)


# ------------------------------------------------------------------------------------------------------------
# C4 (configs[3]): 63 rotations of 2*pi/63 at 32^6 through bsl6d_rotate, full depth on sampled planes
# ------------------------------------------------------------------------------------------------------------
def test_C4_full_size_rotation_63_steps():
    _need(28)
    w = wl.C4
    nsteps = 63
    dt = 2.0 * math.pi / nsteps                              # reading S7: theta = 2*pi/63 for the return test
    B = (0.0, 0.0, 1.0)
    f0 = w.make_f("cuda")
    ps = PlaneSample(w, 2004)
    ref = ps.gather(f0)
    ref0 = ref.copy()
    a = f0.clone()
    b = torch.empty_like(a)
    with bsl.create(w.n, w.lo, w.dx, w.degree) as ctx:
        for s in range(nsteps):
            ctx.rotate(a, b, B, dt)                          # one fused pass in -> out (or 3 sweeps)
            a, b = b, a
            ref = oracle.rotate(ps.grid, w.degree, ref, B, dt)
            if s in (0, 1, 31, nsteps - 1):
                got = ps.gather(a)
                err = np.max(np.abs(got - ref)) / np.max(np.abs(ref))
                assert err <= TOL, f"C4 step {s}: rel err {err:.3e}"
        assert ctx.launch_count() in (nsteps, 3 * nsteps)    # one fused pass per rotation where available
    # return to the initial state within interpolation error + smoothed noise: the GPU's global deviation is of
    # the size the oracle shows on the sampled planes (C4 is under-resolved in v2: ~3 % of max f)
    dev_oracle = np.max(np.abs(ref - ref0)) / np.max(np.abs(ref0))
    dev_gpu = float((a - f0).abs().max() / f0.abs().max())
    assert dev_gpu < 0.08 and dev_gpu < 3.0 * dev_oracle + 1e-3, (dev_gpu, dev_oracle)


# ------------------------------------------------------------------------------------------------------------
# C5 (configs[4]): Strang steps at 48^3 x 32^3 (29 GB per buffer), degree 9
# ------------------------------------------------------------------------------------------------------------
def test_C5_full_size_strang_step_and_density():
    """(1) bsl6d_strang_step (ping-pong with f_tmp) equals, bit for bit on the whole array, the same twelve
    sweeps issued one by one in place; (2) each of those twelve sweeps is checked against the oracle on sampled
    pencils / planes; (3) the density of the result on sampled x-points.  Together: the full-size Strang step is
    the oracle's, on every sampled element."""
    _need(100)
    w = wl.C5
    og = _ogrid(w)
    E = w.E()
    Ed = [torch.from_numpy(e).cuda() for e in E]
    B = (0.0, 0.0, 1.0)
    f = w.make_f("cuda")
    g = f.clone()
    tmp = torch.empty_like(f)
    with bsl.create(w.n, w.lo, w.dx, w.degree) as ctx:
        ctx.strang_step(f, tmp, Ed, B, w.dt)                 # 12 launches, ping-pong
        del tmp
        torch.cuda.empty_cache()
        half = 0.5 * w.dt
        for d in range(3):
            check_sweep(ctx, w, og, g, g, d, "x", half, 2500 + d, what="x half 1")
        for d in range(3, 6):
            check_sweep(ctx, w, og, g, g, d, "E", w.dt, 2500 + d, E=E, what="E")
        ps = PlaneSample(w, 2510)
        ref = oracle.rotate(ps.grid, w.degree, ps.gather(g), B, w.dt)
        ctx.rotate(g, g, B, w.dt)
        err = np.max(np.abs(ps.gather(g) - ref)) / np.max(np.abs(ref))
        assert err <= TOL, f"C5 rotation: rel err {err:.3e}"
        for d in range(3):
            check_sweep(ctx, w, og, g, g, d, "x", half, 2520 + d, what="x half 2")
        assert torch.equal(f, g)                             # strang_step == the twelve verified sweeps
        del g
        check_density(ctx, w, og, f, 2599)
