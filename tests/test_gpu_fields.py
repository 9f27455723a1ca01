"""Field step on the GPU against the numpy oracle and against the Landau damping closed form."""
from __future__ import annotations

import math

import numpy as np
import pytest
import torch

import bsl6d_workloads as wl
import oracle
import paper_2303_05994_b200 as bsl

pytestmark = pytest.mark.gpu
TOL = 1e-12


def _need_gpu():
    from conftest import need_gpu
    need_gpu()


def _E_bufs(nx):
    return [torch.empty(nx, dtype=torch.float64, device="cuda") for _ in range(3)]


@pytest.mark.parametrize("nx,L", [((16, 9, 10), (4 * math.pi, 2 * math.pi, 6.0)), ((8, 8, 8), (1.0, 2.0, 3.0)),
                                  ((48, 6, 5), (7.0, 1.0, 2.5)), ((32, 32, 32), (4 * math.pi,) * 3)])
@pytest.mark.parametrize("closure", ("poisson", "adiabatic"))
def test_field_solve_matches_oracle(nx, L, closure):
    _need_gpu()
    n = tuple(nx) + (4, 4, 4)
    lo = (0.0, 0.0, 0.0, -2.0, -2.0, -2.0)
    dx = tuple(L[d] / nx[d] for d in range(3)) + (1.0, 1.0, 1.0)
    rng = np.random.default_rng(42)
    moment = 1.0 + 0.1 * rng.random(nx)
    md = torch.from_numpy(moment).cuda()
    E = _E_bufs(nx)
    with bsl.create(n, lo, dx, 3) as ctx:
        if closure == "poisson":
            ctx.field_poisson(md, -1.0, -0.5, E)
            ref = oracle.poisson_E(moment, L, -1.0, -0.5)
        else:
            ctx.field_adiabatic(md, 0.7, 1.5, E)
            ref = oracle.adiabatic_E(moment, L, 0.7, 1.5)
        assert ctx.launch_count() == 13
    scale = max(np.max(np.abs(r)) for r in ref)
    for d in range(3):
        assert np.max(np.abs(E[d].cpu().numpy() - ref[d])) <= TOL * scale, d


def test_field_single_mode_closed_form_on_gpu():
    """The same closed form that pins the oracle, applied to the GPU result directly."""
    _need_gpu()
    nx, L = (16, 12, 10), (4 * math.pi, 2 * math.pi, 6.0)
    ax = [np.arange(nx[d]) * (L[d] / nx[d]) for d in range(3)]
    X = np.meshgrid(*ax, indexing="ij")
    kap = [2 * math.pi * m / l for m, l in zip((2, -1, 1), L)]
    ph = kap[0] * X[0] + kap[1] * X[1] + kap[2] * X[2] + 0.3
    moment = 1.0 + 0.05 * np.cos(ph)
    E = _E_bufs(nx)
    n = tuple(nx) + (4, 4, 4)
    with bsl.create(n, (0.0,) * 6, tuple(L[d] / nx[d] for d in range(3)) + (1.0,) * 3, 3) as ctx:
        ctx.field_poisson(torch.from_numpy(moment).cuda(), 1.0, 1.0, E)
    k2 = sum(k * k for k in kap)
    for d in range(3):
        want = 0.05 * kap[d] * np.sin(ph) / k2
        assert np.max(np.abs(E[d].cpu().numpy() - want)) <= 1e-14


@pytest.mark.parametrize("pingpong", (False, True))
def test_vp_step_matches_oracle(pingpong):
    _need_gpu()
    w = wl.C5.reduced((8, 8, 8, 16, 16, 16))
    og = oracle.Grid(tuple(w.n), tuple(w.lo), tuple(w.dx))
    f = w.make_f("cpu").numpy()
    fd = torch.from_numpy(f).cuda()
    tmp = torch.empty_like(fd) if pingpong else None
    rho = torch.empty(w.n[:3], dtype=torch.float64, device="cuda")
    E = _E_bufs(tuple(w.n[:3]))
    ref = f.copy()
    with bsl.create(w.n, w.lo, w.dx, w.degree) as ctx:
        for step in range(3):
            ctx.vp_step(fd, tmp, rho, E, w.B, w.dt, 0, -1.0, -1.0)
            ref, mom, Eo = oracle.vp_step(og, w.degree, ref, w.B, w.dt, "poisson", -1.0, -1.0)
            assert np.max(np.abs(fd.cpu().numpy() - ref)) <= TOL * np.max(np.abs(ref)), step
            assert np.max(np.abs(rho.cpu().numpy() - mom)) <= TOL * np.max(np.abs(mom))
            es = max(np.max(np.abs(e)) for e in Eo)
            for d in range(3):
                assert np.max(np.abs(E[d].cpu().numpy() - Eo[d])) <= 1e-11 * es + 1e-15
        ctx.vp_step(fd, tmp, rho, E, None, w.dt, 1, 0.5, 1.0)     # adiabatic closure, no B
        ref, _, _ = oracle.vp_step(og, w.degree, ref, None, w.dt, "adiabatic", 0.5, 1.0)
        assert np.max(np.abs(fd.cpu().numpy() - ref)) <= TOL * np.max(np.abs(ref))


def test_landau_damping_on_gpu():
    """1D1V Vlasov-Poisson through bsl6d_vp_step: gamma = -0.1533, omega = 1.4156 (k = 0.5), as for the oracle."""
    _need_gpu()
    nx, nv, vmax = 32, 64, 6.0
    Lx = 4 * math.pi
    n = (nx, 1, 1, nv, 1, 1)
    lo = (0.0, 0.0, 0.0, -vmax, 0.0, 0.0)
    dx = (Lx / nx, 1.0, 1.0, 2 * vmax / nv, 1.0, 1.0)
    x = np.arange(nx) * dx[0]
    v = -vmax + np.arange(nv) * dx[3]
    f = ((1 + 0.01 * np.cos(0.5 * x))[:, None] * (np.exp(-0.5 * v * v) / math.sqrt(2 * math.pi))[None, :]).reshape(n)
    fd = torch.from_numpy(np.ascontiguousarray(f)).cuda()
    rho = torch.empty((nx, 1, 1), dtype=torch.float64, device="cuda")
    E = _E_bufs((nx, 1, 1))
    dt, nsteps = 0.1, 220
    amp = []
    with bsl.create(n, lo, dx, 7) as ctx:
        for _ in range(nsteps):
            ctx.vp_step(fd, None, rho, E, None, dt, 0, -1.0, -1.0)
            amp.append(float(E[0].abs().max()))
    amp = np.array(amp)
    t = (np.arange(nsteps) + 0.5) * dt
    pk = [i for i in range(1, nsteps - 1) if amp[i] > amp[i - 1] and amp[i] >= amp[i + 1] and 1.0 < t[i] < 20.0]
    tp, ap = [], []
    for i in pk:
        y0, y1, y2 = np.log(amp[i - 1]), np.log(amp[i]), np.log(amp[i + 1])
        d = 0.5 * (y0 - y2) / (y0 - 2 * y1 + y2)
        tp.append(t[i] + d * dt)
        ap.append(y1 - 0.25 * (y0 - y2) * d)
    gamma = np.polyfit(tp, ap, 1)[0]
    omega = math.pi / np.mean(np.diff(tp))
    assert abs(gamma + 0.1533) < 0.004 and abs(omega - 1.4156) < 0.01, (gamma, omega)


def test_field_error_paths():
    _need_gpu()
    w = wl.C1
    rho = torch.zeros(w.n[:3], dtype=torch.float64, device="cuda")
    E = _E_bufs(tuple(w.n[:3]))
    f = w.make_f("cuda")
    with bsl.create(w.n, w.lo, w.dx, w.degree) as ctx:
        with pytest.raises(bsl.Bsl6dError) as e:
            ctx.field_poisson(rho, float("nan"), 1.0, E)
        assert e.value.code == bsl.EINVAL
        with pytest.raises(bsl.Bsl6dError) as e:
            ctx.vp_step(f, None, rho, E, (30.0, 40.0, 0.0), 0.2, 0, 1.0, 1.0)    # oblique B, > a full turn
        assert e.value.code == bsl.EUNSUPPORTED
        with pytest.raises(bsl.Bsl6dError) as e:
            ctx.vp_step(f, None, rho, E, None, 0.1, 7, 1.0, 1.0)                 # unknown closure
        assert e.value.code == bsl.EINVAL
        assert ctx.launch_count() == 0
        # an opened x dim (a slab with halo planes) has no spectral field solve: refused before anything is enqueued
        ctx.set_boundary(0, 1)
        f0 = f.clone()
        with pytest.raises(bsl.Bsl6dError) as e:
            ctx.vp_step(f, None, rho, E, None, 0.1, 0, 1.0, 1.0)
        assert e.value.code == bsl.EUNSUPPORTED
        torch.cuda.synchronize()
        assert ctx.launch_count() == 0 and torch.equal(f, f0)
