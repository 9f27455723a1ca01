"""x1-slab decomposition on ONE GPU: a grid is cut into 2 and 4
slabs that live side by side on the device, halos are exchanged with device copies, and every operation on the
slabs must reproduce the same operation on the undivided grid bit for bit (torch.equal) -- displacements of more than
one cell and whole-cell shifts included."""
from __future__ import annotations

import numpy as np
import pytest
import torch

import bsl6d_workloads as wl
import oracle
import paper_2303_05994_b200 as bsl
from paper_2303_05994_b200 import slab

pytestmark = pytest.mark.gpu


def _need_gpu():
    from conftest import need_gpu
    need_gpu()


def _slabs(w, world, max_shift):
    ss = [slab.Slab(w.n, w.lo, w.dx, w.degree, world, r, max_shift) for r in range(world)]
    return ss, [s.plan for s in ss]


def _scatter(ss, f):
    locs = []
    for s in ss:
        t = s.alloc()
        s.scatter_from_global(f, t)
        locs.append(t)
    return locs


def _gather(ss, locs):
    return torch.cat([s.interior(t) for s, t in zip(ss, locs)], dim=0)


@pytest.mark.parametrize("world", (2, 4))
@pytest.mark.parametrize("dt_cells", (0.37, 2.3, "whole"))
def test_x1_sweep_on_slabs_equals_undivided(world, dt_cells):
    _need_gpu()
    w = wl.C2.reduced((32, 4, 2, 8, 4, 8))
    vmax = 6.0
    if dt_cells == "whole":
        dt, max_shift = 2.0 * w.dx[0], 2.0 * vmax               # alpha = -2 v_j: whole cells (v_j = -6 + 1.5 j), |k| up to 12
        # w = 4 + 12 = 16 halo planes: fits L = 16 (two slabs), not L = 8 (four slabs: refused, see below)
    else:
        dt, max_shift = dt_cells * w.dx[0] / vmax, dt_cells
    if dt_cells == "whole" and world == 4:
        with pytest.raises(ValueError):
            _slabs(w, world, max_shift)
        return
    f = w.make_f("cuda")
    with bsl.create(w.n, w.lo, w.dx, w.degree) as ctx:
        ref = ctx.advect(f, torch.empty_like(f), 0, None, dt)
    ss, plans = _slabs(w, world, max_shift)
    locs = _scatter(ss, f)
    slab.exchange_local(plans, locs)
    for s, t in zip(ss, locs):
        s.advect_x1(t, dt)
    out = _gather(ss, locs)
    assert torch.equal(out, ref)
    if dt_cells == "whole":                                     # and an exact permutation it is
        fh = f.cpu().numpy()
        exp = np.empty_like(fh)
        for j in range(w.n[3]):
            exp[:, :, :, j] = np.roll(fh[:, :, :, j], int(round(2.0 * (w.lo[3] + j * w.dx[3]))), axis=0)
        assert np.array_equal(out.cpu().numpy(), exp)
    for s in ss:
        s.destroy()


def test_halo_too_narrow_for_the_time_step_is_refused():
    _need_gpu()
    w = wl.C2.reduced((16, 2, 2, 8, 4, 4))
    s = slab.Slab(w.n, w.lo, w.dx, w.degree, 2, 0, 0.5)
    t = s.alloc()
    with pytest.raises(ValueError):
        s.advect_x1(t, 3.0 * w.dx[0] / 6.0)                      # 3 cells at |v| = 6, planned for 0.5
    s.destroy()


@pytest.mark.parametrize("world", (2, 4))
def test_strang_steps_and_density_on_slabs_equal_undivided(world):
    """Two Strang steps (x halves with halo exchange, E sweeps, rotation) and the density moment: every slab holds
    exactly the planes of the undivided run, and the whole thing agrees with the oracle."""
    _need_gpu()
    w = wl.C5.reduced((32, 4, 4, 8, 8, 8))
    w = wl.replace(w, degree=5)
    f0 = w.make_f("cpu").numpy()
    E = w.E()
    f = torch.from_numpy(f0).cuda()
    Ed = [torch.from_numpy(e).cuda() for e in E]
    rho_ref = torch.empty(w.n[:3], dtype=torch.float64, device="cuda")
    with bsl.create(w.n, w.lo, w.dx, w.degree) as ctx:
        for _ in range(2):
            ctx.strang_step(f, None, Ed, w.B, w.dt)
        ctx.density(f, rho_ref)
    max_shift = 6.0 * 0.5 * w.dt / w.dx[0]
    ss, plans = _slabs(w, world, max_shift)
    locs = _scatter(ss, torch.from_numpy(f0).cuda())
    L = plans[0].L
    Eloc = [[e[r * L:(r + 1) * L].contiguous() for e in Ed] for r in range(world)]
    for _ in range(2):
        # the ranks of a real run proceed in lock step; here the slabs take turns between the exchanges
        slab.exchange_local(plans, locs)
        for s, t in zip(ss, locs):
            s.advect_x1(t, 0.5 * w.dt)
        for r, (s, t) in enumerate(zip(ss, locs)):
            for d in (1, 2):
                s.advect(t, d, None, 0.5 * w.dt)
            for d in (3, 4, 5):
                s.advect(t, d, Eloc[r][d - 3], w.dt)
            s.rotate(t, w.B, w.dt)
        slab.exchange_local(plans, locs)
        for s, t in zip(ss, locs):
            s.advect_x1(t, 0.5 * w.dt)
        for s, t in zip(ss, locs):
            for d in (1, 2):
                s.advect(t, d, None, 0.5 * w.dt)
    out = _gather(ss, locs)
    assert torch.equal(out, f)
    rho = torch.empty_like(rho_ref)
    for r, (s, t) in enumerate(zip(ss, locs)):
        s.density(t, rho[r * L:(r + 1) * L])
    assert torch.equal(rho, rho_ref)
    og = oracle.Grid(tuple(w.n), tuple(w.lo), tuple(w.dx))
    ref = f0.copy()
    for _ in range(2):
        ref = oracle.strang_step(og, w.degree, ref, E, w.B, w.dt)
    assert np.max(np.abs(out.cpu().numpy() - ref)) <= 1e-12 * np.max(np.abs(ref))
    for s in ss:
        s.destroy()


def test_slab_strang_driver_single_rank_ring():
    """Slab.strang_step with world = 1 (the ring closes on itself: the halos are the slab's own far planes) equals
    bsl6d_strang_step on the plain periodic grid."""
    _need_gpu()
    w = wl.replace(wl.C5.reduced((16, 4, 4, 8, 8, 8)), degree=7)
    f0 = w.make_f("cuda")
    Ed = [torch.from_numpy(e).cuda() for e in w.E()]
    ref = f0.clone()
    with bsl.create(w.n, w.lo, w.dx, w.degree) as ctx:
        ctx.strang_step(ref, None, Ed, w.B, w.dt)
    s = slab.Slab(w.n, w.lo, w.dx, w.degree, 1, 0, 6.0 * 0.5 * w.dt / w.dx[0])
    t = s.scatter_from_global(f0, s.alloc())
    s.strang_step(t, Ed, w.B, w.dt, lambda x: slab.exchange(s.plan, x))
    assert torch.equal(s.interior(t), ref)
    s.destroy()


@pytest.mark.parametrize("world,n0", [(2, 32), (4, 32), (2, 12)])
def test_overlapped_strang_steps_on_slabs_equal_undivided(world, n0):
    """The overlapped step (boundary regions first, exchange posted, middle planes while the halos travel) on 2 and 4
    slabs, phases in the lock step of a real run with the exchange emulated by device copies: bit-identical to the
    undivided grid.  (4, 32): L = 2w, no middle; (2, 12): L < 2w, the whole interior is boundary."""
    _need_gpu()
    w = wl.replace(wl.C5.reduced((n0, 4, 4, 8, 8, 8)), degree=5)
    f = w.make_f("cuda")
    Ed = [torch.from_numpy(e).cuda() for e in w.E()]
    ref = f.clone()
    with bsl.create(w.n, w.lo, w.dx, w.degree) as ctx:
        for _ in range(2):
            ctx.strang_step(ref, None, Ed, w.B, w.dt)
    ss, plans = _slabs(w, world, 6.0 * 0.5 * w.dt / w.dx[0])
    L, hw = plans[0].L, plans[0].w
    assert (plans[0].regions is None) == (L < 2 * hw)
    locs = _scatter(ss, f)
    Eloc = [[e[r * L:(r + 1) * L].contiguous() for e in Ed] for r in range(world)]
    half = 0.5 * w.dt
    seq_x = [(1, None, 0, half / w.dx[1]), (2, None, 0, half / w.dx[2])]
    first, later = ss[0].step_regions()
    slab.exchange_local(plans, locs)
    for _ in range(2):
        for s, t in zip(ss, locs):
            s.advect_x1(t, half)
        for r, (s, t) in enumerate(zip(ss, locs)):
            for reg in first:
                s.local_ops(t, reg, seq_x, Eloc[r], w.B, w.dt, w.dt)
        slab.exchange_local(plans, locs)                     # posted here in a real run ...
        for r, (s, t) in enumerate(zip(ss, locs)):
            for reg in later:                                # ... while the middle planes are advanced
                s.local_ops(t, reg, seq_x, Eloc[r], w.B, w.dt, w.dt)
        for s, t in zip(ss, locs):
            s.advect_x1(t, half)
        for s, t in zip(ss, locs):
            for reg in first:
                s.local_ops(t, reg, seq_x, None, None, None, None)
        slab.exchange_local(plans, locs)
        for s, t in zip(ss, locs):
            for reg in later:
                s.local_ops(t, reg, seq_x, None, None, None, None)
    assert torch.equal(_gather(ss, locs), ref)
    for s in ss:
        s.destroy()


def test_overlapped_strang_driver_single_rank_ring():
    """Slab.strang_step_overlapped with world = 1, two steps chained through the pending handle."""
    _need_gpu()
    w = wl.replace(wl.C5.reduced((16, 4, 4, 8, 8, 8)), degree=5)
    f0 = w.make_f("cuda")
    Ed = [torch.from_numpy(e).cuda() for e in w.E()]
    ref = f0.clone()
    with bsl.create(w.n, w.lo, w.dx, w.degree) as ctx:
        for _ in range(2):
            ctx.strang_step(ref, None, Ed, w.B, w.dt)
    s = slab.Slab(w.n, w.lo, w.dx, w.degree, 1, 0, 6.0 * 0.5 * w.dt / w.dx[0])
    assert s.plan.regions is not None
    t = s.scatter_from_global(f0, s.alloc())
    h = s.strang_step_overlapped(t, Ed, w.B, w.dt)
    h = s.strang_step_overlapped(t, Ed, w.B, w.dt, pending=h)
    slab.exchange_finish(h)
    assert torch.equal(s.interior(t), ref)
    s.destroy()
