"""Slabs WITHOUT halo planes: bsl6d_advect_x1_peer reads the neighbours' planes where they
are, so the halo exchange is the sweep's own loads.  Here the "peers" are other slabs on the same device (one process),
and -- through CUDA IPC, the mechanism a one-process-per-GPU run uses -- another PROCESS on the same device.  Every
result must equal the same operation on the undivided periodic grid bit for bit."""
from __future__ import annotations

import os
import socket

import numpy as np
import pytest
import torch

import bsl6d_workloads as wl
import paper_2303_05994_b200 as bsl
from paper_2303_05994_b200 import slab

pytestmark = pytest.mark.gpu


def _need_gpu():
    from conftest import need_gpu
    need_gpu()


def _ring(w, world, max_shift, f):
    ss = [slab.PeerSlab(w.n, w.lo, w.dx, w.degree, world, r, max_shift) for r in range(world)]
    L = ss[0].plan.L
    for r, s in enumerate(ss):
        s.alloc()
        s.f.copy_(f[r * L:(r + 1) * L])
    for r, s in enumerate(ss):
        s.connect(ss[s.plan.left].buf, ss[s.plan.right].buf)
    return ss


def _gather(ss):
    return torch.cat([s.f for s in ss], dim=0)


def test_x1_peer_sweep_refuses_a_step_longer_than_planned():
    """A dt above the one the slab was planned for would read beyond the promised neighbour planes (silently zeros)."""
    _need_gpu()
    w = wl.C2.reduced((32, 4, 2, 8, 4, 8))
    f = w.make_f("cuda")
    ss = _ring(w, 2, 0.5, f)                                    # planned for half a cell
    before = ss[0].ctx.launch_count()
    with pytest.raises(ValueError):
        ss[0].advect_x1(1.7 * w.dx[0] / 6.0)                    # 1.7 cells
    assert ss[0].ctx.launch_count() == before and ss[0].cur == 0
    ss[0].advect_x1(0.4 * w.dx[0] / 6.0)                        # within the plan
    for s in ss:
        s.destroy()


@pytest.mark.parametrize("world", (1, 2, 4))
@pytest.mark.parametrize("dt_cells", (0.37, 2.3, "whole"))
def test_x1_peer_sweep_equals_undivided(world, dt_cells):
    _need_gpu()
    w = wl.C2.reduced((32, 4, 2, 8, 4, 8))
    vmax = 6.0
    if dt_cells == "whole":
        dt, max_shift = 2.0 * w.dx[0], 2.0 * vmax               # alpha = -2 v_j: whole cells, |k| up to 12
    else:
        dt, max_shift = dt_cells * w.dx[0] / vmax, dt_cells
    if dt_cells == "whole" and world == 4:                      # w = 16 > L = 8: refused by the plan
        with pytest.raises(ValueError):
            slab.plan_slab(w.n, w.degree, world, 0, max_shift)
        return
    f = w.make_f("cuda")
    with bsl.create(w.n, w.lo, w.dx, w.degree) as ctx:
        ref = ctx.advect(f, torch.empty_like(f), 0, None, dt)
    ss = _ring(w, world, max_shift, f)
    for s in ss:                                                # every slab reads the others' UNCHANGED input buffers
        s.advect_x1(dt)
    got = _gather(ss)
    assert torch.equal(got, ref)
    # and against the oracle directly (the undivided GPU sweep is compared with it in test_gpu_parity.py as well)
    import oracle
    og = oracle.Grid(tuple(w.n), tuple(w.lo), tuple(w.dx))
    oref = oracle.advect(og, w.degree, f.cpu().numpy(), 0, None, dt)
    if dt_cells == "whole":
        assert np.array_equal(got.cpu().numpy(), oref)
    else:
        assert np.max(np.abs(got.cpu().numpy() - oref)) <= 1e-12 * np.max(np.abs(oref))
    for s in ss:
        s.destroy()


@pytest.mark.parametrize("n0,world", [(24, 2), (20, 1), (36, 3), (30, 2)])
def test_x1_peer_sweep_runtime_extent_kernel(n0, world):
    """Slab thicknesses without a compiled instance (12, 20, 12, 15 planes) take sweep_peer_kernel (run-time extent,
    pencil and neighbour planes staged in shared memory); q = 8 and q = 4."""
    _need_gpu()
    for degree in (7, 3):
        w = wl.replace(wl.C2.reduced((n0, 3, 2, 8, 4, 5)), degree=degree)
        dt = 1.7 * w.dx[0] / 6.0
        f = w.make_f("cuda")
        with bsl.create(w.n, w.lo, w.dx, w.degree) as ctx:
            ref = ctx.advect(f, torch.empty_like(f), 0, None, dt)
        ss = _ring(w, world, 1.7, f)
        for s in ss:
            s.advect_x1(dt)
        assert torch.equal(_gather(ss), ref), (n0, world, degree)
        for s in ss:
            s.destroy()


@pytest.mark.parametrize("world", (2, 4))
def test_peer_strang_steps_equal_undivided(world):
    _need_gpu()
    w = wl.replace(wl.C5.reduced((32, 4, 4, 8, 8, 8)), degree=5)
    f = w.make_f("cuda")
    Ed = [torch.from_numpy(e).cuda() for e in w.E()]
    ref = f.clone()
    with bsl.create(w.n, w.lo, w.dx, w.degree) as ctx:
        for _ in range(2):
            ctx.strang_step(ref, None, Ed, w.B, w.dt)
    ss = _ring(w, world, 6.0 * 0.5 * w.dt / w.dx[0], f)
    L = ss[0].plan.L
    Eloc = [[e[r * L:(r + 1) * L].contiguous() for e in Ed] for r in range(world)]
    half = 0.5 * w.dt
    for _ in range(2):                                          # the phases of PeerSlab.strang_step, slabs in lock step
        for s in ss:
            s.advect_x1(half)
        for r, s in enumerate(ss):
            s.local_part(Eloc[r], w.B, half, w.dt, w.dt)
        for s in ss:
            s.advect_x1(half)
        for s in ss:
            s.local_part(None, None, half, None, None)
    assert torch.equal(_gather(ss), ref)
    for s in ss:
        s.destroy()


def test_peer_sweep_error_codes():
    _need_gpu()
    n = (16, 2, 2, 8, 2, 2)
    f = torch.zeros(n, dtype=torch.float64, device="cuda")
    g = torch.zeros_like(f)
    with bsl.create(n, (0.0,) * 3 + (-6.0,) * 3, (1.0,) * 6, 7) as ctx:
        for bad in (lambda: ctx.advect_x1_peer(f, f, f, f, 5, None, 0.1),        # in place
                    lambda: ctx.advect_x1_peer(f, g, f, g, 5, None, 0.1)):       # the output is a neighbour's input
            with pytest.raises(bsl.Bsl6dError) as e:
                bad()
            assert e.value.code == bsl.EALIAS
        for halo in (3, 17):                                                     # below q/2; more than the slab has
            with pytest.raises(bsl.Bsl6dError) as e:
                ctx.advect_x1_peer(f, f, f, g, halo, None, 0.1)
            assert e.value.code == bsl.EINVAL
        assert ctx.launch_count() == 0


# ---- two PROCESSES on one device: the neighbours' arrays arrive through CUDA IPC ----------------------------------
def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _ipc_worker(rank, world, port, out_path):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        torch.cuda.set_device(0)
        w = wl.replace(wl.C5.reduced((16, 4, 4, 8, 8, 8)), degree=5)
        f = w.make_f("cuda")                                   # every rank builds the same seeded global grid
        Ed = [torch.from_numpy(e).cuda() for e in w.E()]
        s = slab.PeerSlab(w.n, w.lo, w.dx, w.degree, world, rank, 6.0 * 0.5 * w.dt / w.dx[0])
        L = s.plan.L
        s.alloc()
        s.f.copy_(f[rank * L:(rank + 1) * L])
        descs = [None] * world
        dist.all_gather_object(descs, slab.share_buffers(s.buf))
        s.connect(slab.open_peer_buffers(descs[s.plan.left]), slab.open_peer_buffers(descs[s.plan.right]))
        Eloc = [e[rank * L:(rank + 1) * L].contiguous() for e in Ed]
        for _ in range(2):
            s.strang_step(Eloc, w.B, w.dt, sync=slab.ring_sync)
        slab.ring_sync()
        mine = s.f.cpu()
        parts = [torch.empty_like(mine) for _ in range(world)]
        dist.all_gather(parts, mine)
        if rank == 0:
            ref = f.clone()
            with bsl.create(w.n, w.lo, w.dx, w.degree) as ctx:
                for _ in range(2):
                    ctx.strang_step(ref, None, Ed, w.B, w.dt)
            torch.cuda.synchronize()
            with open(out_path, "w") as fh:
                fh.write("equal" if torch.equal(torch.cat(parts, dim=0), ref.cpu()) else "different")
        dist.barrier()                                         # nobody frees arrays a neighbour may still have mapped
        s.destroy()
    finally:
        dist.destroy_process_group()


def test_peer_strang_steps_two_processes_cuda_ipc(tmp_path):
    _need_gpu()
    import torch.multiprocessing as mp
    out = str(tmp_path / "result.txt")
    mp.spawn(_ipc_worker, args=(2, _free_port(), out), nprocs=2, join=True)
    assert open(out).read() == "equal"
