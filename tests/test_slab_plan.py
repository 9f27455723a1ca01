"""x1-slab decomposition: host-side planning and the ring halo
exchange, on CPU.  The exchange is pure torch.distributed plumbing, so it runs here with the gloo backend and
world_size 2 and 3; the sweeps themselves are covered on the GPU (tests/test_gpu_slab.py)."""
import os
import socket
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from paper_2303_05994_b200 import slab  # noqa: E402


def test_plan_geometry():
    p = slab.plan_slab((32, 4, 4, 8, 8, 8), degree=7, world=4, rank=1, max_shift_cells=2.3)
    assert (p.L, p.w, p.q) == (8, 4 + 3, 8)                    # q/2 + ceil(2.3)
    assert p.local_shape == (8 + 14, 4, 4, 8, 8, 8) and p.plane == 4 * 4 * 8 * 8 * 8
    assert (p.left, p.right, p.x1_offset) == (0, 2, 8)
    assert p.interior == (7, 15) and p.recv_lo == (0, 7) and p.recv_hi == (15, 22)
    assert p.send_lo == (7, 14) and p.send_hi == (8, 15)
    assert p.halo_bytes_per_side == 8 * 7 * p.plane
    ring0 = slab.plan_slab((32, 4, 4, 8, 8, 8), 7, 4, 0, 0.5)
    assert (ring0.left, ring0.right, ring0.w) == (3, 1, 5)    # periodic ring; ceil(0.5) = 1
    one = slab.plan_slab((8, 2, 2, 2, 2, 2), 3, 1, 0, 0.0)
    assert (one.left, one.right, one.w, one.L) == (0, 0, 2, 8)


def test_planes_needed_by_an_x1_sweep():
    """Half the stencil plus the largest |v1| dt / dx1, rounded up -- what both slab forms check before an x1 sweep."""
    n = (32, 4, 4, 8, 8, 8)
    lo = (0.0, 0.0, 0.0, -6.0, -6.0, -6.0)
    dx = (0.25, 1.0, 1.0, 1.5, 1.5, 1.5)                          # v1 nodes -6 .. 4.5: |v1| <= 6
    assert slab.x1_planes_needed(lo, dx, n, 8, 0.0) == 4
    assert slab.x1_planes_needed(lo, dx, n, 8, 0.01) == 5         # 0.24 cells
    assert slab.x1_planes_needed(lo, dx, n, 8, -0.1) == 4 + 3     # 2.4 cells, the sign of dt does not matter
    assert slab.x1_planes_needed(lo, dx, n, 6, 0.125) == 3 + 3    # exactly 3 cells
    lo2 = (0.0, 0.0, 0.0, -3.0, -6.0, -6.0)                       # v1 nodes -3 .. 7.5: the upper end decides
    assert slab.x1_planes_needed(lo2, dx, n, 8, 0.1) == 4 + 3
    # consistent with the plan: a slab planned for that displacement accepts the step
    p = slab.plan_slab(n, 7, 2, 0, 6.0 * 0.1 / 0.25)
    assert slab.x1_planes_needed(lo, dx, n, p.q, 0.1) == p.w


def test_plan_rejects_what_the_halo_cannot_serve():
    with pytest.raises(ValueError):
        slab.plan_slab((30, 4, 4, 8, 8, 8), 7, 4, 0, 1.0)     # 30 planes do not divide among 4 ranks
    with pytest.raises(ValueError):
        slab.plan_slab((32, 4, 4, 8, 8, 8), 7, 8, 0, 1.5)     # L = 4 < w = 6: halo would reach past the neighbour
    with pytest.raises(ValueError):
        slab.plan_slab((32, 4, 4, 8, 8, 8), 7, 4, 4, 1.0)


def _coded(plan, r):
    """Local array whose interior plane j holds the value 1000*r + j (global plane id would do as well)."""
    t = torch.full(plan.local_shape, -1.0, dtype=torch.float64)
    for j in range(plan.L):
        t[plan.w + j] = 1000.0 * r + j
    return t


def _check_halos(plan, t):
    L, w = plan.L, plan.w
    for h in range(w):
        assert torch.all(t[h] == 1000.0 * plan.left + (L - w + h)), (plan.rank, h)          # left neighbour's top planes
        assert torch.all(t[w + L + h] == 1000.0 * plan.right + h), (plan.rank, h)           # right neighbour's bottom
    for j in range(L):
        assert torch.all(t[w + j] == 1000.0 * plan.rank + j)                                 # interior untouched


@pytest.mark.parametrize("world", (1, 2, 4))
def test_exchange_local_fills_every_halo(world):
    n = (16, 2, 3, 2, 2, 2)
    plans = [slab.plan_slab(n, 3, world, r, 1.2) for r in range(world)]
    locs = [_coded(p, r) for r, p in enumerate(plans)]
    slab.exchange_local(plans, locs)
    for p, t in zip(plans, locs):
        _check_halos(p, t)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        plan = slab.plan_slab((12, 2, 3, 2, 2, 2), 3, world, rank, 0.7)
        t = _coded(plan, rank)
        slab.exchange(plan, t)
        _check_halos(plan, t)
        # a second exchange after the interior changed must carry the new values
        t[plan.w:plan.w + plan.L] += 0.5
        slab.exchange(plan, t)
        assert torch.all(t[0] == 1000.0 * plan.left + (plan.L - plan.w) + 0.5)
        # the two halves on a thicker slab: post, change planes that are neither sent nor received, finish
        plan = slab.plan_slab((24, 2, 3, 2, 2, 2), 3, world, rank, 0.7)
        reg = plan.regions
        assert reg is not None and reg[2][1] > reg[2][0] and reg[0] == plan.send_lo and reg[1] == plan.send_hi
        t = _coded(plan, rank)
        h = slab.exchange_start(plan, t)
        t[reg[2][0]:reg[2][1]] += 7.0                        # middle planes: work that overlaps the transfers
        slab.exchange_finish(h)
        for k in range(plan.w):
            assert torch.all(t[k] == 1000.0 * plan.left + (plan.L - plan.w + k))
            assert torch.all(t[plan.w + plan.L + k] == 1000.0 * plan.right + k)
        assert torch.all(t[reg[2][0]] == 1000.0 * rank + (reg[2][0] - plan.w) + 7.0)
        assert slab.plan_slab((12, 2, 3, 2, 2, 2), 3, 3, 0, 0.7).regions is None      # L = 4 < 2w = 6
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", (2, 3))
def test_exchange_over_torch_distributed_gloo(world):
    mp.spawn(_worker, args=(world, _free_port()), nprocs=world, join=True)


def test_exchange_single_rank_wraps_onto_itself():
    plan = slab.plan_slab((8, 2, 2, 2, 2, 2), 3, 1, 0, 0.5)
    t = _coded(plan, 0)
    slab.exchange(plan, t)
    _check_halos(plan, t)
