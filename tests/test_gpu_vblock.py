"""Whole-v-block passes (paper_2303_05994_b200/csrc/vblock_kernels.cuh): a run of velocity-space
sweeps executed as ONE pass -- TMA-staged tile per CTA, v3 sweeps through distributed shared memory across the
cluster -- must give, bit for bit, what the same sweeps give one launch at a time, must agree with the oracle
within 1e-12, and must take the number of passes the planner promises."""
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


def _need_gpu(gb=0.0):
    from conftest import need_gpu
    need_gpu(gb)


def ogrid(w):
    return oracle.Grid(tuple(w.n), tuple(w.lo), tuple(w.dx))


def rel_err(gpu: torch.Tensor, ref: np.ndarray) -> float:
    return float(np.max(np.abs(gpu.cpu().numpy() - ref)) / np.max(np.abs(ref)))


def v_chain(w, amp, rng):
    """A chain over all three velocity dims whose shift sources depend on x (E-like, any size up to `amp` cells,
    both signs, so that the v3 sweep reads from every CTA of the cluster) and on another velocity (shear-like)."""
    nx = w.n[:3]
    E = [amp * w.dx[3 + d] * (2.0 * rng.random(nx) - 1.0) for d in range(3)]      # |alpha| <= amp cells at scale 1/dx
    sw_host = [(3 + d, E[d], 0x7, 1.0 / w.dx[3 + d]) for d in range(3)]
    # shears: v1 by v2, v2 by v1, v3 by v1, v1 by v3, v2 by v3, v3 by v2 (every source/target pairing)
    for a, b, s in ((3, 4, 0.11), (4, 3, -0.2), (5, 3, 0.15), (3, 5, -0.07), (4, 5, 0.3), (5, 4, -0.25)):
        nodes = np.array([w.lo[b] + i * w.dx[b] for i in range(w.n[b])])
        sw_host.append((a, nodes, 1 << b, s / w.dx[a]))
    return sw_host


def run_oracle(w, f, sw_host):
    ref = f
    for dim, src, mask, scale in sw_host:
        ref = oracle.sweep(ref, dim, np.ascontiguousarray(src), mask, scale, w.degree + 1)
    return ref


@pytest.mark.parametrize("nv", (8, 16, 32))
@pytest.mark.parametrize("degree", (5, 7, 9))
def test_v_chain_one_pass_equals_single_sweeps_and_oracle(nv, degree):
    _need_gpu()
    w = wl.replace(wl.C5.reduced((2, 3, 2, nv, nv, nv)), degree=degree)
    rng = np.random.default_rng(100 * nv + degree)
    f = w.make_f("cpu").numpy()
    sw_host = v_chain(w, 2.6, rng)
    sw = [(d, torch.from_numpy(np.ascontiguousarray(s)).cuda(), m, sc) for d, s, m, sc in sw_host]
    fd = torch.from_numpy(f).cuda()
    with bsl.create(w.n, w.lo, w.dx, w.degree) as ctx:
        default_passes = ctx.seq_passes(sw)                       # default policy: v3 sweeps stay passes of their own
        assert 1 < default_passes < len(sw)
        by_policy = ctx.advect_seq(fd, torch.empty_like(fd), sw)
        ctx.set_fusion(2)                                         # everything the kernels can do
        assert ctx.seq_passes(sw) == 1                            # nine velocity-space sweeps, one pass
        l0 = ctx.launch_count()
        one = ctx.advect_seq(fd, torch.empty_like(fd), sw)
        assert ctx.launch_count() - l0 == 1
        inplace = fd.clone()
        ctx.advect_seq(inplace, inplace, sw)
        ctx.set_fusion(0)
        assert ctx.seq_passes(sw) == len(sw)
        single = ctx.advect_seq(fd, torch.empty_like(fd), sw)
    assert torch.equal(one, single) and torch.equal(inplace, single) and torch.equal(by_policy, single)
    assert rel_err(one, run_oracle(w, f, sw_host)) <= TOL


def test_whole_cell_shifts_stay_exact_through_a_v_block_pass():
    _need_gpu()
    w = wl.C2.reduced((2, 2, 2, 32, 32, 32))
    f = w.make_f("cpu").numpy()
    fd = torch.from_numpy(f).cuda()
    one = torch.ones(1, dtype=torch.float64, device="cuda")
    with bsl.create(w.n, w.lo, w.dx, w.degree) as ctx:
        sw = [(3, one, 0, 2.0), (4, one, 0, -3.0), (5, one, 0, 9.0), (5, one, 0, -20.0)]   # alpha = -2, +3, -9, +20
        ctx.set_fusion(2)
        assert ctx.seq_passes(sw) == 1
        out = ctx.advect_seq(fd, torch.empty_like(fd), sw).cpu().numpy()
    ref = f                                                       # shift with zero fill, sweep by sweep
    for dim, a in ((3, -2), (4, 3), (5, -9), (5, 20)):
        nxt = np.zeros_like(ref)
        idx_out = [slice(None)] * 6
        idx_in = [slice(None)] * 6
        n = ref.shape[dim]
        if a < 0:
            idx_out[dim], idx_in[dim] = slice(-a, n), slice(0, n + a)
        else:
            idx_out[dim], idx_in[dim] = slice(0, n - a), slice(a, n)
        nxt[tuple(idx_out)] = ref[tuple(idx_in)]
        ref = nxt
    assert np.array_equal(out, ref)


@pytest.mark.parametrize("pingpong", (False, True))
def test_strang_step_passes_and_matches(pingpong):
    """Fusion mode 2: x1+x2 | x3 | the whole velocity part in ONE pass | x1+x2 | x3 -- five launches.  Default policy:
    x1 | x2+x3 | v1+v2 | v3 | the three shears | x1 | x2+x3 -- seven.  All of them bit-identical to twelve sweeps."""
    _need_gpu()
    w = wl.C5.reduced((6, 8, 8, 32, 32, 32))
    w = wl.replace(w, degree=7)
    f = w.make_f("cpu").numpy()
    E = w.E()
    Ed = [torch.from_numpy(e).cuda() for e in E]
    a = torch.from_numpy(f).cuda()
    tmp = torch.empty_like(a) if pingpong else None
    b = a.clone()
    with bsl.create(w.n, w.lo, w.dx, w.degree) as ctx:
        l0 = ctx.launch_count()
        ctx.strang_step(a, tmp, Ed, w.B, w.dt)
        assert ctx.launch_count() - l0 == 7
        c5 = b.clone()
        ctx.set_fusion(2)
        l0 = ctx.launch_count()
        ctx.strang_step(c5, tmp, Ed, w.B, w.dt)
        assert ctx.launch_count() - l0 == 5
        c3 = b.clone()
        ctx.set_fusion(3)                                         # round 1's two-dim tile passes only
        ctx.strang_step(c3, None, Ed, w.B, w.dt)
        ctx.set_fusion(0)
        l0 = ctx.launch_count()
        ctx.strang_step(b, None, Ed, w.B, w.dt)
        assert ctx.launch_count() - l0 == 12
    assert torch.equal(a, b) and torch.equal(c5, b) and torch.equal(c3, b)
    assert rel_err(a, oracle.strang_step(ogrid(w), w.degree, f.copy(), E, w.B, w.dt)) <= TOL


def test_oblique_B_rotation_in_v_block_passes():
    _need_gpu()
    w = wl.C4.reduced((2, 1, 2, 32, 32, 32))
    f = w.make_f("cpu").numpy()
    B, dt = (0.4, -0.3, 0.6), 0.5
    fd = torch.from_numpy(f).cuda()
    with bsl.create(w.n, w.lo, w.dx, w.degree) as ctx:
        by_policy = ctx.rotate(fd, torch.empty_like(fd), B, dt)
        ctx.set_fusion(2)
        l0 = ctx.launch_count()
        out = ctx.rotate(fd, torch.empty_like(fd), B, dt)
        npass = ctx.launch_count() - l0
        ctx.set_fusion(0)
        single = ctx.rotate(fd, torch.empty_like(fd), B, dt)
    assert npass <= 2, npass                                      # 15 shears: two passes of <= 12 sweeps
    assert torch.equal(out, single) and torch.equal(by_policy, single)
    assert rel_err(out, oracle.rotate(ogrid(w), w.degree, f, B, dt)) <= TOL


def test_full_size_C2_v_block_pass_on_sampled_x_points():
    """32^6 at full size, in the launch configuration bench.py times: the six velocity-space sweeps of the step in
    one pass; the oracle runs the same sweeps on sampled x-points (a v-block never couples different x-points)."""
    _need_gpu(20.0)
    w = wl.C2
    fd = w.make_f("cuda")
    E = w.E()
    Ed = [torch.from_numpy(e).cuda() for e in E]
    th = 0.1
    t, s = math.tan(0.5 * th), math.sin(th)
    v1 = torch.tensor([w.lo[3] + i * w.dx[3] for i in range(w.n[3])], dtype=torch.float64)
    v2 = torch.tensor([w.lo[4] + i * w.dx[4] for i in range(w.n[4])], dtype=torch.float64)
    chain_host = [(3 + d, E[d], 0x7, w.dt / w.dx[3 + d]) for d in range(3)] + \
                 [(3, v2.numpy(), 1 << 4, t / w.dx[3]), (4, v1.numpy(), 1 << 3, -s / w.dx[4]),
                  (3, v2.numpy(), 1 << 4, t / w.dx[3])]
    chain = [(d, torch.from_numpy(np.ascontiguousarray(sr)).cuda(), m, sc) for d, sr, m, sc in chain_host]
    rng = np.random.default_rng(2002)
    xs = rng.integers(0, 32, size=(24, 3))
    xs[0] = (0, 0, 0)
    xs[1] = (31, 31, 31)
    before = np.stack([fd[i, j, k].cpu().numpy() for i, j, k in xs])          # [24][32][32][32]
    with bsl.create(w.n, w.lo, w.dx, w.degree) as ctx:
        ctx.set_fusion(2)
        assert ctx.seq_passes(chain) == 1
        ctx.advect_seq(fd, fd, chain)                                          # in place, one launch
    after = np.stack([fd[i, j, k].cpu().numpy() for i, j, k in xs])
    # oracle on the sampled x-points, as a (24,1,1,32,32,32) grid with the matching E values
    sub = before.reshape(24, 1, 1, 32, 32, 32).copy()
    ref = sub
    for dim, src, mask, scale in chain_host:
        if mask == 0x7:
            src = np.array([src[i, j, k] for i, j, k in xs]).reshape(24, 1, 1)
        ref = oracle.sweep(ref, dim, np.ascontiguousarray(src), mask, scale, w.degree + 1)
    err = np.max(np.abs(after.reshape(ref.shape) - ref)) / np.max(np.abs(ref))
    assert err <= TOL, err
