"""Fused multi-sweep passes (include/bsl6d.h "sequences of sweeps"): a chain of sweeps run
through the planner must give, bit for bit, what the same sweeps give one launch at a time, must agree with the
oracle within 1e-12, and must take the number of passes the header promises."""
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


def ogrid(w):
    return oracle.Grid(tuple(w.n), tuple(w.lo), tuple(w.dx))


def six_sweeps(w, Ed):
    """(dim, src, mask, scale) of x1,x2,x3 (grid nodes) then v1,v2,v3 (E_d over x)."""
    sw = [(d, None, 0, w.dt / w.dx[d]) for d in range(3)]
    sw += [(3 + d, Ed[d], 0x7, w.dt / w.dx[3 + d]) for d in range(3)]
    return sw


def rel_err(gpu: torch.Tensor, ref: np.ndarray) -> float:
    return float(np.max(np.abs(gpu.cpu().numpy() - ref)) / np.max(np.abs(ref)))


# grids whose extents all have fused kernels, for every stencil width; (n, degree, expected passes of the six sweeps)
GRIDS = [
    ((8, 8, 8, 8, 8, 8), 7, 4),           # (x1,x2) (x3,v1) v2 v3
    ((8, 8, 8, 16, 16, 16), 5, 4),        # mixed (8,16) x3-v1 pair
    ((16, 16, 16, 16, 16, 16), 9, 4),
]


@pytest.mark.parametrize("n,degree,npass", GRIDS)
def test_six_sweeps_fused_equals_unfused_and_oracle(n, degree, npass):
    _need_gpu()
    w = wl.C2.reduced(n)
    w = wl.replace(w, degree=degree)
    f = w.make_f("cpu").numpy()
    E = w.E()
    Ed = [torch.from_numpy(e).cuda() for e in E]
    fd = torch.from_numpy(f).cuda()
    with bsl.create(w.n, w.lo, w.dx, w.degree) as ctx:
        sw = six_sweeps(w, Ed)
        assert ctx.seq_passes(sw) == npass
        fused = ctx.advect_seq(fd, torch.empty_like(fd), sw)
        l_fused = ctx.launch_count()
        assert l_fused == npass
        assert ctx.set_fusion(False) == 1
        assert ctx.seq_passes(sw) == 6
        plain = ctx.advect_seq(fd, torch.empty_like(fd), sw)
        assert ctx.launch_count() - l_fused == 6
        inplace = fd.clone()
        ctx.set_fusion(True)
        ctx.advect_seq(inplace, inplace, sw)                 # fused passes in place
    assert torch.equal(fused, plain)
    assert torch.equal(fused, inplace)
    ref = f
    for d in range(6):
        ref = oracle.advect(ogrid(w), w.degree, ref, d, None if d < 3 else E[d - 3], w.dt)
    assert rel_err(fused, ref) <= TOL


@pytest.mark.parametrize("n,degree", [((2, 3, 2, 8, 8, 8), 7), ((2, 2, 2, 16, 16, 16), 5), ((1, 2, 1, 32, 32, 32), 7),
                                      ((1, 1, 2, 48, 48, 8), 9), ((1, 1, 1, 64, 64, 16), 5)])
def test_rotation_fused_equals_unfused_and_oracle(n, degree):
    """B along x3: the three shears v1, v2, v1 are one ABA pass; |alpha| reaches 1.6 cells (k != 0)."""
    _need_gpu()
    w = wl.C4.reduced(n)
    w = wl.replace(w, degree=degree)
    f = w.make_f("cpu").numpy()
    fd = torch.from_numpy(f).cuda()
    B, dt = (0.0, 0.0, 1.0), 0.1
    with bsl.create(w.n, w.lo, w.dx, w.degree) as ctx:
        fused = ctx.rotate(fd, torch.empty_like(fd), B, dt)
        assert ctx.launch_count() == 1
        ctx.set_fusion(False)
        plain = ctx.rotate(fd, torch.empty_like(fd), B, dt)
        assert ctx.launch_count() == 4
        ctx.set_fusion(True)
        inplace = fd.clone()
        ctx.rotate(inplace, inplace, B, -dt)                 # negative angle, in place
        ctx.set_fusion(False)
        plain_neg = ctx.rotate(fd, torch.empty_like(fd), B, -dt)
    assert torch.equal(fused, plain)
    assert torch.equal(inplace, plain_neg)
    assert rel_err(fused, oracle.rotate(ogrid(w), w.degree, f, B, dt)) <= TOL


def test_rotation_other_axes_fall_back_to_single_sweeps():
    """B along x1 / x2 involves the unit-stride dim v3: no fused kernel, three launches, same numbers as before."""
    _need_gpu()
    w = wl.C4.reduced((2, 2, 2, 16, 16, 16))
    f = w.make_f("cpu").numpy()
    fd = torch.from_numpy(f).cuda()
    with bsl.create(w.n, w.lo, w.dx, w.degree) as ctx:
        for ax in (0, 1):
            B = [0.0, 0.0, 0.0]
            B[ax] = 1.0
            before = ctx.launch_count()
            out = ctx.rotate(fd, torch.empty_like(fd), B, 0.1)
            assert ctx.launch_count() - before == 3
            assert rel_err(out, oracle.rotate(ogrid(w), w.degree, f, B, 0.1)) <= TOL


@pytest.mark.parametrize("pingpong", (False, True))
def test_strang_step_fused_equals_unfused_and_oracle(pingpong):
    _need_gpu()
    w = wl.C5.reduced((8, 8, 8, 16, 16, 16))
    f = w.make_f("cpu").numpy()
    E = w.E()
    Ed = [torch.from_numpy(e).cuda() for e in E]
    a = torch.from_numpy(f).cuda()
    b = a.clone()
    tmp = torch.empty_like(a) if pingpong else None
    with bsl.create(w.n, w.lo, w.dx, w.degree) as ctx:
        for _ in range(2):
            ctx.strang_step(a, tmp, Ed, w.B, w.dt)
        # (x1,x2) (x3,v1) v2 v3 (v1,v2,v1) (x1,x2) x3 = 7 passes per step
        assert ctx.launch_count() == 14
        ctx.set_fusion(False)
        for _ in range(2):
            ctx.strang_step(b, tmp, Ed, w.B, w.dt)
        assert ctx.launch_count() == 14 + 24
    assert torch.equal(a, b)
    ref = f.copy()
    for _ in range(2):
        ref = oracle.strang_step(ogrid(w), w.degree, ref, E, w.B, w.dt)
    assert rel_err(a, ref) <= TOL


def test_integer_shifts_stay_bit_exact_through_fused_passes():
    """Whole-cell displacements in both sweeps of a fused pair: the pass is an exact permutation (x, periodic)
    followed by an exact shift with zero fill (v)."""
    _need_gpu()
    w = wl.C2.reduced((8, 8, 8, 8, 8, 8))
    f = w.make_f("cpu").numpy()
    fd = torch.from_numpy(f).cuda()
    one = torch.ones(1, dtype=torch.float64, device="cuda")
    with bsl.create(w.n, w.lo, w.dx, w.degree) as ctx:
        sw = [(0, one, 0, 3.0), (1, one, 0, -2.0), (2, one, 0, 1.0), (3, one, 0, 2.0)]   # alpha = -3, +2, -1, -2 cells
        assert ctx.seq_passes(sw) == 2
        out = ctx.advect_seq(fd, torch.empty_like(fd), sw).cpu().numpy()
    ref = np.roll(np.roll(np.roll(f, 3, axis=0), -2, axis=1), 1, axis=2)
    exp = np.zeros_like(ref)
    exp[:, :, :, 2:] = ref[:, :, :, :-2]                     # out[j] = in[j-2], zero fill
    assert np.array_equal(out, exp)


def test_sequence_error_paths_enqueue_nothing():
    _need_gpu()
    w = wl.C1
    fd = w.make_f("cuda")
    one = torch.ones(w.n[1], dtype=torch.float64, device="cuda")   # sized for the mask, so the C check is what fires
    with bsl.create(w.n, w.lo, w.dx, w.degree) as ctx:
        with pytest.raises(bsl.Bsl6dError) as e:
            ctx.advect_seq(fd, fd, [(0, None, 0, 0.1), (3, None, 0x7, 0.1)])   # v sweep without a source
        assert e.value.code == bsl.EINVAL
        with pytest.raises(bsl.Bsl6dError) as e:
            ctx.advect_seq(fd, fd, [(0, None, 0, 0.1), (1, one, 1 << 1, 0.1)])  # mask contains the swept dim
        assert e.value.code == bsl.EINVAL
        with pytest.raises(bsl.Bsl6dError):
            ctx.advect_seq(fd, fd, [(0, None, 0, float("inf"))])
        assert ctx.launch_count() == 0
        out = ctx.advect_seq(fd, torch.empty_like(fd), [])   # empty chain copies
        assert torch.equal(out, fd)


@pytest.mark.parametrize("B,dt", [((0.4, -0.3, 0.6), 0.5), ((1.0, 1.0, 0.0), 0.4), ((0.0, 1.0, 1.0), 2.5),
                                  ((-2.0, 0.1, -1.0), 0.9)])
def test_oblique_B_rotation_matches_oracle(B, dt):
    """B in general position = five axis rotations of three shears each (same plan as the oracle);
    the Rz factors run as fused passes.  GPU == oracle within 1e-12, fused == unfused bit for bit."""
    _need_gpu()
    w = wl.C4.reduced((2, 1, 2, 16, 16, 16))
    f = w.make_f("cpu").numpy()
    fd = torch.from_numpy(f).cuda()
    nrot = len(oracle.rotation_plan(B, dt))
    with bsl.create(w.n, w.lo, w.dx, w.degree) as ctx:
        fused = ctx.rotate(fd, torch.empty_like(fd), B, dt)
        nfused = ctx.launch_count()
        ctx.set_fusion(0)
        plain = ctx.rotate(fd, torch.empty_like(fd), B, dt)
        assert ctx.launch_count() - nfused == 3 * nrot
        assert nfused < 3 * nrot
        inplace = fd.clone()
        ctx.rotate(inplace, inplace, B, dt)
    assert torch.equal(fused, plain) and torch.equal(inplace, plain)
    assert rel_err(fused, oracle.rotate(ogrid(w), w.degree, f, B, dt)) <= TOL


def test_strang_step_is_capturable_in_a_cuda_graph():
    """Every entry point only enqueues work on the caller's stream (no allocation, no synchronisation in steady state),
    so a launch-bound loop of small steps can be captured once and replayed as a CUDA graph (C1 is 2 MiB: L2-resident,
    launch-latency-bound).  Replays must reproduce eager execution bit for bit -- persistent TMA-fed passes included."""
    _need_gpu()
    w = wl.C2.reduced((8, 8, 8, 16, 16, 16))
    f0 = w.make_f("cuda")
    Ed = [torch.from_numpy(e).cuda() for e in w.E()]
    with bsl.create(w.n, w.lo, w.dx, w.degree) as ctx:
        eager = f0.clone()
        tmp = torch.empty_like(eager)
        for _ in range(4):
            ctx.strang_step(eager, tmp, Ed, w.B if any(w.B) else (0.0, 0.0, 1.0), w.dt)
        g_f = f0.clone()
        g_tmp = torch.empty_like(g_f)
        B = w.B if any(w.B) else (0.0, 0.0, 1.0)
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):                           # warm-up on the capture stream (first-use attributes)
            ctx.strang_step(g_f, g_tmp, Ed, B, w.dt, stream=side)
        torch.cuda.current_stream().wait_stream(side)
        torch.cuda.synchronize()
        g_f.copy_(f0)
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph):
            ctx.strang_step(g_f, g_tmp, Ed, B, w.dt, stream=torch.cuda.current_stream())
        g_f.copy_(f0)
        for _ in range(4):
            graph.replay()
        torch.cuda.synchronize()
    assert torch.equal(g_f, eager)


@pytest.mark.parametrize("n,degree,seed", [((8, 8, 8, 8, 8, 8), 7, 1), ((4, 16, 16, 16, 16, 16), 5, 2),
                                            ((2, 2, 32, 32, 32, 32), 9, 3), ((3, 32, 32, 32, 32, 8), 7, 4)])
def test_random_chains_every_planner_mode_equals_single_sweeps(n, degree, seed):
    """Random chains of sweeps (any order of dims, repeats, sources over random subsets of the other dims, displacements
    of up to ~2.5 cells): whatever grouping the planner picks in modes 1-4 -- persistent tile passes with chains like
    b,a,b,a, v-block passes with re-tiling, round-1 pairs and triples -- the result equals the sweeps launched one by
    one, bit for bit, in place and out of place; and the first chain also agrees with the oracle."""
    _need_gpu()
    rng = np.random.default_rng(seed)
    w = wl.replace(wl.C5.reduced(n), degree=degree)
    f = w.make_f("cpu").numpy()
    fd = torch.from_numpy(f).cuda()
    with bsl.create(w.n, w.lo, w.dx, w.degree) as ctx:
        for trial in range(6):
            ns = int(rng.integers(2, 11))
            chain_host = []
            dims = rng.integers(0, 6, size=ns) if trial % 2 else rng.choice([3, 4, 5, 3, 4, 2], size=ns)
            for d in dims:
                others = [k for k in range(6) if k != d]
                mask = 0
                for k in rng.choice(others, size=int(rng.integers(0, 3)), replace=False):
                    mask |= 1 << int(k)
                shape = [w.n[k] for k in range(6) if mask >> k & 1]
                src = 2.5 * (2.0 * rng.random(shape if shape else (1,)) - 1.0)
                chain_host.append((int(d), src, mask, 1.0))
            chain = [(d, torch.from_numpy(np.ascontiguousarray(s)).cuda(), m, sc) for d, s, m, sc in chain_host]
            ctx.set_fusion(0)
            single = ctx.advect_seq(fd, torch.empty_like(fd), chain)
            for mode in (1, 2, 3, 4, 5):
                ctx.set_fusion(mode)
                npass = ctx.seq_passes(chain)
                assert 1 <= npass <= ns
                out = ctx.advect_seq(fd, torch.empty_like(fd), chain)
                assert torch.equal(out, single), (trial, mode, [c[0] for c in chain_host])
                inp = fd.clone()
                ctx.advect_seq(inp, inp, chain)
                assert torch.equal(inp, single), (trial, mode, "in place")
            if trial == 0:
                ref = f
                for d, s, m, sc in chain_host:
                    ref = oracle.sweep(ref, d, np.ascontiguousarray(s), m, sc, w.degree + 1)
                assert rel_err(single, ref) <= TOL


@pytest.mark.parametrize("n,degree", [((4, 8, 8, 32, 32, 8), 7), ((2, 16, 16, 16, 16, 16), 5), ((2, 8, 32, 32, 8, 8), 9)])
def test_tile_passes_with_displacements_of_many_cells(n, degree):
    """Chains over two dims with |alpha| up to 11 cells, both signs, varying per pencil: the persistent tile pass takes
    its streaming form for some pencils (first stencil row above -q) and the all-loads-first form for the others in the
    same warp; zero-extended and periodic dims.  Bit-identical to the sweeps one by one, in and out of place."""
    _need_gpu()
    w = wl.replace(wl.C2.reduced(n), degree=degree)
    rng = np.random.default_rng(sum(n) + degree)
    fd = w.make_f("cuda")
    for a, b in ((3, 4), (2, 3), (1, 2)):
        chain = []
        for d in (a, b, a, b):
            mask = sum(1 << k for k in range(6) if k not in (d,) and k in (a, b, 0, 5))
            shape = [w.n[k] for k in range(6) if mask >> k & 1]
            src = torch.from_numpy(11.0 * (2.0 * rng.random(shape) - 1.0)).cuda()
            chain.append((d, src, mask, 1.0))
        with bsl.create(w.n, w.lo, w.dx, w.degree) as ctx:
            ctx.set_fusion(0)
            single = ctx.advect_seq(fd, torch.empty_like(fd), chain)
            for mode in (1, 2, 5):
                ctx.set_fusion(mode)
                assert torch.equal(ctx.advect_seq(fd, torch.empty_like(fd), chain), single), (a, b, mode)
                inp = fd.clone()
                ctx.advect_seq(inp, inp, chain)
                assert torch.equal(inp, single), (a, b, mode, "in place")


@pytest.mark.parametrize("n,degree", [((8, 8, 8, 16, 16, 16), 7), ((4, 4, 4, 32, 32, 32), 9)])
def test_arrays_on_8_byte_boundaries_run_without_tma_passes(n, degree):
    """include/bsl6d.h allows f on an 8-byte boundary; a TMA tensor map needs 16.  The planner must then keep the
    persistent-tile and v-block passes out of the plan instead of failing half way through a step: a Strang step, a
    rotation and a chain on arrays offset by one double give, bit for bit, what the 16-byte aligned arrays give."""
    _need_gpu()
    w = wl.replace(wl.C5.reduced(n), degree=degree)
    f = w.make_f("cuda")
    Ed = [torch.from_numpy(e).cuda() for e in w.E()]
    B = (0.0, 0.0, 1.0)

    def odd(t=None):
        """A copy of t (or an empty array of f's size) that starts one double past a 16-byte boundary."""
        raw = torch.empty(f.numel() + 3, dtype=torch.float64, device="cuda")
        off = 1 if raw.data_ptr() % 16 == 0 else 2
        v = raw[off:off + f.numel()].view(f.shape)
        assert v.data_ptr() % 16 == 8
        if t is not None:
            v.copy_(t)
        return v

    with bsl.create(w.n, w.lo, w.dx, w.degree) as ctx:
        sw = six_sweeps(w, Ed)
        want_step = ctx.strang_step(f.clone(), torch.empty_like(f), Ed, B, w.dt)
        want_rot = ctx.rotate(f, torch.empty_like(f), B, w.dt)
        want_seq = ctx.advect_seq(f, torch.empty_like(f), sw)
        torch.cuda.synchronize()
        got = odd(f)
        ctx.strang_step(got, odd(), Ed, B, w.dt)               # both arrays misaligned, ping-pong
        assert torch.equal(got, want_step)
        got = odd(f)
        ctx.strang_step(got, None, Ed, B, w.dt)                # in place
        assert torch.equal(got, want_step)
        got = f.clone()
        ctx.strang_step(got, odd(), Ed, B, w.dt)               # only the second array misaligned
        assert torch.equal(got, want_step)
        assert torch.equal(ctx.rotate(odd(f), odd(), B, w.dt), want_rot)
        assert torch.equal(ctx.rotate(f, odd(), B, w.dt), want_rot)
        assert torch.equal(ctx.advect_seq(odd(f), odd(), sw), want_seq)
        got = odd(f)
        assert torch.equal(ctx.advect_seq(got, got, sw), want_seq)
