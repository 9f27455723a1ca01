"""Parity of the CUDA path (through the C ABI, via the ctypes binding) against the CPU oracle.

Tolerance (BASELINE.json north_star): bit-exact when every displacement is a whole number of cells,
max|gpu - oracle| <= 1e-12 * max|oracle| otherwise.  All inputs are seeded and synthetic (bsl6d_workloads).
Run on the B200 box:  python -m pytest tests -m gpu
"""
import math

import numpy as np
import pytest
import torch

import bsl6d_workloads as wl
import oracle
import paper_2303_05994_b200 as bsl

pytestmark = pytest.mark.gpu

RTOL = 1e-12


def _need_gpu():
    assert torch.cuda.is_available(), "GPU tests selected but no CUDA device is visible"
    bsl.load_library()


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def assert_close(gpu, ref, what=""):
    gpu = gpu.cpu().numpy() if isinstance(gpu, torch.Tensor) else gpu
    scale = np.max(np.abs(ref))
    err = np.max(np.abs(gpu.reshape(ref.shape) - ref))
    assert err <= RTOL * scale, f"{what}: max|diff| {err:.3e} > {RTOL:g} * {scale:.3e}"
    return err / max(scale, 1e-300)


def ctx_for(w):
    return bsl.create(w.n, w.lo, w.dx, w.degree)


def ogrid(w):
    return oracle.Grid(tuple(w.n), tuple(w.lo), tuple(w.dx))


def mini(n, degree, Lx=4 * math.pi, vmax=6.0, seed=7, kind="maxwell_xyz"):
    return wl._mk("mini", n, Lx, vmax, degree=degree, dt=0.05, seed=seed, noise_amp=1e-3, kind=kind)


# ------------------------------------------------------------------------------------------------
# config 1 (BASELINE.json configs[0]) -- whole grid, element by element
# ------------------------------------------------------------------------------------------------
def test_C1_x1_sweep_and_integer_shifts():
    _need_gpu()
    w = wl.C1
    f = w.make_f("cpu").numpy()
    fd = dev(f)
    with ctx_for(w) as ctx:
        assert ctx.kernel_name(0).startswith("strided<N=8,Q=8,periodic")
        out = torch.empty_like(fd)
        ctx.advect(fd, out, 0, None, w.dt)
        assert_close(out, oracle.advect(ogrid(w), w.degree, f, 0, None, w.dt), "C1 x1")
        # integer case (i): every pencil rolled by exactly one cell (reading S10)
        one = dev(np.array([1.0]))
        for dim in range(6):
            ctx.advect_generic(fd, out, dim, one, 0, 1.0)
            ref = oracle.sweep(f, dim, np.array([1.0]), 0, 1.0, w.q)
            assert np.array_equal(out.cpu().numpy(), ref), f"unit roll dim {dim}"
            if dim < 3:
                assert np.array_equal(ref, np.roll(f, 1, axis=dim))
        # integer case (ii): dt = 2*dx1 -> alpha = -2 v_j, k in {12, 9, .., -9}
        dt = 2.0 * w.dx[0]
        ctx.advect(fd, out, 0, None, dt)
        assert np.array_equal(out.cpu().numpy(), oracle.advect(ogrid(w), w.degree, f, 0, None, dt))
        assert ctx.launch_count() == 8


def test_C1_all_six_sweeps_sequence():
    _need_gpu()
    w = wl.C1
    f = w.make_f("cpu").numpy()
    E = w.E()
    cur = dev(f)
    ref = f.copy()
    with ctx_for(w) as ctx:
        for d in range(3):
            ctx.advect(cur, cur, d, None, w.dt)
            ref = oracle.advect(ogrid(w), w.degree, ref, d, None, w.dt)
        for d in range(3):
            ctx.advect(cur, cur, 3 + d, dev(E[d]), w.dt)
            ref = oracle.advect(ogrid(w), w.degree, ref, 3 + d, E[d], w.dt)
        assert_close(cur, ref, "C1 six sweeps")


def test_workload_generator_cpu_equals_cuda():
    _need_gpu()
    for w in (wl.C1, wl.C3.reduced((4, 4, 4, 16, 16, 16)), wl.C4.reduced((8, 8, 8, 8, 8, 8))):
        assert torch.equal(w.make_f("cuda").cpu(), w.make_f("cpu"))


# ------------------------------------------------------------------------------------------------
# every specialised kernel and the fallback, on grids small enough for the oracle, spanning several
# tiles and ragged tails; displacements of several cells, both signs, varying per lane
# ------------------------------------------------------------------------------------------------
GRIDS = [
    # (extents, degree)  -- kernels exercised
    ((32, 8, 16, 32, 8, 32), 7),      # C2/C4-like: strided<32,8> periodic+zero, unit<32,8>, strided<8>, <16>
    ((48, 4, 8, 8, 48, 48), 9),       # C5-like: strided<48,10> periodic+zero, unit<48,10>; n=4 < q -> generic
    ((16, 16, 8, 64, 8, 64), 5),      # C3-like: strided<64,6> zero, unit<64,6>, strided<16,6> periodic
    ((64, 8, 8, 8, 64, 8), 7),        # strided<64,8> periodic + zero, unit<8,8>
    ((5, 7, 9, 11, 13, 6), 3),        # ragged: strided generic + unit generic, q=4
    ((9, 3, 12, 6, 10, 14), 11),      # q=12 has no specialised instance -> generic everywhere
    ((8, 16, 32, 16, 32, 16), 3),     # q=4 instances
    ((3, 2, 2, 2, 3, 200), 7),        # long unit-stride pencils (fallback), tiny everything else
    ((5, 3, 9, 1, 1, 1), 3),          # degenerate: x3 is periodic AND unit-stride (inner == 1) -> strided fallback
    ((1, 1, 1, 7, 5, 11), 5),         # no x extent at all
    ((13, 1, 1, 21, 1, 1), 1),        # 1D1V, linear interpolation (q = 2)
    ((2, 1, 37, 1, 1, 40), 7),        # the paper's extent 37 (periodic, inner = 40) + unit-stride fallback (40)
    ((37, 2, 2, 37, 2, 37), 7),       # strided<37,8> periodic + zero with flattened pencil indexing, unit<37,8>
    ((3, 37, 37, 37, 37, 37), 9),     # strided<37,10> on inner extents 37^k (no multiple of the warp width), unit<37,10>
    ((36, 3, 2, 36, 2, 36), 5),       # extent 36: no specialised instance -> generic strided + generic unit, q = 6
    ((64, 2, 48, 4, 4, 8), 9),        # long periodic pencils: out of place = sweep_stream_kernel<64,10>, <48,10>; in place = strided
    ((48, 3, 5, 2, 3, 7), 5),         # sweep_stream_kernel<48,6> with a ragged inner extent (flattened pencil index)
    ((5, 64, 3, 3, 1, 2), 3),         # sweep_stream_kernel<64,4>, inner = 18
]


@pytest.mark.parametrize("n,degree", GRIDS)
def test_sweeps_every_dim_every_kernel(n, degree):
    _need_gpu()
    w = mini(n, degree, seed=sum(n))
    q = w.q
    f = w.make_f("cpu").numpy()
    fd = dev(f)
    rng = np.random.default_rng(sum(n) + degree)
    with ctx_for(w) as ctx:
        out = torch.empty_like(fd)
        for dim in range(6):
            others = [d for d in range(6) if d != dim]
            masks = [[(dim + 3) % 6], others, [d for d in (0, 2, 5) if d != dim], [d for d in (1, 3, 4) if d != dim]]
            for mi, md in enumerate(masks):
                mask = sum(1 << d for d in md)
                src = rng.uniform(-1.0, 1.0, size=[n[d] for d in sorted(md)])
                scale = (0.7, 3.3, 11.0, 0.05)[mi]          # sub-cell ... many cells
                ctx.advect_generic(fd, out, dim, dev(src), mask, scale)
                ref = oracle.sweep(f, dim, src, mask, scale, q)
                assert_close(out, ref, f"n={n} q={q} dim={dim} mask={md} kernel={ctx.kernel_name(dim)}")
            # in place == out of place, bit for bit
            g = fd.clone()
            ctx.advect_generic(g, g, dim, dev(src), mask, scale)
            assert torch.equal(g, out), f"in-place differs, dim {dim}"


@pytest.mark.parametrize("n,degree", [((32, 4, 4, 32, 4, 32), 7), ((6, 48, 6, 48, 6, 48), 9), ((4, 4, 64, 4, 64, 64), 5)])
def test_integer_shifts_bit_exact_all_kernels(n, degree):
    """Whole-cell displacements (per-pencil different, up to +-(n+3) cells) are exact permutations."""
    _need_gpu()
    w = mini(n, degree, seed=3)
    f = w.make_f("cpu").numpy()
    fd = dev(f)
    rng = np.random.default_rng(5)
    with ctx_for(w) as ctx:
        out = torch.empty_like(fd)
        for dim in range(6):
            md = [d for d in range(6) if d != dim]
            src = rng.integers(-n[dim] - 3, n[dim] + 4, size=[n[d] for d in md]).astype(np.float64)
            ctx.advect_generic(fd, out, dim, dev(src), sum(1 << d for d in md), 1.0)
            ref = oracle.sweep(f, dim, src, sum(1 << d for d in md), 1.0, w.q)
            assert np.array_equal(out.cpu().numpy(), ref), (n, dim, ctx.kernel_name(dim))


def test_theta_rounds_to_one_and_tiny_shifts():
    """Reading S4: alpha = -tiny gives k = -1, theta = 1.0 exactly; the result must still be f itself."""
    _need_gpu()
    w = mini((8, 8, 8, 16, 16, 32), 7)
    f = w.make_f("cpu").numpy()
    fd = dev(f)
    with ctx_for(w) as ctx:
        out = torch.empty_like(fd)
        for dim in (0, 3, 5):
            for a in (1e-30, -1e-30, 1e-17, -1e-17, 0.0, -0.0):
                s = np.array([a])
                ctx.advect_generic(fd, out, dim, dev(s), 0, 1.0)
                ref = oracle.sweep(f, dim, s, 0, 1.0, w.q)
                if a >= 0.0 or a == -1e-30:
                    # alpha = -a: theta is exactly 0 or rounds to exactly 1 -> unit weights -> f itself, bit for bit
                    # (alpha = +1e-30 has theta = 1e-30: every tap but one is below half an ulp of f)
                    assert np.array_equal(out.cpu().numpy(), ref)
                    assert np.array_equal(ref, f)
                else:
                    # alpha = +1e-17: a genuine sub-cell shift; results move by at most an ulp
                    assert_close(out, ref, "tiny shift")
                    assert np.max(np.abs(ref - f)) <= 1e-15 * np.max(np.abs(f))


# ------------------------------------------------------------------------------------------------
# reduced copies of configs 2-5: the named sweeps, rotation, Strang steps, density
# ------------------------------------------------------------------------------------------------
def test_C2_reduced_six_sweeps():
    _need_gpu()
    w = wl.C2.reduced((16,) * 6)
    f = w.make_f("cpu").numpy()
    E = w.E()
    cur, ref = dev(f), f.copy()
    tmp = torch.empty_like(cur)
    with ctx_for(w) as ctx:
        for d in range(6):
            ss = None if d < 3 else E[d - 3]
            ctx.advect(cur, tmp, d, None if ss is None else dev(ss), w.dt)
            cur, tmp = tmp, cur
            ref = oracle.advect(ogrid(w), w.degree, ref, d, ss, w.dt)
            assert_close(cur, ref, f"C2r after sweep {d}")


def test_C3_reduced_six_sweeps_k_nonzero():
    _need_gpu()
    w = wl.C3.reduced((16, 8, 8, 64, 16, 64))            # keeps dx1 and dv1: |alpha| = 1.0186 at v1 = -8
    assert abs(8.0 * w.dt / w.dx[0]) > 1.0
    f = w.make_f("cpu").numpy()
    E = w.E()
    cur, ref = dev(f), f.copy()
    with ctx_for(w) as ctx:
        for d in range(6):
            ss = None if d < 3 else E[d - 3]
            ctx.advect(cur, cur, d, None if ss is None else dev(ss), w.dt)
            ref = oracle.advect(ogrid(w), w.degree, ref, d, ss, w.dt)
        assert_close(cur, ref, "C3r six sweeps")


@pytest.mark.parametrize("axis", (0, 1, 2))
def test_rotation_each_axis(axis):
    _need_gpu()
    w = wl.C4.reduced((4, 6, 4, 32, 32, 32))
    f = w.make_f("cpu").numpy()
    B = [0.0, 0.0, 0.0]
    B[axis] = -1.3
    with ctx_for(w) as ctx:
        out = torch.empty_like(dev(f))
        ctx.rotate(dev(f), out, B, 0.4)
        assert_close(out, oracle.rotate(ogrid(w), w.degree, f, B, 0.4), f"rotate axis {axis}")
        g = dev(f)
        ctx.rotate(g, g, B, 0.4)
        assert torch.equal(g, out)
        z = torch.empty_like(g)
        ctx.rotate(g, z, [0.0, 0.0, 0.0], 0.4)               # B = 0: copy
        assert torch.equal(z, g)


@pytest.mark.parametrize("axis", (0, 1, 2))
@pytest.mark.parametrize("theta", (3.0, -2.0, 6.2))
def test_rotation_large_angle_each_axis(axis, theta):
    """Reading R2: an axis rotation above pi/2 runs in equal pieces (the library and the oracle plan it alike);
    more than a full turn is BSL6D_EUNSUPPORTED."""
    _need_gpu()
    w = wl.C4.reduced((2, 3, 2, 32, 32, 32))
    f = w.make_f("cpu").numpy()
    B = [0.0, 0.0, 0.0]
    B[axis] = theta / 0.5
    with ctx_for(w) as ctx:
        out = torch.empty_like(dev(f))
        ctx.rotate(dev(f), out, B, 0.5)
        assert_close(out, oracle.rotate(ogrid(w), w.degree, f, B, 0.5), f"rotate axis {axis} by {theta}")
        assert float(out.abs().max()) > 0.05                  # not shorn off the grid
        ctx.set_fusion(0)
        out2 = torch.empty_like(out)
        ctx.rotate(dev(f), out2, B, 0.5)
        assert torch.equal(out, out2)
        B[axis] = 13.0
        with pytest.raises(bsl.Bsl6dError) as ei:
            ctx.rotate(dev(f), out, B, 0.5)
        assert ei.value.code == bsl.EUNSUPPORTED


def test_binding_checks_counts_and_device():
    """api.py validates what the C ABI cannot see: element counts of every tensor argument."""
    _need_gpu()
    w = wl.C1
    f = dev(w.make_f("cpu").numpy())
    out = torch.empty_like(f)
    nx = w.n[0] * w.n[1] * w.n[2]
    good_E = [torch.zeros(nx, dtype=torch.float64, device="cuda") for _ in range(3)]
    bad = torch.zeros(nx - 1, dtype=torch.float64, device="cuda")
    with ctx_for(w) as ctx:
        with pytest.raises(ValueError):
            ctx.advect(f, out, 0, bad, 0.1)                  # x sweep wants n[3] values
        with pytest.raises(ValueError):
            ctx.advect(f, out, 3, bad, 0.1)                  # v sweep wants nx values
        with pytest.raises(ValueError):
            ctx.strang_step(f, out[..., :-1].contiguous(), good_E, None, 0.1)
        with pytest.raises(ValueError):
            ctx.strang_step(f, None, [good_E[0], bad, good_E[2]], None, 0.1)
        with pytest.raises(ValueError):
            ctx.advect_seq(f, out, [(3, bad, 0x7, 1.0)])
        with pytest.raises(ValueError):
            ctx.density(f, bad)
        with pytest.raises(ValueError):
            ctx.field_poisson(bad, 1.0, 1.0, good_E)
        ctx.advect(f, out, 3, good_E[0], 0.1)                # and the well-formed call still goes through


def test_C4_reduced_rotation_return_63_steps():
    """configs[3] at reduced x extent, full depth: 63 steps of theta = 2*pi/63 (reading S7), GPU == oracle
    after all 189 sweeps, and both return to the start within interpolation error."""
    _need_gpu()
    w = wl.C4.reduced((2, 4, 2, 32, 32, 32))
    f0 = w.make_f("cpu", noise=False).numpy()
    theta = 2 * math.pi / 63
    cur, ref = dev(f0), f0.copy()
    with ctx_for(w) as ctx:
        for _ in range(63):
            ctx.rotate(cur, cur, w.B, theta)
            ref = oracle.rotate(ogrid(w), w.degree, ref, w.B, theta)
        rel = assert_close(cur, ref, "C4r 63 rotations")
        assert ctx.launch_count() in (63, 189)                # one fused pass per rotation, or three sweeps
    back = np.max(np.abs(ref - f0)) / np.max(np.abs(f0))
    assert back < 0.06, back                                  # under-resolved on purpose (sigma_v2 = 0.5, dv = 0.375)
    print(f"C4r: gpu-vs-oracle {rel:.2e}, return error {back:.3e}")


@pytest.mark.parametrize("pingpong", (False, True))
def test_C5_reduced_strang_steps_and_density(pingpong):
    _need_gpu()
    w = wl.C5.reduced((12, 12, 12, 16, 16, 16))
    f = w.make_f("cpu").numpy()
    E = w.E()
    cur, ref = dev(f), f.copy()
    tmp = torch.empty_like(cur) if pingpong else None
    Ed = [dev(e) for e in E]
    rho = torch.empty(w.n[:3], dtype=torch.float64, device="cuda")
    with ctx_for(w) as ctx:
        for step in range(3):
            ctx.strang_step(cur, tmp, Ed, w.B, w.dt)
            ref = oracle.strang_step(ogrid(w), w.degree, ref, E, w.B, w.dt)
            assert_close(cur, ref, f"C5r step {step}")
            ctx.density(cur, rho)
            assert_close(rho, oracle.density(ogrid(w), ref), f"C5r rho step {step}")
        assert ctx.launch_count() in (3 * 10, 3 * 13)         # fused v1v2 + fused shears, or 12 sweeps; + density
        # no E, no B: 6 sweeps; E only: 9 sweeps (odd count with ping-pong still lands in f)
        before = ctx.launch_count()
        ctx.strang_step(cur, tmp, None, None, w.dt)
        ref = oracle.strang_step(ogrid(w), w.degree, ref, [None] * 3, None, w.dt)
        ctx.strang_step(cur, tmp, Ed, None, w.dt)
        ref = oracle.strang_step(ogrid(w), w.degree, ref, E, None, w.dt)
        assert ctx.launch_count() - before in (14, 15)
        assert_close(cur, ref, "C5r partial steps")


@pytest.mark.parametrize("n", [(3, 2, 4, 5, 6, 7), (2, 2, 2, 64, 32, 32), (4, 4, 4, 8, 8, 8), (2, 3, 2, 31, 33, 35),
                               (16, 2, 2, 32, 32, 32)])
def test_density(n):
    _need_gpu()
    w = mini(n, 7, seed=11, kind="maxwell_x1")
    f = w.make_f("cpu").numpy()
    rho = torch.empty(n[:3], dtype=torch.float64, device="cuda")
    with ctx_for(w) as ctx:
        ctx.density(dev(f), rho)
        r1 = rho.clone()
        ctx.density(dev(f), rho)
    assert torch.equal(r1, rho)                               # deterministic
    ref = oracle.density(ogrid(w), f)
    # fp64 tree sum vs long-double reference: error <= log2(S) ulp of sum|f|
    assert np.max(np.abs(rho.cpu().numpy() - ref)) <= 1e-14 * np.max(np.abs(ref))
    if n == (16, 2, 2, 32, 32, 32):
        # closed form on the noise-free f: trapezoid sum of a Maxwellian on [-6,6)^3 is 1 to ~1e-8
        f0 = w.make_f("cpu", noise=False).numpy()
        with ctx_for(w) as ctx:
            ctx.density(dev(f0), rho)
        x1 = w.nodes(0)
        assert np.max(np.abs(rho.cpu().numpy()[:, 0, 0] - (1 + 0.01 * np.cos(0.5 * x1)))) < 1e-7


def test_run_host_matches_device_path():
    _need_gpu()
    w = wl.C5.reduced((8, 8, 8, 16, 16, 16))
    f = w.make_f("cpu")
    E = [torch.from_numpy(e) for e in w.E()]
    ops = [dict(kind="advect", dim=d, dt=0.5 * w.dt) for d in range(3)]
    ops += [dict(kind="advect", dim=3 + d, dt=w.dt, shift_source=E[d]) for d in range(3)]
    ops += [dict(kind="rotate", B=w.B, dt=w.dt)]
    ops += [dict(kind="advect", dim=d, dt=0.5 * w.dt) for d in range(3)]
    rho_h = torch.empty(w.n[:3], dtype=torch.float64)
    ops += [dict(kind="density", rho_host=rho_h)]
    out_h = torch.empty_like(f)
    with ctx_for(w) as ctx:
        ctx.run_host(f.pin_memory(), out_h, ops)
        g = f.cuda()
        ctx.strang_step(g, None, [e.cuda() for e in E], w.B, w.dt)
        rho = torch.empty(w.n[:3], dtype=torch.float64, device="cuda")
        ctx.density(g, rho)
        torch.cuda.synchronize()
    assert torch.equal(out_h, g.cpu()) and torch.equal(rho_h, rho.cpu())
    ref = oracle.strang_step(ogrid(w), w.degree, f.numpy().copy(), w.E(), w.B, w.dt)
    assert_close(out_h.numpy(), ref, "run_host strang")
    # two problems in flight (bsl6d_run_host_begin / _end on slots 0 and 1, then a third queued behind slot 0):
    # the same numbers as one after the other
    ins = [f.pin_memory(), (f * 0.5 + 0.01).pin_memory(), (f * 2.0).pin_memory()]
    outs = [torch.empty_like(f).pin_memory() for _ in ins]
    rhos = [torch.empty(w.n[:3], dtype=torch.float64).pin_memory() for _ in ins]
    with ctx_for(w) as ctx:
        for k in range(3):
            ctx.run_host_begin(ins[k], outs[k], ops[:-1] + [dict(kind="density", rho_host=rhos[k])], k % 2)
        ctx.run_host_end(0)
        ctx.run_host_end(1)
        for k in range(3):
            o1 = torch.empty_like(f)
            r1 = torch.empty(w.n[:3], dtype=torch.float64)
            ctx.run_host(ins[k], o1, ops[:-1] + [dict(kind="density", rho_host=r1)])
            assert torch.equal(outs[k], o1) and torch.equal(rhos[k], r1), k
        with pytest.raises(bsl.Bsl6dError) as e:
            ctx.run_host_begin(ins[0], outs[0], ops, 2)
        assert e.value.code == bsl.EINVAL
        ctx.run_host_end(1)                                  # nothing pending: returns at once


def test_run_host_two_slots_with_split_v_blocks():
    """v-blocks above 32768 points are reduced through scratch partial sums: each host-path slot has scratch of its
    own, so two density moments in flight at once do not disturb each other."""
    _need_gpu()
    w = mini((2, 2, 3, 64, 32, 32), 5, seed=11)
    rng = np.random.default_rng(3)
    ins = [torch.from_numpy(rng.random(w.n)).pin_memory() for _ in range(4)]
    outs = [torch.empty(w.n, dtype=torch.float64).pin_memory() for _ in ins]
    rhos = [torch.empty(w.n[:3], dtype=torch.float64).pin_memory() for _ in ins]
    with ctx_for(w) as ctx:
        for k in range(4):
            ops = [dict(kind="advect", dim=5, dt=0.3, shift_source=torch.ones(w.n[:3], dtype=torch.float64)),
                   dict(kind="density", rho_host=rhos[k])]
            ctx.run_host_begin(ins[k], outs[k], ops, k % 2)
        ctx.run_host_end(0)
        ctx.run_host_end(1)
        for k in range(4):
            g = ins[k].cuda()
            ctx.advect(g, g, 5, torch.ones(w.n[:3], dtype=torch.float64, device="cuda"), 0.3)
            rho = torch.empty(w.n[:3], dtype=torch.float64, device="cuda")
            ctx.density(g, rho)
            assert torch.equal(outs[k], g.cpu()) and torch.equal(rhos[k], rho.cpu()), k


def test_error_codes():
    _need_gpu()
    with pytest.raises(bsl.Bsl6dError) as e:
        bsl.create([8] * 6, [0.0] * 6, [1.0] * 6, 6)          # even degree
    assert e.value.code == bsl.EINVAL
    with pytest.raises(bsl.Bsl6dError):
        bsl.create([8, 8, 0, 8, 8, 8], [0.0] * 6, [1.0] * 6, 7)
    with pytest.raises(bsl.Bsl6dError):
        bsl.create([8] * 6, [0.0] * 6, [1.0, 1.0, -1.0, 1.0, 1.0, 1.0], 7)
    w = wl.C1
    with ctx_for(w) as ctx:
        buf = torch.zeros(w.npts + 64, dtype=torch.float64, device="cuda")
        a, b = buf[:w.npts], buf[64:]
        with pytest.raises(bsl.Bsl6dError) as e:
            ctx.advect(a, b, 0, None, 0.1)                    # partial overlap
        assert e.value.code == bsl.EALIAS
        with pytest.raises(bsl.Bsl6dError) as e:
            ctx.advect(a, a, 3, None, 0.1)                    # E sweep needs a source
        assert e.value.code == bsl.EINVAL
        with pytest.raises(bsl.Bsl6dError) as e:
            ctx.advect_generic(a, a, 2, a[:w.n[2]], 1 << 2, 1.0)   # mask contains the swept dim
        assert e.value.code == bsl.EINVAL
        with pytest.raises(bsl.Bsl6dError) as e:
            ctx.advect(a, a, 0, None, float("nan"))
        assert e.value.code == bsl.EINVAL
        with pytest.raises(bsl.Bsl6dError) as e:
            ctx.rotate(a, a, [30.0, 40.0, 0.0], 0.2)          # oblique B, more than a full turn
        assert e.value.code == bsl.EUNSUPPORTED
        assert ctx.launch_count() == 0                        # failed calls enqueue nothing


def test_density_with_caller_scratch_on_two_streams():
    """bsl6d_density_scratch: two moments of ONE context in flight on two streams, each with a work array of its own,
    give the bits of bsl6d_density (whose single work array two overlapping calls would race on)."""
    _need_gpu()
    n = (6, 4, 4, 64, 32, 40)                                  # v-block of 81920 points: 3 chunks per x-point
    w = mini(n, 7, seed=12, kind="maxwell_x1")
    f1 = dev(w.make_f("cpu").numpy())
    f2 = (f1 * 1.5 + 0.25).contiguous()
    with ctx_for(w) as ctx:
        need = ctx.density_scratch_doubles()
        assert need == 6 * 4 * 4 * 3
        want1 = ctx.density(f1, torch.empty(n[:3], dtype=torch.float64, device="cuda")).clone()
        want2 = ctx.density(f2, torch.empty(n[:3], dtype=torch.float64, device="cuda")).clone()
        torch.cuda.synchronize()
        s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
        w1 = torch.full((need,), float("nan"), dtype=torch.float64, device="cuda")
        w2 = torch.full((need,), float("nan"), dtype=torch.float64, device="cuda")
        r1 = torch.empty(n[:3], dtype=torch.float64, device="cuda")
        r2 = torch.empty(n[:3], dtype=torch.float64, device="cuda")
        torch.cuda.synchronize()
        for _ in range(20):                                   # interleaved launches on the two streams
            ctx.density_scratch(f1, r1, w1, stream=s1)
            ctx.density_scratch(f2, r2, w2, stream=s2)
        torch.cuda.synchronize()
        assert torch.equal(r1, want1) and torch.equal(r2, want2)
        with pytest.raises(ValueError):
            ctx.density_scratch(f1, r1, None)
    small = mini((3, 2, 4, 5, 6, 7), 7, seed=11, kind="maxwell_x1")   # one chunk: no work array needed
    fs = dev(small.make_f("cpu").numpy())
    with ctx_for(small) as ctx:
        assert ctx.density_scratch_doubles() == 0
        a = ctx.density_scratch(fs, torch.empty(small.n[:3], dtype=torch.float64, device="cuda"), None)
        b = ctx.density(fs, torch.empty(small.n[:3], dtype=torch.float64, device="cuda"))
        assert torch.equal(a, b)
