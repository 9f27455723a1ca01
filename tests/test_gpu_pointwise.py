"""Odd-q / per-point-displacement sweep on the GPU against the oracle."""
from __future__ import annotations

import numpy as np
import pytest
import torch

import bsl6d_workloads as wl
import oracle
import paper_2303_05994_b200 as bsl

pytestmark = pytest.mark.gpu
TOL = 1e-12


def _need(gb=0.0):
    from conftest import need_gpu
    need_gpu(gb)


def _ctx(n):
    return bsl.create(n, (0.0,) * 3 + (-6.0,) * 3, (1.0,) * 6, 7)


GRIDS = [(8, 16, 32, 37, 8, 16), (37, 8, 8, 16, 32, 37), (16, 37, 8, 8, 37, 32), (32, 8, 37, 8, 16, 8),
         (48, 8, 4, 64, 8, 48), (4, 64, 8, 8, 48, 64)]
#: extents without a compiled instance -> the run-time-extent kernels (any n, n < q and n = 1 included)
GENERIC_GRIDS = [(12, 5, 36, 7, 40, 11), (3, 20, 2, 130, 1, 100), (36, 2, 1, 3, 9, 1), (1, 1, 6, 1, 1, 210)]


@pytest.mark.parametrize("n", GRIDS)
@pytest.mark.parametrize("q", (3, 5, 7, 9))
def test_every_dim_random_shifts(n, q):
    _need()
    rng = np.random.default_rng(q)
    f = rng.random(n)
    alpha = wl.random_shifts(n, 77 + q).numpy()
    fd, ad = torch.from_numpy(f).cuda(), torch.from_numpy(alpha).cuda()
    out = torch.empty_like(fd)
    with _ctx(n) as ctx:
        for dim in range(6):
            ctx.advect_pointwise(fd, out, dim, ad, q)
            ref = oracle.sweep_pointwise(f, dim, alpha, q)
            err = np.max(np.abs(out.cpu().numpy() - ref)) / np.max(np.abs(ref))
            assert err <= TOL, (dim, err)
            inplace = fd.clone()
            ctx.advect_pointwise(inplace, inplace, dim, ad, q)     # in place
            assert torch.equal(inplace, out), dim
        assert ctx.launch_count() == 12


@pytest.mark.parametrize("n", GENERIC_GRIDS)
@pytest.mark.parametrize("q", (1, 3, 5, 7, 9, 11))
def test_runtime_extent_kernels(n, q):
    """Any extent, widths 1..11, every dim, in place == out of place."""
    _need()
    rng = np.random.default_rng(100 + q)
    f = rng.random(n)
    alpha = wl.random_shifts(n, 31 + q).numpy()
    fd, ad = torch.from_numpy(f).cuda(), torch.from_numpy(alpha).cuda()
    out = torch.empty_like(fd)
    with _ctx(n) as ctx:
        for dim in range(6):
            ctx.advect_pointwise(fd, out, dim, ad, q)
            ref = oracle.sweep_pointwise(f, dim, alpha, q)
            err = np.max(np.abs(out.cpu().numpy() - ref)) / np.max(np.abs(ref))
            assert err <= TOL, (dim, err)
            inplace = fd.clone()
            ctx.advect_pointwise(inplace, inplace, dim, ad, q)
            assert torch.equal(inplace, out), dim


@pytest.mark.parametrize("q", (3, 9))
@pytest.mark.parametrize("n", [(37, 8, 16, 32, 8, 37), (36, 5, 12, 33, 8, 35)])
def test_whole_cell_shifts_are_bit_exact(q, n):
    _need()
    f = np.random.default_rng(1).random(n)
    alpha = wl.random_shifts(n, 5, whole_cells=True).numpy()
    assert set(np.unique(alpha)) == {-1.0, 0.0, 1.0}
    fd, ad = torch.from_numpy(f).cuda(), torch.from_numpy(alpha).cuda()
    out = torch.empty_like(fd)
    with _ctx(n) as ctx:
        for dim in range(6):
            ctx.advect_pointwise(fd, out, dim, ad, q)
            assert np.array_equal(out.cpu().numpy(), oracle.sweep_pointwise(f, dim, alpha, q)), dim
    # and the expected value needs no oracle at all: out[j] = in[j + alpha_j] (periodic dim 0)
    with _ctx(n) as ctx:
        got = ctx.advect_pointwise(fd, out, 0, ad, q).cpu().numpy()
    j = np.arange(n[0]).reshape(n[0], 1, 1, 1, 1, 1)
    src = (j + alpha.astype(np.int64)) % n[0]
    assert np.array_equal(got, np.take_along_axis(f, src, axis=0))


@pytest.mark.parametrize("n", [(37, 8, 4, 32, 8, 37), (13, 3, 10, 9, 4, 21)])
def test_whole_cell_shifts_up_to_half_width(n):
    """alpha in {-h..h} per point (beyond the paper's |alpha| < dx): still an exact gather, compiled and run-time kernels."""
    _need()
    rng = np.random.default_rng(7)
    f = rng.random(n)
    for q in (5, 9):
        h = (q - 1) // 2
        alpha = rng.integers(-h, h + 1, n).astype(np.float64)
        fd, ad = torch.from_numpy(f).cuda(), torch.from_numpy(alpha).cuda()
        out = torch.empty_like(fd)
        with _ctx(n) as ctx:
            for dim in range(6):
                ctx.advect_pointwise(fd, out, dim, ad, q)
                assert np.array_equal(out.cpu().numpy(), oracle.sweep_pointwise(f, dim, alpha, q)), (q, dim)


def test_generator_cpu_equals_cuda():
    _need()
    a = wl.random_shifts((5, 4, 3, 2, 3, 4), 9)
    assert torch.equal(a, wl.random_shifts((5, 4, 3, 2, 3, 4), 9, device="cuda").cpu())
    assert float(a.min()) >= -1.0 and float(a.max()) < 1.0


def test_error_codes():
    _need()
    n = (8, 8, 8, 8, 8, 500)
    f = torch.zeros(n, dtype=torch.float64, device="cuda")
    a = torch.zeros_like(f)
    with _ctx(n) as ctx:
        with pytest.raises(bsl.Bsl6dError) as e:
            ctx.advect_pointwise(f, f, 0, a, 4)              # even width
        assert e.value.code == bsl.EINVAL
        with pytest.raises(bsl.Bsl6dError) as e:
            ctx.advect_pointwise(f, f, 0, f, 3)              # alpha aliases the output
        assert e.value.code == bsl.EALIAS
        with pytest.raises(bsl.Bsl6dError) as e:
            ctx.advect_pointwise(f, f, 5, a, 3)              # unit-stride extent 500: no shared-memory staging
        assert e.value.code == bsl.EUNSUPPORTED
        with pytest.raises(bsl.Bsl6dError) as e:
            ctx.advect_pointwise(f, f, 0, a, 13)             # width 13 has no kernel
        assert e.value.code == bsl.EUNSUPPORTED
        assert ctx.launch_count() == 0


def test_paper_benchmark_grid_full_size_sampled():
    """37^6 (20.5 GB per array, three arrays), width 7, every direction: oracle on sampled pencils of f and alpha."""
    _need(70)
    w = wl.P37
    f = w.make_f("cuda")
    alpha = wl.random_shifts(w.n, w.seed + 1, device="cuda")
    out = torch.empty_like(f)
    rng = np.random.default_rng(2037)
    P, N = 1024, 37
    with bsl.create(w.n, w.lo, w.dx, w.degree) as ctx:
        for dim in range(6):
            outer = int(np.prod(w.n[:dim], dtype=np.int64))
            inner = int(np.prod(w.n[dim + 1:], dtype=np.int64))
            o = torch.from_numpy(rng.integers(0, outer, P)).cuda()
            i = torch.from_numpy(rng.integers(0, inner, P)).cuda()
            ctx.advect_pointwise(f, out, dim, alpha, 7)
            g = lambda t: t.view(outer, N, inner)[o, :, i].cpu().numpy()          # (P, N)
            gi, ga, go = g(f), g(alpha), g(out)
            if dim < 3:      # mini-grid: swept dim at position 0 (periodic), samples at position 3
                ref = oracle.sweep_pointwise(np.ascontiguousarray(gi.T).reshape(N, 1, 1, P, 1, 1), 0,
                                             np.ascontiguousarray(ga.T).reshape(N, 1, 1, P, 1, 1), 7).reshape(N, P).T
            else:            # swept dim at position 3 (zero-extended), samples at position 0
                ref = oracle.sweep_pointwise(gi.reshape(P, 1, 1, N, 1, 1), 3, ga.reshape(P, 1, 1, N, 1, 1), 7).reshape(P, N)
            err = np.max(np.abs(go - ref)) / np.max(np.abs(ref))
            assert err <= TOL, (dim, err)
