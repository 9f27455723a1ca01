"""bsl6d_density_static -- the density moment for callers that cannot allocate device memory.

Some users of this library run where cudaMalloc / cudaFree must not be called while the simulation is going: the
library sits inside an application that hands out all GPU memory from its own pool, or the moment is a diagnostic
taken between time steps that must not pay for the synchronisation an allocation can cause.  Every other entry point
needs a context, and creating one allocates.  bsl6d_density_static takes plain arguments and keeps the partial sums
of long velocity blocks in a 2 MiB array that is compiled into the library (262144 doubles per GPU, never freed).

Checked here: on two calls in a row -- different grids, different data, nothing cleared in between -- the result
equals what Context.density (the path with cudaMalloc'ed scratch) returns, within the 1e-14 * max|rho| the density
parity test uses and in fact bit for bit; grids beyond the array's size are refused with ESCRATCH before anything is
launched; the calls leave the amount of free device memory unchanged.

The file name sorts last on purpose: `pytest -x` stops at the first failure, and this test must not hide the others.
It has no state in common with them and passes alone in a fresh process as well as after the rest of the suite.
"""
import ctypes as C
import math

import pytest
import torch

import bsl6d_workloads as wl
import paper_2303_05994_b200 as bsl

pytestmark = pytest.mark.gpu

RTOL = 1e-14          # the tolerance of test_gpu_parity.test_density


def _need_gpu():
    assert torch.cuda.is_available(), "GPU tests selected but no CUDA device is visible"
    bsl.load_library()


def _problem(n, seed):
    w = wl._mk("static", n, 4 * math.pi, 6.0, degree=7, dt=0.05, seed=seed, noise_amp=1e-3, kind="maxwell_x1")
    return w, w.make_f("cpu").cuda()


def _chunks(n):
    """G of include/bsl6d.h: the number of chunks of <= 32768 doubles (even length) a v-block is cut into."""
    seg = n[3] * n[4] * n[5]
    G = -(-seg // 32768)
    chunk = (-(-seg // G) + 1) & ~1
    return -(-seg // chunk)


def _existing_path(w, f):
    rho = torch.empty(w.n[:3], dtype=torch.float64, device="cuda")
    with bsl.create(w.n, w.lo, w.dx, w.degree) as ctx:
        ctx.density(f, rho)
        torch.cuda.synchronize()
    return rho


def _same(got, want, what):
    err = (got - want).abs().max().item()
    assert err <= RTOL * want.abs().max().item(), f"{what}: max|diff| {err:.3e}"
    assert torch.equal(got, want), f"{what}: within tolerance but not the same bits as bsl6d_density"


def test_two_calls_in_a_row_match_the_allocating_path():
    _need_gpu()
    n_a, n_b = (2, 3, 2, 64, 32, 40), (3, 2, 2, 64, 32, 32)       # 3 and 2 chunks per x-point: both use the array
    assert _chunks(n_a) == 3 and _chunks(n_b) == 2
    wa, fa = _problem(n_a, seed=21)
    wb, fb = _problem(n_b, seed=22)
    _, fa2 = _problem(n_a, seed=23)                                # grid A again with other data
    want_a, want_b, want_a2 = _existing_path(wa, fa), _existing_path(wb, fb), _existing_path(wa, fa2)
    assert not torch.equal(want_a, want_a2)

    nan = float("nan")
    got_a = torch.full(n_a[:3], nan, dtype=torch.float64, device="cuda")
    got_b = torch.full(n_b[:3], nan, dtype=torch.float64, device="cuda")
    got_a2 = torch.full(n_a[:3], nan, dtype=torch.float64, device="cuda")
    # back to back on one stream, no synchronisation and no clearing in between: the second call finds the first
    # call's partial sums in the array (three per x-point where it writes two), the third those of the second
    bsl.density_static(n_a, wa.dx[3:], fa, got_a)
    bsl.density_static(n_b, wb.dx[3:], fb, got_b)
    bsl.density_static(n_a, wa.dx[3:], fa2, got_a2)
    torch.cuda.synchronize()
    _same(got_a, want_a, "first call")
    _same(got_b, want_b, "second call")
    _same(got_a2, want_a2, "third call")

    # the same three calls again: the first call on this device is behind us (it looked the array's address up, which
    # may have loaded code onto the GPU), so from here on the free device memory must not move at all
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info()
    for _ in range(2):
        bsl.density_static(n_a, wa.dx[3:], fa, got_a)
        bsl.density_static(n_b, wb.dx[3:], fb, got_b)
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    assert free_after == free_before, (free_before, free_after)
    _same(got_a, want_a, "repeat, grid A")
    _same(got_b, want_b, "repeat, grid B")


def test_short_velocity_blocks_need_no_scratch():
    _need_gpu()
    for n in [(3, 2, 4, 5, 6, 7), (4, 4, 4, 32, 32, 32)]:          # one chunk per x-point, odd and even length
        assert _chunks(n) == 1
        w, f = _problem(n, seed=31)
        got = torch.full(n[:3], float("nan"), dtype=torch.float64, device="cuda")
        bsl.density_static(n, w.dx[3:], f, got)
        torch.cuda.synchronize()
        _same(got, _existing_path(w, f), str(n))


def test_grids_beyond_the_array_are_refused():
    _need_gpu()
    lib = bsl.load_library()
    f = torch.zeros(16, dtype=torch.float64, device="cuda")        # never read: the call must fail before any launch
    rho = torch.full((16,), 7.0, dtype=torch.float64, device="cuda")
    dv = (C.c_double * 3)(0.1, 0.1, 0.1)
    err = C.c_int(123)

    def call(n):
        return lib.bsl6d_density_static((C.c_int32 * 6)(*n), dv, f.data_ptr(), rho.data_ptr(), None, C.byref(err))

    # 2 chunks x 131072 x-points = exactly the array: accepted by the size check (not run: f is a dummy);
    # one x-plane more is one slot too many
    too_big = (128, 32, 33, 64, 32, 32)
    assert 2 * 128 * 32 * 33 > bsl.STATIC_SCRATCH_DOUBLES >= 2 * 128 * 32 * 32
    assert call(too_big) == bsl.ESCRATCH and err.value == 0
    assert lib.bsl6d_strerror(bsl.ESCRATCH).decode().startswith("needs more scratch")
    assert call((0, 1, 1, 8, 8, 8)) == bsl.EINVAL
    assert lib.bsl6d_density_static(None, dv, f.data_ptr(), rho.data_ptr(), None, None) == bsl.EINVAL
    torch.cuda.synchronize()
    assert torch.all(rho == 7.0)                                   # nothing was launched
    # the binding checks shapes before it calls the library
    w, fs = _problem((2, 2, 2, 8, 8, 8), seed=5)
    with pytest.raises(ValueError):
        bsl.density_static(too_big, w.dx[3:], fs, rho)
    # BASELINE config C3 (16^3 x 64^3) needs 8 * 4096 = 32768 slots: fits
    assert _chunks((16, 16, 16, 64, 64, 64)) * 16 ** 3 <= bsl.STATIC_SCRATCH_DOUBLES
