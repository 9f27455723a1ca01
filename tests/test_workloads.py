"""The seeded input generators (bsl6d_workloads) -- CPU checks; the CPU==CUDA bit-equality is in test_gpu_parity."""
import math

import numpy as np
import torch

import bsl6d_workloads as wl


def test_splitmix_torch_matches_pure_python():
    lin = torch.tensor([0, 1, 2, 12345, 2 ** 31, 2 ** 40 + 17, 2 ** 62], dtype=torch.int64)
    for seed in (0, 1001, 2 ** 63 + 5):
        u = wl.uniform_torch(seed, lin).numpy()
        ref = np.array([wl.uniform_py(seed, int(l)) for l in lin])
        assert np.array_equal(u, ref)
        assert np.all((u >= 0) & (u < 1))
    # published splitmix64 test vector: state 0 -> first output 0xE220A8397B1DCDAF
    assert wl.splitmix64_py(0) == 0xE220A8397B1DCDAF


def test_noise_is_uniform_and_white():
    u = wl.uniform_torch(1002, torch.arange(1 << 18, dtype=torch.int64)).numpy()
    assert abs(u.mean() - 0.5) < 5e-3 and abs(u.var() - 1 / 12) < 2e-3
    assert abs(np.corrcoef(u[:-1], u[1:])[0, 1]) < 1e-2


def test_config_tables():
    c = wl.CONFIGS
    assert c["C1"].n == (8,) * 6 and c["C1"].q == 8 and c["C1"].dx[3] == 1.5
    assert c["C2"].npts == 32 ** 6 and c["C3"].n == (16, 16, 16, 64, 64, 64) and c["C3"].q == 6
    assert c["C5"].n == (48, 48, 48, 32, 32, 32) and c["C5"].q == 10 and c["C5"].npts == 3623878656
    assert abs(c["C2"].dx[0] - 4 * math.pi / 32) < 1e-15 and c["C3"].dx[3] == 0.25
    # max |alpha| of SURVEY section 8(d): x sweeps of C2 0.764 cells, C3 1.0186 cells
    assert abs(6.0 * c["C2"].dt / c["C2"].dx[0] - 0.7639) < 1e-3
    assert abs(8.0 * c["C3"].dt / c["C3"].dx[0] - 1.0186) < 1e-3


def test_fill_formula_and_slab_independence():
    w = wl.C1
    f = w.make_f("cpu").numpy()
    fx, fv = w.fx(), w.fv()
    lin = np.arange(w.npts).reshape(w.n)
    for idx in [(0, 0, 0, 0, 0, 0), (7, 7, 7, 7, 7, 7), (3, 1, 4, 1, 5, 2)]:
        ref = fx[idx[:3]] * fv[idx[3:]] + w.noise_amp * wl.uniform_py(w.seed, int(lin[idx]))
        assert f[idx] == ref
    g = torch.empty(w.n, dtype=torch.float64)
    w.fill(g, slab_bytes=8 * w.npts // 8 // 2)          # different slab size, same bits
    assert np.array_equal(g.numpy(), f)
    assert f.min() >= 0 and abs(f.max() - (2 * math.pi) ** -1.5 * 1.01) < 2e-3
    r = wl.C2.reduced((8, 8, 8, 16, 16, 16))
    assert r.dx[0] * 8 == wl.C2.dx[0] * 32 and r.q == 8 and r.make_f().shape == (8, 8, 8, 16, 16, 16)
