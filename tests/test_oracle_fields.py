"""Pins of the field-step oracle (oracle/fields.py) against what the mathematics fixes -- no GPU, no CUDA path.
Closed forms for single Fourier modes on non-cubic boxes (even and odd extents), the Nyquist convention, linearity,
and the textbook linear Landau damping rate for the self-consistent step (eq (2), 74-78)."""
import math

import numpy as np
import pytest

import oracle


def grid_xyz(n, L):
    ax = [np.arange(n[d]) * (L[d] / n[d]) for d in range(3)]
    return np.meshgrid(*ax, indexing="ij")


N, L = (16, 9, 10), (4 * math.pi, 2 * math.pi, 6.0)


@pytest.mark.parametrize("mode", [(1, 0, 0), (0, 2, 0), (0, 0, 3), (2, -1, 1), (-3, 4, 2), (7, 0, 0)])
def test_poisson_single_mode_closed_form(mode):
    """rho_c = a cos(kappa.x + p)  =>  phi = rho_c/|kappa|^2,  E = -grad(phi) = a kappa sin(kappa.x + p)/|kappa|^2."""
    X = grid_xyz(N, L)
    kap = [2 * math.pi * mode[d] / L[d] for d in range(3)]
    ph = kap[0] * X[0] + kap[1] * X[1] + kap[2] * X[2] + 0.3
    a, rho_fac, e_fac = 0.05, -1.0, -2.0
    moment = 1.0 + a * np.cos(ph)
    E = oracle.poisson_E(moment, L, rho_fac, e_fac)
    k2 = sum(k * k for k in kap)
    for d in range(3):
        want = e_fac * rho_fac * a * kap[d] * np.sin(ph) / k2
        assert np.max(np.abs(E[d] - want)) <= 1e-14 * (1 + np.max(np.abs(want))), d


def test_adiabatic_single_mode_closed_form():
    X = grid_xyz(N, L)
    kap = [2 * math.pi * m / l for m, l in zip((2, 1, -1), L)]
    ph = kap[0] * X[0] + kap[1] * X[1] + kap[2] * X[2] - 1.1
    moment = 3.0 + 0.2 * np.sin(ph)
    E = oracle.adiabatic_E(moment, L, 0.7, 1.5)               # phi = 0.7 (moment - mean); E = -1.5 grad(phi)
    for d in range(3):
        want = -1.5 * 0.7 * 0.2 * kap[d] * np.cos(ph)
        assert np.max(np.abs(E[d] - want)) <= 1e-14


def test_mean_is_dropped_and_linearity():
    rng = np.random.default_rng(5)
    m1, m2 = rng.random(N), rng.random(N)
    E1, E2 = oracle.poisson_E(m1, L, 1.0, 1.0), oracle.poisson_E(m2, L, 1.0, 1.0)
    E12 = oracle.poisson_E(2.0 * m1 - 3.0 * m2 + 11.0, L, 1.0, 1.0)      # + constant: the k = 0 mode is dropped (F1)
    for d in range(3):
        assert np.max(np.abs(E12[d] - (2.0 * E1[d] - 3.0 * E2[d]))) <= 1e-12
        assert abs(np.mean(E1[d])) <= 1e-15


def test_nyquist_mode_has_no_gradient_but_enters_the_laplacian():
    """Even n: the alternating mode (-1)^j is its own conjugate; its first derivative is taken as zero (F2), while a
    mixed mode (Nyquist in x1, mode 1 in x2) still feels |kappa|^2 = (pi n/L1)^2 + kappa2^2 in the Laplacian."""
    n, Lb = (8, 6, 4), (2.0, 3.0, 5.0)
    X = grid_xyz(n, Lb)
    j1 = np.arange(n[0])[:, None, None]
    alt = np.where(j1 % 2 == 0, 1.0, -1.0) * np.ones(n)
    E = oracle.poisson_E(alt, Lb, 1.0, 1.0)
    assert all(np.max(np.abs(e)) <= 1e-15 for e in E)
    k2y = 2 * math.pi / Lb[1]
    mixed = alt * np.cos(k2y * X[1])
    E = oracle.poisson_E(mixed, Lb, 1.0, 1.0)
    kn = math.pi * n[0] / Lb[0]
    want = alt * k2y * np.sin(k2y * X[1]) / (kn * kn + k2y * k2y)
    assert np.max(np.abs(E[0])) <= 1e-15
    assert np.max(np.abs(E[1] - want)) <= 1e-14


def test_vp_step_reproduces_linear_landau_damping():
    """1D1V Vlasov-Poisson, k = 0.5, Maxwellian, eps = 0.01: the field amplitude decays as exp(gamma t) cos(omega t)
    with the textbook roots gamma = -0.1533, omega = 1.4156 of the plasma dispersion relation."""
    nx, nv, vmax = 32, 64, 6.0
    Lx = 4 * math.pi
    g = oracle.Grid((nx, 1, 1, nv, 1, 1), (0.0, 0.0, 0.0, -vmax, 0.0, 0.0), (Lx / nx, 1.0, 1.0, 2 * vmax / nv, 1.0, 1.0))
    x, v = g.nodes(0), g.nodes(3)
    f = ((1 + 0.01 * np.cos(0.5 * x))[:, None] * (np.exp(-0.5 * v * v) / math.sqrt(2 * math.pi))[None, :])
    f = np.ascontiguousarray(f.reshape(g.n))
    dt, nsteps = 0.1, 220
    mass0 = np.sum(f)
    amp, t = [], []
    for s in range(nsteps):
        f, moment, E = oracle.vp_step(g, 7, f, None, dt, "poisson", -1.0, -1.0)    # electrons: q = -1, q/m = -1
        amp.append(np.max(np.abs(E[0])))
        t.append((s + 0.5) * dt)                              # the field is evaluated after the first half-step
    amp, t = np.array(amp), np.array(t)
    pk = [i for i in range(1, nsteps - 1) if amp[i] > amp[i - 1] and amp[i] >= amp[i + 1] and 1.0 < t[i] < 20.0]
    assert len(pk) >= 6
    # parabolic refinement of the peak times, then a straight line through log(peak amplitude)
    tp, ap = [], []
    for i in pk:
        y0, y1, y2 = np.log(amp[i - 1]), np.log(amp[i]), np.log(amp[i + 1])
        d = 0.5 * (y0 - y2) / (y0 - 2 * y1 + y2)
        tp.append(t[i] + d * dt)
        ap.append(y1 - 0.25 * (y0 - y2) * d)
    gamma = np.polyfit(tp, ap, 1)[0]
    omega = math.pi / np.mean(np.diff(tp))                    # |E| peaks twice per period
    assert abs(gamma - (-0.1533)) < 0.004, gamma
    assert abs(omega - 1.4156) < 0.01, omega
    assert abs(np.sum(f) - mass0) < 1e-9 * mass0              # particle number conserved (periodic x, f ~ 0 at |v| = 6)
