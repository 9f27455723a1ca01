"""ORACLE (test infrastructure, not the product): the field step of the Vlasov-Poisson system, plain numpy.

PAPER.md:44-48 eq (2):  rho_c = q (int f dv - n0),  -Laplace(phi) = rho_c,  E = -grad(phi);  PAPER.md:78: periodic
boundaries, "pseudo-spectral method based on the Fast Fourier Transform";  PAPER.md:375 eq (11): adiabatic-electron
closure  (n0 q^2 / T_e) phi = rho_c  used instead of Poisson in the ion-Bernstein-wave test.
The FFT itself is numpy's (a library primitive serving as one step); everything else is written out.

Readings:
  F1  n0 is the mean of the moment over the periodic box (neutralising background), i.e. the k = 0 mode of rho_c is
      dropped; without that the periodic Poisson problem has no solution.  phi has zero mean.
  F2  wavenumber of mode index m on n points of period L:  kappa = 2 pi mm / L with mm = m (m < n/2), m - n (m > n/2).
      The Nyquist mode m = n/2 (even n) has |kappa| = pi n / L in the Laplacian, but its first derivative is taken as
      zero (the usual pseudo-spectral convention; it keeps E real).
  F3  the moment passed in is the bare  sum_v f dv^3  of bsl6d_density / oracle.density (reading S9); the caller
      supplies the charge factors:  rho_c = rho_fac * (moment - mean),  output = e_fac * E  (e_fac = q/m so that the
      result is directly the shift source of the v-sweeps).

Pin status (tests/test_oracle_fields.py, -m "not gpu"): poisson_E and adiabatic_E pinned (single-mode closed forms on
non-cubic boxes, div E = rho_c, linearity, Nyquist rule); vp_step pinned by the textbook linear Landau damping rate
(k = 0.5: gamma = -0.1533, omega = 1.4156) on a 1D1V grid.
"""
from __future__ import annotations

from typing import List, Optional, Sequence

import numpy as np


def _wavenumbers(n: int, L: float):
    """(kappa for the Laplacian, kappa for first derivatives) of the n modes of period L  (reading F2)."""
    m = np.arange(n)
    mm = np.where(m < (n + 1) // 2, m, m - n).astype(np.float64)
    if n % 2 == 0:
        mm[n // 2] = n / 2.0
    k_lap = 2.0 * np.pi * mm / L
    k_der = k_lap.copy()
    if n % 2 == 0:
        k_der[n // 2] = 0.0
    return k_lap, k_der


def _spectral_E(rho_c_hat: np.ndarray, phi_hat: np.ndarray, kder, e_fac: float) -> List[np.ndarray]:
    out = []
    for d in range(3):
        shape = [1, 1, 1]
        shape[d] = -1
        E_hat = -1j * kder[d].reshape(shape) * phi_hat            # E = -grad(phi)
        out.append(np.ascontiguousarray(e_fac * np.real(np.fft.ifftn(E_hat))))
    return out


def poisson_E(moment: np.ndarray, L: Sequence[float], rho_fac: float, e_fac: float) -> List[np.ndarray]:
    """e_fac * E_d(x), d = 0,1,2, from -Laplace(phi) = rho_fac * (moment - mean(moment)), periodic box of lengths L."""
    n = moment.shape
    ks = [_wavenumbers(n[d], float(L[d])) for d in range(3)]
    rho_hat = np.fft.fftn(rho_fac * (moment - np.mean(moment)))
    k2 = (ks[0][0] ** 2)[:, None, None] + (ks[1][0] ** 2)[None, :, None] + (ks[2][0] ** 2)[None, None, :]
    phi_hat = np.zeros_like(rho_hat)
    nz = k2 != 0.0
    phi_hat[nz] = rho_hat[nz] / k2[nz]
    return _spectral_E(rho_hat, phi_hat, [k[1] for k in ks], e_fac)


def adiabatic_E(moment: np.ndarray, L: Sequence[float], phi_fac: float, e_fac: float) -> List[np.ndarray]:
    """e_fac * E_d(x) with the closure phi = phi_fac * (moment - mean(moment))  (eq (11): phi_fac = q T_e/(n0 q^2))."""
    n = moment.shape
    ks = [_wavenumbers(n[d], float(L[d])) for d in range(3)]
    phi_hat = np.fft.fftn(phi_fac * (moment - np.mean(moment)))
    return _spectral_E(phi_hat, phi_hat, [k[1] for k in ks], e_fac)


def vp_step(oracle_mod, grid, degree: int, f: np.ndarray, B: Optional[Sequence[float]], dt: float, closure: str,
            c1: float, e_fac: float):
    """One self-consistent Strang step IN PLACE on f (Fig. 1 caption at 114):
    x1,x2,x3 (dt/2) -> moment -> field solve -> v1,v2,v3 with E (dt) -> rotation (theta = B_c dt) -> x1,x2,x3 (dt/2).
    `oracle_mod` is the oracle package (sweeps, density); returns (f, moment, [E0,E1,E2]) of the mid-step."""
    L = [grid.n[d] * grid.dx[d] for d in range(3)]
    half = 0.5 * dt
    for d in range(3):
        f = oracle_mod.advect(grid, degree, f, d, None, half)
    moment = oracle_mod.density(grid, f)
    E = poisson_E(moment, L, c1, e_fac) if closure == "poisson" else adiabatic_E(moment, L, c1, e_fac)
    for d in range(3):
        f = oracle_mod.advect(grid, degree, f, 3 + d, E[d], dt)
    if B is not None and any(b != 0.0 for b in B):
        f = oracle_mod.rotate(grid, degree, f, B, dt)
    for d in range(3):
        f = oracle_mod.advect(grid, degree, f, d, None, half)
    return f, moment, E
