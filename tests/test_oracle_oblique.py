"""Pins of the oblique-B rotation oracle (eq (3): dV/dt = V x B): the axis-rotation
plan multiplies out to Rodrigues' rotation matrix, an anisotropic Gaussian is carried to its closed-form image with
the expected convergence, rotations about an oblique axis compose and return, and the axis-aligned case is untouched."""
import math

import numpy as np
import pytest

import oracle


def R_axis(c, t):
    a, b = (c + 1) % 3, (c + 2) % 3
    M = np.eye(3)
    M[a, a], M[a, b], M[b, a], M[b, b] = math.cos(t), -math.sin(t), math.sin(t), math.cos(t)
    return M


def rodrigues(B, dt):
    B = np.asarray(B, dtype=np.float64)
    bn = np.linalg.norm(B)
    k = B / bn
    th = bn * dt
    K = np.array([[0, -k[2], k[1]], [k[2], 0, -k[0]], [-k[1], k[0], 0]])
    return np.eye(3) + math.sin(th) * K + (1 - math.cos(th)) * (K @ K)


@pytest.mark.parametrize("B,dt", [((0.3, -0.5, 0.8), 0.7), ((1.0, 1.0, 0.0), 0.4), ((-2.0, 0.1, -1.0), 0.9),
                                  ((0.0, 1.0, 1.0), 2.5), ((-1.0, -1e-3, 0.2), 0.05), ((0.5, 0.5, -0.7), -1.3)])
def test_axis_rotation_plan_multiplies_out_to_rodrigues(B, dt):
    """(T_M f)(v) = f(M v); applying T_A after T_M gives T_{M A}: the applied factors multiply left to right."""
    plan = oracle.rotation_plan(B, dt)
    M = np.eye(3)
    for c, t in plan:
        assert abs(t) <= math.pi / 2 + 1e-15
        M = M @ R_axis(c, t)
    assert np.max(np.abs(M - rodrigues(B, dt))) <= 5e-16 * 8
    assert len(plan) <= 16


def gaussian_grid(n, vmax, S):
    v = -vmax + np.arange(n) * (2 * vmax / n)
    V = np.stack(np.meshgrid(v, v, v, indexing="ij"), axis=-1)
    f = np.exp(-0.5 * np.einsum("...i,ij,...j->...", V, S, V))
    return v, V, f


def test_oblique_rotation_carries_a_gaussian_to_its_closed_form_image():
    """f(v) = exp(-v.S.v/2)  ->  f_new(v) = f(R v) = exp(-(Rv).S.(Rv)/2); error falls with resolution (q = 8)."""
    S = np.diag([1.0, 2.5, 0.6])
    B, dt = (0.4, -0.3, 0.6), 0.5
    R = rodrigues(B, dt)
    errs = []
    for n in (16, 32):
        vmax = 6.0
        v, V, f = gaussian_grid(n, vmax, S)
        g = oracle.Grid((1, 1, 1, n, n, n), (0.0, 0.0, 0.0, -vmax, -vmax, -vmax), (1.0, 1.0, 1.0) + (2 * vmax / n,) * 3)
        out = oracle.rotate(g, 7, np.ascontiguousarray(f.reshape(g.n)), B, dt).reshape(n, n, n)
        RV = np.einsum("ij,...j->...i", R, V)
        want = np.exp(-0.5 * np.einsum("...i,ij,...j->...", RV, S, RV))
        errs.append(np.max(np.abs(out - want)))
    assert errs[1] < 4e-3 and errs[0] / errs[1] > 20.0, errs      # sigma_min = 0.63 against dv = 0.375 at n = 32


def test_oblique_rotations_compose_and_return():
    """Two rotations about the same oblique axis equal (to interpolation error) one by the summed angle; the opposite
    angle undoes a rotation; the sign of the rotation agrees with the axis-aligned primitive."""
    n, vmax = 24, 6.0
    S = np.diag([1.0, 2.0, 0.7])
    v, V, f = gaussian_grid(n, vmax, S)
    g = oracle.Grid((1, 1, 1, n, n, n), (0.0,) * 3 + (-vmax,) * 3, (1.0,) * 3 + (2 * vmax / n,) * 3)
    f6 = np.ascontiguousarray(f.reshape(g.n))
    B = (0.2, 0.5, -0.4)
    a = oracle.rotate(g, 7, oracle.rotate(g, 7, f6, B, 0.3), B, 0.4)
    b = oracle.rotate(g, 7, f6, B, 0.7)
    assert np.max(np.abs(a - b)) < 2e-2
    back = oracle.rotate(g, 7, b, B, -0.7)
    assert np.max(np.abs(back - f6)) < 2e-2
    # nearly axis-aligned oblique B ~ the axis-aligned primitive (continuity across the special case)
    c = oracle.rotate(g, 7, f6, (1e-9, 0.0, 1.0), 0.5)
    d = oracle.rotate(g, 7, f6, (0.0, 0.0, 1.0), 0.5)
    assert np.max(np.abs(c - d)) < 1e-6
