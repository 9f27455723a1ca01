"""Pins of the odd-q / per-point-displacement oracle (eq (6), 194)."""
from fractions import Fraction

import numpy as np
import pytest

import oracle


def exact_weights(q, alpha: Fraction):
    h = (q - 1) // 2
    out = []
    for m in range(-h, h + 1):
        num, den = Fraction(1), Fraction(1)
        for n in range(-h, h + 1):
            if n != m:
                num *= alpha - n
                den *= m - n
        out.append(num / den)
    return out


def test_q3_closed_form():
    for a in (-0.75, -0.25, 0.0, 0.3, 1.0):
        w = oracle.lagrange_weights_odd(3, a)
        assert np.allclose(w, [(a * a - a) / 2, 1 - a * a, (a * a + a) / 2], rtol=0, atol=2e-16)


def test_q5_textbook_values_at_half():
    # nodes -2..2 at alpha = 1/2: (3, -20, 90, 60, -5)/128
    assert np.array_equal(oracle.lagrange_weights_odd(5, 0.5), np.array([3, -20, 90, 60, -5]) / 128.0)


@pytest.mark.parametrize("q", (3, 5, 7, 9))
def test_weights_against_exact_rationals_and_moments(q):
    h = (q - 1) // 2
    for a in (Fraction(-7, 8), Fraction(-1, 3), Fraction(1, 4), Fraction(5, 7), Fraction(1, 1), Fraction(0, 1)):
        w = oracle.lagrange_weights_odd(q, float(a))
        ex = exact_weights(q, Fraction(float(a)))             # exact weights of the rounded alpha
        assert np.max(np.abs(w - np.array([float(e) for e in ex]))) <= 8e-16
        m = np.arange(-h, h + 1, dtype=np.float64)
        for p in range(q):                                    # sum_m m^p l_m(alpha) = alpha^p
            assert abs(np.dot(m ** p, w) - float(a) ** p) <= 1e-12 * max(1.0, h ** p)
    for k in range(-h, h + 1):                                # whole-cell displacement: exact unit vector
        assert np.array_equal(oracle.lagrange_weights_odd(q, float(k)), np.eye(q)[k + h])


@pytest.mark.parametrize("dim", (0, 2, 3, 5))
@pytest.mark.parametrize("q", (3, 7, 9))
def test_pointwise_sweep_reproduces_polynomials_and_matches_numpy(dim, q):
    rng = np.random.default_rng(10 * dim + q)
    n = [3, 2, 4, 3, 2, 4]
    n[dim] = 13
    f = rng.random(n)
    alpha = rng.uniform(-1.0, 1.0, n)
    out = oracle.sweep_pointwise(f, dim, alpha, q)
    h = (q - 1) // 2
    fm = np.moveaxis(f, dim, -1).reshape(-1, 13)
    am = np.moveaxis(alpha, dim, -1).reshape(-1, 13)
    om = np.moveaxis(out, dim, -1).reshape(-1, 13)
    for p in range(0, fm.shape[0], 7):                        # every 7th pencil: numpy polynomial through the stencil
        for j in range(13):
            idx = np.arange(j - h, j + h + 1)
            vals = fm[p, idx % 13] if dim < 3 else np.where((idx >= 0) & (idx < 13), fm[p, np.clip(idx, 0, 12)], 0.0)
            c = np.polyfit(np.arange(-h, h + 1, dtype=np.float64), vals, q - 1)
            assert abs(np.polyval(c, am[p, j]) - om[p, j]) <= 1e-10
    # degree q-1 polynomial data on a zero-extended dim: interior points are reproduced at x_j + alpha_j
    if dim >= 3:
        coef = rng.standard_normal(q)
        j = np.arange(13, dtype=np.float64)
        shape = [1] * 6
        shape[dim] = 13
        fp = np.broadcast_to(np.polyval(coef, j).reshape(shape), n).copy()
        op = oracle.sweep_pointwise(fp, dim, alpha, q)
        want = np.polyval(coef, j.reshape(shape) + alpha)
        sl = [slice(None)] * 6
        sl[dim] = slice(h, 13 - h)
        assert np.max(np.abs(op[tuple(sl)] - want[tuple(sl)])) <= 1e-9 * np.max(np.abs(want))


def test_whole_cell_alpha_is_an_exact_roll_or_shift():
    rng = np.random.default_rng(3)
    f = rng.random((6, 2, 2, 7, 2, 2))
    for k in (-1, 0, 1):
        a = np.full(f.shape, float(k))
        assert np.array_equal(oracle.sweep_pointwise(f, 0, a, 7), np.roll(f, -k, axis=0))     # out[j] = in[j+k]
        exp = np.zeros_like(f)
        if k == 0:
            exp = f.copy()
        elif k == 1:
            exp[:, :, :, :-1] = f[:, :, :, 1:]
        else:
            exp[:, :, :, 1:] = f[:, :, :, :-1]
        assert np.array_equal(oracle.sweep_pointwise(f, 3, a, 7), exp)
