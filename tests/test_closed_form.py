"""Pins of workloads/analytic.py (App. A in reading G8): the closed form must
satisfy the boundary-value problem it claims to solve, and reproduce the constants in
tests/golden/layered_channel_constants.txt."""
import os

import numpy as np
import pytest

from workloads import layered_channel_closed_form

CASES = [
    dict(a=64.0, b=64.0, L=256.0, T_h=20.0, T_c=10.0, T_0=4.0, k_r=1.0, mu_r=1.0, mu_B=0.2, sigma_T=-5e-4),
    dict(a=64.0, b=64.0, L=256.0, T_h=20.0, T_c=10.0, T_0=4.0, k_r=0.2, mu_r=1.0, mu_B=0.2, sigma_T=-5e-4),
    dict(a=40.0, b=70.0, L=200.0, T_h=20.0, T_c=10.0, T_0=4.0, k_r=3.0, mu_r=2.5, mu_B=0.1, sigma_T=-3e-4),
]


def _eval(kw, x, y):
    return layered_channel_closed_form(np.asarray(x, float), np.asarray(y, float), **kw)


@pytest.mark.parametrize("kw", CASES)
def test_wall_and_interface_conditions(kw):
    a, b, L = kw["a"], kw["b"], kw["L"]
    x = np.linspace(0, L, 41)
    w = 2 * np.pi / L
    e = 1e-6
    u, v, T, _ = _eval(kw, x, np.full_like(x, -b))
    assert np.allclose(T, kw["T_h"] + kw["T_0"] * np.cos(w * x), atol=1e-10)      # eq. 30
    assert np.allclose(u, 0, atol=1e-12) and np.allclose(v, 0, atol=1e-12)         # no slip
    u, v, T, _ = _eval(kw, x, np.full_like(x, a))
    assert np.allclose(T, kw["T_c"], atol=1e-10)                                    # eq. 31
    assert np.allclose(u, 0, atol=1e-12) and np.allclose(v, 0, atol=1e-12)
    # continuity of T, u, v and of the heat flux k dT/dy across y = 0
    up = _eval(kw, x, np.full_like(x, e))
    lo = _eval(kw, x, np.full_like(x, -e))
    for i in range(3):
        assert np.allclose(up[i], lo[i], atol=1e-7)
    dT_up = (_eval(kw, x, np.full_like(x, 2 * e))[2] - up[2]) / e
    dT_lo = (lo[2] - _eval(kw, x, np.full_like(x, -2 * e))[2]) / e
    assert np.allclose(kw["k_r"] * dT_up, dT_lo, atol=1e-4)
    # normal velocity vanishes on the flat interface
    assert np.allclose(_eval(kw, x, np.zeros_like(x))[1], 0, atol=1e-12)


@pytest.mark.parametrize("kw", CASES)
def test_laplace_and_divergence_free(kw):
    a, b, L = kw["a"], kw["b"], kw["L"]
    h = 1e-3
    rng = np.random.default_rng(0)
    x = rng.uniform(0, L, 50)
    for lo_, hi_ in ((-b + 1, -1.0), (1.0, a - 1)):
        y = rng.uniform(lo_, hi_, 50)
        f = lambda dx, dy: _eval(kw, x + dx, y + dy)
        c, xp, xm, yp, ym = f(0, 0), f(h, 0), f(-h, 0), f(0, h), f(0, -h)
        lapT = (xp[2] + xm[2] + yp[2] + ym[2] - 4 * c[2]) / h ** 2
        assert np.abs(lapT).max() < 1e-4                                            # steady conduction
        div = (xp[0] - xm[0]) / (2 * h) + (yp[1] - ym[1]) / (2 * h)
        assert np.abs(div).max() < 1e-9 * max(1.0, abs(c[3]) / 1e-4)                # continuity, eq. 1


@pytest.mark.parametrize("kw", CASES)
def test_marangoni_stress_jump(kw):
    """mu_A du/dy|_0+ - mu_B du/dy|_0- = -sigma_T dT/dx at the interface (tangential balance
    behind eq. 8's Marangoni term)."""
    L = kw["L"]
    x = np.linspace(0, L, 33)
    e = 1e-5
    mu_A = kw["mu_r"] * kw["mu_B"]
    du_up = (_eval(kw, x, np.full_like(x, 2 * e))[0] - _eval(kw, x, np.full_like(x, e))[0]) / e
    du_lo = (_eval(kw, x, np.full_like(x, -e))[0] - _eval(kw, x, np.full_like(x, -2 * e))[0]) / e
    dTdx = (_eval(kw, x + e, np.zeros_like(x))[2] - _eval(kw, x - e, np.zeros_like(x))[2]) / (2 * e)
    lhs = mu_A * du_up - mu_B_times(kw, du_lo)
    assert np.allclose(lhs, -kw["sigma_T"] * dTdx, atol=2e-9)


def mu_B_times(kw, v):
    return kw["mu_B"] * v


def test_constants_match_golden(golden_dir):
    vals = {}
    for line in open(os.path.join(golden_dir, "layered_channel_constants.txt")):
        if line.startswith("#") or not line.strip():
            continue
        k, v = line.split()
        vals[k] = float(v)
    kw = CASES[0]
    *_, U_max = _eval(kw, [0.0], [0.0])
    assert U_max == pytest.approx(vals["U_max"], rel=2e-6)
    w = 2 * np.pi / kw["L"]
    ar = kw["a"] * w
    f = 1.0 / (2 * np.sinh(ar) * np.cosh(ar))      # A.5 with k_r = 1, a = b
    assert f == pytest.approx(vals["f"], rel=2e-6)
    assert np.sinh(ar) * f == pytest.approx(vals["g"], rel=2e-6)
