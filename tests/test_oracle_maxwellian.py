"""Pins of the oracle's Maxwellian equilibrium (`equilibrium = 1`, D3Q27 lattices): the continuous Maxwell-Boltzmann
distribution taken in central-moment space, in place of the second-order equilibria the paper prints (eqs. 12, 18).
Definition-level pins with numpy (central moments; the textbook product form), and the closed forms every equilibrium
must still satisfy: the advected heat sinusoid (Poiseuille and the Laplace law see moments up to second order
only, which the two equilibria share; the GPU parity tests run both flows with it)."""
import numpy as np
import pytest

import workloads as W
from oracle import tcpo

MX = dict(equilibrium=1, thermal="lb_d3q27")


def _product_form(c, s, u):
    """the textbook discrete Maxwellian on D3Q27: s * prod_axis p(c_a; u_a), p(0) = 2/3 - u^2, p(+-1) = 1/6 +- u/2 + u^2/2"""
    out = np.full(len(c), s, dtype=float)
    for a in range(3):
        p = np.where(c[:, a] == 0, 2 / 3 - u[a] ** 2, 1 / 6 + c[:, a] * u[a] / 2 + u[a] ** 2 / 2)
        out = out * p
    return out


def test_equilibrium_populations_are_the_product_form_and_have_maxwellian_central_moments():
    """One collision with every rate 1 and no force returns the equilibrium itself.  Oracle route: dense solve K(u) a = kappa^M.
    Expected: the product form, written out here; its central moments of order 3 vanish and kappa_220 = s / 9,
    kappa_222 = s / 27, where the printed second-order equilibrium leaves remnants (-s u_x^2 u_y, s (1 + 27 u_x^2 u_y^2) / 9)."""
    rng = np.random.default_rng(5)
    c, w, opp, order = tcpo.lattice(27)
    cf = c.astype(float)
    s0, u = 0.83, np.array([0.07, -0.04, 0.09])
    a_in = w * s0 * (1 + 0.1 * rng.standard_normal(27))
    a_in *= s0 / a_in.sum()
    # the oracle's Maxwellian enters through a full step only; here: one cell, all rates 1, via a 1-cell periodic box
    o = tcpo.Oracle(1, 1, 1, dict(MX, xi=1e30, kappa_H=1 / 6, kappa_L=1 / 6))       # omega_T = 1 / (1/2 + 3 kappa) = 1
    o.init_fields(np.zeros((1, 1, 1)), u=u.reshape(3, 1, 1, 1), T=np.full((1, 1, 1), s0))
    f0 = o.read_populations(2).ravel()                                             # f~ = f_eq^M(T, u) at initialisation
    want = _product_form(c, s0, u)
    assert np.abs(f0 - want).max() < 1e-15
    d = cf - u
    mom = lambda a, b, cc: (want * d[:, 0] ** a * d[:, 1] ** b * d[:, 2] ** cc).sum()
    assert abs(mom(2, 1, 0)) < 1e-16 and abs(mom(1, 1, 1)) < 1e-16 and abs(mom(1, 2, 2)) < 1e-16
    assert mom(2, 0, 0) == pytest.approx(s0 / 3, abs=1e-15)
    assert mom(2, 2, 0) == pytest.approx(s0 / 9, abs=1e-15)
    assert mom(2, 2, 2) == pytest.approx(s0 / 27, abs=1e-15)
    cu = cf @ u
    printed = s0 * w * (1 + 3 * cu + 4.5 * cu ** 2 - 1.5 * u @ u)
    assert (printed * d[:, 0] ** 2 * d[:, 1]).sum() == pytest.approx(-s0 * u[0] ** 2 * u[1], abs=1e-15)
    o.step(1)                                                                      # a uniform state at equilibrium stays there
    assert np.abs(o.read_populations(2).ravel() - want).max() < 1e-15
    g0 = o.read_populations(1).ravel()                                             # g~ = w (p* - 1) + a^M(1, u), p* = 0
    assert np.abs(g0 - (_product_form(c, 1.0, u) - w)).max() < 1e-15
    o.close()


def test_advected_heat_sinusoid_with_the_maxwellian():
    # (Poiseuille is left to the other equilibrium: it sees second moments only, which the two equilibria share)
    n, kap, U, steps = 48, 0.1, 0.04, 120
    k = 2 * np.pi / n
    T0 = (1 + 0.5 * np.sin(k * np.arange(n))).reshape(1, 1, n)
    u0 = np.zeros((3, 1, 1, n)); u0[0] = U
    o = tcpo.Oracle(n, 1, 1, dict(MX, kappa_H=kap, kappa_L=kap, xi=1e30))
    o.init_fields(np.zeros((1, 1, n)), u=u0, T=T0)
    o.step(steps)
    T = o.read_fields()[3].ravel()
    o.close()
    Fm = np.fft.rfft(T - 1)[1]
    assert -np.log(2 * np.abs(Fm) / n / 0.5) / steps == pytest.approx(kap * k * k, rel=0.02)
    assert (-np.angle(Fm) - np.pi / 2) / k == pytest.approx(U * steps, rel=0.01)


def test_only_d3q27_lattices_take_the_maxwellian():
    for bad in (dict(equilibrium=1, thermal="lb_d3q7"), dict(equilibrium=1, thermal="lb_d3q27", hydro_lattice=19)):
        with pytest.raises(tcpo.OracleError):
            tcpo.Oracle(4, 4, 4, bad)
    tcpo.Oracle(4, 4, 4, dict(equilibrium=1, thermal="rk2")).close()
