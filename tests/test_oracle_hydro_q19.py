"""Pins of the oracle's D3Q19 hydrodynamic lattice (`hydro_lattice = 19`; "hydrodynamic LBM solvers often
rely on a D3Q19 or D3Q27 stencil"; weights App. B.3, central-moment basis of reading S2: the 19 monomials
x^a y^b z^c with a, b, c <= 2 and abc = 0).  Closed forms only -- nothing here compares the oracle with itself except the
last test, which says how close the two lattices must be on a smooth flow."""
import numpy as np
import pytest

import workloads as W
from oracle import tcpo


def test_weights_and_basis_of_the_q19_hydrodynamic_lattice():
    c, w, opp, order = tcpo.lattice(19)
    assert w.sum() == pytest.approx(1.0, abs=1e-15)
    for a in range(3):
        assert (w * c[:, a] ** 2).sum() == pytest.approx(1 / 3, abs=1e-15)
        assert (w * c[:, a] ** 4).sum() == pytest.approx(1 / 3, abs=1e-15)
    assert (w * c[:, 0] ** 2 * c[:, 1] ** 2).sum() == pytest.approx(1 / 9, abs=1e-15)       # fourth-order isotropy
    assert sorted(order) == [0] + [1] * 3 + [2] * 6 + [3] * 6 + [4] * 3
    K = tcpo.central_moment_matrix(19, np.array([0.05, -0.03, 0.08]))
    assert np.linalg.cond(K) < 100


def test_poiseuille_profile_on_q19():
    """Single phase, body force, halfway bounce-back: u = g_x y (H - y) / (2 nu), nu = tau c_s^2 (A13, S6)."""
    ny, nu, gx = 20, 0.2, 1e-6
    o = tcpo.Oracle(1, ny, 1, dict(bc=("periodic", "walls", "periodic"), tau_H=3 * nu, tau_L=3 * nu, gravity=(gx, 0, 0),
                                   xi=1e30, hydro_lattice=19))
    o.init_fields(np.zeros((1, ny, 1)))
    o.step(6000)
    phi, u, p, T = o.read_fields()
    o.close()
    yy = np.arange(ny) + 0.5
    exact = gx / (2 * nu) * yy * (ny - yy)
    assert np.abs(u[0].ravel() - exact).max() / exact.max() < 2e-3
    assert np.abs(u[1:]).max() < 1e-15


def test_poiseuille_in_a_diagonal_channel_direction_on_q19():
    """Force along z between x walls: exercises the other axes of the lattice tables (19 velocities, bounce-back pairs)."""
    nx, nu, gz = 20, 0.15, 2e-6
    o = tcpo.Oracle(nx, 1, 1, dict(bc=("walls", "periodic", "periodic"), tau_H=3 * nu, tau_L=3 * nu, gravity=(0, 0, gz),
                                   xi=1e30, hydro_lattice=19))
    o.init_fields(np.zeros((1, 1, nx)))
    o.step(7000)
    u = o.read_fields()[1]
    o.close()
    xx = np.arange(nx) + 0.5
    exact = gz / (2 * nu) * xx * (nx - xx)
    assert np.abs(u[2].ravel() - exact).max() / exact.max() < 3e-3


def test_laplace_law_quasi_2d_droplet_on_q19():
    """dp = sigma / R within 5 %, spurious currents small, sum(phi) conserved (same bar as the D3Q27 pin)."""
    n, R = 32, 7.0
    wl = W.static_droplet(n=n, R=R, nz=1)
    o = tcpo.Oracle(n, n, 1, dict(wl.params, hydro_lattice=19))
    o.init_fields(wl.phi.numpy())
    o.step(600)
    phi, u, p, T = o.read_fields()
    o.close()
    dp = p[0, n // 2 - 1:n // 2 + 1, n // 2 - 1:n // 2 + 1].mean() - p[0, 0, 0]
    assert dp / (wl.params["sigma_ref"] / R) == pytest.approx(1.0, abs=0.05)
    assert np.abs(u).max() < 2e-6
    assert abs(phi.sum() - float(wl.phi.sum())) / float(wl.phi.sum()) < 1e-12


def test_bgk_mode_on_q19_is_plain_bgk_with_guo_forcing():
    """All rates equal on the Q19 basis: K^-1 (w I) K = w I, so one collision equals (1 - w) g + w g_eq + (1 - w/2) F
    computed here from the printed equilibrium (eq. 18) and Guo's populations with the D3Q19 weights."""
    rng = np.random.default_rng(2)
    c, w, opp, _ = tcpo.lattice(19)
    u = np.array([0.03, -0.02, 0.05]); a = np.array([1e-3, 2e-3, -1.5e-3]); om, ps = 1.3, 0.01
    g = w * (1 + 0.1 * rng.standard_normal(19))
    cu = c @ u
    geq = w * (ps + 3 * cu + 4.5 * cu ** 2 - 1.5 * u @ u)
    F = w * (3 * ((c - u) @ a) + 9 * cu * (c @ a))
    want = (1 - om) * g + om * geq + (1 - om / 2) * F
    got = tcpo.collide_cell(19, 1, [om] * 5, u, ps, a, g)
    assert np.abs(got - want).max() < 1e-15


def test_q19_and_q27_agree_on_a_smooth_marangoni_flow():
    """Both lattices discretise the same equations: on the layered channel (App. A set-up) after 400 steps the velocity
    fields agree to a few per cent of u_max (they differ in their O(u^2), O(dx^2) error terms only)."""
    wl = W.layered_channel(nx=24, ny=12, nz=1)
    res = []
    for Q in (27, 19):
        o = tcpo.Oracle(24, 12, 1, dict(wl.params, hydro_lattice=Q))
        for (ax, fc), plane in wl.wall_T.items():
            o.set_wall_temperature(ax, fc, plane.numpy())
        o.init_fields(wl.phi.numpy(), None, wl.T.numpy())
        o.step(400)
        res.append(o.read_fields()[1])
        o.close()
    assert np.abs(res[0]).max() > 5e-5
    assert np.abs(res[0] - res[1]).max() < 0.03 * np.abs(res[0]).max()
