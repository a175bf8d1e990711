"""Dynamic pins of the CPU oracle against what the paper and the mathematics fix
(SURVEY.md 8(c) P2-P7, P9-P11).  CPU only; sized so the file runs in about two minutes.

None of these compares the oracle with itself: every expected value is a closed form, a
conservation law, or a number the paper prints.
"""
import numpy as np
import pytest
from scipy.optimize import curve_fit

import workloads as W
from oracle import tcpo

THERMALS = ["lb_d3q7", "lb_d3q15", "lb_d3q19", "lb_d3q27", "rk2", "rk4"]


def _amp(field, mean, n):
    return 2 * np.abs(np.fft.rfft(field - mean)[1]) / n


# ---- P4: mobility (eq. 11 read as a rate, G3) --------------------------------------------------

def test_mobility_decay_rate():
    """Sharpening force off (xi -> inf): a phi sinusoid decays as exp(-M k^2 t)  (eq. 3 with the
    normal term removed is a diffusion equation with diffusivity M)."""
    n, M = 64, 0.05
    k = 2 * np.pi / n
    x = np.arange(n)
    o = tcpo.Oracle(n, 1, 1, dict(M=M, xi=1e30))
    o.init_fields((0.5 + 0.1 * np.sin(k * x)).reshape(1, 1, n))
    o.step(100); a1 = _amp(o.read_fields()[0].ravel(), 0.5, n)
    o.step(300); a2 = _amp(o.read_fields()[0].ravel(), 0.5, n)
    rate = -np.log(a2 / a1) / 300
    assert rate == pytest.approx(M * k * k, rel=0.01)


# ---- P5: heat equation closed forms, all six thermal variants ---------------------------------

@pytest.mark.parametrize("thermal", THERMALS)
@pytest.mark.parametrize("axis", [0, 1, 2])
def test_heat_sinusoid_decay_and_advection(thermal, axis):
    """u uniform, rho c_p = 1, uniform kappa: T = 1 + A sin(k (x - u t)) exp(-kappa k^2 t)
    (eq. 4 / eqs. 27-29).  Pins omega_T <-> kappa (G4), the advection term's sign and the axis
    bookkeeping of every stencil."""
    n, kap, U, steps = 48, 0.1, 0.04, 120
    k = 2 * np.pi / n
    shape = [1, 1, 1]; shape[2 - axis] = n
    s = np.arange(n)
    T0 = (1 + 0.5 * np.sin(k * s)).reshape(shape)
    u0 = np.zeros([3] + shape); u0[axis] = U
    o = tcpo.Oracle(shape[2], shape[1], shape[0], dict(thermal=thermal, kappa_H=kap, kappa_L=kap, xi=1e30))
    o.init_fields(np.zeros(shape), u=u0, T=T0)
    o.step(steps)
    T = o.read_fields()[3].ravel()
    F = np.fft.rfft(T - 1)[1]
    decay = -np.log(2 * np.abs(F) / n / 0.5) / steps
    shift_cells = (-np.angle(F) - np.pi / 2) / k
    assert decay == pytest.approx(kap * k * k, rel=0.02)
    assert shift_cells == pytest.approx(U * steps, rel=0.01)
    assert T.sum() == pytest.approx(T0.sum(), abs=1e-10)          # energy conserved (periodic)


@pytest.mark.parametrize("thermal", THERMALS)
def test_uniform_heat_source_raises_temperature_linearly(thermal):
    """q_T of eqs. 4 / 27 on a uniform, quiescent periodic box: dT/dt = q exactly.  RK: T^n = T0 + n q.
    LB: the + w_i q_T of eq. 27 is added after the collision, so it shows in T = sum f one step later:
    T^n = T0 + (n - 1) q."""
    n, q, T0, steps = 6, 2.5e-3, 0.7, 40
    o = tcpo.Oracle(n, n, n, dict(thermal=thermal, xi=1e30))
    o.set_heat_source(np.full((n, n, n), q))
    o.init_fields(np.zeros((n, n, n)), T=np.full((n, n, n), T0))
    o.step(steps)
    T = o.read_fields()[3]
    expect = T0 + (steps - 1 if thermal.startswith("lb") else steps) * q
    assert np.abs(T - expect).max() < 1e-12


@pytest.mark.parametrize("thermal", THERMALS)
def test_two_wall_conduction_is_linear_through_wall_values(thermal):
    """S9: Dirichlet walls half a cell outside the end cells; steady profile linear and equal to
    T_w at y = -1/2 and y = ny - 1/2, also across a conductivity jump-free slab."""
    ny = 12
    p = dict(thermal=thermal, bc=("periodic", "walls", "periodic"), kappa_H=0.25, kappa_L=0.25,
             wall_T=((0, 0), (2.0, 5.0), (0, 0)))
    o = tcpo.Oracle(1, ny, 1, p)
    o.init_fields(np.zeros((1, ny, 1)), T=np.full((1, ny, 1), 3.0))
    o.step(2500)
    T = o.read_fields()[3].ravel()
    exact = 2.0 + 3.0 * (np.arange(ny) + 0.5) / ny
    assert np.abs(T - exact).max() < 1e-9


@pytest.mark.parametrize("thermal", ["lb_d3q7", "rk2"])
def test_two_layer_conduction_follows_conductivity_ratio(thermal):
    """Steady 1-D conduction through two layers with k_H/k_L = 1/5 (k* = 1/5):
    heat flux continuity gives the piecewise-linear closed form (the linear part of App. A, G8).
    Pins S11 (omega_T from the local kappa(phi)) and G5."""
    ny = 64
    wl = W.layered_channel(nx=1, ny=ny, nz=1, thermal=thermal, kappa_upper=0.04)
    wl.params["sigma_T"] = 0.0
    wl.params["sigma_ref"] = 0.0
    a = b = ny / 2.0
    k_r = 0.2
    yi = np.arange(ny) - (ny / 2 - 0.5)
    den = a + k_r * b
    exact = np.where(yi > 0, ((10.0 - 20.0) * yi + k_r * 10.0 * b + 20.0 * a) / den,
                     (k_r * (10.0 - 20.0) * yi + k_r * 10.0 * b + 20.0 * a) / den)
    o = tcpo.Oracle(1, ny, 1, wl.params)
    # start from a deliberately wrong (single-slope) profile so the kink has to form by itself
    o.init_fields(wl.phi.numpy(), T=(20.0 - 10.0 * (np.arange(ny) + 0.5) / ny).reshape(1, ny, 1))
    o.set_wall_temperature(1, 0, np.full((1, 1), 20.0))
    o.step(25000)
    T = o.read_fields()[3].ravel()
    # diffuse interface (xi = 4) smears the kink: the paper's own l2(T) at k*=1/5 is 5.6e-3 (Table 1)
    l2 = np.sqrt(((T - exact) ** 2).sum() / (exact ** 2).sum())
    assert l2 < 8e-3
    assert np.abs(T[[0, -1]] - exact[[0, -1]]).max() < 0.05


# ---- P6: Poiseuille ---------------------------------------------------------------------------

def test_poiseuille_profile():
    """Single phase, body force g_x, halfway bounce-back walls: u = g_x y (H - y) / (2 nu),
    H = ny, nu = tau c_s^2 (A13; S6 half-force velocity)."""
    ny, nu, gx = 24, 0.2, 1e-6
    o = tcpo.Oracle(1, ny, 1, dict(bc=("periodic", "walls", "periodic"), tau_H=3 * nu, tau_L=3 * nu,
                                   gravity=(gx, 0, 0), xi=1e30))
    o.init_fields(np.zeros((1, ny, 1)))
    o.step(9000)
    phi, u, p, T = o.read_fields()
    yy = np.arange(ny) + 0.5
    exact = gx / (2 * nu) * yy * (ny - yy)
    assert np.abs(u[0].ravel() - exact).max() / exact.max() < 2e-3
    assert np.abs(u[1:]).max() < 1e-15


def test_two_layer_poiseuille_with_density_contrast():
    """Body-force driven two-layer channel with rho_H/rho_L = 3 and equal kinematic viscosity:
    F_b = rho g (eq. 7) so the acceleration is uniform and, with equal nu, the sharp-interface
    solution is again the single-phase parabola only if F_p and F_mu (eqs. 20-21) supply the
    rho-gradient terms of eq. 6 correctly.  A wrong sign of F_mu gives a kink of several per cent."""
    ny, nu, gx = 32, 0.2, 1e-6
    wl = W.layered_channel(nx=1, ny=ny, nz=1, rho_upper=3.0)
    wl.params.update(sigma_T=0.0, sigma_ref=1e-3, gravity=(gx, 0.0, 0.0))
    o = tcpo.Oracle(1, ny, 1, wl.params)
    o.init_fields(wl.phi.numpy(), T=np.full((1, ny, 1), 10.0))
    o.step(12000)
    phi, u, p, T = o.read_fields()
    # sharp-interface closed form: mu_i u_i'' = -rho_i g, continuity of u and of mu u' at the interface
    yy = np.arange(ny) + 0.5
    h = ny / 2.0
    mu1, mu2, r1, r2 = nu * 1.0, nu * 3.0, 1.0, 3.0      # lower (L), upper (H)
    # u1 = -r1 g y^2/(2 mu1) + A1 y ;  u2 = -r2 g (y-H)^2/(2 mu2) + A2 (y-H)
    H = float(ny)
    Am = np.array([[h, -(h - H)], [mu1, -mu2]])
    rhs = np.array([r1 * gx * h ** 2 / (2 * mu1) - r2 * gx * (h - H) ** 2 / (2 * mu2),
                    r1 * gx * h - r2 * gx * (h - H)])
    A1, A2 = np.linalg.solve(Am, rhs)
    exact = np.where(yy < h, -r1 * gx * yy ** 2 / (2 * mu1) + A1 * yy,
                     -r2 * gx * (yy - H) ** 2 / (2 * mu2) + A2 * (yy - H))
    err = np.abs(u[0].ravel() - exact).max() / exact.max()
    assert err < 0.02


# ---- P2, P3: conservation and the tanh profile ------------------------------------------------

def test_flat_interface_relaxes_to_tanh_of_width_xi_and_conserves_phi():
    """Eqs. 3, 15, 35 with readings S7, G1: started too wide (W = 6) the interface sharpens to
    phi = 1/2 [1 + tanh(2 (x - x0) / xi)], xi = 4; sum(phi) is conserved to round-off (P2)."""
    n, xi = 64, 4.0
    x = np.arange(n)
    phi0 = 0.5 * (np.tanh(2 * (x - 15.5) / 6.0) - np.tanh(2 * (x - 47.5) / 6.0))
    o = tcpo.Oracle(n, 1, 1, dict(M=0.05, xi=xi))
    o.init_fields(phi0.reshape(1, 1, n))
    o.step(1500)
    phi = o.read_fields()[0].ravel()
    f = lambda x, x0, Wd: 0.5 * (1 + np.tanh(2 * (x - x0) / Wd))
    (x0, Wd), _ = curve_fit(f, x[:32], phi[:32], p0=(15.5, 5.0))
    assert Wd == pytest.approx(xi, rel=0.02)
    assert x0 == pytest.approx(15.5, abs=1e-3)
    assert abs(phi.sum() - phi0.sum()) / phi0.sum() < 1e-12
    assert phi.min() > -1e-6 and phi.max() < 1 + 1e-6


# ---- P7: Laplace law ---------------------------------------------------------------------------

def test_laplace_law_quasi_2d_droplet():
    """Static cylinder, rho ratio 10 (config 1 fluid): dp = sigma / R within 5 %, spurious
    currents tiny, sum(phi) conserved (eq. 8 calibration with mu_phi of S5; p = c_s^2 rho p*, A12)."""
    n, R = 40, 8.0
    wl = W.static_droplet(n=n, R=R, nz=1)
    o = tcpo.Oracle(n, n, 1, wl.params)
    o.init_fields(wl.phi.numpy())
    o.step(800)
    phi, u, p, T = o.read_fields()
    dp = p[0, n // 2 - 1:n // 2 + 1, n // 2 - 1:n // 2 + 1].mean() - p[0, 0, 0]
    assert dp / (wl.params["sigma_ref"] / R) == pytest.approx(1.0, abs=0.05)
    assert np.abs(u).max() < 2e-6
    assert abs(phi.sum() - float(wl.phi.sum())) / float(wl.phi.sum()) < 1e-12


def test_laplace_law_3d_droplet_config1_short():
    """BASELINE.json configs[0] at reduced size/steps (24^3, R = 6, 150 steps): dp -> 2 sigma / R."""
    n, R = 24, 6.0
    wl = W.static_droplet(n=n, R=R)
    o = tcpo.Oracle(n, n, n, wl.params)
    o.init_fields(wl.phi.numpy())
    o.step(150)
    phi, u, p, T = o.read_fields()
    c = n // 2
    dp = p[c - 1:c + 1, c - 1:c + 1, c - 1:c + 1].mean() - p[0, 0, 0]
    assert dp / (2 * wl.params["sigma_ref"] / R) == pytest.approx(1.0, abs=0.08)
    assert abs(phi.sum() - float(wl.phi.sum())) / float(wl.phi.sum()) < 1e-12


# ---- P9, P10: layered thermocapillary channel vs App. A ----------------------------------------

def _l2(num, ana):
    return np.sqrt(((np.abs(num) - np.abs(ana)) ** 2).sum() / (ana ** 2).sum())      # eq. 36


@pytest.fixture(scope="module")
def channel_runs():
    nx, ny, steps = 48, 24, 1800
    out = {}
    xn = np.arange(nx)[None, :]
    yn = (np.arange(ny) - (ny / 2 - 0.5))[:, None]
    ua, va, Ta, Umax = W.layered_channel_closed_form(xn, yn, a=ny / 2, b=ny / 2, L=float(nx), T_h=20, T_c=10,
                                                     T_0=4, k_r=1.0, mu_r=1.0, mu_B=0.2, sigma_T=-5e-4)
    for th in ("lb_d3q7", "lb_d3q19", "rk2"):
        wl = W.layered_channel(nx, ny, 1, thermal=th)
        o = tcpo.Oracle(nx, ny, 1, wl.params)
        o.init_fields(wl.phi.numpy(), T=wl.T.numpy())
        for (ax, fc), v in wl.wall_T.items():
            o.set_wall_temperature(ax, fc, v.numpy())
        o.step(steps)
        out[th] = o.read_fields()
    return out, (ua, va, Ta, Umax)


def test_layered_channel_matches_closed_form(channel_runs):
    """P9: u, v, T of the two-layer heated channel against App. A (G8).  At this
    resolution the diffuse interface smears the velocity cusp: the paper itself has l2(u) = 9.2e-2 at
    512x256 (Table 1); what must hold is the flow pattern (correlation), its sign and its scale."""
    runs, (ua, va, Ta, Umax) = channel_runs
    phi, u, p, T = runs["lb_d3q7"]
    assert _l2(T[0], Ta) < 1e-3
    cu = np.corrcoef(u[0, 0].ravel(), ua.ravel())[0, 1]
    cv = np.corrcoef(u[1, 0].ravel(), va.ravel())[0, 1]
    assert cu > 0.99 and cv > 0.99                                  # sign and pattern of the Marangoni flow
    assert _l2(u[0, 0], ua) < 0.30 and _l2(u[1, 0], va) < 0.30
    peak = np.abs(u[0, 0]).max() / np.abs(ua).max()
    assert 0.6 < peak < 1.05
    assert np.abs(u[2]).max() < 1e-15


def test_thermal_variants_agree_on_channel(channel_runs):
    """P10: Tables 1-2: the thermal stencil / RK choice does not change the result."""
    runs, _ = channel_runs
    ref = runs["lb_d3q7"]
    for th in ("lb_d3q19", "rk2"):
        got = runs[th]
        assert np.abs(got[3] - ref[3]).max() / np.abs(ref[3]).max() < 2e-3          # T
        assert np.abs(got[1] - ref[1]).max() / np.abs(ref[1]).max() < 2e-2          # u


# ---- P11: Marangoni direction ------------------------------------------------------------------

def test_droplet_migrates_toward_hot_wall():
    """sigma_T < 0 (eq. 9): the droplet of config 3 moves toward the hot wall (+z); thermal LB and
    RK4 agree on the displacement."""
    zc = {}
    for th in ("lb_d3q19", "rk4"):
        wl = W.droplet_in_gradient(nx=32, ny=1, nz=40, thermal=th, R=7.0, zc=17.0, grad_T=0.05)
        o = tcpo.Oracle(32, 1, 40, wl.params)
        o.init_fields(wl.phi.numpy(), T=wl.T.numpy())
        o.step(600)
        phi = o.read_fields()[0]
        zc[th] = float((phi * np.arange(40)[:, None, None]).sum() / phi.sum())
        assert abs(phi.sum() - float(wl.phi.sum())) / float(wl.phi.sum()) < 1e-12
    assert zc["lb_d3q19"] - 17.0 > 0.02
    assert zc["lb_d3q19"] == pytest.approx(zc["rk4"], abs=1e-3)


# ---- NEXT-1 ingredients: moving wall and temperature pre-initialisation ----

def _wall_u(axis, face, vec):
    w = [[[0.0] * 3 for _ in range(2)] for _ in range(3)]
    w[axis][face] = list(vec)
    return w


def test_couette_flow_from_a_moving_wall():
    """Top wall moving with U_w, bottom wall at rest (reading S18: velocity bounce-back on g):
    steady u(y) = U_w (y + 1/2) / H, walls half a cell outside the end cells."""
    ny, U, nu = 16, 0.01, 0.2
    o = tcpo.Oracle(3, ny, 2, dict(bc=("periodic", "walls", "periodic"), tau_H=3 * nu, tau_L=3 * nu, xi=1e30,
                                   wall_u=_wall_u(1, 1, (U, 0.0, 0.0))))
    o.init_fields(np.zeros((2, ny, 3)))
    o.step(7000)
    u = o.read_fields()[1]
    exact = U * (np.arange(ny) + 0.5) / ny
    assert np.abs(u[0, 0, :, 0] - exact).max() < 1e-8
    assert np.abs(u[1:]).max() < 1e-15


def test_two_layer_couette_with_viscosity_contrast():
    """Two layers with nu_H / nu_L = 4 (tau interpolated by phi, eq. 22) sheared by a moving top wall:
    the stress mu du/dy is uniform, so the sharp-interface profile is piecewise linear with slopes in the
    ratio nu_L / nu_H."""
    ny, U = 32, 0.01
    wl = W.layered_channel(nx=1, ny=ny, nz=1)
    wl.params.update(sigma_T=0.0, sigma_ref=0.0, tau_H=1.2, tau_L=0.3, wall_u=_wall_u(1, 1, (U, 0.0, 0.0)))
    o = tcpo.Oracle(1, ny, 1, wl.params)
    o.init_fields(wl.phi.numpy(), T=np.full((1, ny, 1), 10.0))
    o.step(15000)
    u = o.read_fields()[1][0].ravel()
    h = ny / 2.0
    nuL, nuH = 0.3 / 3, 1.2 / 3                       # lower layer = L, upper = H
    sL = U / (h + h * nuL / nuH)                      # slope in the lower layer; upper slope = sL nuL / nuH
    yy = np.arange(ny) + 0.5
    exact = np.where(yy < h, sL * yy, sL * h + sL * nuL / nuH * (yy - h))
    assert np.abs(u - exact).max() / U < 0.04          # diffuse interface (xi = 4) rounds the kink
    slope_lo = (u[8] - u[2]) / 6.0
    slope_up = (u[29] - u[23]) / 6.0
    assert slope_lo / slope_up == pytest.approx(nuH / nuL, rel=0.03)     # uniform shear stress


@pytest.mark.parametrize("thermal", ["lb_d3q7", "lb_d3q19", "rk2", "rk4"])
def test_temperature_preinitialisation_reaches_steady_conduction(thermal):
    """tcpo_relax_temperature: the thermal solver alone, phi / u / h / g frozen, relaxes a uniform initial
    temperature to the steady conduction field of the heated channel, App. A (k* = 1: harmonic T)."""
    nx, ny = 32, 16
    wl = W.layered_channel(nx, ny, 1, thermal=thermal)
    o = tcpo.Oracle(nx, ny, 1, wl.params)
    for (ax, fc), v in wl.wall_T.items():
        o.set_wall_temperature(ax, fc, v.numpy())
    o.init_fields(wl.phi.numpy(), T=np.full((1, ny, nx), 15.0))
    h0, g0 = o.read_populations(0), o.read_populations(1)
    o.relax_temperature(2500)
    phi, u, p, T = o.read_fields()
    Ta = wl.T.numpy()
    assert np.sqrt(((T - Ta) ** 2).sum() / (Ta ** 2).sum()) < 1e-3
    assert np.array_equal(h0, o.read_populations(0)) and np.array_equal(g0, o.read_populations(1))
    assert np.array_equal(phi, wl.phi.numpy()) and np.abs(u).max() == 0.0
