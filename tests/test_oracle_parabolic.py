"""Pins of the oracle's parabolic surface tension sigma(T) = sigma_ref + sigma_T (T - T_ref) + sigma_TT (T - T_ref)^2 / 2
(fluids with "a parabolic (or non-linear) relation between surface tension and temperature";
SURVEY.md 8(f) NEXT-4; reading S19).  The paper prints no worked example for it, so the pins are what the
mathematics fixes: a polynomial may be expanded about any reference temperature, a parabola seen from far away is a
straight line of slope sigma_TT (T - T_ref), and along a sinusoidally heated interface d sigma/dx changes sign four
times per period instead of twice.  CPU only.
"""
import numpy as np

import workloads as W
from oracle import tcpo

NX, NY = 32, 16          # the oracle solves three dense 27 x 27 systems per cell and step: keep it small


def _run(extra, steps=300, thermal="lb_d3q7", walls=None):
    """Config-2 channel; walls = (T_h, T_c) replaces the 20 / 10 of the config (bottom wall T_h + 4 cos(2 pi x / L))."""
    wl = W.layered_channel(NX, NY, 1, thermal=thermal)
    params = dict(wl.params, eps_normal=1e-8)      # S8: keeps the bulk normal well conditioned, so that
    params.update(extra)                           # round-off differences between two runs stay round-off
    T0, Tw = wl.T.numpy(), {k: v.numpy() for k, v in wl.wall_T.items()}
    if walls is not None:
        T_h, T_c = walls
        xn = np.arange(NX)[None, :]
        yn = (np.arange(NY) - (NY / 2 - 0.5))[:, None]
        T0 = W.layered_channel_closed_form(xn, yn, a=NY / 2, b=NY / 2, L=float(NX), T_h=T_h, T_c=T_c, T_0=4, k_r=1.0,
                                           mu_r=1.0, mu_B=0.2, sigma_T=-5e-4)[2][None]
        Tw = {(1, 0): (T_h + 4.0 * np.cos(2 * np.pi * np.arange(NX) / NX))[None, :]}
        params["wall_T"] = ((0.0, 0.0), (T_h, T_c), (0.0, 0.0))
    o = tcpo.Oracle(NX, NY, 1, params)
    o.init_fields(wl.phi.numpy(), T=T0)
    for (ax, fc), v in Tw.items():
        o.set_wall_temperature(ax, fc, v)
    o.step(steps)
    out = o.read_fields()
    o.close()
    return out


def test_expansion_about_another_reference_temperature_changes_nothing():
    """sigma and d sigma/dT of the same parabola written about T_ref and about T_ref + d: a dropped 1/2, a sign or a
    mismatch between sigma (chemical potential) and d sigma/dT (Marangoni term) breaks the equality."""
    s0, s1, s2, Tr, d = 2.5e-2, -5e-4, 4e-5, 10.0, 7.3
    a = _run(dict(sigma_ref=s0, sigma_T=s1, sigma_TT=s2, T_ref=Tr))
    b = _run(dict(sigma_ref=s0 + s1 * d + 0.5 * s2 * d * d, sigma_T=s1 + s2 * d, sigma_TT=s2, T_ref=Tr + d))
    assert np.abs(a[1]).max() > 1e-5                      # there is a flow to compare
    for fa, fb in zip(a, b):
        assert np.abs(fa - fb).max() <= 1e-10 * max(1.0, np.abs(fa).max())
    # and the parabolic term is not a no-op
    lin = _run(dict(sigma_ref=s0, sigma_T=s1, sigma_TT=0.0, T_ref=Tr))
    assert np.abs(a[1] - lin[1]).max() > 0.2 * np.abs(lin[1]).max()


def test_far_from_its_vertex_a_parabola_is_the_linear_law():
    """sigma_TT means d^2 sigma / dT^2: with the vertex 2015 K below the channel, d sigma/dT = sigma_TT (T - T_ref) is the
    linear law's sigma_T to within 0.5 %, and so is the flow (a factor 2 or 1/2 anywhere gives 50-100 %)."""
    sT, Tm, far = -5e-4, 15.0, -2000.0
    sTT = sT / (Tm - far)
    lin = _run(dict(sigma_ref=2.5e-2, sigma_T=sT, sigma_TT=0.0, T_ref=Tm))
    par = _run(dict(sigma_ref=2.5e-2 - 0.5 * sTT * (Tm - far) ** 2, sigma_T=0.0, sigma_TT=sTT, T_ref=far))
    scale = np.abs(lin[1]).max()
    assert scale > 1e-5
    assert np.abs(par[1] - lin[1]).max() < 0.02 * scale
    assert np.abs(par[3] - lin[3]).max() < 1e-6 * np.abs(lin[3]).max()


def test_surface_flow_toward_the_larger_surface_tension_doubles_its_wavenumber():
    """Vertex at the mean interface temperature, sigma_TT > 0 (a self-rewetting fluid): along the interface
    T = T_m + dT cos(kx), so d sigma/dx = -sigma_TT dT^2 k sin(2kx)/2 -- the interface is pulled toward BOTH the hottest
    (x = 0) and the coldest (x = L/2) point, four convection-cell boundaries per period, while the linear law
    (sigma_T < 0) pulls it from the hot toward the cold point only."""
    # both walls at 15 on average: no temperature gradient across the (four cells wide) diffuse interface
    par = _run(dict(sigma_ref=2.5e-2, sigma_T=0.0, sigma_TT=2e-4, T_ref=15.0), steps=400, walls=(15.0, 15.0))
    lin = _run(dict(sigma_ref=2.5e-2, sigma_T=-5e-4, sigma_TT=0.0, T_ref=15.0), steps=400, walls=(15.0, 15.0))
    row = NY // 2                                           # cell row just above the interface
    spec = lambda f: np.abs(np.fft.rfft(f[1][0, 0, row, :]))
    sp, sl = spec(par), spec(lin)
    assert sp[2] > 10 * sp[1] and sp[2] > 10 * sp[3:].max()
    assert sl[1] > 10 * sl[2]
    ux = par[1][0, 0, row, :]
    assert ux[NX // 8] < 0 < ux[3 * NX // 8] and ux[5 * NX // 8] < 0 < ux[7 * NX // 8]
    uxl = lin[1][0, 0, row, :]
    assert uxl[NX // 4] > 0 > uxl[3 * NX // 4]             # hot (x = 0) to cold (x = L/2) on both sides
