"""Pins of reading S20, the wetting (contact-angle) boundary condition (PAPER.md:307 names it and cites refs. [34], [35];
no formula is printed): ghost value of phi behind a wall from  n_w . grad phi = -(4 / xi) cos(theta) phi_w (1 - phi_w).

None of these compares the oracle with itself:
  * the ghost rule against the closed-form equilibrium profile (eq. 35) of a planar interface that meets the
    wall at the angle theta -- the analytic wall-normal gradient, second-order convergence;
  * theta = 90 degrees is the mirror ghost of S9, bit for bit;
  * a sessile 2-D droplet started as a half disc (90 degrees) relaxes to a circular cap whose height / base-half-width
    ratio is tan(theta / 2) (geometry of a circular segment), within 3 degrees, for theta = 60 and 120;
  * sum(phi) stays conserved to round-off (the ghost rule touches the stencils, not the populations).
"""
import numpy as np
import pytest

from oracle import tcpo


def _inclined_profile(nx, ny, xi, theta_deg, x0, top=False):
    """phi = 1/2 [1 + tanh(2 s / xi)], s = signed distance into the phi = 1 fluid, of a planar interface through the
    wall point (x0, Y = 0) with contact angle theta inside phi = 1 (which lies on the side x < x0).  Y = distance from the
    wall (bottom wall: y + 1/2; top wall: ny - 1/2 - y)."""
    th = np.radians(theta_deg)
    x = np.arange(nx)[None, :] - x0
    Y = (np.arange(ny)[:, None] + 0.5) if not top else (ny - 0.5 - np.arange(ny)[:, None])
    s = -np.sin(th) * x - np.cos(th) * Y
    phi = 0.5 * (1 + np.tanh(2 * s / xi))
    dphi_dY = (4 / xi) * phi * (1 - phi) * (-np.cos(th))          # wall-normal derivative, pointing into the fluid
    return phi, dphi_dY


@pytest.mark.parametrize("theta", [30.0, 60.0, 120.0, 150.0])
@pytest.mark.parametrize("top", [False, True])
def test_ghost_rule_reproduces_the_wall_normal_gradient_of_the_inclined_tanh_profile(theta, top):
    nx, ny = 96, 24
    errs = []
    for xi in (6.0, 12.0):
        phi, dY = _inclined_profile(nx, ny, xi, theta, x0=47.3, top=top)
        angles = [[90.0, 90.0], [90.0, 90.0], [90.0, 90.0]]
        angles[1][1 if top else 0] = theta
        o = tcpo.Oracle(nx, ny, 1, dict(bc=("periodic", "walls", "periodic"), xi=xi, wall_contact_angle=angles))
        grad, lap = o.fd(phi.reshape(1, ny, nx), is_temp=False)
        o.close()
        row = ny - 1 if top else 0
        gy = grad[1][0, row] * (-1.0 if top else 1.0)             # derivative along the wall normal into the fluid
        sl = slice(20, 76)                                       # away from the periodic seam of the (non-periodic) profile
        scale = np.abs(dY[row, sl]).max()
        errs.append(np.abs(gy[sl] - dY[row, sl]).max() / scale)
        # the same row with the neutral (mirror) ghost is wrong by O(1): the pin discriminates
        o = tcpo.Oracle(nx, ny, 1, dict(bc=("periodic", "walls", "periodic"), xi=xi))
        g0, _ = o.fd(phi.reshape(1, ny, nx), is_temp=False)
        o.close()
        assert np.abs(g0[1][0, row, sl] * (-1.0 if top else 1.0) - dY[row, sl]).max() / scale > 0.4
    assert errs[0] < 0.08 and errs[1] < 0.02
    assert errs[0] / errs[1] > 3.0                               # second order in 1 / xi


def test_neutral_angle_is_the_mirror_ghost_bit_for_bit():
    rng = np.random.default_rng(4)
    nx, ny, nz = 9, 7, 5
    phi = rng.random((nz, ny, nx))
    bc = ("walls", "walls", "walls")
    a = tcpo.Oracle(nx, ny, nz, dict(bc=bc))
    b = tcpo.Oracle(nx, ny, nz, dict(bc=bc, wall_contact_angle=((90.0, 90.0),) * 3))
    ga, la = a.fd(phi, is_temp=False)
    gb, lb = b.fd(phi, is_temp=False)
    assert np.array_equal(ga, gb) and np.array_equal(la, lb)
    # and the mirror ghost means: zero wall-normal gradient contribution from the ghost layer on a field constant along y
    c = tcpo.Oracle(nx, ny, nz, dict(bc=bc, wall_contact_angle=((90.0, 90.0), (60.0, 90.0), (90.0, 90.0))))
    gc, _ = c.fd(phi, is_temp=False)
    assert not np.array_equal(gc[1][:, 0], ga[1][:, 0])           # the low-y wall now differs ...
    assert np.array_equal(gc[1][:, 2:], ga[1][:, 2:])             # ... and only there
    for o in (a, b, c):
        o.close()


def _cap_angle(phi):
    """Contact angle of a circular cap from its height H (sharp-interface equivalent: integral of phi up the symmetry
    column) and its base width at the wall (row widths at Y = 1/2, 3/2 extrapolated to Y = 0): tan(theta/2) = H / (base/2)."""
    nx = phi.shape[1]
    xc = (phi.sum(axis=0) * np.arange(nx)).sum() / phi.sum()
    lo = int(np.floor(xc)); w = xc - lo
    H = (1 - w) * phi[:, lo].sum() + w * phi[:, lo + 1].sum()
    w0, w1 = phi[0].sum(), phi[1].sum()
    base = w0 + 0.5 * (w0 - w1)
    return 2 * np.degrees(np.arctan(H / (0.5 * base)))


@pytest.mark.parametrize("theta,steps", [(60.0, 1200), (120.0, 1000)])
def test_sessile_droplet_relaxes_to_the_prescribed_contact_angle(theta, steps):
    nx, ny, R, xi = 46, 18, 8.0, 4.0
    x = np.arange(nx)[None, :]; Y = np.arange(ny)[:, None] + 0.5
    phi0 = 0.5 * (1 - np.tanh(2 * (np.sqrt((x - (nx - 1) / 2) ** 2 + Y ** 2) - R) / xi))      # half disc: 90 degrees
    assert _cap_angle(phi0) == pytest.approx(90.0, abs=1.5)
    p = dict(bc=("periodic", "walls", "periodic"), xi=xi, M=0.05, sigma_ref=5e-2, tau_H=0.5, tau_L=0.5, eps_normal=1e-9,
             wall_contact_angle=((90.0, 90.0), (theta, 90.0), (90.0, 90.0)))
    o = tcpo.Oracle(nx, ny, 1, p)
    o.init_fields(phi0.reshape(1, ny, nx))
    o.step(steps)
    phi, u, _, _ = o.read_fields()
    o.close()
    assert _cap_angle(phi[0]) == pytest.approx(theta, abs=3.0)       # measured 61.3 / 117.6 at these step counts; 59.2 / 118.3 after 3000
    assert abs(phi.sum() - phi0.sum()) / phi0.sum() < 1e-12
    assert np.abs(u).max() < 1e-3                                      # settling, not flying apart
