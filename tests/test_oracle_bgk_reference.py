"""Pin P8: with `high_rate_equals_shear=1` every collision of the oracle must be
plain BGK + Guo.  The coupled step is re-coded here independently (numpy, np.roll, its own
velocity ordering, periodic box) as the textbook scheme and compared after a few steps.

A second implementation agreeing with the first is not proof that either reads the paper
correctly, but it does catch what a pin of a steady state cannot: a wrong pull direction, a
transposed index, a wrong time level, a dropped force term in a transient.
"""
import itertools

import numpy as np
import pytest

from oracle import tcpo

C27 = np.array(list(itertools.product((-1, 0, 1), repeat=3)))          # (cx, cy, cz), own order
W1 = {0: 2.0 / 3.0, 1: 1.0 / 6.0, -1: 1.0 / 6.0}
W27 = np.array([W1[a] * W1[b] * W1[c] for a, b, c in C27])            # = B.4 as a tensor product
C7 = np.array([(0, 0, 0), (1, 0, 0), (-1, 0, 0), (0, 1, 0), (0, -1, 0), (0, 0, 1), (0, 0, -1)])
W7 = np.array([0.0] + [1.0 / 6.0] * 6)


def shift(a, c):
    """a(x + c) on the periodic box; arrays are [z][y][x]."""
    return np.roll(a, (-c[2], -c[1], -c[0]), axis=(0, 1, 2))


def grad_lap(psi):
    g = np.zeros((3,) + psi.shape)
    lap = np.zeros_like(psi)
    for c, w in zip(C27, W27):
        v = shift(psi, c)
        for al in range(3):
            g[al] += 3.0 * w * c[al] * v
        lap += 6.0 * w * (v - psi)
    return g, lap


def eq(C, W, s, u, hydro=False):
    uu = (u ** 2).sum(0)
    out = []
    for c, w in zip(C, W):
        cu = c[0] * u[0] + c[1] * u[1] + c[2] * u[2]
        poly = 3 * cu + 4.5 * cu ** 2 - 1.5 * uu
        out.append(w * (s + poly) if hydro else s * w * (1 + poly))
    return np.array(out)


def guo(C, W, a, u):
    out = []
    for c, w in zip(C, W):
        cu = c[0] * u[0] + c[1] * u[1] + c[2] * u[2]
        out.append(w * sum((3 * (c[al] - u[al]) + 9 * cu * c[al]) * a[al] for al in range(3)))
    return np.array(out)


def pull(pop, C):
    return np.array([shift(pop[i], -C[i]) for i in range(len(C))])


class BGKReference:
    def __init__(self, p, phi, u, T, thermal):
        self.p, self.thermal = p, thermal
        self.phi, self.u, self.T = phi.copy(), u.copy(), T.copy()
        self.h = eq(C27, W27, phi, u)
        self.g = eq(C27, W27, 0.0 * phi, u, hydro=True)
        self.f = eq(C7, W7, T, u)

    def rhs(self, Y, phi, u):
        p = self.p
        gY, lY = grad_lap(Y)
        gP, _ = grad_lap(phi)
        kap = p["kappa_L"] + phi * (p["kappa_H"] - p["kappa_L"])
        rcp = (p["rho_L"] + phi * (p["rho_H"] - p["rho_L"])) * (p["cp_L"] + phi * (p["cp_H"] - p["cp_L"]))
        return -(u * gY).sum(0) + ((p["kappa_H"] - p["kappa_L"]) * (gP * gY).sum(0) + kap * lY) / rcp

    def step(self):
        p = self.p
        phi_n, u_n, T_n = self.phi, self.u, self.T
        # phase field (eqs. 10-15), force from phi^n, equilibrium from phi'
        hp = pull(self.h, C27)
        phi_new = hp.sum(0)
        G, lap = grad_lap(phi_n)
        nrm = np.sqrt((G ** 2).sum(0) + p["eps_normal"])
        a = (1.0 / 3.0) * 4 * phi_n * (1 - phi_n) / p["xi"] * G / nrm
        w_phi = 1.0 / (0.5 + 3.0 * p["M"])
        self.h = hp - w_phi * (hp - eq(C27, W27, phi_new, u_n)) + (1 - w_phi / 2) * guo(C27, W27, a, u_n)
        # hydrodynamics (eqs. 16-22), everything from phi^n (S16) and T^n
        gp = pull(self.g, C27)
        ps = gp.sum(0)
        j = np.einsum("ia,izyx->azyx", C27.astype(float), gp)
        rho = p["rho_L"] + phi_n * (p["rho_H"] - p["rho_L"])
        tau = p["tau_L"] + phi_n * (p["tau_H"] - p["tau_L"])
        Th, _ = grad_lap(T_n)
        sig = p["sigma_ref"] + p["sigma_T"] * (T_n - p["T_ref"])
        mu = 4 * (12 * sig / p["xi"]) * phi_n * (phi_n - 1) * (phi_n - 0.5) - 1.5 * sig * p["xi"] * lap
        GG, TG = (G * G).sum(0), (Th * G).sum(0)
        drho = p["rho_H"] - p["rho_L"]
        grav = np.array(p["gravity"]).reshape(3, 1, 1, 1)
        F0 = mu * G + 1.5 * p["xi"] * p["sigma_T"] * (GG * Th - TG * G) + rho * grav - ps / 3.0 * drho * G
        ustar = j + F0 / (2 * rho)
        neq = gp - eq(C27, W27, ps, ustar, hydro=True)
        Pi = np.einsum("ia,ib,izyx->abzyx", C27.astype(float), C27.astype(float), neq)
        Fmu = -(tau / (tau + 0.5)) * drho * np.einsum("abzyx,bzyx->azyx", Pi, G)
        F = F0 + Fmu
        u_new = j + F / (2 * rho)
        om = 1.0 / (tau + 0.5)
        self.g = gp - om * (gp - eq(C27, W27, ps, u_new, hydro=True)) + (1 - om / 2) * guo(C27, W27, F / rho, u_new)
        # temperature, with phi^{n+1} and u^{n+1}
        if self.thermal == "lb_d3q7":
            fp = pull(self.f, C7)
            T_new = fp.sum(0)
            kap = p["kappa_L"] + phi_new * (p["kappa_H"] - p["kappa_L"])
            w_T = 1.0 / (0.5 + 3.0 * kap)
            self.f = fp - w_T * (fp - eq(C7, W7, T_new, u_new))
        elif self.thermal == "rk2":
            K1 = self.rhs(T_n, phi_new, u_new)
            T_new = T_n + self.rhs(T_n + 0.5 * K1, phi_new, u_new)
        else:
            K1 = self.rhs(T_n, phi_new, u_new)
            K2 = self.rhs(T_n + 0.5 * K1, phi_new, u_new)
            K3 = self.rhs(T_n + 0.5 * K2, phi_new, u_new)
            K4 = self.rhs(T_n + K3, phi_new, u_new)
            T_new = T_n + K1 / 6 + K2 / 3 + K3 / 3 + K4 / 6
        self.phi, self.u, self.T = phi_new, u_new, T_new

    def pressure(self):
        rho = self.p["rho_L"] + self.phi * (self.p["rho_H"] - self.p["rho_L"])
        return rho * self.g.sum(0) / 3.0


@pytest.mark.parametrize("thermal", ["lb_d3q7", "rk2", "rk4"])
def test_oracle_bgk_mode_equals_textbook_bgk(thermal):
    nx, ny, nz = 10, 8, 6
    rng = np.random.default_rng(42)
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    r = np.sqrt((x - 4.3) ** 2 + (y - 3.6) ** 2 + (z - 2.8) ** 2)
    phi = 0.5 * (1 - np.tanh(2 * (r - 2.5) / 3.0))
    u = 0.02 * rng.standard_normal((3, nz, ny, nx))
    T = 1.0 + 0.5 * np.sin(2 * np.pi * x / nx) * np.cos(2 * np.pi * y / ny) + 0.1 * rng.random((nz, ny, nx))
    p = dict(tcpo.DEFAULTS)
    p.update(thermal=thermal, rho_H=5.0, rho_L=1.0, tau_H=0.7, tau_L=0.3, xi=3.0, M=0.03,
             sigma_ref=5e-3, sigma_T=-4e-4, T_ref=0.5, kappa_H=0.15, kappa_L=0.05, cp_H=2.0, cp_L=1.0,
             gravity=(1e-5, -2e-5, 3e-5), high_rate_equals_shear=1)
    o = tcpo.Oracle(nx, ny, nz, p)
    o.init_fields(phi, u, T)
    ref = BGKReference(p, phi, u, T, thermal)
    for _ in range(4):
        o.step(1)
        ref.step()
    ophi, ou, op, oT = o.read_fields()
    assert np.abs(ophi - ref.phi).max() < 1e-13
    assert np.abs(ou - ref.u).max() < 1e-13
    assert np.abs(oT - ref.T).max() < 1e-12
    assert np.abs(op - ref.pressure()).max() < 1e-13
    # the fields moved: this is not a comparison of two zeros
    assert np.abs(ou - u).max() > 1e-4 and np.abs(oT - T).max() > 1e-3 and np.abs(ophi - phi).max() > 1e-3
