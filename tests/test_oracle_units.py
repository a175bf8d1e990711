"""Unit-level pins of the CPU oracle (oracle/tcpo.c): lattices, central-moment operator,
finite-difference operators, ghost rules.  CPU only."""
import os
from fractions import Fraction

import numpy as np
import pytest

from oracle import tcpo

QS = (7, 15, 19, 27)


# ---- P1: lattice weights (App. B) -------------------------------------------

def _golden_weights(golden_dir):
    out = {}
    for line in open(os.path.join(golden_dir, "appendix_b_weights.txt")):
        if line.startswith("#") or not line.strip():
            continue
        name, cls, cnt, num, den = line.split()
        out.setdefault(int(name[3:]), {})[int(cls)] = (int(cnt), Fraction(int(num), int(den)))
    return out


@pytest.mark.parametrize("Q", QS)
def test_weights_match_appendix_b(Q, golden_dir):
    gold = _golden_weights(golden_dir)[Q]
    c, w, opp, order = tcpo.lattice(Q)
    assert len(set(map(tuple, c))) == Q
    cls = (c ** 2).sum(1)
    for k, (cnt, frac) in gold.items():
        assert (cls == k).sum() == cnt
        assert np.allclose(w[cls == k], float(frac), rtol=0, atol=1e-17)
    assert set(cls) == set(gold)
    # isotropy conditions the method relies on: sum w = 1, sum w c = 0, sum w c c = c_s^2 I, c_s^2 = 1/3
    assert w.sum() == pytest.approx(1.0, abs=1e-15)
    assert np.allclose(w @ c, 0, atol=1e-16)
    assert np.allclose(np.einsum("i,ia,ib->ab", w, c, c), np.eye(3) / 3, atol=1e-15)
    # opposite directions
    assert np.array_equal(c[opp], -c)
    assert order[0] == 0 and sorted(order[1:4]) == [1, 1, 1]


def test_thermal_bytes_formula(golden_dir):
    """n_b = (2Q+4)*8 -> 144 B for D3Q7 (sanity of the byte accounting in DESIGN.md)."""
    q, nb = map(int, [l for l in open(os.path.join(golden_dir, "thermal_lb_bytes.txt")) if not l.startswith("#")][0].split())
    assert (2 * q + 4) * 8 == nb


# ---- central-moment matrix and generic collision (readings S1, S2) ----------------------------

@pytest.mark.parametrize("Q", QS)
def test_central_moment_matrix_properties(Q):
    rng = np.random.default_rng(Q)
    c, w, opp, order = tcpo.lattice(Q)
    K0 = tcpo.central_moment_matrix(Q, np.zeros(3))
    assert np.allclose(K0[0], 1.0)                               # zeroth moment row
    rows = lambda A: sorted(map(tuple, np.round(A, 12)))
    assert rows(K0[1:4]) == rows(c.T.astype(float))              # first raw moments (any axis order)
    for _ in range(5):
        u = rng.uniform(-0.3, 0.3, 3)
        K = tcpo.central_moment_matrix(Q, u)
        assert rows(K[1:4]) == rows((c - u).T)                   # central: shifted by u
        # unisolvent, and the raw->central shift has determinant 1 (SURVEY.md 8(c) "facts verified")
        assert np.linalg.cond(K) < 100
        assert np.linalg.det(K @ np.linalg.inv(K0)) == pytest.approx(1.0, abs=1e-10)
        # translation invariance: K(u) K(0)^-1 is lower triangular w.r.t. moment order
        S = K @ np.linalg.inv(K0)
        for m in range(Q):
            for k in range(Q):
                if order[k] > order[m]:
                    assert abs(S[m, k]) < 1e-12


def _eq_scalar(c, w, s, u):
    cu = c @ u
    return s * w * (1 + 3 * cu + 4.5 * cu ** 2 - 1.5 * u @ u)


def _eq_hydro(c, w, p, u):
    cu = c @ u
    return w * (p + 3 * cu + 4.5 * cu ** 2 - 1.5 * u @ u)


def _guo(c, w, a, u):
    cu = c @ u
    return w * (3 * ((c - u) @ a) + 9 * cu * (c @ a))


@pytest.mark.parametrize("Q", QS)
@pytest.mark.parametrize("kind", (0, 1))
def test_bgk_reduction_cell(Q, kind):
    """P8 (cell level): with every rate equal to omega the central-moment operator is exactly
    BGK + Guo:  a~ = a - omega (a - a_eq) + (1 - omega/2) F_i   (textbook special case, S1)."""
    rng = np.random.default_rng(100 + Q + kind)
    c, w, *_ = tcpo.lattice(Q)
    c = c.astype(float)
    for _ in range(4):
        u = rng.uniform(-0.15, 0.15, 3)
        a_vec = rng.uniform(-1e-2, 1e-2, 3)
        a_in = w * (1 + rng.uniform(-0.2, 0.2, Q)) + rng.uniform(0, 0.01, Q)
        s0 = a_in.sum()
        om = rng.uniform(0.6, 1.9)
        out = tcpo.collide_cell(Q, kind, [om] * 5, u, s0, a_vec, a_in)
        eq = _eq_scalar(c, w, s0, u) if kind == 0 else _eq_hydro(c, w, s0, u)
        ref = a_in - om * (a_in - eq) + (1 - om / 2) * _guo(c, w, a_vec, u)
        assert np.allclose(out, ref, rtol=0, atol=2e-14)


@pytest.mark.parametrize("Q", QS)
def test_collision_moment_balance(Q):
    """What any correct central-moment collision must do, whatever the rates: conserve the zeroth
    moment, change the first moment by -r1 (j - j_eq) + (1 - r1/2) a, and leave post-collision
    central moments of order k at  kappa - r_k (kappa - kappa_eq) + (1 - r_k/2) kappa_F."""
    rng = np.random.default_rng(7 * Q)
    c, w, opp, order = tcpo.lattice(Q)
    cf = c.astype(float)
    for trial in range(4):
        u = rng.uniform(-0.1, 0.1, 3)
        a_vec = rng.uniform(-1e-2, 1e-2, 3)
        a_in = w * (1 + rng.uniform(-0.2, 0.2, Q)) + rng.uniform(0, 0.01, Q)
        s0 = a_in.sum()
        r = dict(r0=1.0, r1=rng.uniform(0.5, 1.9), r2s=rng.uniform(0.5, 1.9), r2b=rng.uniform(0.5, 1.9),
                 r3=rng.uniform(0.5, 1.9))
        out = tcpo.collide_cell(Q, 0, [r["r0"], r["r1"], r["r2s"], r["r2b"], r["r3"]], u, s0, a_vec, a_in)
        eq = _eq_scalar(cf, w, s0, u)
        F = _guo(cf, w, a_vec, u)
        assert out.sum() == pytest.approx(a_in.sum(), abs=1e-14)
        j_in, j_eq, j_out = cf.T @ a_in, cf.T @ eq, cf.T @ out
        assert np.allclose(j_out, j_in - r["r1"] * (j_in - j_eq) + (1 - r["r1"] / 2) * a_vec, atol=1e-14)
        K = tcpo.central_moment_matrix(Q, u)
        k_in, k_eq, k_F, k_out = K @ a_in, K @ eq, K @ F, K @ out
        for m in range(Q):
            if order[m] == 2:
                continue
            rate = {0: r["r0"], 1: r["r1"]}.get(order[m], r["r3"])
            assert k_out[m] == pytest.approx(k_in[m] - rate * (k_in[m] - k_eq[m]) + (1 - rate / 2) * k_F[m], abs=1e-13)
        # second order: off-diagonals and deviatoric diagonal at r2s, trace at r2b
        d = cf - u
        def second(pop):
            return np.einsum("i,ia,ib->ab", pop, d, d)
        P_in, P_eq, P_F, P_out = second(a_in), second(eq), second(F), second(out)
        dev = lambda P: P - np.eye(3) * np.trace(P) / 3
        want = dev(P_in) - r["r2s"] * dev(P_in - P_eq) + (1 - r["r2s"] / 2) * dev(P_F)
        assert np.allclose(np.diag(dev(P_out)), np.diag(want), atol=1e-13)
        if Q != 7:   # D3Q7's basis has no xy, xz, yz moments (S2)
            assert np.allclose(dev(P_out), want, atol=1e-13)
        assert np.trace(P_out) == pytest.approx(
            np.trace(P_in) - r["r2b"] * np.trace(P_in - P_eq) + (1 - r["r2b"] / 2) * np.trace(P_F), abs=1e-13)


def test_guo_populations_central_moments():
    """on D3Q27 the Guo populations have central moments 0 (orders 0 and 2)
    and a (order 1).  Seen through the oracle: with rates (1,1,1,1,1) and a = a_eq the
    post-collision populations are a_eq + F/2."""
    rng = np.random.default_rng(3)
    c, w, *_ = tcpo.lattice(27)
    cf = c.astype(float)
    u = rng.uniform(-0.1, 0.1, 3)
    a_vec = rng.uniform(-1e-2, 1e-2, 3)
    eq = _eq_hydro(cf, w, 0.3, u)
    out = tcpo.collide_cell(27, 1, [1.0] * 5, u, 0.3, a_vec, eq)
    F = out - eq                      # = F_i / 2
    d = cf - u
    assert abs(F.sum()) < 1e-16
    assert np.allclose(d.T @ F, a_vec / 2, atol=1e-16)
    assert np.allclose(np.einsum("i,ia,ib->ab", F, d, d), 0, atol=1e-16)


# ---- finite-difference operators and ghosts (readings S3, S9) ---------------------------------

def test_fd_exact_on_quadratics_periodic_interior():
    nx, ny, nz = 9, 8, 7
    o = tcpo.Oracle(nx, ny, nz, {})
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    rng = np.random.default_rng(5)
    A = rng.normal(size=(3, 3)); A = A + A.T
    b = rng.normal(size=3); c0 = 0.7
    X = np.stack([x, y, z]).astype(float)
    psi = c0 + np.einsum("a,a...->...", b, X) + 0.5 * np.einsum("ab,a...,b...->...", A, X, X)
    for is_temp in (0, 1):
        grad, lap = o.fd(psi, is_temp)
        exact = b[:, None, None, None] + np.einsum("ab,b...->a...", A, X)
        inner = (slice(None), slice(1, -1), slice(1, -1), slice(1, -1))
        assert np.allclose(grad[inner], exact[inner], atol=1e-12)
        assert np.allclose(lap[1:-1, 1:-1, 1:-1], np.trace(A), atol=1e-12)


def test_fd_second_order_convergence():
    errs = []
    for n in (16, 32, 64):
        o = tcpo.Oracle(n, n, 1, {})
        y, x = np.meshgrid(np.arange(n), np.arange(n), indexing="ij")
        k = 2 * np.pi / n
        psi = (np.sin(k * x) * np.cos(2 * k * y))[None]
        grad, lap = o.fd(psi, 0)
        ex = k * np.cos(k * x) * np.cos(2 * k * y)
        el = -5 * k * k * psi[0]
        errs.append((np.abs(grad[0, 0] - ex).max() / k, np.abs(lap[0] - el).max() / (k * k)))
        assert np.abs(grad[2]).max() < 1e-15            # nz = 1 periodic: no z-gradient
    for a, b in zip(errs[:-1], errs[1:]):
        assert 3.5 < a[0] / b[0] < 4.5 and 3.5 < a[1] / b[1] < 4.5


def test_wall_ghost_rules():
    """S9: phi ghost = mirror cell (even extension, zero normal gradient at the wall); temperature
    ghost = 2 T_w - T(mirror): a linear profile through T_w at the half-cell wall is differentiated
    exactly, T_w taken at the ghost cell's tangential position."""
    nx, ny, nz = 6, 5, 4
    p = dict(bc=("periodic", "walls", "periodic"), wall_T=((0, 0), (2.0, 7.0), (0, 0)))
    o = tcpo.Oracle(nx, ny, nz, p)
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    T = 2.0 + (y + 0.5) * (7.0 - 2.0) / ny
    grad, lap = o.fd(T, 1)
    assert np.allclose(grad[1], 1.0, atol=1e-13) and np.allclose(lap, 0, atol=1e-12)
    assert np.allclose(grad[0], 0, atol=1e-13) and np.allclose(grad[2], 0, atol=1e-13)
    phi = np.cos(np.pi * (y + 0.5) / ny) + 0.0 * x      # even about both walls
    grad, lap = o.fd(phi, 0)
    # mirror ghosts: the wall cells see phi(-1) = phi(0): gradient = (phi(1) - phi(0)) / 2
    assert np.allclose(grad[1][:, 0, :], (phi[:, 1, :] - phi[:, 0, :]) / 2, atol=1e-14)
    assert np.allclose(grad[1][:, -1, :], (phi[:, -1, :] - phi[:, -2, :]) / 2, atol=1e-14)
    # wall temperature plane varying along x: ghost uses T_w at the ghost's own x
    Tw = 3.0 + np.arange(nx, dtype=float)[None, :].repeat(nz, 0)
    o.set_wall_temperature(1, 0, Tw)
    T0 = np.zeros((nz, ny, nx))
    grad, lap = o.fd(T0, 1)
    # cell (x, y=0): neighbours at y=-1 hold 2 T_w(x+cx): grad_y = -(2/2) * sum_cx w1d(cx) T_w(x+cx)
    w1 = {-1: 1 / 6, 0: 2 / 3, 1: 1 / 6}
    for xx in range(nx):
        s = sum(w1[cx] * Tw[0, (xx + cx) % nx] for cx in (-1, 0, 1))
        assert grad[1][0, 0, xx] == pytest.approx(-s, abs=1e-13)
