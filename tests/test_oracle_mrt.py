"""Pins of the oracle's raw-moment (MRT) collision space (`collision_space = 1`: the same basis and rates as reading S2,
about the lattice at rest instead of about u; PAPER.md:180 names MRT next to SRT as the methods in widespread use).
Expected values come from numpy moment sums coded here and from closed forms, not from the oracle."""
import numpy as np
import pytest

from oracle import tcpo

QS = [7, 15, 19, 27]


def _eq_scalar(c, w, s, u):
    cu = c @ u
    return s * w * (1 + 3 * cu + 4.5 * cu ** 2 - 1.5 * u @ u)


def _guo(c, w, a, u):
    return w * (3 * ((c - u) @ a) + 9 * (c @ u) * (c @ a))


@pytest.mark.parametrize("Q", QS)
def test_raw_moment_balance(Q):
    """What any MRT collision must do, whatever the rates: every RAW basis moment m_k of the populations goes to
    m_k - r_k (m_k - m_k^eq) + (1 - r_k / 2) m_k^F; second order: deviatoric part at r2s, trace at r2b.  The raw basis
    moments are formed here with numpy from the lattice velocities (K(0) of the oracle is only used to read off which
    monomial each basis row is: it is checked against the velocities first)."""
    rng = np.random.default_rng(11 * Q)
    c, w, opp, order = tcpo.lattice(Q)
    cf = c.astype(float)
    K0 = tcpo.central_moment_matrix(Q, np.zeros(3))
    # rows of K(0) are sums of monomials of the velocities: entries are integers in {-1, 0, 1, 2, 3}
    assert np.array_equal(K0, np.round(K0))
    assert np.array_equal(K0[0], np.ones(Q))
    for trial in range(4):
        u = rng.uniform(-0.1, 0.1, 3)
        a_vec = rng.uniform(-1e-2, 1e-2, 3)
        a_in = w * (1 + rng.uniform(-0.2, 0.2, Q)) + rng.uniform(0, 0.01, Q)
        s0 = a_in.sum()
        r = [1.0, rng.uniform(0.5, 1.9), rng.uniform(0.5, 1.9), rng.uniform(0.5, 1.9), rng.uniform(0.5, 1.9)]
        out = tcpo.collide_cell_space(Q, 0, r, u, s0, a_vec, a_in, raw_space=1)
        eq, F = _eq_scalar(cf, w, s0, u), _guo(cf, w, a_vec, u)
        assert out.sum() == pytest.approx(a_in.sum(), abs=1e-14)
        j = lambda p: cf.T @ p
        assert np.allclose(j(out), j(a_in) - r[1] * (j(a_in) - j(eq)) + (1 - r[1] / 2) * a_vec, atol=1e-14)
        m_in, m_eq, m_F, m_out = K0 @ a_in, K0 @ eq, K0 @ F, K0 @ out
        for m in range(Q):
            if order[m] == 2:
                continue
            rate = {0: r[0], 1: r[1]}.get(order[m], r[4])
            assert m_out[m] == pytest.approx(m_in[m] - rate * (m_in[m] - m_eq[m]) + (1 - rate / 2) * m_F[m], abs=1e-13)
        second = lambda p: np.einsum("i,ia,ib->ab", p, cf, cf)                 # RAW second moments
        P_in, P_eq, P_F, P_out = second(a_in), second(eq), second(F), second(out)
        dev = lambda P: P - np.eye(3) * np.trace(P) / 3
        want = dev(P_in) - r[2] * dev(P_in - P_eq) + (1 - r[2] / 2) * dev(P_F)
        assert np.allclose(np.diag(dev(P_out)), np.diag(want), atol=1e-13)
        if Q != 7:
            assert np.allclose(dev(P_out), want, atol=1e-13)
        assert np.trace(P_out) == pytest.approx(np.trace(P_in) - r[3] * np.trace(P_in - P_eq) + (1 - r[3] / 2) * np.trace(P_F), abs=1e-13)
        # it is a different operator from the central-moment one unless u = 0 or all rates are equal
        cm = tcpo.collide_cell_space(Q, 0, r, u, s0, a_vec, a_in, raw_space=0)
        assert np.abs(cm - out).max() > 1e-8
        at_rest = [tcpo.collide_cell_space(Q, 0, r, np.zeros(3), s0, a_vec, a_in, raw_space=k) for k in (0, 1)]
        assert np.array_equal(at_rest[0], at_rest[1])
        bgk = [tcpo.collide_cell_space(Q, 0, [1.3] * 5, u, s0, a_vec, a_in, raw_space=k) for k in (0, 1)]
        assert np.abs(bgk[0] - bgk[1]).max() < 1e-15


def test_poiseuille_and_heat_decay_in_raw_moment_space():
    """The physical rates are the same in both spaces: nu = tau c_s^2 (Poiseuille, A13) and kappa (heat sinusoid, G4)."""
    ny, nu, gx = 20, 0.2, 1e-6
    o = tcpo.Oracle(1, ny, 1, dict(bc=("periodic", "walls", "periodic"), tau_H=3 * nu, tau_L=3 * nu, gravity=(gx, 0, 0),
                                   xi=1e30, collision_space=1))
    o.init_fields(np.zeros((1, ny, 1)))
    o.step(6000)
    u = o.read_fields()[1]
    o.close()
    yy = np.arange(ny) + 0.5
    exact = gx / (2 * nu) * yy * (ny - yy)
    assert np.abs(u[0].ravel() - exact).max() / exact.max() < 2e-3
    n, kap, U, steps = 48, 0.1, 0.04, 120
    k = 2 * np.pi / n
    for thermal in ("lb_d3q7", "lb_d3q19", "lb_d3q27"):
        T0 = (1 + 0.5 * np.sin(k * np.arange(n))).reshape(1, 1, n)
        u0 = np.zeros((3, 1, 1, n)); u0[0] = U
        o = tcpo.Oracle(n, 1, 1, dict(thermal=thermal, kappa_H=kap, kappa_L=kap, xi=1e30, collision_space=1))
        o.init_fields(np.zeros((1, 1, n)), u=u0, T=T0)
        o.step(steps)
        T = o.read_fields()[3].ravel()
        o.close()
        Fm = np.fft.rfft(T - 1)[1]
        assert -np.log(2 * np.abs(Fm) / n / 0.5) / steps == pytest.approx(kap * k * k, rel=0.02)
        assert (-np.angle(Fm) - np.pi / 2) / k == pytest.approx(U * steps, rel=0.01)
