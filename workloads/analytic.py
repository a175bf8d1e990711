"""Closed-form solution of the two-layer heated channel, PAPER.md:452-493 (Appendix A, after
Pendse & Esmaeeli, ref. [33]), in the de-garbled reading G8 of SURVEY.md 8(c):

  * the printed T(x,y) has its two case labels swapped and the lower-layer linear part lost a
    k_r; the version below satisfies both wall conditions, continuity of T and of k dT/dy at
    y = 0 and Laplace's equation (tests/test_closed_form.py checks all of that numerically);
  * u, v as printed, superscript a for the upper layer (0 < y < a), b for the lower (-b < y <= 0).

Used (i) as the initial temperature of config 2 and (ii) as the expected field of pin P9.
Upper layer = fluid A, lower layer = fluid B; k_r = k_A/k_B, mu_r = mu_A/mu_B, mu_B is the
viscosity in U_max ("mu_h": the fluid next to the heated wall).
"""
import numpy as np


def layered_channel_closed_form(x, y, *, a, b, L, T_h, T_c, T_0, k_r, mu_r, mu_B, sigma_T):
    """x, y: numpy arrays (broadcastable); y measured from the interface, wall at y=-b is the
    heated one (T = T_h + T_0 cos(w x)), wall at y=a is at T_c.  Returns (u, v, T, U_max)."""
    x = np.asarray(x, dtype=np.float64)
    y = np.asarray(y, dtype=np.float64)
    w = 2.0 * np.pi / L                     # PAPER.md:208 (reading G7: omega = 2 pi / L)
    ar, br = a * w, b * w                   # A.4
    f = 1.0 / (k_r * np.sinh(br) * np.cosh(ar) + np.sinh(ar) * np.cosh(br))   # A.5
    da = np.sinh(ar) ** 2 - ar ** 2
    db = np.sinh(br) ** 2 - br ** 2
    C1a, C1b = np.sinh(ar) ** 2 / da, np.sinh(br) ** 2 / db                  # A.6
    C2a, C2b = -a * ar / da, -b * br / db                                    # A.7
    C3a = (2 * ar - np.sinh(2 * ar)) / (2 * da)                              # A.8
    C3b = (-2 * br + np.sinh(2 * br)) / (2 * db)
    g = np.sinh(ar) * f                                                      # A.10
    h = da * db / (mu_r * db * (np.sinh(2 * ar) - 2 * ar) + da * (np.sinh(2 * br) - 2 * br))  # A.11
    U_max = -(T_0 * sigma_T / mu_B) * g * h                                  # A.9
    up = y > 0
    C1 = np.where(up, C1a, C1b)
    C2 = np.where(up, C2a, C2b)
    C3 = np.where(up, C3a, C3b)
    ch, sh = np.cosh(w * y), np.sinh(w * y)
    u = U_max * ((C1 + w * (C2 + C3 * y)) * ch + (C3 + w * C1 * y) * sh) * np.sin(w * x)       # A.1
    v = -w * U_max * (C1 * y * ch + (C2 + C3 * y) * sh) * np.cos(w * x)                        # A.2
    den = a + k_r * b
    T_up = ((T_c - T_h) * y + k_r * T_c * b + T_h * a) / den + T_0 * f * np.sinh(ar - w * y) * np.cos(w * x)
    T_lo = (k_r * (T_c - T_h) * y + k_r * T_c * b + T_h * a) / den \
        + T_0 * f * (np.sinh(ar) * ch - k_r * sh * np.cosh(ar)) * np.cos(w * x)
    T = np.where(up, T_up, T_lo)
    return u, v, T, float(U_max)
