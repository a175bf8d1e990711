"""ctypes wrapper of the CPU oracle (oracle/tcpo.c).  TEST INFRASTRUCTURE, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
import this module.  It imports nothing from paper_2401_03041_b200 and declares its own copy of
the parameter struct (the oracle and the CUDA path share no code).
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

THERMAL = {"lb_d3q7": 0, "lb_d3q15": 1, "lb_d3q19": 2, "lb_d3q27": 3, "rk2": 4, "rk4": 5}
BC = {"periodic": 0, "walls": 1}


class Params(C.Structure):
    _fields_ = [
        ("struct_size", C.c_uint),
        ("precision", C.c_int), ("thermal", C.c_int), ("streaming", C.c_int),
        ("bc", C.c_int * 3),
        ("rho_H", C.c_double), ("rho_L", C.c_double),
        ("tau_H", C.c_double), ("tau_L", C.c_double),
        ("xi", C.c_double), ("M", C.c_double),
        ("sigma_ref", C.c_double), ("sigma_T", C.c_double), ("T_ref", C.c_double),
        ("kappa_H", C.c_double), ("kappa_L", C.c_double), ("cp_H", C.c_double), ("cp_L", C.c_double),
        ("gravity", C.c_double * 3),
        ("wall_T", (C.c_double * 2) * 3),
        ("s_bulk", C.c_double), ("s_high", C.c_double),
        ("high_rate_equals_shear", C.c_int),
        ("eps_normal", C.c_double),
        ("wall_u", ((C.c_double * 3) * 2) * 3),
        ("sigma_TT", C.c_double),
        ("wall_contact_angle", (C.c_double * 2) * 3),   # degrees, reading S20
        ("hydro_lattice", C.c_int),        # 27 or 19
        ("collision_space", C.c_int),      # 0 central moments, 1 raw moments (MRT)
        ("equilibrium", C.c_int),          # 0 printed second-order (eqs. 12, 18), 1 Maxwellian in central-moment space
        ("hydro_phi_level", C.c_int),      # oracle-only (reading S16): 0 = phi^n, 1 = phi^{n+1}
    ]


DEFAULTS = dict(
    thermal="lb_d3q7", bc=("periodic", "periodic", "periodic"),
    rho_H=1.0, rho_L=1.0, tau_H=0.6, tau_L=0.6, xi=4.0, M=0.05,
    sigma_ref=0.0, sigma_T=0.0, T_ref=0.0,
    kappa_H=0.2, kappa_L=0.2, cp_H=1.0, cp_L=1.0,
    gravity=(0.0, 0.0, 0.0), wall_T=((0.0, 0.0), (0.0, 0.0), (0.0, 0.0)),
    s_bulk=1.0, s_high=1.0, high_rate_equals_shear=0, eps_normal=1e-32,
    wall_u=(((0.0,) * 3,) * 2,) * 3,
    sigma_TT=0.0,
    wall_contact_angle=((90.0, 90.0), (90.0, 90.0), (90.0, 90.0)),
    hydro_lattice=27,
    equilibrium=0,
    collision_space=0,
    hydro_phi_level=0,
)


def make_params(d: dict) -> Params:
    """dict (keys of DEFAULTS; 'precision'/'streaming' are ignored) -> Params."""
    unknown = set(d) - set(DEFAULTS) - {"precision", "streaming"}
    if unknown:
        raise KeyError(f"unknown parameter(s): {sorted(unknown)}")
    v = dict(DEFAULTS)
    v.update(d)
    p = Params()
    p.struct_size = C.sizeof(Params)
    p.precision = 0
    p.streaming = 0
    p.thermal = THERMAL[v["thermal"]] if isinstance(v["thermal"], str) else int(v["thermal"])
    for a in range(3):
        b = v["bc"][a]
        p.bc[a] = BC[b] if isinstance(b, str) else int(b)
        p.gravity[a] = float(v["gravity"][a])
        for f in range(2):
            p.wall_T[a][f] = float(v["wall_T"][a][f])
            p.wall_contact_angle[a][f] = float(v["wall_contact_angle"][a][f])
    for k in ("rho_H", "rho_L", "tau_H", "tau_L", "xi", "M", "sigma_ref", "sigma_T", "sigma_TT", "T_ref",
              "kappa_H", "kappa_L", "cp_H", "cp_L", "s_bulk", "s_high", "eps_normal"):
        setattr(p, k, float(v[k]))
    p.high_rate_equals_shear = int(v["high_rate_equals_shear"])
    p.hydro_phi_level = int(v["hydro_phi_level"])
    p.hydro_lattice = int(v["hydro_lattice"])
    eqm = v["equilibrium"]
    p.equilibrium = {"second_order": 0, "maxwellian": 1}[eqm] if isinstance(eqm, str) else int(eqm)
    cs = v["collision_space"]
    p.collision_space = {"central": 0, "raw": 1}[cs] if isinstance(cs, str) else int(cs)
    for a in range(3):
        for f in range(2):
            for c in range(3):
                p.wall_u[a][f][c] = float(v["wall_u"][a][f][c])
    return p


_lib = None


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        dp = C.POINTER(C.c_double)
        ip = C.POINTER(C.c_int)
        L.tcpo_create.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(Params), C.POINTER(C.c_void_p)]
        L.tcpo_destroy.argtypes = [C.c_void_p]
        L.tcpo_init_fields.argtypes = [C.c_void_p, dp, dp, dp]
        L.tcpo_set_wall_temperature.argtypes = [C.c_void_p, C.c_int, C.c_int, dp]
        L.tcpo_set_heat_source.argtypes = [C.c_void_p, dp]
        L.tcpo_step.argtypes = [C.c_void_p, C.c_int]
        L.tcpo_relax_temperature.argtypes = [C.c_void_p, C.c_int]
        L.tcpo_read_fields.argtypes = [C.c_void_p, dp, dp, dp, dp]
        L.tcpo_read_populations.argtypes = [C.c_void_p, C.c_int, dp]
        L.tcpo_lattice.argtypes = [C.c_int, ip, dp, ip, ip]
        L.tcpo_collide_cell.argtypes = [C.c_int, C.c_int, dp, dp, C.c_double, dp, dp, dp]
        L.tcpo_collide_cell_space.argtypes = [C.c_int, C.c_int, dp, dp, C.c_double, dp, dp, dp, C.c_int]
        L.tcpo_central_moment_matrix.argtypes = [C.c_int, dp, dp]
        L.tcpo_fd.argtypes = [C.c_void_p, dp, C.c_int, dp, dp]
        L.tcpo_last_error.restype = C.c_char_p
        L.tcpo_num_threads.restype = C.c_int
        L.tcpo_set_num_threads.argtypes = [C.c_int]
        L.tcpo_set_num_threads.restype = None
        _lib = L
    return _lib


def _dp(a):
    return None if a is None else a.ctypes.data_as(C.POINTER(C.c_double))


def _f64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


class OracleError(RuntimeError):
    pass


def _check(rc):
    if rc != 0:
        raise OracleError(f"tcpo error {rc}: {lib().tcpo_last_error().decode()}")


def num_threads() -> int:
    return int(lib().tcpo_num_threads())


_MAX_THREADS = None


def threads_for(cells: int) -> int:
    """One thread per 288 cells (a 48 x 24 channel gets 4), at most what OpenMP offers.  On the small grids of the pins a parallel region
    costs more than it saves, and with spinning OpenMP barriers a busy box makes it far worse (measured: 512 cells,
    8 threads, two processes at once: 30-60 ms per step against 12 ms with one thread)."""
    global _MAX_THREADS
    if _MAX_THREADS is None:
        _MAX_THREADS = num_threads()
    return max(1, min(_MAX_THREADS, cells // 288))


class Oracle:
    """One oracle simulation.  Arrays are [nz][ny][nx] (x fastest); u is [3][nz][ny][nx]."""

    def __init__(self, nx, ny, nz, params: dict):
        self.shape = (nz, ny, nx)
        self.n = nx * ny * nz
        self.params = params
        self._p = make_params(params)
        self._h = C.c_void_p()
        _check(lib().tcpo_create(nx, ny, nz, C.byref(self._p), C.byref(self._h)))
        qt = {0: 7, 1: 15, 2: 19, 3: 27}
        self.q_thermal = qt.get(self._p.thermal)

    def close(self):
        if self._h:
            lib().tcpo_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def init_fields(self, phi, u=None, T=None):
        phi, u, T = _f64(phi), _f64(u), _f64(T)
        assert phi.size == self.n and (u is None or u.size == 3 * self.n) and (T is None or T.size == self.n)
        _check(lib().tcpo_init_fields(self._h, _dp(phi), _dp(u), _dp(T)))

    def set_wall_temperature(self, axis, face, Tw):
        Tw = _f64(Tw)
        _check(lib().tcpo_set_wall_temperature(self._h, axis, face, _dp(Tw)))

    def set_heat_source(self, q):
        q = _f64(q)
        _check(lib().tcpo_set_heat_source(self._h, _dp(q)))

    def step(self, n=1):
        lib().tcpo_set_num_threads(threads_for(self.n))
        _check(lib().tcpo_step(self._h, int(n)))

    def relax_temperature(self, n=1):
        lib().tcpo_set_num_threads(threads_for(self.n))
        _check(lib().tcpo_relax_temperature(self._h, int(n)))

    def read_fields(self):
        nz, ny, nx = self.shape
        phi = np.empty((nz, ny, nx)); u = np.empty((3, nz, ny, nx)); p = np.empty((nz, ny, nx)); T = np.empty((nz, ny, nx))
        _check(lib().tcpo_read_fields(self._h, _dp(phi), _dp(u), _dp(p), _dp(T)))
        return phi, u, p, T

    def read_populations(self, which):
        q = 27 if which == 0 else (self._p.hydro_lattice if which == 1 else self.q_thermal)
        out = np.empty((q,) + self.shape)
        _check(lib().tcpo_read_populations(self._h, which, _dp(out)))
        return out

    def fd(self, psi, is_temp):
        psi = _f64(psi)
        grad = np.empty((3,) + self.shape); lap = np.empty(self.shape)
        _check(lib().tcpo_fd(self._h, _dp(psi), int(is_temp), _dp(grad), _dp(lap)))
        return grad, lap


def lattice(Q):
    c = np.empty((Q, 3), dtype=np.int32); w = np.empty(Q); opp = np.empty(Q, dtype=np.int32); order = np.empty(Q, dtype=np.int32)
    ip = C.POINTER(C.c_int)
    _check(lib().tcpo_lattice(Q, c.ctypes.data_as(ip), _dp(w), opp.ctypes.data_as(ip), order.ctypes.data_as(ip)))
    return c, w, opp, order


def collide_cell(Q, kind, rates5, u, s0, avec, a_in):
    rates5, u, avec, a_in = _f64(rates5), _f64(u), _f64(avec), _f64(a_in)
    out = np.empty(Q)
    _check(lib().tcpo_collide_cell(Q, kind, _dp(rates5), _dp(u), float(s0), _dp(avec), _dp(a_in), _dp(out)))
    return out


def collide_cell_space(Q, kind, rates5, u, s0, avec, a_in, raw_space):
    rates5, u, avec, a_in = _f64(rates5), _f64(u), _f64(avec), _f64(a_in)
    out = np.empty(Q)
    _check(lib().tcpo_collide_cell_space(Q, kind, _dp(rates5), _dp(u), float(s0), _dp(avec), _dp(a_in), _dp(out), int(raw_space)))
    return out


def central_moment_matrix(Q, u):
    u = _f64(u)
    K = np.empty((Q, Q))
    _check(lib().tcpo_central_moment_matrix(Q, _dp(u), _dp(K)))
    return K
