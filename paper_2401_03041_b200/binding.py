"""Thin Python binding of the C ABI in include/tcp.h (argument marshalling only).

Every step of the path runs in the CUDA kernels of libtcp.so; PyTorch is used for device memory
(the workspace handed to `tcp_create_in`) and for the CUDA stream.  There is no CPU fallback:
if libtcp.so cannot be loaded, or there is no CUDA device, the calls raise.
"""
import ctypes as C

import numpy as np
import torch

from . import build as _build

TCP_OK, TCP_EINVAL, TCP_ENOMEM, TCP_ECUDA, TCP_EUNSUPPORTED, TCP_ESTATE = 0, -1, -2, -3, -4, -5
PRECISION = {"f64": 0, "f32": 1}
THERMAL = {"lb_d3q7": 0, "lb_d3q15": 1, "lb_d3q19": 2, "lb_d3q27": 3, "rk2": 4, "rk4": 5}
BC = {"periodic": 0, "walls": 1}
STREAMING = {"two_grid": 0, "aa": 1}
SPACE = {"central": 0, "raw": 1}
EQUILIBRIUM = {"second_order": 0, "maxwellian": 1}


class tcp_params(C.Structure):
    """Mirror of `struct tcp_params` (include/tcp.h)."""
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
        ("wall_contact_angle", (C.c_double * 2) * 3),
        ("hydro_lattice", C.c_int),
        ("collision_space", C.c_int),
        ("equilibrium", C.c_int),
    ]


PARAM_DEFAULTS = dict(
    precision="f64", thermal="lb_d3q7", streaming="two_grid", bc=("periodic", "periodic", "periodic"),
    rho_H=1.0, rho_L=1.0, tau_H=0.6, tau_L=0.6, xi=4.0, M=0.05,
    sigma_ref=0.0, sigma_T=0.0, T_ref=0.0,
    kappa_H=0.2, kappa_L=0.2, cp_H=1.0, cp_L=1.0,
    gravity=(0.0, 0.0, 0.0), wall_T=((0.0, 0.0), (0.0, 0.0), (0.0, 0.0)),
    s_bulk=1.0, s_high=1.0, high_rate_equals_shear=0, eps_normal=1e-32,
    wall_u=(((0.0,) * 3,) * 2,) * 3,
    sigma_TT=0.0,
    wall_contact_angle=((90.0, 90.0), (90.0, 90.0), (90.0, 90.0)),
    hydro_lattice=27,
    collision_space="central",
    equilibrium="second_order",
)


def make_params(d: dict) -> tcp_params:
    unknown = set(d) - set(PARAM_DEFAULTS)
    if unknown:
        raise KeyError(f"unknown tcp_params field(s): {sorted(unknown)}")
    v = dict(PARAM_DEFAULTS)
    v.update(d)
    p = tcp_params()
    p.struct_size = C.sizeof(tcp_params)
    enum = lambda table, x: table[x] if isinstance(x, str) else int(x)
    p.precision = enum(PRECISION, v["precision"])
    p.thermal = enum(THERMAL, v["thermal"])
    p.streaming = enum(STREAMING, v["streaming"])
    for a in range(3):
        p.bc[a] = enum(BC, v["bc"][a])
        p.gravity[a] = float(v["gravity"][a])
        for f in range(2):
            p.wall_T[a][f] = float(v["wall_T"][a][f])
            p.wall_contact_angle[a][f] = float(v["wall_contact_angle"][a][f])
    for k in ("rho_H", "rho_L", "tau_H", "tau_L", "xi", "M", "sigma_ref", "sigma_T", "sigma_TT", "T_ref",
              "kappa_H", "kappa_L", "cp_H", "cp_L", "s_bulk", "s_high", "eps_normal"):
        setattr(p, k, float(v[k]))
    p.high_rate_equals_shear = int(v["high_rate_equals_shear"])
    p.hydro_lattice = int(v["hydro_lattice"])
    p.collision_space = enum(SPACE, v["collision_space"])
    p.equilibrium = enum(EQUILIBRIUM, v["equilibrium"])
    for a in range(3):
        for f in range(2):
            for c in range(3):
                p.wall_u[a][f][c] = float(v["wall_u"][a][f][c])
    return p


EXPORTS = ["tcp_params_default", "tcp_workspace_bytes", "tcp_create", "tcp_create_in", "tcp_init_fields", "tcp_set_wall_temperature",
           "tcp_set_heat_source", "tcp_step", "tcp_relax_temperature", "tcp_read_fields", "tcp_synchronize", "tcp_launch_count",
           "tcp_last_step_ms", "tcp_pattern_copy_ms", "tcp_read_pressure_static", "tcp_destroy", "tcp_last_error",
           "tcp_set_halo", "tcp_halo_phases", "tcp_halo_message_bytes", "tcp_halo_bytes", "tcp_step_begin", "tcp_step_advance",
           "tcp_step_end"]

_lib = None


def library_path() -> str:
    return _build.LIB


def lib():
    """Load libtcp.so (building it in-tree if the sources are newer).  Raises if that fails."""
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        vp, pp = C.c_void_p, C.POINTER(tcp_params)
        L.tcp_params_default.argtypes = [pp]
        L.tcp_workspace_bytes.argtypes = [C.c_int, C.c_int, C.c_int, pp, C.POINTER(C.c_size_t)]
        L.tcp_create.argtypes = [C.c_int, C.c_int, C.c_int, pp, C.POINTER(vp)]
        L.tcp_create_in.argtypes = [C.c_int, C.c_int, C.c_int, pp, vp, C.c_size_t, vp, C.POINTER(vp)]
        L.tcp_init_fields.argtypes = [vp, vp, vp, vp]
        L.tcp_set_wall_temperature.argtypes = [vp, C.c_int, C.c_int, vp]
        L.tcp_set_heat_source.argtypes = [vp, vp]
        L.tcp_step.argtypes = [vp, C.c_int]
        L.tcp_relax_temperature.argtypes = [vp, C.c_int]
        L.tcp_read_fields.argtypes = [vp, vp, vp, vp, vp]
        L.tcp_read_pressure_static.argtypes = [vp, vp]
        L.tcp_synchronize.argtypes = [vp]
        L.tcp_launch_count.argtypes = [vp]
        L.tcp_launch_count.restype = C.c_longlong
        L.tcp_last_step_ms.argtypes = [vp, C.POINTER(C.c_float)]
        L.tcp_pattern_copy_ms.argtypes = [vp, C.c_int, C.POINTER(C.c_float)]
        L.tcp_destroy.argtypes = [vp]
        L.tcp_set_halo.argtypes = [vp, C.c_int, C.c_int, vp, vp, vp, vp, vp]
        L.tcp_halo_bytes.argtypes = [vp, C.POINTER(C.c_size_t)]
        L.tcp_halo_phases.argtypes = [vp, C.POINTER(C.c_int)]
        L.tcp_halo_message_bytes.argtypes = [vp, C.c_int, C.POINTER(C.c_size_t)]
        L.tcp_step_advance.argtypes = [vp, C.POINTER(C.c_int)]
        L.tcp_step_begin.argtypes = [vp]
        L.tcp_step_end.argtypes = [vp]
        L.tcp_last_error.restype = C.c_char_p
        _lib = L
    return _lib


class TcpError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"tcp error {code}: {msg}")
        self.code = code


def _check(rc):
    if rc != TCP_OK:
        raise TcpError(rc, lib().tcp_last_error().decode())


def _ptr(a):
    """host numpy array / torch tensor (cpu or cuda) / None -> void*"""
    if a is None:
        return None
    if isinstance(a, torch.Tensor):
        assert a.is_contiguous()
        return C.c_void_p(a.data_ptr())
    assert a.flags["C_CONTIGUOUS"]
    return C.c_void_p(a.ctypes.data)


# ---- the ABI, name for name -------------------------------------------------------------------

def tcp_params_default() -> tcp_params:
    p = tcp_params()
    _check(lib().tcp_params_default(C.byref(p)))
    return p


def tcp_workspace_bytes(nx, ny, nz, params: tcp_params) -> int:
    n = C.c_size_t()
    _check(lib().tcp_workspace_bytes(nx, ny, nz, C.byref(params), C.byref(n)))
    return n.value


def tcp_create(nx, ny, nz, params: tcp_params):
    h = C.c_void_p()
    _check(lib().tcp_create(nx, ny, nz, C.byref(params), C.byref(h)))
    return h


def tcp_create_in(nx, ny, nz, params: tcp_params, workspace: torch.Tensor, stream: "torch.cuda.Stream | None" = None):
    h = C.c_void_p()
    sp = C.c_void_p(stream.cuda_stream if stream is not None else 0)
    _check(lib().tcp_create_in(nx, ny, nz, C.byref(params), C.c_void_p(workspace.data_ptr()),
                               workspace.numel() * workspace.element_size(), sp, C.byref(h)))
    return h


def tcp_init_fields(sim, phi, u=None, T=None):
    _check(lib().tcp_init_fields(sim, _ptr(phi), _ptr(u), _ptr(T)))


def tcp_set_wall_temperature(sim, axis, face, Tw):
    _check(lib().tcp_set_wall_temperature(sim, axis, face, _ptr(Tw)))


def tcp_set_heat_source(sim, q):
    _check(lib().tcp_set_heat_source(sim, _ptr(q)))


def tcp_step(sim, nsteps=1):
    _check(lib().tcp_step(sim, int(nsteps)))


def tcp_relax_temperature(sim, nsteps=1):
    _check(lib().tcp_relax_temperature(sim, int(nsteps)))


def tcp_read_fields(sim, phi=None, u=None, p=None, T=None):
    _check(lib().tcp_read_fields(sim, _ptr(phi), _ptr(u), _ptr(p), _ptr(T)))


TCP_STATIC_SCRATCH_BYTES = 8 << 20


def tcp_read_pressure_static(sim, p):
    _check(lib().tcp_read_pressure_static(sim, _ptr(p)))


def tcp_synchronize(sim):
    _check(lib().tcp_synchronize(sim))


def tcp_launch_count(sim) -> int:
    return int(lib().tcp_launch_count(sim))


def tcp_last_step_ms(sim) -> float:
    ms = C.c_float()
    _check(lib().tcp_last_step_ms(sim, C.byref(ms)))
    return float(ms.value)


def tcp_pattern_copy_ms(sim, nlaunches=10) -> float:
    ms = C.c_float()
    _check(lib().tcp_pattern_copy_ms(sim, int(nlaunches), C.byref(ms)))
    return float(ms.value)


def tcp_set_halo(sim, lo, hi, comm_stream: "torch.cuda.Stream | None", send_lo=None, send_hi=None, recv_lo=None, recv_hi=None):
    sp = C.c_void_p(comm_stream.cuda_stream if comm_stream is not None else 0)
    _check(lib().tcp_set_halo(sim, int(lo), int(hi), sp, _ptr(send_lo), _ptr(send_hi), _ptr(recv_lo), _ptr(recv_hi)))


def tcp_halo_bytes(sim) -> int:
    n = C.c_size_t()
    _check(lib().tcp_halo_bytes(sim, C.byref(n)))
    return n.value


def tcp_halo_phases(sim) -> int:
    n = C.c_int()
    _check(lib().tcp_halo_phases(sim, C.byref(n)))
    return n.value


def tcp_halo_message_bytes(sim, phase) -> int:
    n = C.c_size_t()
    _check(lib().tcp_halo_message_bytes(sim, int(phase), C.byref(n)))
    return n.value


def tcp_step_begin(sim):
    _check(lib().tcp_step_begin(sim))


def tcp_step_advance(sim) -> int:
    """-> transfers left in this step (0: the step is complete)"""
    n = C.c_int()
    _check(lib().tcp_step_advance(sim, C.byref(n)))
    return n.value


def tcp_step_end(sim):
    _check(lib().tcp_step_end(sim))


def tcp_destroy(sim):
    _check(lib().tcp_destroy(sim))


def tcp_last_error() -> str:
    return lib().tcp_last_error().decode()


# ---- convenience wrapper: torch owns the device memory and the stream ---------------------------

class Simulation:
    """One simulation on the current CUDA device.  Arrays are [nz][ny][nx] (x fastest)."""

    def __init__(self, nx, ny, nz, params: dict, stream: "torch.cuda.Stream | None" = None, device="cuda"):
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2401_03041_b200 needs a CUDA device: there is no CPU path")
        self.nx, self.ny, self.nz = nx, ny, nz
        self.shape = (nz, ny, nx)
        self.params = make_params(params)
        self.np_dtype = np.float64 if self.params.precision == 0 else np.float32
        self.torch_dtype = torch.float64 if self.params.precision == 0 else torch.float32
        self.device = torch.device(device)
        nbytes = tcp_workspace_bytes(nx, ny, nz, self.params)
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)   # 512-B aligned by the caching allocator
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self._h = tcp_create_in(nx, ny, nz, self.params, self.workspace, self.stream)

    def _as(self, a):
        if a is None:
            return None
        if isinstance(a, torch.Tensor):
            return a.to(self.torch_dtype).contiguous()
        return np.ascontiguousarray(a, dtype=self.np_dtype)

    def init_fields(self, phi, u=None, T=None):
        tcp_init_fields(self._h, self._as(phi), self._as(u), self._as(T))

    def set_wall_temperature(self, axis, face, Tw):
        tcp_set_wall_temperature(self._h, axis, face, self._as(Tw))

    def set_heat_source(self, q):
        tcp_set_heat_source(self._h, self._as(q))

    def step(self, n=1):
        tcp_step(self._h, n)

    def relax_temperature(self, n=1):
        tcp_relax_temperature(self._h, n)

    def read_fields(self):
        """-> phi, u, p, T as host numpy arrays in the simulation's precision."""
        nz, ny, nx = self.shape
        phi = np.empty((nz, ny, nx), self.np_dtype); u = np.empty((3, nz, ny, nx), self.np_dtype)
        p = np.empty((nz, ny, nx), self.np_dtype); T = np.empty((nz, ny, nx), self.np_dtype)
        tcp_read_fields(self._h, phi, u, p, T)
        return phi, u, p, T

    def read_fields_device(self):
        nz, ny, nx = self.shape
        mk = lambda *s: torch.empty(*s, dtype=self.torch_dtype, device=self.device)
        phi, u, p, T = mk(nz, ny, nx), mk(3, nz, ny, nx), mk(nz, ny, nx), mk(nz, ny, nx)
        tcp_read_fields(self._h, phi, u, p, T)
        return phi, u, p, T

    def synchronize(self):
        tcp_synchronize(self._h)

    @property
    def launches(self):
        return tcp_launch_count(self._h)

    def last_step_ms(self):
        return tcp_last_step_ms(self._h)

    def pattern_copy_ms(self, nlaunches=10):
        return tcp_pattern_copy_ms(self._h, nlaunches)

    def close(self):
        if getattr(self, "_h", None):
            tcp_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
