"""Out-of-bounds guard: every kernel family runs on a caller-owned workspace (tcp_create_in) that sits between two guard
bands filled with a byte pattern; afterwards the bands must be untouched and the fields finite.  (Writes that stay inside
the workspace but hit a neighbouring array are what the element-wise parity tests catch.)"""
import numpy as np
import pytest
import torch

import paper_2401_03041_b200 as tcp
import workloads as W

pytestmark = pytest.mark.gpu
GUARD = 1 << 20


def _run_guarded(wl, extra, precision, steps=5, relax=0):
    params = tcp.make_params(dict(wl.params, precision=precision, **extra))
    nbytes = tcp.tcp_workspace_bytes(wl.nx, wl.ny, wl.nz, params)
    buf = torch.full((GUARD + nbytes + GUARD,), 0xA5, dtype=torch.uint8, device="cuda")
    ws = buf[GUARD:GUARD + nbytes]
    assert ws.data_ptr() % 256 == 0
    h = tcp.tcp_create_in(wl.nx, wl.ny, wl.nz, params, ws, torch.cuda.current_stream())
    dt = np.float64 if precision == "f64" else np.float32
    as_np = lambda t: None if t is None else np.ascontiguousarray(t.numpy(), dtype=dt)
    for (ax, fc), plane in wl.wall_T.items():
        tcp.tcp_set_wall_temperature(h, ax, fc, as_np(plane))
    tcp.tcp_init_fields(h, as_np(wl.phi), as_np(wl.u), as_np(wl.T))
    if relax:
        tcp.tcp_relax_temperature(h, relax)
    tcp.tcp_step(h, steps)
    shape = (wl.nz, wl.ny, wl.nx)
    phi, u, p, T = np.empty(shape, dt), np.empty((3,) + shape, dt), np.empty(shape, dt), np.empty(shape, dt)
    tcp.tcp_read_fields(h, phi, u, p, T)
    tcp.tcp_destroy(h)
    assert all(np.all(np.isfinite(a)) for a in (phi, u, p, T))
    assert bool((buf[:GUARD] == 0xA5).all()) and bool((buf[GUARD + nbytes:] == 0xA5).all()), "write outside the workspace"


@pytest.mark.parametrize("precision", ["f64", "f32"])
@pytest.mark.parametrize("thermal", ["lb_d3q7", "lb_d3q19", "lb_d3q27", "rk2", "rk4"])
def test_periodic_boxes(thermal, precision):
    for extra in (dict(), dict(streaming="aa"), dict(hydro_lattice=19), dict(collision_space="raw")):
        # 20 x 14 x 9: even nx (pair kernel in fp32), blocks that end inside a row, a ragged last block
        _run_guarded(W.perf_box(20, thermal=thermal, ny=14, nz=9, r_min=3.0, r_max=4.0, seed=2), extra, precision)
    _run_guarded(W.perf_box(21, thermal=thermal, ny=13, nz=7, r_min=3.0, r_max=4.0, seed=2), dict(), precision)     # odd nx
    if thermal in ("lb_d3q27", "rk2"):
        _run_guarded(W.perf_box(16, thermal=thermal, ny=12, nz=8, r_min=3.0, r_max=4.0, seed=2), dict(equilibrium="maxwellian"), precision)


@pytest.mark.parametrize("precision", ["f64", "f32"])
def test_boxes_with_walls(precision):
    wl = W.layered_channel(nx=24, ny=14, nz=3, thermal="lb_d3q19", rho_upper=2.0)
    for extra in (dict(wall_contact_angle=((90, 90), (60, 120), (90, 90))), dict(streaming="aa"), dict(s_high=1.3),
                  dict(high_rate_equals_shear=1), dict(hydro_lattice=19)):
        _run_guarded(wl, extra, precision, relax=2)
    wl3 = W.perf_box(12, thermal="lb_d3q15", ny=10, nz=8, r_min=3.0, r_max=4.0, seed=3, volume_fraction=0.3)
    wl3.params.update(bc=("walls", "walls", "walls"), eps_normal=1e-9, wall_contact_angle=((30, 150), (60, 120), (45, 100)))
    _run_guarded(wl3, dict(), precision)
    _run_guarded(wl3, dict(streaming="aa"), precision, steps=6)


def test_box_large_enough_for_the_l2_prefetch_to_run():
    # > 300 blocks: blocks issue their bulk L2 prefetch, which is clamped to the arrays (a hint, but it must stay a valid range)
    wl = W.perf_box(48, thermal="lb_d3q7", ny=40, nz=24, r_min=4.0, r_max=6.0, seed=5)
    for precision in ("f64", "f32"):
        _run_guarded(wl, dict(), precision, steps=3)
        _run_guarded(wl, dict(streaming="aa"), precision, steps=4)
