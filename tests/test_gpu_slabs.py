"""Block decomposition along z (include/tcp.h: tcp_set_halo / tcp_step_begin / tcp_step_end).

A box cut into z-slabs with ghost planes must give, cell for cell, the BITS of the undivided box: every cell
sees the same neighbour values and runs the same instructions.  All slabs live on the one GPU of the test box
(`LocalSlabs`: the transfer between neighbours is a device copy), launched one after the other -- no kernel
waits for another.  One case is also compared with the oracle directly.
"""
import numpy as np
import pytest
import torch

import paper_2401_03041_b200 as tcp
from paper_2401_03041_b200 import binding as B
from paper_2401_03041_b200.slab import LocalSlabs
from parity_util import _np, assert_parity_f64, run_gpu, run_oracle
from workloads import configs

pytestmark = pytest.mark.gpu


def run_slabs(wl, nslabs, steps, q=None, extra=None, precision="f64"):
    params = dict(wl.params)
    if extra:
        params.update(extra)
    params["precision"] = precision
    box = LocalSlabs(wl.nx, wl.ny, wl.nz, nslabs, params)
    for (ax, fc), plane in wl.wall_T.items():
        box.set_wall_temperature(ax, fc, _np(plane))
    if q is not None:
        box.set_heat_source(_np(q))
    box.init_fields(_np(wl.phi), _np(wl.u), _np(wl.T))
    box.step(steps)
    out = box.read_fields()
    launches = box.launches
    box.close()
    return out, launches


def assert_same_bits(got, want):
    for name, g, w in zip(("phi", "u", "p", "T"), got, want):
        assert g.shape == w.shape and g.dtype == w.dtype
        assert np.array_equal(g, w), f"{name}: {np.count_nonzero(g != w)} cells differ, max {np.abs(g - w).max():.3e}"


@pytest.mark.parametrize("thermal", ["lb_d3q7", "lb_d3q15", "lb_d3q19", "lb_d3q27"])
@pytest.mark.parametrize("nslabs", [2, 5])
def test_periodic_box_in_slabs_is_bit_identical(thermal, nslabs):
    wl = configs.perf_box(24, thermal=thermal, ny=20, nz=22, seed=11, r_min=4.0, r_max=6.0)   # 5 slabs: 5,5,4,4,4 planes
    want, _ = run_gpu(wl, 20)
    got, _ = run_slabs(wl, nslabs, 20)
    assert_same_bits(got, want)


def test_slabs_match_the_oracle():
    wl = configs.perf_box(20, thermal="lb_d3q7", ny=18, nz=21, seed=5, r_min=4.0, r_max=5.0)
    got, _ = run_slabs(wl, 3, 100)
    assert_parity_f64(got, run_oracle(wl, 100))


def test_one_plane_slabs():
    wl = configs.perf_box(16, thermal="lb_d3q19", ny=12, nz=4, seed=3, r_min=2.0, r_max=3.0)
    want, _ = run_gpu(wl, 12)
    got, _ = run_slabs(wl, 4, 12)          # every slab: one plane of its own between two ghost planes
    assert_same_bits(got, want)


def test_walls_in_z_droplet_in_gradient():
    # config-3 set-up at reduced size: the first / last slab keeps the wall on its outer face
    wl = configs.droplet_in_gradient(nx=20, ny=22, nz=30, thermal="lb_d3q19", R=6.0, zc=11.0)
    want, _ = run_gpu(wl, 25)
    got, _ = run_slabs(wl, 3, 25)
    assert_same_bits(got, want)


def test_walls_in_y_with_wall_temperature_rows_and_moving_wall():
    # config-2 set-up extruded in z (periodic): the y-wall temperature planes [nz][nx] are cut with ghost rows
    wl = configs.layered_channel(nx=32, ny=16, nz=6)
    rng = np.random.default_rng(7)
    wl.wall_T[(1, 0)] = torch.from_numpy(20.0 + rng.standard_normal((6, 32)))   # varies along z as well
    wl.phi = wl.phi + 0.0
    wl.T = wl.T + torch.from_numpy(0.01 * rng.standard_normal((6, 16, 32)))
    wall_u = [[[0.0] * 3, [0.0] * 3] for _ in range(3)]
    wall_u[1][1] = [0.01, 0.0, 0.004]
    extra = dict(wall_u=wall_u)
    want, _ = run_gpu(wl, 20, extra=extra)
    got, _ = run_slabs(wl, 2, 20, extra=extra)
    assert_same_bits(got, want)


def test_tweezer_with_heat_source_and_initial_velocity():
    wl = configs.thermal_tweezer(nx=24, ny=20, nz=18, thermal="lb_d3q15", R=5.0, offset=4.0, A=2.0, s=5.0)
    q = configs.laser_source(24, 20, 18, Q_s=0.01, w_s=4.0, d_s=5.0)
    want, _ = run_gpu(wl, 20, q=q)
    got, _ = run_slabs(wl, 3, 20, q=q)
    assert_same_bits(got, want)


@pytest.mark.parametrize("nx", [24, 23])
def test_fp32_slabs(nx):
    # even nx: the packed-pair kernel; odd nx: one cell per thread
    wl = configs.perf_box(nx, thermal="lb_d3q7", ny=16, nz=15, seed=2, r_min=4.0, r_max=5.0)
    want, _ = run_gpu(wl, 15, precision="f32")
    got, _ = run_slabs(wl, 3, 15, precision="f32")
    assert_same_bits(got, want)


@pytest.mark.parametrize("thermal", ["rk2", "rk4"])
def test_runge_kutta_slabs(thermal):
    # Algorithm 2: one transfer after the fused kernel and one after every stage (3 / 5 per step)
    wl = configs.perf_box(36, thermal=thermal, ny=20, nz=23, seed=4, r_min=4.0, r_max=5.0)   # x spans two 32-wide tiles
    want, _ = run_gpu(wl, 12)
    got, _ = run_slabs(wl, 3, 12)
    assert_same_bits(got, want)


def test_runge_kutta_tweezer_walls_in_z():
    # config-4 set-up at reduced size (RK2, wall-temperature plane on the bottom wall, initial velocity)
    wl = configs.thermal_tweezer(nx=24, ny=20, nz=18, thermal="rk2", R=5.0, offset=4.0, A=2.0, s=5.0)
    q = configs.laser_source(24, 20, 18, Q_s=0.01, w_s=4.0, d_s=5.0)
    want, _ = run_gpu(wl, 20, q=q)
    got, _ = run_slabs(wl, 4, 20, q=q)
    assert_same_bits(got, want)
    assert_parity_f64(got, run_oracle(wl, 20, q=q))


def test_runge_kutta_phases_and_messages():
    wl = configs.perf_box(16, thermal="rk4", ny=12, nz=12, seed=1, r_min=3.0, r_max=4.0)
    plane = 16 * 12 * 8
    # equal conductivities (the benchmark fluid): stage 1 runs inside the fused kernel, its output travels with phase 0
    box = LocalSlabs(16, 12, 12, 2, dict(wl.params))
    h = box.slabs[0].sim._h
    assert wl.params["kappa_H"] == wl.params["kappa_L"]
    assert B.tcp_halo_phases(h) == 4
    assert [B.tcp_halo_message_bytes(h, p) for p in range(4)] == [20 * plane] + [plane] * 3
    assert B.tcp_halo_bytes(h) == 20 * plane
    box.close()
    box = LocalSlabs(16, 12, 12, 2, dict(wl.params, thermal="rk2"))
    assert B.tcp_halo_phases(box.slabs[0].sim._h) == 2
    box.close()
    # different conductivities: every stage is a kernel of its own
    wl.params["kappa_H"] = 0.1
    box = LocalSlabs(16, 12, 12, 2, dict(wl.params))
    h = box.slabs[0].sim._h
    assert B.tcp_halo_phases(h) == 5
    assert [B.tcp_halo_message_bytes(h, p) for p in range(5)] == [19 * plane] + [plane] * 4
    assert B.tcp_halo_bytes(h) == 19 * plane
    box.init_fields(_np(wl.phi), None, _np(wl.T))
    B.tcp_step_begin(h)
    with pytest.raises(tcp.TcpError) as e:
        B.tcp_step_end(h)                      # four stages and their transfers are still to come
    assert e.value.code == B.TCP_ESTATE
    assert [B.tcp_step_advance(h) for _ in range(5)] == [4, 3, 2, 1, 0]
    with pytest.raises(tcp.TcpError) as e:
        B.tcp_step_advance(h)
    assert e.value.code == B.TCP_ESTATE
    box.close()
    box = LocalSlabs(16, 12, 12, 2, dict(wl.params, thermal="rk2"))
    assert B.tcp_halo_phases(box.slabs[0].sim._h) == 3
    box.close()


def test_general_rates_and_bgk_in_slabs():
    wl = configs.perf_box(16, thermal="lb_d3q7", ny=14, nz=12, seed=9, r_min=3.0, r_max=4.0)
    for extra in (dict(s_high=1.5, s_bulk=0.8), dict(high_rate_equals_shear=1)):
        want, _ = run_gpu(wl, 10, extra=extra)
        got, _ = run_slabs(wl, 2, 10, extra=extra)
        assert_same_bits(got, want)


def test_launch_count_and_messages():
    wl = configs.perf_box(16, thermal="lb_d3q27", ny=12, nz=12, seed=1, r_min=3.0, r_max=4.0)
    params = dict(wl.params)
    box = LocalSlabs(16, 12, 12, 2, params)
    s0 = box.slabs[0]
    assert B.tcp_halo_bytes(s0.sim._h) == (9 + 9 + 9 + 2) * 16 * 12 * 8
    box.init_fields(_np(wl.phi), None, _np(wl.T))
    before = box.launches
    box.step(3)
    box.synchronize()
    # per slab and step: two boundary planes, the interior, one gather, one scatter
    assert box.launches - before == 2 * 3 * 5
    assert s0.sim.last_step_ms() > 0.0
    box.close()


def test_state_errors():
    wl = configs.perf_box(16, thermal="lb_d3q7", ny=12, nz=8, seed=1, r_min=3.0, r_max=4.0)
    box = LocalSlabs(16, 12, 8, 2, dict(wl.params))
    h = box.slabs[0].sim._h
    with pytest.raises(tcp.TcpError) as e:
        B.tcp_step_begin(h)                       # not initialised
    assert e.value.code == B.TCP_ESTATE
    box.init_fields(_np(wl.phi), None, _np(wl.T))
    with pytest.raises(tcp.TcpError) as e:
        B.tcp_step(h, 1)
    assert e.value.code == B.TCP_ESTATE
    with pytest.raises(tcp.TcpError) as e:
        B.tcp_step_end(h)
    assert e.value.code == B.TCP_ESTATE
    B.tcp_step_begin(h)
    with pytest.raises(tcp.TcpError) as e:
        B.tcp_step_begin(h)
    assert e.value.code == B.TCP_ESTATE
    B.tcp_step_end(h)
    with pytest.raises(tcp.TcpError) as e:
        B.tcp_relax_temperature(h, 2)
    assert e.value.code == B.TCP_EUNSUPPORTED
    box.close()
    # a plain box has no split step; AA boxes take no ghost planes
    sim = tcp.Simulation(16, 12, 8, dict(wl.params))
    with pytest.raises(tcp.TcpError) as e:
        B.tcp_step_begin(sim._h)
    assert e.value.code == B.TCP_ESTATE
    sim.close()
    buf = torch.zeros(64 * 16 * 12, dtype=torch.float64, device="cuda")
    sim = tcp.Simulation(16, 12, 8, dict(wl.params, streaming="aa"))
    with pytest.raises(tcp.TcpError) as e:
        B.tcp_set_halo(sim._h, 1, 1, torch.cuda.Stream(), buf, buf, buf, buf)
    assert e.value.code == B.TCP_EUNSUPPORTED
    sim.close()
    sim = tcp.Simulation(16, 12, 2, dict(wl.params))
    with pytest.raises(tcp.TcpError) as e:
        B.tcp_set_halo(sim._h, 1, 1, torch.cuda.Stream(), buf, buf, buf, buf)     # no plane of its own left
    assert e.value.code == B.TCP_EINVAL
    with pytest.raises(tcp.TcpError) as e:
        B.tcp_set_halo(sim._h, 1, 0, torch.cuda.Stream(), None, None, None, None)  # missing buffers
    assert e.value.code == B.TCP_EINVAL
    sim.close()
