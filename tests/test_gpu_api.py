"""GPU tests of the C ABI itself (include/tcp.h): both creation paths, pointer kinds, error codes,
resetting optional inputs, two simulations side by side.  Run with `pytest -m gpu` on a B200."""
import ctypes as C

import numpy as np
import pytest
import torch

import paper_2401_03041_b200 as tcp
import workloads as W
from parity_util import assert_parity_f64, run_oracle

pytestmark = pytest.mark.gpu


def _wl():
    return W.droplet_in_gradient(nx=16, ny=12, nz=20, thermal="lb_d3q7", R=4.0, zc=8.0, grad_T=0.05)


def test_tcp_create_owns_memory_and_stream_host_pointers():
    """tcp_create (library-allocated workspace, own stream) with plain host numpy arrays."""
    wl = _wl()
    want = run_oracle(wl, 20)
    p = tcp.make_params(wl.params)
    h = tcp.tcp_create(wl.nx, wl.ny, wl.nz, p)
    try:
        tcp.tcp_init_fields(h, wl.phi.numpy(), None, wl.T.numpy())
        tcp.tcp_step(h, 20)
        shape = (wl.nz, wl.ny, wl.nx)
        phi, u, pr, T = np.empty(shape), np.empty((3,) + shape), np.empty(shape), np.empty(shape)
        tcp.tcp_read_fields(h, phi, u, pr, T)
        assert_parity_f64((phi, u, pr, T), want)
        assert tcp.tcp_launch_count(h) >= 20
        assert tcp.tcp_last_step_ms(h) > 0
        # partial read-back: any pointer may be NULL
        T2 = np.empty(shape)
        tcp.tcp_read_fields(h, None, None, None, T2)
        assert np.array_equal(T2, T)
    finally:
        tcp.tcp_destroy(h)


def test_state_and_argument_errors():
    wl = _wl()
    h = tcp.tcp_create(wl.nx, wl.ny, wl.nz, tcp.make_params(wl.params))
    try:
        with pytest.raises(tcp.TcpError) as e:
            tcp.tcp_step(h, 1)
        assert e.value.code == tcp.TCP_ESTATE
        with pytest.raises(tcp.TcpError) as e:
            tcp.tcp_read_fields(h, None, None, None, np.empty(4))
        assert e.value.code == tcp.TCP_ESTATE
        with pytest.raises(tcp.TcpError) as e:
            tcp.tcp_last_step_ms(h)
        assert e.value.code == tcp.TCP_ESTATE
        with pytest.raises(tcp.TcpError) as e:
            tcp.tcp_init_fields(h, None)
        assert e.value.code == tcp.TCP_EINVAL
        tcp.tcp_init_fields(h, wl.phi.numpy(), None, wl.T.numpy())
        with pytest.raises(tcp.TcpError) as e:
            tcp.tcp_step(h, -1)
        assert e.value.code == tcp.TCP_EINVAL
        with pytest.raises(tcp.TcpError) as e:
            tcp.tcp_set_wall_temperature(h, 3, 0, None)
        assert e.value.code == tcp.TCP_EINVAL
        assert "axis" in tcp.tcp_last_error()
        tcp.tcp_step(h, 1)                      # still usable after the errors
    finally:
        tcp.tcp_destroy(h)
    # undersized / misaligned caller workspace
    p = tcp.make_params(wl.params)
    need = tcp.tcp_workspace_bytes(wl.nx, wl.ny, wl.nz, p)
    small = torch.empty(need // 2, dtype=torch.uint8, device="cuda")
    with pytest.raises(tcp.TcpError) as e:
        tcp.tcp_create_in(wl.nx, wl.ny, wl.nz, p, small)
    assert e.value.code == tcp.TCP_EINVAL
    big = torch.empty(need + 512, dtype=torch.uint8, device="cuda")
    with pytest.raises(tcp.TcpError) as e:
        tcp.tcp_create_in(wl.nx, wl.ny, wl.nz, p, big[8:])
    assert e.value.code == tcp.TCP_EINVAL


def test_optional_inputs_can_be_reset():
    """Wall plane -> NULL restores the constant wall_T; heat source -> NULL removes it."""
    wl = _wl()
    rng = np.random.default_rng(0)
    plane = 0.3 + 0.2 * rng.random((wl.ny, wl.nx))
    q = 1e-3 * rng.random((wl.nz, wl.ny, wl.nx))
    want = run_oracle(wl, 15)                                     # constant walls, no source
    sim = tcp.Simulation(wl.nx, wl.ny, wl.nz, wl.params)
    sim.set_wall_temperature(2, 0, plane)
    sim.set_heat_source(q)
    sim.init_fields(wl.phi.numpy(), None, wl.T.numpy())
    sim.step(3)
    assert np.abs(sim.read_fields()[3] - run_oracle(wl, 3)[3]).max() > 1e-6      # the plane and the source did act
    sim.set_wall_temperature(2, 0, None)
    sim.set_heat_source(None)
    sim.init_fields(wl.phi.numpy(), None, wl.T.numpy())           # re-initialising restarts the run
    sim.step(15)
    assert_parity_f64(sim.read_fields(), want)
    sim.close()


def test_two_simulations_on_two_streams():
    """Independent simulations (different streams, different variants) interleaved step by step."""
    wa = W.perf_box(16, thermal="lb_d3q19", ny=14, nz=12, r_min=3.0, r_max=4.0, seed=2)
    wb = W.layered_channel(nx=24, ny=16, nz=1, thermal="rk2")
    sa = tcp.Simulation(wa.nx, wa.ny, wa.nz, wa.params, stream=torch.cuda.Stream())
    sb = tcp.Simulation(wb.nx, wb.ny, wb.nz, dict(wb.params, streaming="aa"), stream=torch.cuda.Stream())
    for (ax, fc), pl in wb.wall_T.items():
        sb.set_wall_temperature(ax, fc, pl.numpy())
    sa.init_fields(wa.phi.numpy(), None, wa.T.numpy())
    sb.init_fields(wb.phi.numpy(), None, wb.T.numpy())
    for _ in range(10):
        sa.step(2)
        sb.step(3)
    assert_parity_f64(sa.read_fields(), run_oracle(wa, 20))
    assert_parity_f64(sb.read_fields(), run_oracle(wb, 30))
    sa.close(); sb.close()
