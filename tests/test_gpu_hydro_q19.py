"""D3Q19 hydrodynamic lattice (`hydro_lattice = 19`): the CUDA path against the oracle, element by
element, for every thermal variant, with walls (bounce-back, moving wall, wall-temperature plane, wetting), both streaming
patterns, BGK mode, the fp32 kernels and slabs."""
import numpy as np
import pytest
import torch

import paper_2401_03041_b200 as tcp
import workloads as W
from parity_util import assert_parity_f32, assert_parity_f64, run_gpu, run_oracle

pytestmark = pytest.mark.gpu
Q19 = dict(hydro_lattice=19)


@pytest.mark.parametrize("thermal", ["lb_d3q7", "lb_d3q15", "lb_d3q19", "lb_d3q27", "rk2", "rk4"])
def test_periodic_box_all_thermal_variants(thermal):
    wl = W.perf_box(24, thermal=thermal, ny=20, nz=18, r_min=3.0, r_max=5.0, seed=7)
    want = run_oracle(wl, 100, extra=Q19)
    got, _ = run_gpu(wl, 100, extra=Q19)
    assert_parity_f64(got, want)
    # it is a different lattice: the D3Q27 result differs by far more than the bar
    got27, _ = run_gpu(wl, 100)
    assert np.abs(got27[1] - got[1]).max() > 1e-8


@pytest.mark.parametrize("streaming", ["two_grid", "aa"])
@pytest.mark.parametrize("thermal", ["lb_d3q7", "rk2"])
def test_channel_with_walls_moving_wall_and_wetting(streaming, thermal):
    wl = W.layered_channel(nx=44, ny=26, nz=3, thermal=thermal, rho_upper=2.0)
    wu = [[[0.0] * 3 for _ in range(2)] for _ in range(3)]
    wu[1][1] = [2e-3, 0.0, -1e-3]
    extra = dict(Q19, wall_u=wu, streaming=streaming, wall_contact_angle=((90.0, 90.0), (70.0, 110.0), (90.0, 90.0)))
    for steps in (60, 61):
        want = run_oracle(wl, steps, extra=extra)
        got, _ = run_gpu(wl, steps, extra=extra)
        assert_parity_f64(got, want)


def test_walls_on_every_axis_and_bgk_mode():
    wl = W.perf_box(16, thermal="lb_d3q19", ny=14, nz=12, r_min=3.0, r_max=5.0, seed=13, volume_fraction=0.3)
    wl.params.update(bc=("walls", "walls", "walls"), wall_T=((0.2, 0.9), (0.4, 0.6), (0.1, 0.8)), eps_normal=1e-9)
    for extra in (dict(Q19), dict(Q19, high_rate_equals_shear=1), dict(Q19, s_bulk=0.8)):
        want = run_oracle(wl, 50, extra=extra)
        got, _ = run_gpu(wl, 50, extra=extra)
        assert_parity_f64(got, want)


def test_initial_state_pressure_and_chunked_stepping_aa():
    wl = W.droplet_in_gradient(nx=16, ny=12, nz=20, thermal="lb_d3q7", R=4.0, zc=8.0, grad_T=0.05)
    rng = np.random.default_rng(3)
    wl.u = torch.from_numpy(0.01 * rng.standard_normal((3, 20, 12, 16)))
    extra = dict(Q19, streaming="aa")
    assert_parity_f64(run_gpu(wl, 0, extra=extra)[0], run_oracle(wl, 0, extra=Q19), tol=1e-15)
    got, _ = run_gpu(wl, 25, extra=extra, chunks=[1, 2, 0, 5, 17])
    assert_parity_f64(got, run_oracle(wl, 25, extra=Q19))


@pytest.mark.parametrize("nx", [36, 35])
def test_fp32_pair_and_scalar_kernels(nx):
    wl = W.thermal_tweezer(nx=nx, ny=20, nz=18, thermal="lb_d3q7", R=5.0, offset=7.0, A=2.0, s=4.0)
    for extra in (dict(Q19), dict(Q19, streaming="aa")):
        want = run_oracle(wl, 41, extra=Q19)
        got, _ = run_gpu(wl, 41, extra=extra, precision="f32")
        assert_parity_f32(got, want, sigma=0.0, label=f"tweezer {nx}x20x18 hydro D3Q19 {extra.get('streaming', 'two_grid')}")


def test_slabs_are_bit_identical():
    from test_gpu_slabs import assert_same_bits, run_slabs
    for thermal in ("lb_d3q19", "rk4"):
        wl = W.perf_box(24, thermal=thermal, ny=20, nz=22, seed=11, r_min=4.0, r_max=6.0)
        want, _ = run_gpu(wl, 15, extra=Q19)
        got, _ = run_slabs(wl, 3, 15, extra=Q19)
        assert_same_bits(got, want)


def test_general_rates_are_refused_and_the_workspace_is_smaller():
    with pytest.raises(tcp.TcpError) as e:
        tcp.tcp_workspace_bytes(8, 8, 8, tcp.make_params(dict(hydro_lattice=19, s_high=1.3)))
    assert e.value.code == tcp.TCP_EUNSUPPORTED
    with pytest.raises(tcp.TcpError) as e:
        tcp.tcp_workspace_bytes(8, 8, 8, tcp.make_params(dict(hydro_lattice=15)))
    assert e.value.code == tcp.TCP_EINVAL
    sim = tcp.Simulation(8, 8, 8, Q19)          # the calibration kernel exists for the D3Q27 layout only
    sim.init_fields(np.zeros((8, 8, 8)))
    with pytest.raises(tcp.TcpError) as e:
        sim.pattern_copy_ms(1)
    assert e.value.code == tcp.TCP_EUNSUPPORTED
    sim.close()
    n = 64
    b27 = tcp.tcp_workspace_bytes(n, n, n, tcp.make_params({}))
    b19 = tcp.tcp_workspace_bytes(n, n, n, tcp.make_params(Q19))
    assert b27 - b19 == pytest.approx(16 * n ** 3 * 8, rel=1e-3)


def test_full_size_sampled_parity_400_cubed_hydro_q19():
    from test_gpu_fullsize import _sampled_parity
    worst = _sampled_parity(400, "lb_d3q7", steps=5, samples=18, half=12, extra=Q19)
    assert max(v[0] for v in worst.values()) <= 1e-10
