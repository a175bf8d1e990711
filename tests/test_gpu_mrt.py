"""Raw-moment (MRT) collision space (`collision_space = "raw"`): the CUDA path against the oracle.  On the GPU
it is the central-moment kernel with the carrier populations of the relaxed moments taken about the lattice at rest
(DESIGN.md section 5), so every kernel variant is covered by one flag: thermal stencils, walls, general rates, the D3Q19
hydrodynamic lattice, AA, fp32."""
import numpy as np
import pytest

import paper_2401_03041_b200 as tcp
import workloads as W
from parity_util import assert_parity_f32, assert_parity_f64, run_gpu, run_oracle

pytestmark = pytest.mark.gpu
RAW = dict(collision_space="raw")


@pytest.mark.parametrize("thermal", ["lb_d3q7", "lb_d3q15", "lb_d3q19", "lb_d3q27", "rk2"])
def test_periodic_box(thermal):
    wl = W.perf_box(24, thermal=thermal, ny=20, nz=18, r_min=3.0, r_max=5.0, seed=7)
    rng = np.random.default_rng(1)
    import torch
    wl.u = torch.from_numpy(0.02 * rng.standard_normal((3, 18, 20, 24)))     # u != 0: the two spaces differ at O(u)
    want = run_oracle(wl, 100, extra=RAW)
    got, _ = run_gpu(wl, 100, extra=RAW)
    assert_parity_f64(got, want)
    cm, _ = run_gpu(wl, 100)
    assert np.abs(cm[1] - got[1]).max() > 1e-7          # a different operator from the central-moment one


@pytest.mark.parametrize("extra", [dict(s_high=1.4, s_bulk=0.9), dict(high_rate_equals_shear=1), dict(hydro_lattice=19, s_bulk=0.8),
                                   dict(streaming="aa")])
def test_channel_with_walls_in_other_modes(extra):
    wl = W.layered_channel(nx=44, ny=26, nz=2, thermal="lb_d3q19", rho_upper=2.0)
    wu = [[[0.0] * 3 for _ in range(2)] for _ in range(3)]
    wu[1][1] = [5e-3, 0.0, 2e-3]
    e = dict(RAW, wall_u=wu, **extra)
    for steps in (50, 51):
        want = run_oracle(wl, steps, extra=e)
        got, _ = run_gpu(wl, steps, extra=e)
        assert_parity_f64(got, want)


@pytest.mark.parametrize("nx", [36, 35])
def test_fp32(nx):
    wl = W.thermal_tweezer(nx=nx, ny=20, nz=18, thermal="lb_d3q7", R=5.0, offset=7.0, A=2.0, s=4.0)
    want = run_oracle(wl, 40, extra=RAW)
    got, _ = run_gpu(wl, 40, extra=RAW, precision="f32")
    assert_parity_f32(got, want, sigma=0.0, label=f"tweezer {nx}x20x18 raw-moment space")


def test_bad_value_is_refused():
    with pytest.raises(tcp.TcpError) as e:
        tcp.tcp_workspace_bytes(8, 8, 8, tcp.make_params(dict(collision_space=2)))
    assert e.value.code == tcp.TCP_EINVAL
