"""Maxwellian equilibrium in central-moment space (`equilibrium = "maxwellian"`, D3Q27 lattices): the CUDA path (product
form added to the closed-form collisions) against the oracle (dense solve K(u) a = kappa^M)."""
import numpy as np
import pytest
import torch

import paper_2401_03041_b200 as tcp
import workloads as W
from parity_util import assert_parity_f32, assert_parity_f64, run_gpu, run_oracle

pytestmark = pytest.mark.gpu
MX = dict(equilibrium="maxwellian")


def _with_velocity(wl, amp=0.03, seed=1):
    rng = np.random.default_rng(seed)
    wl.u = torch.from_numpy(amp * rng.standard_normal((3, wl.nz, wl.ny, wl.nx)))     # the equilibria differ at O(u^3)
    return wl


@pytest.mark.parametrize("thermal", ["lb_d3q27", "rk2", "rk4"])
def test_periodic_box(thermal):
    wl = _with_velocity(W.perf_box(24, thermal=thermal, ny=20, nz=18, r_min=3.0, r_max=5.0, seed=7))
    assert_parity_f64(run_gpu(wl, 0, extra=MX)[0], run_oracle(wl, 0, extra=MX), tol=1e-14)     # initial equilibria
    want = run_oracle(wl, 100, extra=MX)
    got, _ = run_gpu(wl, 100, extra=MX)
    assert_parity_f64(got, want)
    printed, _ = run_gpu(wl, 100)
    assert np.abs(printed[1] - got[1]).max() > 1e-8


@pytest.mark.parametrize("extra", [dict(s_bulk=0.9), dict(collision_space="raw"), dict(streaming="aa"), dict(thermal="rk2")])
def test_channel_with_walls_in_other_modes(extra):
    wl = W.layered_channel(nx=44, ny=26, nz=2, thermal="lb_d3q27", rho_upper=2.0)
    wu = [[[0.0] * 3 for _ in range(2)] for _ in range(3)]
    wu[1][1] = [2e-2, 0.0, 1e-2]
    e = dict(MX, wall_u=wu, **extra)
    for steps in (50, 51):
        want = run_oracle(wl, steps, extra=e)
        got, _ = run_gpu(wl, steps, extra=e)
        assert_parity_f64(got, want)


@pytest.mark.parametrize("nx", [36, 35])
def test_fp32(nx):
    wl = W.thermal_tweezer(nx=nx, ny=20, nz=18, thermal="lb_d3q27", R=5.0, offset=7.0, A=2.0, s=4.0)
    want = run_oracle(wl, 40, extra=MX)
    got, _ = run_gpu(wl, 40, extra=MX, precision="f32")
    assert_parity_f32(got, want, sigma=0.0, label=f"tweezer {nx}x20x18 Maxwellian equilibrium")


def test_other_lattices_are_refused():
    for bad in (dict(MX, thermal="lb_d3q7"), dict(MX, thermal="lb_d3q27", hydro_lattice=19), dict(MX, thermal="rk2", s_high=1.3),
                dict(MX, thermal="rk2", high_rate_equals_shear=1)):
        with pytest.raises(tcp.TcpError) as e:
            tcp.tcp_workspace_bytes(8, 8, 8, tcp.make_params(bad))
        assert e.value.code == tcp.TCP_EUNSUPPORTED
    assert tcp.tcp_workspace_bytes(8, 8, 8, tcp.make_params(dict(MX, thermal="rk4"))) > 0


@pytest.mark.parametrize("streaming", ["two_grid", "aa"])
def test_temperature_preinitialisation_with_the_maxwellian(streaming):
    """tcp_relax_temperature runs the thermal-only kernel: its Maxwellian instantiation (D3Q27 thermal LB)."""
    from oracle import tcpo
    wl = _with_velocity(W.layered_channel(nx=20, ny=14, nz=6, thermal="lb_d3q27"), amp=0.02, seed=3)
    p = dict(wl.params, equilibrium=1)
    o = tcpo.Oracle(wl.nx, wl.ny, wl.nz, p)
    sim = tcp.Simulation(wl.nx, wl.ny, wl.nz, dict(p, streaming=streaming))
    for (ax, fc), plane in wl.wall_T.items():
        o.set_wall_temperature(ax, fc, plane.numpy()); sim.set_wall_temperature(ax, fc, plane.numpy())
    o.init_fields(wl.phi.numpy(), wl.u.numpy(), wl.T.numpy()); sim.init_fields(wl.phi.numpy(), wl.u.numpy(), wl.T.numpy())
    o.relax_temperature(20); sim.relax_temperature(20)
    o.step(5); sim.step(5)
    want, got = o.read_fields(), sim.read_fields()
    o.close(); sim.close()
    assert_parity_f64(got, want)
