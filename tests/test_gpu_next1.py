"""NEXT-1 ingredients of the droplet-capture workload on the GPU against the oracle:
moving wall (reading S18) and temperature pre-initialisation."""
import numpy as np
import pytest
import torch

import paper_2401_03041_b200 as tcp
import workloads as W
from oracle import tcpo
from parity_util import assert_parity_f64, run_gpu, run_oracle

pytestmark = pytest.mark.gpu


def _wall_u(entries):
    w = [[[0.0] * 3 for _ in range(2)] for _ in range(3)]
    for (axis, face), vec in entries.items():
        w[axis][face] = list(vec)
    return w


@pytest.mark.parametrize("streaming", ["two_grid", "aa"])
@pytest.mark.parametrize("thermal", ["lb_d3q7", "rk2"])
def test_sheared_droplet_under_a_moving_wall(thermal, streaming):
    """Droplet next to the bottom wall of a channel whose top wall moves (the paper's shear set-up,
    PAPER.md:295), heated by the laser source of eq. 37."""
    wl = W.thermal_tweezer(nx=32, ny=18, nz=16, thermal=thermal, R=4.5, offset=5.0, A=0.0, s=4.0)
    q = W.laser_source(32, 18, 16, Q_s=0.02, centre=(12.0, 8.5, 5.0), w_s=4.0, d_s=5.0)
    extra = dict(wall_u=_wall_u({(2, 1): (2e-3, 1e-3, 0.0), (2, 0): (-1e-3, 0.0, 0.0)}), streaming=streaming)
    for steps in (60, 61):
        want = run_oracle(wl, steps, q=q.numpy(), extra=extra)
        got, _ = run_gpu(wl, steps, q=q.numpy(), extra=extra)
        assert_parity_f64(got, want)
    assert np.abs(want[1][0]).max() > 5e-4                   # the walls did drag the fluid


def test_moving_walls_on_two_axes_and_bgk():
    wl = W.perf_box(14, thermal="lb_d3q19", ny=12, nz=10, r_min=3.0, r_max=4.0, seed=11)
    wl.params["bc"] = ("walls", "periodic", "walls")
    extra = dict(wall_u=_wall_u({(0, 0): (0.0, 1e-3, -1e-3), (2, 1): (2e-3, 0.0, 0.0)}))
    for more in ({}, dict(high_rate_equals_shear=1), dict(streaming="aa"), dict(s_high=1.2)):
        e = dict(extra, **more)
        want = run_oracle(wl, 41, extra=e)
        got, _ = run_gpu(wl, 41, extra=e)
        assert_parity_f64(got, want)


def _relax_both(wl, n_relax, n_step, extra=None, precision="f64"):
    params = dict(wl.params, **(extra or {}))
    o = tcpo.Oracle(wl.nx, wl.ny, wl.nz, params)
    sim = tcp.Simulation(wl.nx, wl.ny, wl.nz, dict(params, precision=precision))
    for (ax, fc), pl in wl.wall_T.items():
        o.set_wall_temperature(ax, fc, pl.numpy()); sim.set_wall_temperature(ax, fc, pl.numpy())
    T0 = np.full((wl.nz, wl.ny, wl.nx), 15.0)
    o.init_fields(wl.phi.numpy(), None, T0); sim.init_fields(wl.phi.numpy(), None, T0)
    o.relax_temperature(n_relax); sim.relax_temperature(n_relax)
    mid = (o.read_fields(), sim.read_fields())
    o.step(n_step); sim.step(n_step)
    o.relax_temperature(2); sim.relax_temperature(2)        # also in the middle of a run
    o.step(3); sim.step(3)
    out = (o.read_fields(), sim.read_fields())
    o.close(); sim.close()
    return mid, out


@pytest.mark.parametrize("thermal", ["lb_d3q7", "lb_d3q15", "lb_d3q19", "lb_d3q27", "rk2", "rk4"])
@pytest.mark.parametrize("streaming", ["two_grid", "aa"])
def test_temperature_preinitialisation_then_coupled_steps(thermal, streaming):
    wl = W.layered_channel(nx=36, ny=18, nz=2, thermal=thermal, kappa_upper=0.08)
    mid, out = _relax_both(wl, 80, 30, extra=dict(streaming=streaming))
    assert_parity_f64(mid[1], mid[0])
    assert np.array_equal(mid[1][0], wl.phi.numpy()) and np.abs(mid[1][1]).max() == 0.0   # phi, u frozen
    assert np.abs(mid[0][3] - 15.0).max() > 1.0                                            # T did relax
    assert_parity_f64(out[1], out[0])


def test_relaxation_argument_checks():
    wl = W.layered_channel(nx=12, ny=8, nz=1, thermal="lb_d3q7")
    sim = tcp.Simulation(wl.nx, wl.ny, wl.nz, dict(wl.params, streaming="aa"))
    with pytest.raises(tcp.TcpError) as e:
        sim.relax_temperature(2)
    assert e.value.code == tcp.TCP_ESTATE
    sim.init_fields(wl.phi.numpy(), None, wl.T.numpy())
    with pytest.raises(tcp.TcpError) as e:
        sim.relax_temperature(3)                            # AA + thermal LB: even counts only
    assert e.value.code == tcp.TCP_EINVAL
    with pytest.raises(tcp.TcpError) as e:
        sim.relax_temperature(-1)
    assert e.value.code == tcp.TCP_EINVAL
    sim.relax_temperature(0); sim.relax_temperature(4)
    sim.close()
