"""AA in-place streaming (`streaming="aa"`, PAPER.md:357 discusses it; one grid of populations): a
storage permutation only, so it must meet the same bar as the two-grid kernel: max-abs error <= 1e-10
against the oracle (which knows nothing about AA) after an even AND after an odd number of steps (the
populations sit in different places then, which the pressure read-back has to undo)."""
import numpy as np
import pytest
import torch

import paper_2401_03041_b200 as tcp
import workloads as W
from parity_util import assert_parity_f32, assert_parity_f64, run_gpu, run_oracle

pytestmark = pytest.mark.gpu
AA = dict(streaming="aa")


@pytest.mark.parametrize("thermal", ["lb_d3q7", "lb_d3q15", "lb_d3q19", "lb_d3q27", "rk2", "rk4"])
@pytest.mark.parametrize("steps", [100, 37])
def test_aa_periodic_box(thermal, steps):
    wl = W.perf_box(24, thermal=thermal, ny=20, nz=18, r_min=3.0, r_max=5.0, seed=7)
    want = run_oracle(wl, steps)
    got, _ = run_gpu(wl, steps, extra=AA)
    assert_parity_f64(got, want)


@pytest.mark.parametrize("thermal", ["lb_d3q7", "lb_d3q19", "rk2"])
@pytest.mark.parametrize("steps", [60, 61])
def test_aa_channel_with_walls_and_wall_temperature_plane(thermal, steps):
    wl = W.layered_channel(nx=44, ny=26, nz=2, thermal=thermal, rho_upper=2.0)
    want = run_oracle(wl, steps)
    got, _ = run_gpu(wl, steps, extra=AA)
    assert_parity_f64(got, want)


@pytest.mark.parametrize("bc", [("walls", "walls", "walls"), ("walls", "periodic", "walls")])
def test_aa_walls_on_several_axes(bc):
    rng = np.random.default_rng(5)
    wl = W.perf_box(14, thermal="lb_d3q27", ny=12, nz=10, r_min=3.0, r_max=4.0, seed=11)
    wl.params["bc"] = bc
    wl.params["wall_T"] = ((0.2, 0.9), (0.4, 0.6), (0.1, 0.8))
    wl.wall_T = {(0, 0): torch.from_numpy(0.2 + 0.1 * rng.random((10, 12))), (2, 1): torch.from_numpy(0.7 + 0.1 * rng.random((12, 14)))}
    for steps in (40, 41):
        want = run_oracle(wl, steps)
        got, _ = run_gpu(wl, steps, extra=AA)
        assert_parity_f64(got, want)


def test_aa_initial_state_and_chunked_stepping():
    wl = W.droplet_in_gradient(nx=16, ny=12, nz=20, thermal="lb_d3q7", R=4.0, zc=8.0, grad_T=0.05)
    rng = np.random.default_rng(3)
    wl.u = torch.from_numpy(0.01 * rng.standard_normal((3, 20, 12, 16)))
    got, _ = run_gpu(wl, 0, extra=AA)                       # pressure gathered from the pushed initial layout
    want = run_oracle(wl, 0)
    assert_parity_f64(got, want, tol=1e-15)
    want = run_oracle(wl, 25)
    got, _ = run_gpu(wl, 25, extra=AA, chunks=[1, 2, 0, 5, 17])
    assert_parity_f64(got, want)


def test_aa_other_collision_modes_and_fp32():
    wl = W.perf_box(20, thermal="lb_d3q19", ny=16, nz=12, r_min=3.0, r_max=4.0, seed=3)
    for extra in (dict(high_rate_equals_shear=1), dict(s_high=1.3, s_bulk=0.9)):
        want = run_oracle(wl, 51, extra=extra)
        got, _ = run_gpu(wl, 51, extra=dict(extra, **AA))
        assert_parity_f64(got, want)
    want = run_oracle(wl, 100)
    got, _ = run_gpu(wl, 100, extra=AA, precision="f32")
    assert_parity_f32(got, want, sigma=wl.params.get("sigma_ref", 0.0))


def test_aa_halves_population_memory():
    p2 = tcp.make_params(dict(thermal="lb_d3q7"))
    pa = tcp.make_params(dict(thermal="lb_d3q7", streaming="aa"))
    n = 64
    b2, ba = tcp.tcp_workspace_bytes(n, n, n, p2), tcp.tcp_workspace_bytes(n, n, n, pa)
    assert (b2 - ba) == pytest.approx(61 * n ** 3 * 8, rel=1e-3)
    assert ba / b2 < 0.56


@pytest.mark.parametrize("streaming", ["aa", "two_grid"])
@pytest.mark.parametrize("thermal", ["lb_d3q7", "lb_d3q27", "rk2"])
def test_wall_temperature_set_after_init_and_mid_run(streaming, thermal):
    """tcp_set_wall_temperature may be called at any time between steps (include/tcp.h).  With AA streaming the
    wall links of f~ are stored already anti-bounced after tcp_init_fields and after every odd step, i.e. they carry
    the wall plane of that moment; the library folds the change into them (aa_wall_repush_kernel).  Sequence: init
    with the constant walls -> set plane A (pushed layout) -> 1 step -> set plane B (natural layout, odd parity) ->
    1 step -> set constant walls again (pushed layout again) -> 4 steps; same calls on the oracle."""
    from oracle import tcpo
    wl = W.layered_channel(nx=20, ny=14, nz=6, thermal=thermal)
    rng = np.random.default_rng(17)
    plane_a = 20.0 + rng.random((6, 20))
    plane_b = 10.0 + 2.0 * rng.random((6, 20))
    o = tcpo.Oracle(wl.nx, wl.ny, wl.nz, wl.params)
    sim = tcp.Simulation(wl.nx, wl.ny, wl.nz, dict(wl.params, streaming=streaming))
    phi0, T0 = wl.phi.numpy(), wl.T.numpy()
    o.init_fields(phi0, None, T0)
    sim.init_fields(phi0, None, T0)
    for (ax, fc, plane, steps) in ((1, 0, plane_a, 1), (1, 1, plane_b, 1), (1, 0, None, 4)):
        if plane is None:
            o.set_wall_temperature(ax, fc, np.full((6, 20), wl.params["wall_T"][ax][fc]))
        else:
            o.set_wall_temperature(ax, fc, plane)
        sim.set_wall_temperature(ax, fc, plane)
        o.step(steps)
        sim.step(steps)
    want, got = o.read_fields(), sim.read_fields()
    o.close(); sim.close()
    assert_parity_f64(got, want)
