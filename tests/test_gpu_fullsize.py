"""Parity at the sizes and in the launch configurations bench.py times (BASELINE configs[4]): every kernel of the
sweep on its full-size box, compared with the oracle on sampled cells, plus properties that hold at any size.

The oracle cannot run 64-134 M cells, so for each sampled cell it runs on the (2*half+1)^3 sub-box of the INITIAL
state around the cell; the periodic wrap of the sub-box only pollutes cells within 2*steps+1 of its faces, so with
half >= 2*steps+2 the centre cell is exact.  Samples cover what only a full-size launch exercises: more than one wave
of blocks, the L2-prefetch clamping at the array ends (first / last blocks, the last prefetch group), 64-bit plane
offsets q*N > 2^31 elements, the periodic seams."""
import gc

import numpy as np
import pytest
import torch

import paper_2401_03041_b200 as tcp
import workloads as W
from parity_util import run_oracle

pytestmark = pytest.mark.gpu


def test_fp64_sum_phi_and_energy_conservation_long_run():
    """Properties that hold at any size: over 2000 steps of the periodic bench box sum(phi) is
    conserved to round-off and (thermal LB, no walls, no source) so is sum(T)."""
    n = 96
    wl = W.perf_box(n, thermal="lb_d3q7", seed=5, device="cuda")
    sim = tcp.Simulation(n, n, n, wl.params)
    sim.init_fields(wl.phi, None, wl.T)
    sim.step(2000)
    phi, u, p, T = sim.read_fields_device()
    sim.close()
    assert bool(torch.isfinite(phi).all()) and bool(torch.isfinite(u).all())
    assert abs(float(phi.sum()) - float(wl.phi.sum())) / float(wl.phi.sum()) < 1e-11
    assert abs(float(T.sum()) - float(wl.T.sum())) / float(wl.T.sum()) < 1e-11
    assert float(phi.min()) > -1e-3 and float(phi.max()) < 1 + 1e-3


def _sample_cells(wl, n, samples, rng):
    # a third on droplet interfaces (where the forces live), the rest anywhere ...
    cand = torch.nonzero((wl.phi > 0.2) & (wl.phi < 0.8))
    picks = [tuple(int(v) for v in cand[int(rng.integers(len(cand)))]) for _ in range(samples // 3)]
    picks += [tuple(int(v) for v in rng.integers(0, n, 3)) for _ in range(samples - samples // 3)]
    # ... plus the places only a full-size launch reaches: the periodic seams, the first and the last block (cells
    # 0.. and ..N-1), the first / last z-plane, and the last prefetch group (the last ~70 blocks = the last ~22 rows of
    # the last plane), where the bulk L2 prefetch is clamped to the array
    picks += [(0, 0, 0), (0, 0, 77), (n - 1, n - 1, n - 1), (n - 1, n - 1, n - 100), (0, n - 1, n // 2), (n // 2, 0, n - 1)]
    picks += [(0, int(rng.integers(n)), int(rng.integers(n))) for _ in range(3)]
    picks += [(n - 1, int(rng.integers(n)), int(rng.integers(n))) for _ in range(3)]
    picks += [(n - 1, n - 1 - int(rng.integers(22)), int(rng.integers(n))) for _ in range(4)]
    return picks


def _sampled_parity(n, thermal, steps, samples, half, precision="f64", streaming="two_grid", extra=None, box=None):
    """-> dict field -> (worst abs error over the samples, max |oracle| over the samples)"""
    assert half >= 2 * steps + 2
    wl = W.perf_box(n, thermal=thermal, device="cuda", **(box or {}))
    torch.cuda.empty_cache()
    tdt = torch.float64 if precision == "f64" else torch.float32
    if extra:
        wl.params.update(extra)
    sim = tcp.Simulation(n, n, n, dict(wl.params, precision=precision, streaming=streaming))
    sim.init_fields(wl.phi.to(tdt), None, wl.T.to(tdt))
    sim.step(steps)
    got = sim.read_fields_device()
    launches = sim.launches
    sim.close()
    torch.cuda.empty_cache()
    assert launches >= steps
    rng = np.random.default_rng(n)
    m = 2 * half + 1
    idx = torch.arange(-half, half + 1, device="cuda")
    names = ("phi", "ux", "uy", "uz", "p", "T")
    worst = {k: [0.0, 0.0] for k in names}
    picks = _sample_cells(wl, n, samples, rng)
    assert len(picks) >= 32
    for (z, y, x) in picks:
        iz, iy, ix = ((z + idx) % n).view(-1, 1, 1), ((y + idx) % n).view(1, -1, 1), ((x + idx) % n).view(1, 1, -1)
        sub = W.Workload("sub", m, m, m, wl.params, wl.phi[iz, iy, ix].cpu(), T=wl.T[iz, iy, ix].cpu())
        want = run_oracle(sub, steps)
        c = (half, half, half)
        vals = {"phi": (float(got[0][z, y, x]), want[0][c]), "p": (float(got[2][z, y, x]), want[2][c]),
                "T": (float(got[3][z, y, x]), want[3][c])}
        for a, k in enumerate(("ux", "uy", "uz")):
            vals[k] = (float(got[1][a, z, y, x]), want[1][(a,) + c])
        for k, (g, w) in vals.items():
            assert np.isfinite(g), f"{k} at {(z, y, x)} is not finite"
            worst[k][0] = max(worst[k][0], abs(g - w))
            worst[k][1] = max(worst[k][1], abs(w))
    print(f"sampled parity {n}^3 {thermal} {precision} {streaming} {steps} steps, {len(picks)} cells: "
          + "  ".join(f"{k}: {v[0]:.2e} / {v[1]:.2e}" for k, v in worst.items()))
    return worst


@pytest.mark.parametrize("thermal,streaming,steps", [
    ("lb_d3q7", "two_grid", 5),      # the headline kernel: h, g, f staged, three blocks per SM
    ("lb_d3q19", "two_grid", 5),     # h pulled straight into registers (h_direct)
    ("lb_d3q27", "two_grid", 5),     # two blocks per SM, prefetch distance TCP_PF2; 27 * 64e6 * 3 planes
    ("rk2", "two_grid", 5),          # fused kernel with stage 1 inside + the z-marching stage kernel
    ("rk4", "two_grid", 5),
    ("lb_d3q7", "aa", 5),            # AA in place, odd step count: populations left in the pushed layout
    ("lb_d3q7", "aa", 6),            # ... and even
])
def test_full_size_sampled_parity_400_cubed(thermal, streaming, steps):
    """The bench workload itself, 400^3 fp64 (plane offsets q*N up to 26 * 64e6 = 1.7e9 elements, 13 GB)."""
    worst = _sampled_parity(400, thermal, steps=steps, samples=18, half=2 * steps + 2, streaming=streaming)
    assert max(v[0] for v in worst.values()) <= 1e-10


@pytest.mark.parametrize("thermal", ["lb_d3q7", "rk2"])
def test_full_size_sampled_parity_512_cubed_fp32(thermal):
    """The fp32 bench box, 512^3 (packed-pair kernel; q*N up to 26 * 134e6 = 3.5e9 elements > 2^31): sampled cells
    against the fp64 oracle at the fp32 bar -- 1e-5 relative to the largest sampled value of each field; for the
    velocity components and p the fp32 force-noise floor of parity_util.assert_parity_f32 applies (sigma_ref = 5e-3)."""
    worst = _sampled_parity(512, thermal, steps=5, samples=18, half=12, precision="f32")
    sig = W.BENCH_FLUID["sigma_ref"]
    umax = max(worst[k][1] for k in ("ux", "uy", "uz"))
    assert worst["phi"][0] <= 1e-5 * worst["phi"][1]
    assert worst["T"][0] <= 1e-5 * worst["T"][1]
    assert worst["p"][0] <= max(1e-5 * worst["p"][1], 1e-6 * sig)
    for k in ("ux", "uy", "uz"):
        assert worst[k][0] <= max(1e-5 * umax, 2e-6 * sig)


@pytest.mark.parametrize("n,thermal,precision,streaming,steps", [
    (624, "lb_d3q7", "f64", "aa", 5),         # 243 M cells, 134 GB: 32-bit in-group offsets up to 10 N = 2.4e9 > 2^31 (fp64 kernel)
    (640, "lb_d3q7", "f32", "two_grid", 5),   # 262 M cells, 136 GB: the same in the fp32 pair kernel
    (752, "lb_d3q7", "f32", "aa", 6),         # 425 M cells, 117 GB: the largest cube under the N <= 429 496 729 limit of tcp_create
    (640, "rk2", "f64", "aa", 5),             # 132 GB: the z-marching Runge-Kutta stage kernel at 262 M cells
    (680, "lb_d3q27", "f32", "aa", 5),        # 314 M cells, 81 population planes: plane offsets up to 80 N = 2.5e10 elements
])
def test_largest_boxes_sampled_parity(n, thermal, precision, streaming, steps):
    """Maximum sizes: the largest boxes one B200 holds (fp64 only with AA in place), where plane offsets reach
    26 N = 1.1e10 elements and the 32-bit offsets inside a group of nine planes (tcp_step.cuh) pass 2^31."""
    gc.collect()
    torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info()
    need = tcp.tcp_workspace_bytes(n, n, n, tcp.make_params(dict(W.BENCH_FLUID, thermal=thermal, precision=precision,
                                                                 streaming=streaming))) + 80 * n ** 3
    if free < need:
        pytest.skip(f"{free / 1e9:.0f} GB free, {need / 1e9:.0f} GB needed")
    worst = _sampled_parity(n, thermal, steps=steps, samples=18, half=2 * steps + 2, precision=precision,
                            streaming=streaming, box=dict(r_min=24.0, r_max=48.0))
    if precision == "f64":
        assert max(v[0] for v in worst.values()) <= 1e-10
    else:
        sig = W.BENCH_FLUID["sigma_ref"]
        umax = max(worst[k][1] for k in ("ux", "uy", "uz"))
        assert worst["phi"][0] <= 1e-5 * worst["phi"][1] and worst["T"][0] <= 1e-5 * worst["T"][1]
        assert worst["p"][0] <= max(1e-5 * worst["p"][1], 1e-6 * sig)
        for k in ("ux", "uy", "uz"):
            assert worst[k][0] <= max(1e-5 * umax, 2e-6 * sig)


def test_box_beyond_the_memory_is_refused_and_the_library_stays_usable():
    n = 700                                                             # fp64 two-grid D3Q27: 467 GB
    with pytest.raises(tcp.TcpError) as e:                              # tcp_create: the library's own cudaMalloc
        tcp.tcp_create(n, n, n, tcp.make_params(dict(W.BENCH_FLUID, thermal="lb_d3q27")))
    assert e.value.code == tcp.TCP_ENOMEM
    with pytest.raises(tcp.TcpError) as e:                              # 760^3 > 429 496 729 cells
        tcp.Simulation(760, 760, 760, dict(W.BENCH_FLUID, thermal="rk2", precision="f32", streaming="aa"))
    assert e.value.code in (tcp.TCP_EINVAL, tcp.TCP_EUNSUPPORTED)
    wl = W.static_droplet(n=16, R=4.0)
    sim = tcp.Simulation(16, 16, 16, wl.params)
    sim.init_fields(wl.phi.numpy())
    sim.step(3)
    assert np.isfinite(sim.read_fields()[2]).all()
    sim.close()
