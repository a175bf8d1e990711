"""tcp_read_pressure_static (include/tcp.h): the pressure read-back for callers that must not allocate.  Its scratch is a
file-scope `static __device__` array of TCP_STATIC_SCRATCH_BYTES (8 MiB) instead of a buffer of the workspace; the array
is shared by every simulation on the GPU and keeps the last call's contents, so the checks below make two calls in a row
(a larger box first, then a smaller one whose result must not show any of the first call's values) and compare each with
the existing path, tcp_read_fields, bit for bit.  Collected last on purpose (file name): the suite runs with pytest -x.
Passes alone in a fresh process and after the other tests (nothing here depends on earlier state)."""
import os
import re

import numpy as np
import pytest
import torch

import paper_2401_03041_b200 as tcp
import workloads as W



def _sim(wl, steps, **extra):
    sim = tcp.Simulation(wl.nx, wl.ny, wl.nz, dict(wl.params, **extra))
    for (ax, fc), plane in wl.wall_T.items():
        sim.set_wall_temperature(ax, fc, plane.numpy())
    sim.init_fields(wl.phi.numpy(), None if wl.u is None else wl.u.numpy(), None if wl.T is None else wl.T.numpy())
    sim.step(steps)
    return sim


@pytest.mark.gpu
@pytest.mark.parametrize("precision,streaming", [("f64", "two_grid"), ("f32", "two_grid"), ("f64", "aa")])
def test_static_scratch_pressure_equals_read_fields_on_two_calls_in_a_row(precision, streaming):
    big = W.perf_box(40, thermal="lb_d3q7", ny=36, nz=30, r_min=4.0, r_max=6.0, seed=21)
    small = W.layered_channel(nx=24, ny=14, nz=3, thermal="rk2", rho_upper=2.0)
    a = _sim(big, 7, precision=precision, streaming=streaming)          # AA: odd step count, pushed layout
    b = _sim(small, 4, precision=precision, streaming=streaming)
    dt = np.float64 if precision == "f64" else np.float32
    for sim, wl in ((a, big), (b, small), (a, big)):                    # calls in a row share the one static array
        want = sim.read_fields()[2]                                     # existing path: scratch in the workspace
        l0 = sim.launches
        got_host = np.full((wl.nz, wl.ny, wl.nx), np.nan, dtype=dt)
        tcp.tcp_read_pressure_static(sim._h, got_host)                  # host destination
        got_dev = torch.full((wl.nz, wl.ny, wl.nx), float("nan"), dtype=sim.torch_dtype, device="cuda")
        tcp.tcp_read_pressure_static(sim._h, got_dev)                   # device destination
        assert sim.launches - l0 == 2
        assert np.all(np.isfinite(got_host)) and np.abs(want).max() > 0
        # same kernel, same inputs: bit-identical (well inside the 1e-10 / fp32 bars of the parity tests)
        assert np.array_equal(got_host, want)
        assert np.array_equal(got_dev.cpu().numpy(), want)
    # the simulations are unchanged by the read-backs: they keep stepping and agree with a fresh run
    a.step(2)
    fresh = _sim(big, 9, precision=precision, streaming=streaming)
    assert np.array_equal(a.read_fields()[2], fresh.read_fields()[2])
    for s in (a, b, fresh):
        s.close()


@pytest.mark.gpu
def test_static_scratch_rejects_boxes_beyond_its_size_and_bad_state():
    n = 104                                                            # 104^3 * 8 B = 9.0 MB > 8 MiB
    sim = tcp.Simulation(n, n, n, dict(W.BENCH_FLUID, thermal="rk2"))
    out = torch.empty((n, n, n), dtype=torch.float64, device="cuda")
    with pytest.raises(tcp.TcpError) as e:                             # not initialised
        tcp.tcp_read_pressure_static(sim._h, out)
    assert e.value.code == tcp.TCP_ESTATE
    sim.init_fields(torch.zeros((n, n, n), dtype=torch.float64, device="cuda"))
    with pytest.raises(tcp.TcpError) as e:
        tcp.tcp_read_pressure_static(sim._h, out)
    assert e.value.code == tcp.TCP_EUNSUPPORTED and "TCP_STATIC_SCRATCH_BYTES" in str(e.value)
    sim.close()
    assert n ** 3 * 8 > tcp.TCP_STATIC_SCRATCH_BYTES >= 101 ** 3 * 8
    # the same box in fp32 fits (2^21 cells)
    sim = tcp.Simulation(n, n, n, dict(W.BENCH_FLUID, thermal="rk2", precision="f32"))
    sim.init_fields(torch.zeros((n, n, n), dtype=torch.float32, device="cuda"))
    out = torch.empty((n, n, n), dtype=torch.float32, device="cuda")
    tcp.tcp_read_pressure_static(sim._h, out)
    assert float(out.abs().max()) == 0.0                               # p* = 0 initially
    sim.close()


def test_entry_point_source_allocates_nothing():
    """CPU check of the source: the body of tcp_read_pressure_static calls no cudaMalloc / cudaFree / allocating routine,
    resolves the array with cudaGetSymbolAddress and checks its return code (CK)."""
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    src = open(os.path.join(root, "paper_2401_03041_b200", "csrc", "tcp_api.cu")).read()
    body = src[src.index("int tcp_read_pressure_static("):src.index("int tcp_pattern_copy_ms(")]
    assert not re.search(r"cudaMalloc|cudaFree|cudaHostAlloc|cudaMallocAsync|\bnew\b|malloc\(", body)
    assert "CK(cudaGetSymbolAddress(&addr, g_static_scratch))" in body
    assert re.search(r"static __device__ __align__\(256\) unsigned char g_static_scratch\[TCP_STATIC_SCRATCH_BYTES\]", src)
