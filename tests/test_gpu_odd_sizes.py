"""Odd, prime and degenerate box sizes: the cell -> (x, y, z) decomposition by multiply-high (fast_div), rows that
straddle warps and blocks, planes whose byte offsets are not 16-byte multiples (fp32, odd N), a box with a single
cell along an axis, and a box large enough (> 300 blocks) that the L2 prefetch of the staged kernels is active.
fp64 against the oracle at the north-star tolerance; fp32 (odd nx -> one cell per thread, even nx -> packed pairs)
at 1e-5 relative."""
import numpy as np
import pytest
import torch

import workloads as W
from parity_util import assert_parity_f32, assert_parity_f64, run_gpu, run_oracle

pytestmark = pytest.mark.gpu


def smooth_box(nx, ny, nz, thermal, seed):
    """Periodic box with a smooth two-phase field and temperature (any size >= 1 per axis)."""
    rng = np.random.default_rng(seed)
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    ph = rng.uniform(0, 2 * np.pi, 6)
    s = (np.cos(2 * np.pi * x / nx + ph[0]) + np.cos(2 * np.pi * y / ny + ph[1]) + np.cos(2 * np.pi * z / nz + ph[2])) / 3.0
    phi = 0.5 * (1.0 + np.tanh(2.5 * s))
    T = 0.5 + 0.3 * np.sin(2 * np.pi * x / nx + ph[3]) * np.cos(2 * np.pi * y / ny + ph[4]) + 0.1 * np.cos(2 * np.pi * z / nz + ph[5])
    u = 1e-3 * rng.standard_normal((3, nz, ny, nx))
    params = dict(W.BENCH_FLUID, thermal=thermal, bc=("periodic", "periodic", "periodic"))
    return W.Workload(f"smooth_{nx}x{ny}x{nz}", nx, ny, nz, params, torch.from_numpy(phi), torch.from_numpy(u), torch.from_numpy(T))


SIZES = [(17, 13, 11), (33, 5, 3), (1, 9, 7), (7, 1, 9), (5, 6, 1), (129, 3, 2), (3, 3, 3)]


@pytest.mark.parametrize("shape", SIZES)
@pytest.mark.parametrize("thermal", ["lb_d3q7", "rk4"])
def test_odd_sizes_f64(shape, thermal):
    wl = smooth_box(*shape, thermal, seed=sum(shape))
    want = run_oracle(wl, 12)
    got, _ = run_gpu(wl, 12, chunks=[1, 11])
    assert_parity_f64(got, want)


@pytest.mark.parametrize("streaming", ["two_grid", "aa"])
def test_odd_sizes_streaming_d3q27(streaming):
    wl = smooth_box(19, 7, 5, "lb_d3q27", seed=5)
    want = run_oracle(wl, 9)
    got, _ = run_gpu(wl, 9, extra=dict(streaming=streaming))
    assert_parity_f64(got, want)


@pytest.mark.parametrize("shape,thermal", [((37, 35, 31), "lb_d3q7"), ((41, 33, 29), "rk2"), ((38, 35, 31), "lb_d3q19")])
def test_prefetch_active_odd_box(shape, thermal):
    """> 300 blocks of 128 cells: blocks do issue their L2 prefetch, rows are not multiples of anything."""
    wl = smooth_box(*shape, thermal, seed=shape[0])
    assert wl.cells > 300 * 128
    want = run_oracle(wl, 6)
    got, _ = run_gpu(wl, 6)
    assert_parity_f64(got, want)
    got32, _ = run_gpu(wl, 6, precision="f32")          # odd nx: scalar kernel; even nx: packed pairs
    assert_parity_f32(got32, want, sigma=wl.params.get("sigma_ref", 0.0))
