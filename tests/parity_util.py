"""Helpers shared by the GPU parity tests: run the same seeded workload through the CPU oracle
(oracle/, test infrastructure) and through the CUDA path (C ABI via the Python binding)."""
import numpy as np
import torch

import paper_2401_03041_b200 as tcp
from oracle import tcpo


def _np(t):
    return None if t is None else (t.detach().cpu().numpy() if isinstance(t, torch.Tensor) else np.asarray(t))


def run_oracle(wl, steps, q=None, extra=None):
    params = dict(wl.params)
    if extra:
        params.update(extra)
    o = tcpo.Oracle(wl.nx, wl.ny, wl.nz, params)
    for (ax, fc), plane in wl.wall_T.items():
        o.set_wall_temperature(ax, fc, _np(plane))
    if q is not None:
        o.set_heat_source(_np(q))
    o.init_fields(_np(wl.phi), _np(wl.u), _np(wl.T))
    o.step(steps)
    out = o.read_fields()
    o.close()
    return out


def run_gpu(wl, steps, q=None, extra=None, precision="f64", chunks=None, device_inputs=False):
    """chunks: split `steps` over several tcp_step calls (e.g. [1, 0, steps-1]) to exercise the
    buffer parity bookkeeping."""
    params = dict(wl.params)
    if extra:
        params.update(extra)
    params["precision"] = precision
    sim = tcp.Simulation(wl.nx, wl.ny, wl.nz, params)
    conv = (lambda t: None if t is None else torch.as_tensor(_np(t)).cuda()) if device_inputs else _np
    for (ax, fc), plane in wl.wall_T.items():
        sim.set_wall_temperature(ax, fc, conv(plane))
    if q is not None:
        sim.set_heat_source(conv(q))
    sim.init_fields(conv(wl.phi), conv(wl.u), conv(wl.T))
    for n in (chunks or [steps]):
        sim.step(n)
    out = sim.read_fields()
    launches = sim.launches
    sim.close()
    return out, launches


NAMES = ("phi", "u", "p", "T")


def assert_parity_f64(got, want, tol=1e-10):
    """north_star: max-abs error <= 1e-10 on phi, u, p and T (fp64, 100 steps)."""
    for name, g, w in zip(NAMES, got, want):
        assert g.shape == w.shape
        assert np.all(np.isfinite(g)), f"{name} has non-finite values"
        err = np.abs(g - w).max()
        assert err <= tol, f"{name}: max-abs error {err:.3e} > {tol:.1e}"


def assert_parity_f32(got, want, rel=1e-5):
    """north_star: fp32 variant <= 1e-5 relative (to the field's own scale: max |oracle|; for u and p,
    whose scale can be ~1e-6 in a quiescent set-up, the scale is floored so that round-off of the
    O(1) populations they are differences of still counts as relative error of those populations)."""
    floors = dict(phi=1.0, u=1.0, p=1.0 / 3.0, T=1.0)
    for name, g, w in zip(NAMES, got, want):
        assert np.all(np.isfinite(g)), f"{name} has non-finite values"
        scale = max(np.abs(w).max(), floors[name])
        err = np.abs(g.astype(np.float64) - w).max() / scale
        assert err <= rel, f"{name}: relative error {err:.3e} > {rel:.1e}"
