"""Seeded synthetic inputs shaped like the paper's workloads (BASELINE.json configs 1-5).

This module serves BOTH the CPU oracle and the CUDA path and holds none of the method's
arithmetic: it only produces parameter dicts and initial fields (phi0, u0, T0, wall-temperature
planes).  It imports neither `oracle` nor `paper_2401_03041_b200`.  The paper's set-ups are
themselves synthetic (tanh interfaces, droplets, prescribed wall temperatures: PAPER.md:198-230,
317-321), so no external data set stands behind them; the recipe of every config is restated in
DESIGN.md.

All arrays are torch float64 tensors laid out [nz][ny][nx] (x fastest); u0 is [3][nz][ny][nx].
"""
from .configs import (Workload, static_droplet, layered_channel, droplet_in_gradient,
                      thermal_tweezer, perf_box, laser_source, laser_channel, BENCH_FLUID)
from .analytic import layered_channel_closed_form

__all__ = ["Workload", "static_droplet", "layered_channel", "droplet_in_gradient",
           "thermal_tweezer", "perf_box", "laser_source", "laser_channel", "BENCH_FLUID", "layered_channel_closed_form"]
