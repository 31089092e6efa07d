"""Seeded synthetic inputs for the Helios-r2 batched forward model.

This module is shared by the oracle tests and by the CUDA path's tests / bench.
It holds NONE of the method's arithmetic (no interpolation, optical depth,
Planck function, radiative transfer, convolution, binning or likelihood): it
only draws random tables, parameter vectors and noise, and describes the five
BASELINE.json workloads.  See DESIGN.md "Input recipe".

The opacity tables, line lists, SpeX/ISAAC spectra of the paper
 are not available; these inputs take their shapes.
"""
from .configs import CONFIGS, WorkloadConfig, get_config
from .generate import (
    Workload,
    make_workload,
    make_tables,
    draw_params,
    true_params,
    near_truth_params,
    observation_grid,
    load_observation,
    golden_dir,
)

__all__ = [
    "CONFIGS", "WorkloadConfig", "get_config", "Workload", "make_workload",
    "make_tables", "draw_params", "true_params", "near_truth_params",
    "observation_grid", "load_observation", "golden_dir",
]
