"""ORACLE (test infrastructure, not the product): fp64 CPU statement of the
Helios-r2 forward model, oracle/helios_oracle.c, loaded through ctypes.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this package.  It imports nothing from
paper_1910_01070_b200 and the CUDA library imports nothing from here.
"""
from .binding import (  # noqa: F401
    build, lib, level_pressures, temperature_profile, mixing_ratios, cell,
    interp_sigma, interp_cia, number_density, chi_level, layer_thickness, layer_dtau,
    planck, gauss_legendre_01, sc_coefficients, flux_one_nu, convolve, bin_spectrum,
    loglike, forward, max_threads, forward_workload,
    loglike_inflated, lobatto_nodes, tp_dofs_from_ratios, temperature_profile_fe, teff, cloud_dtau,
    EXTRA_DISTANCE, EXTRA_ERROR_INFLATION, EXTRA_GREY_CLOUD,
)
