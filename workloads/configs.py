"""The five BASELINE.json workloads as plain data (no arithmetic of the method).

Index i here is BASELINE.json `configs[i]`.  Readings of BASELINE's wording
 are repeated in DESIGN.md.
"""
from dataclasses import dataclass, field
from typing import Optional, Tuple


@dataclass(frozen=True)
class WorkloadConfig:
    index: int
    name: str
    seed: int
    # opacity table
    n_species: int
    n_cia: int
    T_grid: Tuple[float, ...]          # K, strictly increasing
    log10p_grid: Tuple[float, ...]     # log10(bar), strictly increasing
    nu0: float                         # cm^-1, first grid point
    dnu: float                         # cm^-1
    n_nu: int
    n_lines: int                       # Lorentzian lines per species
    # atmosphere
    n_levels: int
    p_bottom_bar: float
    p_top_bar: float
    n_knots: int
    n_angles: int
    mean_mol_weight: float
    he_to_h2: float
    flux_const: float
    # observation
    n_bins: int
    fwhm_cm1: Optional[float]          # None -> one bin width
    # batch
    batch: int
    n_calls: int = 1                   # config 4: 16 back-to-back calls
    spectra_out: bool = True
    fixed_params: Optional[Tuple[float, ...]] = None   # config 0
    tables_from: Optional[int] = None  # config 4 reuses config 3's tables


def _lin(a, b, n):
    return tuple(a + (b - a) * i / (n - 1) for i in range(n))


_COMMON = dict(p_bottom_bar=300.0, p_top_bar=1e-3, mean_mol_weight=2.3,
               he_to_h2=0.17, flux_const=1.0)

CONFIGS = (
    WorkloadConfig(
        index=0, name="tiny", seed=0,
        n_species=1, n_cia=0,
        T_grid=(500.0, 1000.0, 1500.0, 2000.0),
        log10p_grid=(-3.0, -1.0, 1.0, 2.5),
        nu0=4000.0, dnu=1.0, n_nu=1000, n_lines=20,
        n_levels=20, n_knots=2, n_angles=2,
        n_bins=50, fwhm_cm1=20.0, batch=1,
        # log10 g, f, T_knot (bottom, top), log10 VMR
        fixed_params=(5.0, 1.0, 2000.0, 800.0, -3.0),
        **_COMMON),
    WorkloadConfig(
        index=1, name="bd_nearir_medium", seed=1,
        n_species=4, n_cia=2,
        T_grid=_lin(100.0, 3000.0, 27), log10p_grid=_lin(-4.0, 2.5, 17),
        nu0=4000.0, dnu=1.0, n_nu=8501, n_lines=5000,
        n_levels=100, n_knots=6, n_angles=4,
        n_bins=120, fwhm_cm1=None, batch=64, **_COMMON),
    WorkloadConfig(
        index=2, name="jwst_broadband", seed=2,
        n_species=8, n_cia=2,
        T_grid=_lin(100.0, 3000.0, 27), log10p_grid=_lin(-4.0, 2.5, 17),
        nu0=357.0, dnu=1.0, n_nu=16311, n_lines=10000,
        n_levels=100, n_knots=6, n_angles=4,
        n_bins=1000, fwhm_cm1=None, batch=256, **_COMMON),
    WorkloadConfig(
        index=3, name="highres_opacity_sampling", seed=3,
        n_species=6, n_cia=2,
        T_grid=_lin(100.0, 3500.0, 40), log10p_grid=_lin(-5.0, 3.0, 20),
        nu0=4000.0, dnu=0.1, n_nu=85001, n_lines=20000,
        n_levels=150, n_knots=6, n_angles=8,
        n_bins=300, fwhm_cm1=None, batch=1024, **_COMMON),
    WorkloadConfig(
        index=4, name="loglike_stream", seed=4,
        n_species=6, n_cia=2,
        T_grid=_lin(100.0, 3500.0, 40), log10p_grid=_lin(-5.0, 3.0, 20),
        nu0=4000.0, dnu=0.1, n_nu=85001, n_lines=20000,
        n_levels=150, n_knots=6, n_angles=8,
        n_bins=300, fwhm_cm1=None, batch=4096, n_calls=16,
        spectra_out=False, tables_from=3, **_COMMON),
)


def get_config(index: int) -> WorkloadConfig:
    return CONFIGS[index]
