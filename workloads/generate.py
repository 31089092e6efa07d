"""Seeded generators: opacity tables, parameter vectors, observation grids.

Recipe (BASELINE.json `configs`):

* RNG: numpy Generator(PCG64) seeded from SeedSequence(seed).spawn(4), streams
  in this order: lines, params, truth, noise.
* Cross-sections, per species: `n_lines` Lorentzian lines, centres uniform on
  [nu_first, nu_last], strengths log-uniform 1e-24..1e-20 cm^2 cm^-1,
  HWHM gamma(T,p) = 0.05 (p/1 bar) (T/1000 K)^-0.5 cm^-1,
  sigma = 1e-30 + sum_k (S_k/pi) gamma / ((nu-nu_k)^2 + gamma^2),
  each line evaluated on the 2K+1 grid points around the grid point nearest
  its centre, K = round(25 cm^-1 / dnu) (documented wing cut-off), stored fp32,
  layout [S][N_T][N_P][N_nu].
* CIA, pair c: A_c (1 + 0.5 sin(2 pi nu / 2000 cm^-1)) (T/1000 K)^0.5 with
  A = 1e-46 cm^5 (H2-H2), 0.5e-46 cm^5 (H2-He), stored in cm^-1 amagat^-2
  (multiplied by n_L^2), fp32, layout [C][N_T][N_nu].
* Params (configs 1-4): log10 g ~ U(4, 5.5), f ~ U(0.5, 2), K knot temperatures
  ~ U(500, 2800) K sorted hottest (bottom) first, log10 VMR ~ U(-8, -2).

None of this is the method's arithmetic; the Lorentzian sum is data synthesis.
"""
from __future__ import annotations

import hashlib
import math
import os
from dataclasses import dataclass
from typing import Optional

import numpy as np

from .configs import CONFIGS, WorkloadConfig

_LOSCHMIDT = 2.686780111798444e19            # cm^-3, only to convert the CIA magnitude to amagat units
_WING_CUT_CM1 = 25.0
_SIGMA_FLOOR = 1e-30
_FWHM_TO_SIGMA = 1.0 / (2.0 * math.sqrt(2.0 * math.log(2.0)))


def golden_dir() -> str:
    return os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))),
                        "tests", "golden")


@dataclass
class Workload:
    cfg: WorkloadConfig
    T_grid: np.ndarray          # [N_T] float64
    log10p_grid: np.ndarray     # [N_P] float64
    sigma: np.ndarray           # [S][N_T][N_P][N_nu] float32
    cia: np.ndarray             # [C][N_T][N_nu] float32 (C may be 0)
    params: np.ndarray          # [B][P] float64
    bin_edges: np.ndarray       # [J+1] float64
    inst_sigma: np.ndarray      # [N_nu] float64
    obs: Optional[np.ndarray]   # [J] float64 (None if the golden file is absent)
    obs_err: Optional[np.ndarray]

    @property
    def n_params(self) -> int:
        return 2 + self.cfg.n_knots + self.cfg.n_species


def _streams(seed: int):
    ss = np.random.SeedSequence(seed).spawn(4)
    return [np.random.Generator(np.random.PCG64(s)) for s in ss]


def _nu_last(cfg: WorkloadConfig) -> float:
    return cfg.nu0 + cfg.dnu * (cfg.n_nu - 1)


# ----------------------------------------------------------------------------
# opacity tables
# ----------------------------------------------------------------------------
def _line_lists(cfg: WorkloadConfig):
    table_cfg = CONFIGS[cfg.tables_from] if cfg.tables_from is not None else cfg
    rng = _streams(table_cfg.seed)[0]
    lists = []
    for _ in range(cfg.n_species):
        centres = rng.uniform(cfg.nu0, _nu_last(cfg), cfg.n_lines)
        strengths = 10.0 ** rng.uniform(-24.0, -20.0, cfg.n_lines)
        lists.append((centres, strengths))
    return lists


def _species_table_numpy(cfg, centres, strengths, out):
    """out: float32 [N_T][N_P][N_nu] filled in place."""
    K = int(round(_WING_CUT_CM1 / cfg.dnu))
    i0 = np.rint((centres - cfg.nu0) / cfg.dnu).astype(np.int64)
    idx = i0[:, None] + np.arange(-K, K + 1, dtype=np.int64)[None, :]
    valid = (idx >= 0) & (idx < cfg.n_nu)
    d2 = (cfg.nu0 + idx * cfg.dnu - centres[:, None]) ** 2
    s_over_pi = np.broadcast_to((strengths / math.pi)[:, None], idx.shape)[valid]
    idx_v = idx[valid]
    d2_v = d2[valid]
    for iT, T in enumerate(cfg.T_grid):
        for ip, lp in enumerate(cfg.log10p_grid):
            gamma = 0.05 * (10.0 ** lp) * (T / 1000.0) ** -0.5
            val = s_over_pi * gamma / (d2_v + gamma * gamma)
            acc = np.bincount(idx_v, weights=val, minlength=cfg.n_nu)
            out[iT, ip, :] = (acc + _SIGMA_FLOOR).astype(np.float32)


def _species_table_torch(cfg, centres, strengths, out, device):
    import torch
    K = int(round(_WING_CUT_CM1 / cfg.dnu))
    c = torch.as_tensor(centres, dtype=torch.float64, device=device)
    s = torch.as_tensor(strengths, dtype=torch.float64, device=device)
    i0 = torch.round((c - cfg.nu0) / cfg.dnu).long()
    idx = i0[:, None] + torch.arange(-K, K + 1, device=device)[None, :]
    valid = (idx >= 0) & (idx < cfg.n_nu)
    d2 = (cfg.nu0 + idx.double() * cfg.dnu - c[:, None]) ** 2
    s_over_pi = (s / math.pi)[:, None].expand_as(d2)[valid]
    idx_v = idx[valid]
    d2_v = d2[valid]
    m = idx_v.numel()
    n_p = len(cfg.log10p_grid)
    chunk = max(1, min(n_p, (1 << 27) // max(m, 1)))
    p_bar = torch.as_tensor([10.0 ** lp for lp in cfg.log10p_grid], dtype=torch.float64, device=device)
    for iT, T in enumerate(cfg.T_grid):
        gam_all = 0.05 * p_bar * (T / 1000.0) ** -0.5
        for a in range(0, n_p, chunk):
            gam = gam_all[a:a + chunk]
            val = s_over_pi[None, :] * gam[:, None] / (d2_v[None, :] + (gam * gam)[:, None])
            flat = (torch.arange(gam.numel(), device=device)[:, None] * cfg.n_nu + idx_v[None, :])
            acc = torch.zeros(gam.numel() * cfg.n_nu, dtype=torch.float64, device=device)
            acc.index_add_(0, flat.reshape(-1), val.reshape(-1))
            out[iT, a:a + chunk, :] = (acc.view(gam.numel(), cfg.n_nu) + _SIGMA_FLOOR).float()


def _cia_tables(cfg: WorkloadConfig) -> np.ndarray:
    nu = cfg.nu0 + cfg.dnu * np.arange(cfg.n_nu, dtype=np.float64)
    T = np.asarray(cfg.T_grid, dtype=np.float64)
    amp_cm5 = [1e-46, 0.5e-46]
    out = np.zeros((cfg.n_cia, len(T), cfg.n_nu), dtype=np.float32)
    for c in range(cfg.n_cia):
        shape = 1.0 + 0.5 * np.sin(2.0 * math.pi * nu / 2000.0)
        a = amp_cm5[c] * _LOSCHMIDT ** 2
        out[c] = (a * shape[None, :] * np.sqrt(T / 1000.0)[:, None]).astype(np.float32)
    return out


def _cache_path(cfg: WorkloadConfig) -> Optional[str]:
    root = os.environ.get("HELIOS_WORKLOAD_CACHE", "/tmp/helios_workload_cache")
    if root in ("", "0", "off"):
        return None
    table_cfg = CONFIGS[cfg.tables_from] if cfg.tables_from is not None else cfg
    key = repr((table_cfg.seed, cfg.n_species, cfg.T_grid, cfg.log10p_grid, cfg.nu0, cfg.dnu,
                cfg.n_nu, cfg.n_lines, _WING_CUT_CM1, _SIGMA_FLOOR, "v1"))
    h = hashlib.sha256(key.encode()).hexdigest()[:16]
    return os.path.join(root, f"sigma_{h}.npy")


def make_tables(cfg: WorkloadConfig, device: str = "cpu", cache: bool = True):
    """Returns (sigma float32 [S][N_T][N_P][N_nu], cia float32 [C][N_T][N_nu]) as numpy.

    device="cuda" synthesises the line sums with torch on the GPU (input
    preparation only; it is never inside a timed region) and copies back.
    The two devices agree to fp64 summation order, i.e. to the last fp32 bit
    almost everywhere; parity tests feed ONE array to both sides.
    """
    path = _cache_path(cfg) if cache else None
    sigma = None
    if path is not None and os.path.exists(path):
        try:
            sigma = np.load(path)
            if sigma.shape != (cfg.n_species, len(cfg.T_grid), len(cfg.log10p_grid), cfg.n_nu):
                sigma = None
        except Exception:
            sigma = None
    if sigma is None:
        lists = _line_lists(cfg)
        if device == "cpu":
            sigma = np.empty((cfg.n_species, len(cfg.T_grid), len(cfg.log10p_grid), cfg.n_nu), np.float32)
            for s, (centres, strengths) in enumerate(lists):
                _species_table_numpy(cfg, centres, strengths, sigma[s])
        else:
            import torch
            out = torch.empty((cfg.n_species, len(cfg.T_grid), len(cfg.log10p_grid), cfg.n_nu),
                              dtype=torch.float32, device=device)
            for s, (centres, strengths) in enumerate(lists):
                _species_table_torch(cfg, centres, strengths, out[s], device)
            sigma = out.cpu().numpy()
        if path is not None:
            try:
                os.makedirs(os.path.dirname(path), exist_ok=True)
                tmp = path + f".tmp{os.getpid()}"
                with open(tmp, "wb") as fh:
                    np.save(fh, sigma)
                os.replace(tmp, path)
            except OSError:
                pass
    return sigma, _cia_tables(cfg)


# ----------------------------------------------------------------------------
# parameter vectors
# ----------------------------------------------------------------------------
def _draw(rng, cfg: WorkloadConfig, n: int) -> np.ndarray:
    P = 2 + cfg.n_knots + cfg.n_species
    out = np.empty((n, P), dtype=np.float64)
    out[:, 0] = rng.uniform(4.0, 5.5, n)
    out[:, 1] = rng.uniform(0.5, 2.0, n)
    knots = rng.uniform(500.0, 2800.0, (n, cfg.n_knots))
    out[:, 2:2 + cfg.n_knots] = -np.sort(-knots, axis=1)          # hottest (bottom) first
    out[:, 2 + cfg.n_knots:] = rng.uniform(-8.0, -2.0, (n, cfg.n_species))
    return out


def draw_params(cfg: WorkloadConfig, n: Optional[int] = None) -> np.ndarray:
    """[n][P] float64: log10 g, f, T_knot[0..K-1] (bottom -> top), log10 VMR[0..S-1]."""
    n = cfg.batch if n is None else n
    if cfg.fixed_params is not None:
        return np.tile(np.asarray(cfg.fixed_params, dtype=np.float64), (n, 1))
    return _draw(_streams(cfg.seed)[1], cfg, n)


def true_params(cfg: WorkloadConfig) -> np.ndarray:
    """The parameter vector the synthetic observation is made from."""
    src = CONFIGS[cfg.tables_from] if cfg.tables_from is not None else cfg
    if src.fixed_params is not None:
        return np.asarray(src.fixed_params, dtype=np.float64)
    return _draw(_streams(src.seed)[2], src, 1)[0]


def near_truth_params(cfg: WorkloadConfig, n: int, draw: int = 0) -> np.ndarray:
    """n vectors close to true_params (reduced chi^2 of order 1): the subset on
    which an absolute logL tolerance is meaningful (SURVEY.md 8(c) hazards).
    draw > 0: another, independent set of the same recipe (draw 0 is the set of rounds 1-2)."""
    rng = np.random.Generator(np.random.PCG64(np.random.SeedSequence([cfg.seed, 777] + ([draw] if draw else []))))
    t = true_params(cfg)
    out = np.tile(t, (n, 1))
    K = cfg.n_knots
    out[:, 0] += rng.normal(0.0, 0.003, n)
    out[:, 1] *= 1.0 + rng.normal(0.0, 0.002, n)
    out[:, 2:2 + K] += rng.normal(0.0, 0.5, (n, K))
    out[:, 2:2 + K] = -np.sort(-out[:, 2:2 + K], axis=1)
    out[:, 2 + K:] += rng.normal(0.0, 0.003, (n, cfg.n_species))
    out[0] = t
    return out


# ----------------------------------------------------------------------------
# observation
# ----------------------------------------------------------------------------
def observation_grid(cfg: WorkloadConfig):
    """(bin_edges [J+1], inst_sigma [N_nu]): J bins uniform in wavenumber over the
    grid, constant Gaussian instrument profile, FWHM = cfg.fwhm_cm1 or one bin."""
    edges = np.linspace(cfg.nu0, _nu_last(cfg), cfg.n_bins + 1)
    fwhm = cfg.fwhm_cm1 if cfg.fwhm_cm1 is not None else (edges[-1] - edges[0]) / cfg.n_bins
    inst_sigma = np.full(cfg.n_nu, fwhm * _FWHM_TO_SIGMA, dtype=np.float64)
    return edges, inst_sigma


def noise_draw(cfg: WorkloadConfig) -> np.ndarray:
    """eps_j ~ N(0,1), one per bin, for D_j = M_j (1 + 0.02 eps_j)."""
    src = CONFIGS[cfg.tables_from] if cfg.tables_from is not None else cfg
    return _streams(src.seed)[3].standard_normal(src.n_bins)


def load_observation(cfg: WorkloadConfig):
    """(D [J], err [J]) from tests/golden/obs_cfg<i>.txt, written by
    tests/golden/make_golden.py from the ORACLE at true_params; None if absent."""
    src = CONFIGS[cfg.tables_from] if cfg.tables_from is not None else cfg
    path = os.path.join(golden_dir(), f"obs_cfg{src.index}.txt")
    if not os.path.exists(path):
        return None, None
    arr = np.loadtxt(path, comments="#", dtype=np.float64, ndmin=2)
    return arr[:, 0].copy(), arr[:, 1].copy()


def make_workload(index: int, batch: Optional[int] = None, device: str = "cpu",
                  cache: bool = True) -> Workload:
    cfg = CONFIGS[index]
    sigma, cia = make_tables(cfg, device=device, cache=cache)
    edges, inst_sigma = observation_grid(cfg)
    obs, err = load_observation(cfg)
    return Workload(cfg=cfg,
                    T_grid=np.asarray(cfg.T_grid, dtype=np.float64),
                    log10p_grid=np.asarray(cfg.log10p_grid, dtype=np.float64),
                    sigma=sigma, cia=cia,
                    params=draw_params(cfg, batch),
                    bin_edges=edges, inst_sigma=inst_sigma, obs=obs, obs_err=err)
