"""GPU parity of the NEXT rows against the fp64 oracle,
through the C ABI: error-inflated likelihood + distance (NEXT-1), finite-element T-p profile in
nodal and ratio form (NEXT-2), effective temperature (NEXT-3), grey cloud (NEXT-4).
Tolerances as for the hot path: 1e-4 relative on fluxes, logL 1e-4 relative / 1e-3 absolute near
the truth; T_eff 1e-5 relative (a fourth root of an fp32 flux integral).
"""
import numpy as np
import pytest

import workloads as W

pytestmark = pytest.mark.gpu

TOL_FLUX = 1e-4
TOL_FLUX_PROPAGATED = 2e-6     # tests/test_gpu_parity.py: the flux error the all-model logL bound is propagated from


def _logl_bound(wl, M, addvar=0.0):
    """What a binned-flux error of TOL_FLUX_PROPAGATED * M_j can move logL by (Eq. 19; Eq. 22-23 with the inflated
    variance s_j^2 = sigma_j^2 + addvar, whose ln-term does not depend on M), plus north_star's 1e-3 absolute."""
    e = TOL_FLUX_PROPAGATED * np.abs(M)
    s2 = wl.obs_err[None, :] ** 2 + np.reshape(addvar, (-1, 1))
    return ((np.abs(wl.obs[None, :] - M) * e + 0.5 * e * e) / s2).sum(axis=1) + 1e-3


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


@pytest.fixture(scope="module")
def wl1(torch_cuda):
    return W.make_workload(1)


def _relerr(a, ref):
    return float(np.max(np.abs(a / ref - 1.0)))


def _helios(wl):
    from paper_1910_01070_b200 import Helios
    h = Helios(0)
    h.setup_workload(wl)
    return h


@pytest.mark.parametrize("kernel", [1, 2, 3], ids=["direct", "slab", "levelpar"])
def test_distance_inflation_and_cloud(torch_cuda, oracle, wl1, kernel):
    """All three extras at once, in the documented order d, epsilon, (log tau_c, log p_top, log phi)."""
    import paper_1910_01070_b200 as pkg
    torch = torch_cuda
    cfg = wl1.cfg
    rng = np.random.default_rng(11)
    B = 24
    base = wl1.params[:B]
    med_var = float(np.median(wl1.obs_err ** 2))
    extra = np.column_stack([rng.uniform(0.8, 1.5, B),                               # d
                             np.log10(med_var) + rng.uniform(-2.0, 2.0, B),          # epsilon around the data errors
                             rng.uniform(-2.0, 1.0, B),                              # log10 tau_c
                             rng.uniform(-2.5, 1.5, B),                              # log10 p_top [bar]
                             rng.uniform(-1.0, 1.0, B)])                             # log10 phi
    params = np.ascontiguousarray(np.column_stack([base, extra]))
    flags = pkg.HELIOS_EXTRA_DISTANCE | pkg.HELIOS_EXTRA_ERROR_INFLATION | pkg.HELIOS_EXTRA_GREY_CLOUD
    ref = oracle.forward_workload(wl1, params=params, want_flux=True, extras=flags)

    h = _helios(wl1)
    h.set_kernel(kernel)
    h.set_extras(flags)
    assert h.n_params == params.shape[1]
    p = torch.as_tensor(params, device="cuda:0")
    spec, logl = h.forward_batch(p)
    flux = h.forward_highres(p)
    torch.cuda.synchronize()
    h.close()
    assert _relerr(flux.cpu().numpy().astype(np.float64), ref["flux_hr"]) <= TOL_FLUX
    assert _relerr(spec.cpu().numpy().astype(np.float64), ref["spectra"]) <= TOL_FLUX
    dl = np.abs(logl.cpu().numpy() - ref["logl"])
    assert np.all(dl <= _logl_bound(wl1, ref["spectra"], 10.0 ** params[:, base.shape[1] + 1]))
    # the cloud really changed something, so the comparison is not vacuous
    ref0 = oracle.forward_workload(wl1, params=np.ascontiguousarray(params[:, :-3]), want_flux=False,
                                   extras=pkg.HELIOS_EXTRA_DISTANCE | pkg.HELIOS_EXTRA_ERROR_INFLATION)
    assert np.max(np.abs(ref0["spectra"] / ref["spectra"] - 1.0)) > 1e-2


def test_inflated_logl_near_truth_absolute(torch_cuda, oracle, wl1):
    import paper_1910_01070_b200 as pkg
    torch = torch_cuda
    near = W.near_truth_params(wl1.cfg, 8)
    eps = np.log10(np.median(wl1.obs_err ** 2)) + np.linspace(-1.0, 1.0, 8)
    params = np.ascontiguousarray(np.column_stack([near, eps]))
    ref = oracle.forward_workload(wl1, params=params, extras=pkg.HELIOS_EXTRA_ERROR_INFLATION)
    h = _helios(wl1)
    h.set_extras(pkg.HELIOS_EXTRA_ERROR_INFLATION)
    _, logl = h.forward_batch(torch.as_tensor(params, device="cuda:0"))
    torch.cuda.synchronize()
    h.close()
    assert np.max(np.abs(logl.cpu().numpy() - ref["logl"])) <= 1e-3


@pytest.mark.parametrize("order,ratio", [(1, False), (2, False), (2, True), (3, True), (4, False)])
def test_finite_element_profile(torch_cuda, oracle, wl1, order, ratio):
    torch = torch_cuda
    cfg = wl1.cfg
    Ke = 3
    NT = Ke * order + 1
    rng = np.random.default_rng(100 + order)
    B = 16
    if ratio:                                   # T_1 and ratios b_i <= 1 (monotone)
        tpar = np.column_stack([rng.uniform(2200, 2800, B), rng.uniform(0.80, 0.98, (B, NT - 1))])
    else:
        tpar = -np.sort(-rng.uniform(600, 2700, (B, NT)), axis=1)
    S = cfg.n_species
    params = np.ascontiguousarray(np.column_stack([wl1.params[:B, :2], tpar, wl1.params[:B, -S:]]))
    ref = oracle.forward_workload(wl1, params=params, want_flux=True, tp_elements=Ke, tp_order=order, tp_ratio=ratio)
    h = _helios(wl1)
    h.set_tp_elements(Ke, order, ratio)
    assert h.n_params == params.shape[1]
    p = torch.as_tensor(params, device="cuda:0")
    spec, logl = h.forward_batch(p)
    flux = h.forward_highres(p)
    torch.cuda.synchronize()
    st = h.stats()
    h.close()
    assert _relerr(flux.cpu().numpy().astype(np.float64), ref["flux_hr"]) <= TOL_FLUX
    assert _relerr(spec.cpu().numpy().astype(np.float64), ref["spectra"]) <= TOL_FLUX
    assert np.all(np.abs(logl.cpu().numpy() - ref["logl"]) <= _logl_bound(wl1, ref["spectra"]))
    assert st["n_clamped"] == 2 * ref["n_clamped"]


def test_effective_temperature(torch_cuda, oracle, wl1):
    torch = torch_cuda
    cfg = wl1.cfg
    nu_a, nu_b = cfg.nu0 + 100.3, cfg.nu0 + cfg.dnu * (cfg.n_nu - 1) - 57.8      # cuts through grid cells
    B = 32
    params = wl1.params[:B]
    ref = oracle.forward_workload(wl1, params=params, want_spectra=False, want_logl=False, teff_range=(nu_a, nu_b))
    h = _helios(wl1)
    teff = h.teff_batch(torch.as_tensor(params, device="cuda:0"), nu_a, nu_b)
    torch.cuda.synchronize()
    # T_eff does not depend on f, (R/d)^2: change f and get the same numbers
    p2 = params.copy(); p2[:, 1] *= 3.0
    teff2 = h.teff_batch(torch.as_tensor(p2, device="cuda:0"), nu_a, nu_b)
    torch.cuda.synchronize()
    h.close()
    assert _relerr(teff.cpu().numpy(), ref["teff"]) <= 1e-5
    assert torch.equal(teff, teff2)
    assert np.all((ref["teff"] > 200) & (ref["teff"] < 3000))
