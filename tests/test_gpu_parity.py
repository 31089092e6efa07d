"""GPU parity: the CUDA path (through the C ABI) against the fp64 oracle, element
by element on the same seeded inputs.  Tolerances are BASELINE.json's north_star:
max relative error 1e-4 on the binned flux, 1e-3 absolute on logL (near truth;
DESIGN.md "logL tolerance"), plus 1e-4 relative on the high-resolution flux.
"""
import numpy as np
import pytest

import workloads as W

pytestmark = pytest.mark.gpu

TOL_FLUX = 1e-4
TOL_LOGL_ABS = 1e-3
# all-model logL bound: what a binned-flux error of TOL_FLUX_PROPAGATED * M_j can do to logL.  The measured flux error
# is 2e-7..5e-7 (fp32 arithmetic; profiles/r03_parity_summary.json) and its terms partly cancel: the measured |dlogL| is
# <= 0.055 of this bound on every model of every config, a factor ~18.  Rounds 1-2 propagated the full 1e-4 (a factor
# ~1000, which would not have noticed a 50x regression of the arithmetic).
TOL_FLUX_PROPAGATED = 2e-6


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


def _gen_device(torch):
    return "cuda" if torch.cuda.is_available() else "cpu"


@pytest.fixture(scope="module")
def wl0(torch_cuda):
    return W.make_workload(0)


@pytest.fixture(scope="module")
def wl1(torch_cuda):
    return W.make_workload(1)


@pytest.fixture(scope="module")
def wl2(torch_cuda):
    return W.make_workload(2, device=_gen_device(torch_cuda))


@pytest.fixture(scope="module")
def wl3(torch_cuda):
    return W.make_workload(3, device=_gen_device(torch_cuda))


def _run(torch, wl, params, kernel=0, highres=True, models_per_cta=0, nu_order=None, fused=False):
    from paper_1910_01070_b200 import Helios
    h = Helios(0)
    if nu_order is not None:
        h.set_nu_order(nu_order)
    h.set_fused_obs(fused)
    h.setup_workload(wl)
    h.set_kernel(kernel, models_per_cta)
    p = torch.as_tensor(np.ascontiguousarray(params), device="cuda:0")
    spec, logl = h.forward_batch(p, want_logl=wl.obs is not None)
    flux = h.forward_highres(p) if highres else None
    torch.cuda.synchronize()
    st = h.stats()
    h.close()
    return (spec.cpu().numpy().astype(np.float64),
            None if logl is None else logl.cpu().numpy(),
            None if flux is None else flux.cpu().numpy().astype(np.float64), st)


def _relerr(a, ref):
    return float(np.max(np.abs(a / ref - 1.0)))


H_PLANCK, C_LIGHT, K_B = 6.62607015e-27, 2.99792458e10, 1.380649e-16


def _check_flux_bounds(cfg, params, flux, n_t=None, rtol=2e-6):
    """SURVEY.md section 4 invariant, on every model: each intensity is a convex combination of level
    sources, so pi f B_nu(T_min) <= F <= pi f B_nu(T_max) with the extremes of the model's own profile
    (piecewise linear in log p: extremes at the nodes).  Planck is evaluated here, in fp64."""
    n_t = cfg.n_knots if n_t is None else n_t
    nu = cfg.nu0 + cfg.dnu * np.arange(cfg.n_nu)
    c1, c2 = 2 * H_PLANCK * C_LIGHT ** 2, H_PLANCK * C_LIGHT / K_B
    for b in range(params.shape[0]):
        T = params[b, 2:2 + n_t]
        f = params[b, 1] * cfg.flux_const
        lo = np.pi * f * c1 * nu ** 3 / np.expm1(c2 * nu / T.min())
        hi = np.pi * f * c1 * nu ** 3 / np.expm1(c2 * nu / T.max())
        assert np.all(flux[b] >= lo * (1 - rtol)) and np.all(flux[b] <= hi * (1 + rtol)), b


class _Obs:
    def __init__(self, obs, obs_err):
        self.obs, self.obs_err = np.asarray(obs, np.float64), np.asarray(obs_err, np.float64)


def _logl_from_spectrum(wl, spec):
    """Eq. 19 in fp64 (scipy's normal log-density) from a binned spectrum [B][J]."""
    from scipy.stats import norm
    return norm.logpdf(wl.obs[None, :], loc=spec, scale=wl.obs_err[None, :]).sum(axis=1)


def _check_logl(wl, logl, ref, spec_gpu=None, tag=None):
    """logL against the oracle.  north_star's 1e-3 ABSOLUTE bound is asserted wherever it is attainable
    (reduced chi-square of order 1: the near-truth tests).  Far from the truth |logL| reaches 1e5..1e6 and
    a binned-flux error e_j (allowed: 1e-4 M_j) moves logL by up to sum_j (|D_j - M_j| e_j + e_j^2/2)/sigma_j^2:
    that propagated bound is asserted on every model, and -- tighter -- that the chi-square reduction
    itself is exact: logL equals Eq. 19 evaluated in fp64 on the GPU's own binned spectrum."""
    M = ref["spectra"]
    e = TOL_FLUX_PROPAGATED * np.abs(M)
    bound = ((np.abs(wl.obs[None, :] - M) * e + 0.5 * e * e) / wl.obs_err[None, :] ** 2).sum(axis=1)
    d = np.abs(logl - ref["logl"])
    assert np.all(d <= bound + TOL_LOGL_ABS), (float(d.max()), float(bound.min()))
    if spec_gpu is not None:
        own = _logl_from_spectrum(wl, spec_gpu)
        assert np.max(np.abs(logl - own) / np.maximum(1.0, np.abs(own))) <= 1e-9
    _record(tag, max_abs_dlogl=float(d.max()), max_rel_dlogl=float(np.max(d / np.maximum(1.0, np.abs(ref["logl"])))),
            max_abs_logl=float(np.abs(ref["logl"]).max()), n_models=int(len(d)),
            max_dlogl_over_bound=float(np.max(d / (bound + TOL_LOGL_ABS))),
            **({} if spec_gpu is None else {"max_rel_err_binned_flux": _relerr(spec_gpu, M)}))
    return float(d.max())


def _record(tag, **kv):
    """Measured maxima go to gpurun_out/parity_summary.json (scratch); the copy DESIGN.md 'logL tolerance' quotes is
    tracked as profiles/r03_parity_summary.json."""
    if tag is None:
        return
    import json, os
    out = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "gpurun_out")
    try:
        os.makedirs(out, exist_ok=True)
        path = os.path.join(out, "parity_summary.json")
        data = json.load(open(path)) if os.path.exists(path) else {}
        data.setdefault(tag, {}).update(kv)
        json.dump(data, open(path, "w"), indent=1, sort_keys=True)
    except OSError:
        pass


@pytest.mark.parametrize("kernel", [1, 2, 3], ids=["direct", "slab", "levelpar"])
def test_config0_tiny(torch_cuda, oracle, wl0, kernel):
    ref = oracle.forward_workload(wl0, want_flux=True)
    spec, logl, flux, st = _run(torch_cuda, wl0, wl0.params, kernel)
    assert _relerr(flux, ref["flux_hr"]) <= TOL_FLUX
    assert _relerr(spec, ref["spectra"]) <= TOL_FLUX
    assert np.max(np.abs(logl - ref["logl"])) <= TOL_LOGL_ABS
    assert st["n_clamped"] == ref["n_clamped"] * 2          # forward_batch + forward_highres


@pytest.mark.parametrize("kernel", [1, 2, 3], ids=["direct", "slab", "levelpar"])
def test_config1_medium_all_models(torch_cuda, oracle, wl1, kernel):
    ref = oracle.forward_workload(wl1, want_flux=True)
    spec, logl, flux, st = _run(torch_cuda, wl1, wl1.params, kernel)
    assert _relerr(flux, ref["flux_hr"]) <= TOL_FLUX
    assert _relerr(spec, ref["spectra"]) <= TOL_FLUX
    _check_logl(wl1, logl, ref, spec, tag=f"configs[1] all 64 models, kernel {kernel}")
    _check_flux_bounds(wl1.cfg, wl1.params, flux)
    assert st["n_clamped"] == ref["n_clamped"] * 2


@pytest.mark.parametrize("kernel", [1, 2, 3], ids=["direct", "slab", "levelpar"])
@pytest.mark.parametrize("cfg_index", [1, 2])
def test_logl_near_truth_absolute_tolerance(torch_cuda, oracle, wl1, wl2, kernel, cfg_index):
    """north_star's 1e-3 absolute bound on logL, on three independent near-truth sets of 12 (36 models): round 2 had
    one set and a 20 % margin at configs[2]; the maximum over the three is what DESIGN.md quotes."""
    wl = {1: wl1, 2: wl2}[cfg_index]
    params = np.concatenate([W.near_truth_params(wl.cfg, 12, draw=d) for d in range(3)])
    ref = oracle.forward_workload(wl, params=params)
    spec, logl, _, _ = _run(torch_cuda, wl, params, kernel, highres=False)
    assert _relerr(spec, ref["spectra"]) <= TOL_FLUX
    red_chi2 = ((wl.obs[None, :] - ref["spectra"]) ** 2 / wl.obs_err[None, :] ** 2).sum(axis=1) / wl.cfg.n_bins
    assert np.all(red_chi2 < 5.0)                            # the subset really is near the truth
    assert np.max(np.abs(logl - ref["logl"])) <= TOL_LOGL_ABS
    _record(f"configs[{cfg_index}] near truth, kernel {kernel}", max_abs_dlogl=float(np.max(np.abs(logl - ref["logl"]))),
            max_abs_dlogl_per_draw=[float(np.max(np.abs(logl - ref["logl"])[12 * d:12 * d + 12])) for d in range(3)],
            max_reduced_chi2=float(red_chi2.max()), n_models=36)


def test_config2_full_batch_sampled_models(torch_cuda, oracle, wl2):
    """configs[2] at its full size (B = 256) in the launch configuration bench.py times
    (kernel = auto); the oracle recomputes ALL 256 models."""
    spec, logl, flux, st = _run(torch_cuda, wl2, wl2.params, kernel=0)
    ref = oracle.forward_workload(wl2, want_flux=True)
    assert _relerr(flux, ref["flux_hr"]) <= TOL_FLUX
    assert _relerr(spec, ref["spectra"]) <= TOL_FLUX
    _check_logl(wl2, logl, ref, spec, tag="configs[2] all 256 models")
    assert np.isfinite(spec).all() and np.isfinite(logl).all() and (flux > 0).all()
    _check_flux_bounds(wl2.cfg, wl2.params, flux)
    assert st["n_clamped"] == ref["n_clamped"] * 2


def test_config3_full_batch_sampled_models(torch_cuda, oracle, wl3):
    """configs[3] at its full size (B = 1024, 85001 wavenumbers, 150 levels, 8 angles, 1.6 GB of
    tables) in the launch configuration bench.py times; the oracle recomputes a seeded sample."""
    spec, logl, flux, st = _run(torch_cuda, wl3, wl3.params, kernel=0)
    rng = np.random.default_rng(3)
    pick = np.sort(rng.choice(wl3.cfg.batch, 64, replace=False))
    ref = oracle.forward_workload(wl3, params=wl3.params[pick], want_flux=True)
    assert _relerr(flux[pick], ref["flux_hr"]) <= TOL_FLUX
    assert _relerr(spec[pick], ref["spectra"]) <= TOL_FLUX
    _check_logl(wl3, logl[pick], ref, spec[pick], tag="configs[3] 64 of 1024 models")
    # properties that hold for every one of the 1024 models
    assert np.isfinite(spec).all() and np.isfinite(logl).all() and (flux > 0).all()
    own = _logl_from_spectrum(wl3, spec)
    assert np.max(np.abs(logl - own) / np.maximum(1.0, np.abs(own))) <= 1e-9
    _check_flux_bounds(wl3.cfg, wl3.params, flux)


def test_config4_streamed_loglike_only(torch_cuda, oracle, wl3):
    """configs[4]: 4096 parameter vectors as 16 back-to-back helios_loglike_batch calls of 256 on
    one stream, no host synchronisation in between, spectra never written.  logL must equal what
    helios_forward_batch returns for the same vectors, and the oracle's on a seeded sample."""
    from paper_1910_01070_b200 import Helios
    torch = torch_cuda
    cfg4 = W.get_config(4)
    params = W.draw_params(cfg4)
    assert params.shape[0] == 4096
    h = Helios(0)
    h.setup_workload(wl3)                       # config 4 re-uses config 3's tables, grid and observation
    h.set_kernel(2)                             # same kernel for the 256-model calls and the 4-model check
    p = torch.as_tensor(params, device="cuda:0")
    out = torch.empty(4096, dtype=torch.float64, device="cuda:0")
    B = 4096 // cfg4.n_calls
    for c in range(cfg4.n_calls):
        h.loglike_batch(p[c * B:(c + 1) * B], out[c * B:(c + 1) * B])
    pick = np.sort(np.random.default_rng(4).choice(4096, 64, replace=False))
    spec_full, full = h.forward_batch(p[torch.as_tensor(pick, device="cuda:0")].contiguous())
    torch.cuda.synchronize()
    logl = out.cpu().numpy()
    assert np.isfinite(logl).all()
    assert np.array_equal(full.cpu().numpy(), logl[pick])
    ref = oracle.forward_workload(wl3, params=params[pick])
    _check_logl(wl3, logl[pick], ref, spec_full.cpu().numpy().astype(np.float64), tag="configs[4] 64 of 4096 models")
    h.close()


def test_logl_near_truth_config3(torch_cuda, oracle, wl3):
    params = np.concatenate([W.near_truth_params(wl3.cfg, 4, draw=d) for d in range(3)])
    ref = oracle.forward_workload(wl3, params=params)
    spec, logl, _, _ = _run(torch_cuda, wl3, params, 0, highres=False)
    assert _relerr(spec, ref["spectra"]) <= TOL_FLUX
    red_chi2 = ((wl3.obs[None, :] - ref["spectra"]) ** 2 / wl3.obs_err[None, :] ** 2).sum(axis=1) / wl3.cfg.n_bins
    assert np.all(red_chi2 < 5.0)
    assert np.max(np.abs(logl - ref["logl"])) <= TOL_LOGL_ABS
    _record("configs[3] near truth", max_abs_dlogl=float(np.max(np.abs(logl - ref["logl"]))),
            max_reduced_chi2=float(red_chi2.max()), n_models=12)
    # configs[4]'s call shape: the same vectors inside a 256-model logL-only call (spectra never written), the rest of
    # the call filled with configs[4]'s own draws; north_star's absolute bound on the near-truth rows
    from paper_1910_01070_b200 import Helios
    torch = torch_cuda
    block = W.draw_params(W.get_config(4))[:256].copy()
    rows = np.arange(12) * 21 + 3                    # scattered over the call, in several CTAs
    block[rows] = params
    h = Helios(0)
    h.setup_workload(wl3)
    out = h.loglike_batch(torch.as_tensor(block, device="cuda:0"))
    torch.cuda.synchronize()
    h.close()
    d4 = np.abs(out.cpu().numpy()[rows] - ref["logl"])
    assert np.max(d4) <= TOL_LOGL_ABS
    _record("configs[4] near truth (rows of a 256-model logL-only call)", max_abs_dlogl=float(d4.max()), n_models=12)


@pytest.mark.parametrize("kernel", [1, 2, 3], ids=["direct", "slab", "levelpar"])
def test_batch_invariants(torch_cuda, wl1, kernel):
    """Permuting models permutes outputs; a model's result does not depend on the batch
    it is in; repeated runs are bitwise identical."""
    p = wl1.params[:40]
    spec, logl, flux, _ = _run(torch_cuda, wl1, p, kernel)
    perm = np.random.default_rng(0).permutation(40)
    spec_p, logl_p, flux_p, _ = _run(torch_cuda, wl1, p[perm], kernel)
    assert np.array_equal(spec_p, spec[perm]) and np.array_equal(logl_p, logl[perm])
    assert np.array_equal(flux_p, flux[perm])
    spec_1, logl_1, flux_1, _ = _run(torch_cuda, wl1, p[7:8], kernel)
    assert np.array_equal(spec_1[0], spec[7]) and logl_1[0] == logl[7]
    spec_r, logl_r, _, _ = _run(torch_cuda, wl1, p, kernel)
    assert np.array_equal(spec_r, spec) and np.array_equal(logl_r, logl)


@pytest.mark.parametrize("fused", [False, True], ids=["twokernel", "fusedobs"])
@pytest.mark.parametrize("kernel", [1, 2, 3], ids=["direct", "slab", "levelpar"])
def test_ragged_sizes_and_edge_cases(torch_cuda, oracle, kernel, fused):
    """Wavenumber count not a multiple of any tile, odd level count, 1..3 angles,
    single species without CIA, CIA only, bins narrower than a grid cell, no
    instrument profile, clamped temperatures, a non-finite parameter."""
    rng = np.random.default_rng(123)
    nNu, nT, nP = 777, 5, 4
    T_grid = np.array([300.0, 700.0, 1200.0, 1900.0, 3100.0])
    lp_grid = np.array([-4.0, -1.5, 0.5, 2.7])
    for (S, C, L, A, K) in [(1, 0, 7, 1, 1), (3, 2, 33, 3, 4), (0, 2, 12, 2, 2), (5, 1, 51, 8, 6)]:
        sigma = (10.0 ** rng.uniform(-27, -21, (S, nT, nP, nNu))).astype(np.float32)
        cia = (10.0 ** rng.uniform(-9, -7, (C, nT, nNu))).astype(np.float32)
        nu0, dnu = 2500.0, 1.5
        edges = np.concatenate([[nu0, nu0 + 0.4, nu0 + 0.9, nu0 + 20.0],
                                np.linspace(nu0 + 50.0, nu0 + dnu * (nNu - 1), 9)])
        inst = np.where(np.arange(nNu) % 2 == 0, 3.0, 4.5) if A != 2 else None
        B = 5
        params = np.column_stack([rng.uniform(4, 5.5, B), rng.uniform(0.5, 2, B),
                                  -np.sort(-rng.uniform(250, 3300, (B, K)), axis=1),   # some T outside the table
                                  rng.uniform(-8, -2, (B, S))])
        params[3, 1] = np.nan
        obs = np.full(len(edges) - 1, 1e4)
        err = np.full(len(edges) - 1, 1e3)
        ref = oracle.forward(T_grid, lp_grid, nu0, dnu, sigma if S else np.zeros((0, nT, nP, nNu), np.float32),
                             cia if C else None, L, 100.0, 1e-4, K, A, 2.3, 0.17, 0.5,
                             edges, obs, err, inst, params, want_flux=True)

        from paper_1910_01070_b200 import Helios
        torch = torch_cuda
        h = Helios(0)
        sig_arg = sigma if S else np.zeros((0, nT, nP, nNu), np.float32)
        h.load_opacity(T_grid, lp_grid, nu0, dnu, sig_arg, cia if C else None)
        h.set_atmosphere(L, 100.0, 1e-4, K, A, 2.3, 0.17, 0.5)
        h.set_observation(edges, obs, err, inst)
        h.set_kernel(kernel)
        h.set_fused_obs(fused)          # the direct kernel ignores it (it always writes the flux)
        p = torch.as_tensor(params, device="cuda:0")
        spec, logl = h.forward_batch(p)
        flux = h.forward_highres(p)
        torch.cuda.synchronize()
        st = h.stats()
        h.close()
        spec = spec.cpu().numpy().astype(np.float64); logl = logl.cpu().numpy(); flux = flux.cpu().numpy().astype(np.float64)
        ok = np.array([0, 1, 2, 4])
        assert np.isnan(spec[3]).all() and np.isnan(flux[3]).all() and logl[3] == -np.inf
        assert _relerr(flux[ok], ref["flux_hr"][ok]) <= TOL_FLUX, (S, C, L, A, K)
        assert _relerr(spec[ok], ref["spectra"][ok]) <= TOL_FLUX, (S, C, L, A, K)
        _check_logl(_Obs(obs, err), logl[ok], {"spectra": ref["spectra"][ok], "logl": ref["logl"][ok]}, spec[ok])
        assert st["n_clamped"] == 2 * ref["n_clamped"] and st["n_nonfinite"] == 2


def test_host_entry_point_matches_device_entry_point(torch_cuda, wl1):
    from paper_1910_01070_b200 import Helios
    torch = torch_cuda
    h = Helios(0)
    h.setup_workload(wl1)
    p_host = torch.as_tensor(wl1.params).pin_memory()
    spec_h = torch.empty((wl1.cfg.batch, wl1.cfg.n_bins), dtype=torch.float32).pin_memory()
    logl_h = torch.empty((wl1.cfg.batch,), dtype=torch.float64).pin_memory()
    h.forward_batch_host(p_host, spec_h, logl_h)
    spec_d, logl_d = h.forward_batch(p_host.cuda())
    torch.cuda.synchronize()
    assert torch.equal(spec_h, spec_d.cpu()) and torch.equal(logl_h, logl_d.cpu())
    only = h.loglike_batch(p_host.cuda())
    torch.cuda.synchronize()
    assert torch.equal(only.cpu(), logl_h)
    h.close()


def test_error_codes(torch_cuda, wl0):
    import paper_1910_01070_b200 as pkg
    torch = torch_cuda
    h = pkg.Helios(0)
    p = torch.as_tensor(wl0.params, device="cuda:0")
    with pytest.raises(pkg.HeliosError) as ei:
        h.forward_highres(p)
    assert ei.value.code == pkg.HELIOS_ESTATE
    with pytest.raises(pkg.HeliosError) as ei:
        h.load_opacity(np.array([500.0, 400.0]), wl0.log10p_grid, 4000.0, 1.0, wl0.sigma[:, :2])
    assert ei.value.code == pkg.HELIOS_EINVAL
    h.load_opacity(wl0.T_grid, wl0.log10p_grid, 4000.0, 1.0, wl0.sigma)
    with pytest.raises(pkg.HeliosError) as ei:
        h.set_atmosphere(20, 1e-3, 300.0, 2, 2, 2.3, 0.17)       # p_bottom < p_top
    assert ei.value.code == pkg.HELIOS_EINVAL
    h.set_atmosphere(20, 300.0, 1e-3, 2, 2, 2.3, 0.17)
    with pytest.raises(pkg.HeliosError) as ei:
        h.set_observation(np.array([3000.0, 4500.0]))             # edge outside the grid
    assert ei.value.code == pkg.HELIOS_EINVAL
    h.set_observation(wl0.bin_edges, None, None, wl0.inst_sigma)
    with pytest.raises(pkg.HeliosError) as ei:
        h.loglike_batch(p)                                        # no data loaded
    assert ei.value.code == pkg.HELIOS_ESTATE
    spec, _ = h.forward_batch(p, want_logl=False)
    torch.cuda.synchronize()
    assert torch.isfinite(spec).all()
    h.close()


def test_auto_falls_back_to_the_direct_kernel_when_planes_do_not_fit(torch_cuda, oracle):
    """40 species x 30 temperature nodes: one table plane would need 307 KB of shared memory, so the
    automatic choice must be the direct kernel, and forcing the staged kernel must fail loudly."""
    import paper_1910_01070_b200 as pkg
    torch = torch_cuda
    rng = np.random.default_rng(5)
    S, nT, nP, nNu, L, K, A, B = 40, 30, 3, 200, 15, 2, 2, 9
    T_grid = np.linspace(200.0, 3200.0, nT); lp_grid = np.array([-4.0, 0.0, 3.0])
    sigma = (10.0 ** rng.uniform(-27, -22, (S, nT, nP, nNu))).astype(np.float32)
    edges = np.linspace(3000.0, 3000.0 + nNu - 1, 11)
    params = np.column_stack([rng.uniform(4, 5.5, B), rng.uniform(0.5, 2, B),
                              -np.sort(-rng.uniform(500, 2800, (B, K)), axis=1), rng.uniform(-8, -3, (B, S))])
    ref = oracle.forward(T_grid, lp_grid, 3000.0, 1.0, sigma, None, L, 100.0, 1e-3, K, A, 2.3, 0.17, 1.0,
                         edges, None, None, None, params, want_flux=True, want_logl=False)
    h = pkg.Helios(0)
    h.load_opacity(T_grid, lp_grid, 3000.0, 1.0, sigma, None)
    h.set_atmosphere(L, 100.0, 1e-3, K, A, 2.3, 0.17, 1.0)
    h.set_observation(edges)
    p = torch.as_tensor(params, device="cuda:0")
    spec, _ = h.forward_batch(p, want_logl=False)
    flux = h.forward_highres(p)
    torch.cuda.synchronize()
    assert _relerr(flux.cpu().numpy().astype(np.float64), ref["flux_hr"]) <= TOL_FLUX
    assert _relerr(spec.cpu().numpy().astype(np.float64), ref["spectra"]) <= TOL_FLUX
    h.set_kernel(2)
    with pytest.raises(pkg.HeliosError) as ei:
        h.forward_highres(p)
    assert ei.value.code == pkg.HELIOS_EINVAL
    h.close()


@pytest.mark.parametrize("kernel", [2, 3], ids=["slab", "levelpar"])
@pytest.mark.parametrize("seed", range(10))
def test_random_shapes_staged_kernel(torch_cuda, oracle, seed, kernel):
    """Random table / atmosphere shapes through the staged and the level-parallel kernel: pressure grids denser
    than the levels (segments that skip table cells, two new planes per segment), two-node grids, two levels
    (one chunk of one layer), one to eight angles, batches that do not fill a CTA, ring wrap-around with many planes."""
    import paper_1910_01070_b200 as pkg
    torch = torch_cuda
    rng = np.random.default_rng(1000 + seed)
    S = int(rng.integers(0, 6)); C = int(rng.integers(0, 3))
    if S + C == 0:
        S = 1
    nT = int(rng.integers(2, 12)); nP = int(rng.choice([2, 3, 9, 40])); nNu = int(rng.integers(60, 300))
    L = int(rng.choice([2, 3, 7, 30, 90])); A = int(rng.integers(1, 9)); K = int(rng.integers(1, 5))
    B = int(rng.choice([1, 5, 17, 33]))
    T_grid = np.sort(rng.uniform(200.0, 3200.0, nT)); T_grid[0] = 200.0; T_grid[-1] = 3200.0
    T_grid = np.unique(np.round(T_grid, 3))
    nT = len(T_grid)
    if nT < 2:
        T_grid = np.array([200.0, 3200.0]); nT = 2
    lp_grid = np.linspace(-4.5, 2.5, nP) + (rng.uniform(-0.05, 0.05, nP) if nP > 2 else 0.0)
    lp_grid = np.sort(lp_grid)
    sigma = (10.0 ** rng.uniform(-27, -21, (S, nT, nP, nNu))).astype(np.float32)
    cia = (10.0 ** rng.uniform(-9, -7, (C, nT, nNu))).astype(np.float32) if C else None
    nu0, dnu = 3000.0, 0.7
    edges = np.linspace(nu0, nu0 + dnu * (nNu - 1), 7)
    inst = np.full(nNu, 2.0)
    params = np.column_stack([rng.uniform(4, 5.5, B), rng.uniform(0.5, 2, B),
                              -np.sort(-rng.uniform(300, 3000, (B, K)), axis=1), rng.uniform(-8, -2, (B, S))])
    obs = np.full(6, 1e4); err = np.full(6, 1e3)
    ref = oracle.forward(T_grid, lp_grid, nu0, dnu, sigma, cia, L, 200.0, 2e-4, K, A, 2.3, 0.17, 1.0,
                         edges, obs, err, inst, params, want_flux=True)
    h = pkg.Helios(0)
    h.load_opacity(T_grid, lp_grid, nu0, dnu, sigma, cia)
    h.set_atmosphere(L, 200.0, 2e-4, K, A, 2.3, 0.17, 1.0)
    h.set_observation(edges, obs, err, inst)
    h.set_kernel(kernel)
    p = torch.as_tensor(params, device="cuda:0")
    spec, logl = h.forward_batch(p)
    flux = h.forward_highres(p)
    torch.cuda.synchronize()
    st = h.stats()
    h.close()
    shape = dict(S=S, C=C, nT=nT, nP=nP, nNu=nNu, L=L, A=A, K=K, B=B)
    assert _relerr(flux.cpu().numpy().astype(np.float64), ref["flux_hr"]) <= TOL_FLUX, shape
    assert _relerr(spec.cpu().numpy().astype(np.float64), ref["spectra"]) <= TOL_FLUX, shape
    _check_logl(_Obs(obs, err), logl.cpu().numpy(), ref, spec.cpu().numpy().astype(np.float64))
    assert st["n_clamped"] == 2 * ref["n_clamped"], shape


def test_n_params_is_checked(torch_cuda, wl1):
    """A parameter block laid out for another parametrisation (wrong row length) is refused with
    HELIOS_EINVAL by every entry point instead of being read with the wrong stride."""
    import paper_1910_01070_b200 as pkg
    torch = torch_cuda
    h = pkg.Helios(0)
    h.setup_workload(wl1)
    good = torch.as_tensor(wl1.params[:4], device="cuda:0")
    assert good.shape[1] == h.n_params == pkg.helios_get_n_params(h.ctx)
    bad = torch.cat([good, torch.zeros((4, 1), dtype=torch.float64, device="cuda:0")], dim=1).contiguous()
    for call in (lambda p: h.forward_batch(p), lambda p: h.loglike_batch(p), lambda p: h.forward_highres(p),
                 lambda p: h.teff_batch(p, 4000.0, 12000.0),
                 lambda p: h.forward_batch_host(p.cpu().pin_memory(), None, torch.empty(4, dtype=torch.float64).pin_memory())):
        with pytest.raises(pkg.HeliosError) as ei:
            call(bad)
        assert ei.value.code == pkg.HELIOS_EINVAL
    h.set_extras(pkg.HELIOS_EXTRA_DISTANCE)
    h.set_atmosphere(wl1.cfg.n_levels, 300.0, 1e-3, wl1.cfg.n_knots, wl1.cfg.n_angles, 2.3, 0.17, 1.0)
    assert h.n_params == good.shape[1] + 1          # the extras survive set_atmosphere; the wrapper follows the context
    with pytest.raises(pkg.HeliosError):
        h.forward_batch(good)
    with pytest.raises(ValueError):
        h.forward_batch(good[0])                    # 1-D
    with pytest.raises(ValueError):
        h.forward_batch_host(torch.as_tensor(wl1.params[:4], dtype=torch.float32).pin_memory(), None,
                             torch.empty(4, dtype=torch.float64).pin_memory())       # fp32 host tensor
    h.close()


@pytest.mark.parametrize("kernel", [1, 2, 3], ids=["direct", "slab", "levelpar"])
def test_unphysical_models_are_rejected(torch_cuda, oracle, wl1, kernel):
    """Finite but unphysical parameter vectors (R31) give logL = -inf (never NaN) and NaN
    spectra, are counted, and leave their neighbours bit-identical; the oracle applies the same rule."""
    import paper_1910_01070_b200 as pkg
    torch = torch_cuda
    cfg = wl1.cfg
    K, S = cfg.n_knots, cfg.n_species
    base = wl1.params[:8].copy()
    params = base.copy()
    params[1, 2 + K:2 + K + S] = -0.1          # VMRs sum to 3.2 > 1: negative H2/He fill
    params[3, 1] = -0.5                         # f < 0
    params[5, 0] = 400.0                        # g = 10^400 overflows
    params[6, 2 + K - 1] = -50.0                # top temperature node below zero
    ref = oracle.forward_workload(wl1, params=params, want_flux=True)
    bad, good = [1, 3, 5, 6], [0, 2, 4, 7]
    assert np.all(ref["logl"][bad] == -np.inf) and np.isnan(ref["spectra"][bad]).all()
    spec, logl, flux, st = _run(torch, wl1, params, kernel)
    assert np.all(logl[bad] == -np.inf) and np.isnan(spec[bad]).all() and np.isnan(flux[bad]).all()
    assert st["n_nonfinite"] == 2 * len(bad)
    spec0, logl0, flux0, _ = _run(torch, wl1, base, kernel)
    assert np.array_equal(spec[good], spec0[good]) and np.array_equal(logl[good], logl0[good])
    assert np.array_equal(flux[good], flux0[good])
    assert _relerr(spec[good], ref["spectra"][good]) <= TOL_FLUX


def test_small_batches_take_the_level_parallel_kernel_and_agree_with_the_staged_one(torch_cuda, oracle, wl2):
    """configs[2] tables with B = 1, 2, 4 in the launch configuration bench.py times for small batches
    (kernel = auto -> level-parallel up to the measured crossover B = 8): every model against the oracle, and against
    the staged kernel's result for the same vectors (different operation order: agreement to a few ulp, not bitwise)."""
    params = wl2.params[:16]
    ref = oracle.forward_workload(wl2, params=params, want_flux=True)
    spec_s, logl_s, flux_s, _ = _run(torch_cuda, wl2, params, kernel=2)
    for B in (1, 2, 4, 8, 16):
        spec, logl, flux, _ = _run(torch_cuda, wl2, params[:B], kernel=0)
        assert _relerr(flux, ref["flux_hr"][:B]) <= TOL_FLUX
        assert _relerr(spec, ref["spectra"][:B]) <= TOL_FLUX
        _check_logl(wl2, logl, {"spectra": ref["spectra"][:B], "logl": ref["logl"][:B]}, spec)
        assert _relerr(flux, flux_s[:B]) <= 5e-6
        forced = _run(torch_cuda, wl2, params[:B], kernel=3 if B <= 8 else 2)
        assert np.array_equal(forced[0], spec) and np.array_equal(forced[2], flux)     # which kernel auto really took
    near = W.near_truth_params(wl2.cfg, 12)[:8]     # the set of test_logl_near_truth_absolute_tolerance
    refn = oracle.forward_workload(wl2, params=near)
    specn, logln, _, _ = _run(torch_cuda, wl2, near, kernel=0, highres=False)
    assert np.max(np.abs(logln - refn["logl"])) <= TOL_LOGL_ABS
    _record("configs[2] near truth, B = 8 (level-parallel)", max_abs_dlogl=float(np.max(np.abs(logln - refn["logl"]))), n_models=8)


@pytest.mark.parametrize("kernel", [1, 2, 3], ids=["direct", "slab", "levelpar"])
def test_wavenumber_order_tables_give_the_same_results(torch_cuda, oracle, wl1, kernel):
    """HELIOS_OPT_NU_ORDER: the resident tables keep their columns in wavenumber order (0) or sorted by a reference
    opacity (1, the default, which every other test runs).  Both against the oracle, and against each other: in the
    direct kernel a wavenumber's arithmetic does not depend on its neighbours, so the two layouts agree bit for bit;
    the staged and level-parallel kernels pick the thin / thick / general form of a layer's update per WARP, i.e.
    depending on which 64 columns sit together, and those forms differ in the last bits."""
    params = wl1.params[:24]
    ref = oracle.forward_workload(wl1, params=params, want_flux=True)
    out = {}
    for order in (0, 1):
        spec, logl, flux, _ = _run(torch_cuda, wl1, params, kernel=kernel, nu_order=order)
        assert _relerr(flux, ref["flux_hr"]) <= TOL_FLUX and _relerr(spec, ref["spectra"]) <= TOL_FLUX
        _check_logl(wl1, logl, ref, spec)
        out[order] = (spec, logl, flux)
    if kernel == 1:
        assert np.array_equal(out[0][2], out[1][2]) and np.array_equal(out[0][0], out[1][0]) and np.array_equal(out[0][1], out[1][1])
    else:
        assert _relerr(out[0][2], out[1][2]) <= 5e-6 and _relerr(out[0][0], out[1][0]) <= 5e-6


@pytest.mark.parametrize("kernel", [2, 3], ids=["slab", "levelpar"])
def test_fused_observation_epilogue(torch_cuda, oracle, wl1, kernel):
    """HELIOS_OPT_FUSED_OBS: the RT kernel applies convolve + bin in its epilogue with 64-bit integer atomics (no flux
    buffer).  Against the oracle at the usual tolerances; against the two-kernel path (same flux, the sum over a bin
    exact in integers instead of fp32: agreement to a few fp32 ulp); bitwise reproducible from run to run and
    independent of the batch a model is in (integer sums do not depend on the arrival order of the CTAs); rejected
    models still give NaN spectra and logL = -inf."""
    params = wl1.params[:40].copy()
    params[7, 1] = -1.0                                   # f < 0: rejected (R31)
    ref = oracle.forward_workload(wl1, params=params)
    ok = np.ones(40, bool); ok[7] = False
    spec_f, logl_f, _, st = _run(torch_cuda, wl1, params, kernel=kernel, highres=False, fused=True)
    spec_u, logl_u, _, _ = _run(torch_cuda, wl1, params, kernel=kernel, highres=False, fused=False)
    assert _relerr(spec_f[ok], ref["spectra"][ok]) <= TOL_FLUX
    assert np.all(np.isnan(spec_f[7])) and logl_f[7] == -np.inf and st["n_nonfinite"] == 1
    _check_logl(wl1, logl_f[ok], {"spectra": ref["spectra"][ok], "logl": ref["logl"][ok]}, spec_f[ok])
    assert _relerr(spec_f[ok], spec_u[ok]) <= 2e-6
    again = _run(torch_cuda, wl1, params, kernel=kernel, highres=False, fused=True)
    assert np.array_equal(again[0][ok], spec_f[ok]) and np.array_equal(again[1], logl_f)
    sub = _run(torch_cuda, wl1, params[8:13], kernel=kernel, highres=False, fused=True)
    assert np.array_equal(sub[0], spec_f[8:13]) and np.array_equal(sub[1], logl_f[8:13])
    near = W.near_truth_params(wl1.cfg, 12)
    refn = oracle.forward_workload(wl1, params=near)
    _, logln, _, _ = _run(torch_cuda, wl1, near, kernel=kernel, highres=False, fused=True)
    assert np.max(np.abs(logln - refn["logl"])) <= TOL_LOGL_ABS


def test_measured_peaks_are_plausible(torch_cuda, wl0):
    """helios_measure_peaks (the roofline denominators of bench.py): the FP32 pipe of an sm_100 SM has 128 lanes and the
    MUFU unit 16; the micro-benchmarks must land within 10 % below those and never above."""
    from paper_1910_01070_b200 import Helios
    h = Helios(0)
    h.setup_workload(wl0)
    pk = h.measure_peaks()
    h.close()
    assert pk["n_sms"] >= 100 and 500.0 < pk["sm_clock_mhz"] < 3000.0
    assert 0.9 * 128 <= pk["ffma_per_clk_sm"] <= 128.5 and 0.9 * 128 <= pk["ffma2_per_clk_sm"] <= 128.5
    assert 0.9 * 16 <= pk["mufu_per_clk_sm"] <= 16.1
    c1, c2, c3 = pk["ffma2_cycles"]
    assert 1.9 <= c1 <= c2 <= c3 <= 4.5           # a packed FFMA2 holds the dispatch port >= 2 cycles, more with 3 register pairs


def test_stage_timing_mode_gives_the_same_results(torch_cuda, wl1):
    """HELIOS_OPT_TIMING brackets the kernels with events and launches them without the programmatic-dependent-launch
    attribute; results must be bit-identical to the default (dependent) launches, and the stage times positive."""
    import torch
    from paper_1910_01070_b200 import Helios
    p = torch.as_tensor(wl1.params[:32], device="cuda:0")
    out = []
    for timing in (False, True):
        h = Helios(0)
        h.setup_workload(wl1)
        h.set_timing(timing)
        spec, logl = h.forward_batch(p)
        spec2, logl2 = h.forward_batch(p)          # second call: the workspace is reused, nothing may leak from the first
        torch.cuda.synchronize()
        assert torch.equal(spec, spec2) and torch.equal(logl, logl2)
        if timing:
            st = h.stage_ms()
            assert st["n_calls"] == 2 and st["prep_ms"] > 0 and st["rt_ms"] > 0 and st["obs_ms"] > 0
        out.append((spec.cpu().numpy(), logl.cpu().numpy()))
        h.close()
    assert np.array_equal(out[0][0], out[1][0]) and np.array_equal(out[0][1], out[1][1])


def test_tall_atmosphere_falls_back_from_the_level_parallel_kernel(torch_cuda, oracle):
    """More than 8 x 32 + 1 levels: the level-parallel kernel is unavailable (chunks of at most 32 layers), so a small
    batch on kernel = auto takes the staged kernel; forcing the level-parallel kernel is an error, not a wrong answer."""
    from paper_1910_01070_b200 import Helios, HeliosError, HELIOS_EINVAL
    rng = np.random.default_rng(5)
    nNu, nT, nP, S, C, L, A, K = 300, 6, 5, 2, 1, 300, 2, 3
    T_grid = np.linspace(200.0, 3200.0, nT); lp_grid = np.linspace(-4.5, 3.0, nP)
    sigma = (10.0 ** rng.uniform(-26, -22, (S, nT, nP, nNu))).astype(np.float32)
    cia = (10.0 ** rng.uniform(-9, -7, (C, nT, nNu))).astype(np.float32)
    nu0, dnu = 3000.0, 2.0
    edges = np.linspace(nu0, nu0 + dnu * (nNu - 1), 21)
    inst = np.full(nNu, 6.0)
    B = 3
    params = np.column_stack([rng.uniform(4, 5, B), rng.uniform(0.5, 2, B), -np.sort(-rng.uniform(500, 2800, (B, K)), axis=1),
                              rng.uniform(-7, -3, (B, S))])
    obs = np.full(20, 1e4); err = np.full(20, 1e3)
    ref = oracle.forward(T_grid, lp_grid, nu0, dnu, sigma, cia, L, 300.0, 1e-3, K, A, 2.3, 0.17, 1.0, edges, obs, err, inst, params,
                         want_flux=True)
    h = Helios(0)
    h.load_opacity(T_grid, lp_grid, nu0, dnu, sigma, cia)
    h.set_atmosphere(L, 300.0, 1e-3, K, A, 2.3, 0.17, 1.0)
    h.set_observation(edges, obs, err, inst)
    p = torch_cuda.as_tensor(params, device="cuda:0")
    spec, logl = h.forward_batch(p)
    flux = h.forward_highres(p)
    torch_cuda.cuda.synchronize()
    assert _relerr(flux.cpu().numpy().astype(np.float64), ref["flux_hr"]) <= TOL_FLUX
    assert _relerr(spec.cpu().numpy().astype(np.float64), ref["spectra"]) <= TOL_FLUX
    h.set_kernel(3)
    with pytest.raises(HeliosError) as ei:
        h.forward_batch(p)
    assert ei.value.code == HELIOS_EINVAL
    h.close()


def test_cuda_graph_replay_gives_the_same_results(torch_cuda, oracle, wl1):
    """HELIOS_OPT_GRAPHS: a call that repeats with the same batch size and buffers is captured on its second
    occurrence and replayed from the third on.  Replays must be bit-identical to plain launches, follow new
    parameter VALUES in the same buffer, survive other calls in between, and be dropped when the context changes."""
    import torch
    from paper_1910_01070_b200 import Helios
    pA = torch.as_tensor(wl1.params[:6], device="cuda:0")
    pB = torch.as_tensor(wl1.params[6:12], device="cuda:0")
    ref = {}
    h = Helios(0); h.setup_workload(wl1); h.set_graphs(False)
    for name, p in (("A", pA), ("B", pB)):
        s, l = h.forward_batch(p); torch.cuda.synchronize()
        ref[name] = (s.clone(), l.clone())
    h.close()
    h = Helios(0); h.setup_workload(wl1)                       # graphs on (default)
    h.stats(reset=True)
    buf = pA.clone()
    spec = torch.empty((6, h.n_bins), dtype=torch.float32, device="cuda:0")
    logl = torch.empty((6,), dtype=torch.float64, device="cuda:0")
    from paper_1910_01070_b200 import helios_forward_batch, helios_loglike_batch
    for it in range(5):                                        # plain, capture, replay, replay, replay
        spec.zero_(); logl.zero_()
        helios_forward_batch(h.ctx, buf, spec, logl); torch.cuda.synchronize()
        assert torch.equal(spec, ref["A"][0]) and torch.equal(logl, ref["A"][1]), it
    buf.copy_(pB)                                              # same buffer, new values: the graph reads them at replay
    helios_forward_batch(h.ctx, buf, spec, logl); torch.cuda.synchronize()
    assert torch.equal(spec, ref["B"][0]) and torch.equal(logl, ref["B"][1])
    s2, l2 = h.forward_batch(pA); torch.cuda.synchronize()     # another call (fresh buffers) in between
    assert torch.equal(s2, ref["A"][0])
    only = torch.empty((6,), dtype=torch.float64, device="cuda:0")
    for it in range(3):                                        # logL-only call: its own graph
        helios_loglike_batch(h.ctx, buf, only); torch.cuda.synchronize()
        assert torch.equal(only, ref["B"][1])
    st = h.stats()
    assert st["n_launches"] == 3 * 10 and st["n_models"] == 6 * 10     # replays are counted like plain calls
    assert st["n_graph_launches"] == 4 + 1 + 2                          # capture + 3 replays, 1 replay, capture + 1 replay
    h.set_observation(wl1.bin_edges, wl1.obs * 1.01, wl1.obs_err, wl1.inst_sigma)     # context changed: graphs dropped
    for it in range(3):
        helios_forward_batch(h.ctx, buf, spec, logl); torch.cuda.synchronize()
        assert torch.equal(spec, ref["B"][0]) and not torch.equal(logl, ref["B"][1])
    h.close()


def test_cuda_graphs_are_dropped_by_every_context_change(torch_cuda, wl1):
    """A captured call holds its kernels' arguments by value (device pointers, sizes, logl_const, tensor maps).  After
    EVERY setter the same (buffers, B) call must run the new context, not replay the old graph: each change below is one
    whose stale replay gives different numbers (a new logl_const, another bin count, another level count, another
    meaning of the one extra parameter, other tables), the first call after it must not be a graph launch, and the
    results must equal -- bit for bit -- those of a context that never uses graphs."""
    import torch
    import paper_1910_01070_b200 as pkg
    from paper_1910_01070_b200 import Helios, helios_forward_batch
    cfg = wl1.cfg
    B = 6
    base = np.ascontiguousarray(wl1.params[:B])

    def make(graphs):
        h = Helios(0); h.setup_workload(wl1); h.set_graphs(graphs)
        return h

    def run_plain(apply_change, params, n_bins):
        h = make(False)
        for ch in apply_change:
            ch(h)
        p = torch.as_tensor(params, device="cuda:0")
        s = torch.empty((B, n_bins), dtype=torch.float32, device="cuda:0")
        l = torch.empty((B,), dtype=torch.float64, device="cuda:0")
        helios_forward_batch(h.ctx, p, s, l); torch.cuda.synchronize()
        h.close()
        return s, l

    edges2 = np.linspace(wl1.bin_edges[0], wl1.bin_edges[-1], 61)          # 60 bins instead of 120
    obs2, err2 = np.full(60, float(np.mean(wl1.obs))), np.full(60, float(np.mean(wl1.obs_err)))
    changes = [
        # (name, change, parameter block of the calls after it, n_bins after it)
        ("obs_err (logl_const by value)",
         lambda h: h.set_observation(wl1.bin_edges, wl1.obs, wl1.obs_err * 1.5, wl1.inst_sigma), base, cfg.n_bins),
        ("extras: distance", lambda h: h.set_extras(pkg.HELIOS_EXTRA_DISTANCE),
         np.concatenate([base, np.full((B, 1), 1.7)], axis=1), cfg.n_bins),
        ("extras: distance -> error inflation, same P", lambda h: h.set_extras(pkg.HELIOS_EXTRA_ERROR_INFLATION),
         np.concatenate([base, np.full((B, 1), 1.7)], axis=1), cfg.n_bins),
        ("extras off", lambda h: h.set_extras(0), base, cfg.n_bins),
        ("n_bins", lambda h: h.set_observation(edges2, obs2, err2, wl1.inst_sigma), base, 60),
        ("n_levels", lambda h: h.set_atmosphere(cfg.n_levels - 30, cfg.p_bottom_bar, cfg.p_top_bar, cfg.n_knots, cfg.n_angles,
                                                cfg.mean_mol_weight, cfg.he_to_h2, cfg.flux_const), base, 60),
        ("tp ratio form, same P", lambda h: h.set_tp_elements(cfg.n_knots - 1, 1, True),
         np.concatenate([base[:, :3], np.full((B, cfg.n_knots - 1), 0.9), base[:, 2 + cfg.n_knots:]], axis=1), 60),
        ("tables x 2", lambda h: (h.load_opacity(wl1.T_grid, wl1.log10p_grid, cfg.nu0, cfg.dnu, wl1.sigma * 2.0, wl1.cia),
                                  h.set_atmosphere(cfg.n_levels, cfg.p_bottom_bar, cfg.p_top_bar, cfg.n_knots, cfg.n_angles,
                                                   cfg.mean_mol_weight, cfg.he_to_h2, cfg.flux_const),
                                  h.set_observation(wl1.bin_edges, wl1.obs, wl1.obs_err, wl1.inst_sigma)), base, cfg.n_bins),
    ]
    h = make(True)
    p, s, l = (torch.as_tensor(base, device="cuda:0"), torch.empty((B, cfg.n_bins), dtype=torch.float32, device="cuda:0"),
               torch.empty((B,), dtype=torch.float64, device="cuda:0"))
    bufs_first = (p, s, l)
    for it in range(4):                                        # graphs exist before the first change
        helios_forward_batch(h.ctx, p, s, l)
    torch.cuda.synchronize()
    assert h.stats()["n_graph_launches"] == 3
    # buffers that stay put over all changes with the same shapes: (params, spectra, logl) keyed by (P, n_bins)
    bufs = {(base.shape[1], cfg.n_bins): bufs_first}
    applied = []
    last = ((base.shape[1], cfg.n_bins), s.clone(), l.clone())
    for name, change, params, n_bins in changes:
        key = (params.shape[1], n_bins)
        if key not in bufs:
            bufs[key] = (torch.empty((B, params.shape[1]), dtype=torch.float64, device="cuda:0"),
                         torch.empty((B, n_bins), dtype=torch.float32, device="cuda:0"),
                         torch.empty((B,), dtype=torch.float64, device="cuda:0"))
        p, s, l = bufs[key]
        change(h); applied.append(change)
        p.copy_(torch.as_tensor(params))
        ref_s, ref_l = run_plain(applied, params, n_bins)
        h.stats(reset=True)
        for it in range(4):                                    # plain, capture, replay, replay: all must give the new context's numbers
            s.zero_(); l.zero_()
            helios_forward_batch(h.ctx, p, s, l); torch.cuda.synchronize()
            if it == 0:
                assert h.stats()["n_graph_launches"] == 0, name      # the first call after a change is never a graph launch
            assert torch.equal(s, ref_s) and torch.equal(l, ref_l), (name, it)
        assert h.stats()["n_graph_launches"] == 3, name
        if last is not None and last[0] == key:                # same buffers as before the change: the numbers did change
            assert not (torch.equal(last[1], s) and torch.equal(last[2], l)), name
        last = (key, s.clone(), l.clone())
    h.close()
