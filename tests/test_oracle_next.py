"""Pins of the oracle functions behind the NEXT rows of SURVEY.md 8(f):
error-inflated likelihood (Eq. 22-23), finite-element T-p profile (Eq. 12-16), effective
temperature (Sect. 2.6), grey cloud (App. B), distance scaling (Eq. 9).  Closed forms,
library routines and special cases only; nothing here comes from the CUDA path.
"""
import numpy as np
import pytest

SIGMA_SB = 5.670374419e-5          # CODATA 2018, erg s^-1 cm^-2 K^-4
C1 = 1.191042972e-5                # 2 h c^2, erg cm^2 s^-1
C2 = 1.438776877                   # h c / k_B, cm K


def planck(nu, T):
    x = C2 * nu / T
    return C1 * nu ** 3 * np.exp(-x) / (-np.expm1(-x))


# ---------------------------------------------------------------------------- NEXT-1
def test_inflated_likelihood_closed_forms(oracle):
    J, sig = 7, 0.3
    D = np.linspace(1.0, 2.0, J)
    err = np.full(J, sig)
    eps = np.log10(3.0 * sig * sig)                 # s_j^2 = 4 sigma^2 exactly
    # D = M: only the normalisation term survives
    assert oracle.loglike_inflated(D, err, D, eps) == pytest.approx(-0.5 * J * np.log(2 * np.pi * 4 * sig * sig), rel=1e-14)
    # every bin off by k s_j lowers ln L by J k^2 / 2
    k = 1.7
    M = D - k * 2.0 * sig
    assert oracle.loglike_inflated(D, err, M, eps) - oracle.loglike_inflated(D, err, D, eps) == pytest.approx(-0.5 * J * k * k, rel=1e-13)
    # no inflation (10^eps -> 0) is Eq. 19
    M2 = D * 1.05
    assert oracle.loglike_inflated(D, err, M2, -300.0) == pytest.approx(oracle.loglike(D, err, M2), rel=1e-15)
    # inflation dominated: s^2 -> 10^eps for every bin, whatever the individual errors
    err3 = np.linspace(0.1, 0.5, J)
    big = 8.0
    expect = -np.sum((D - M2) ** 2) / (2 * 10.0 ** big) - 0.5 * J * np.log(2 * np.pi * 10.0 ** big)
    assert oracle.loglike_inflated(D, err3, M2, big) == pytest.approx(expect, rel=1e-8)


# ---------------------------------------------------------------------------- NEXT-2
@pytest.mark.parametrize("q", [1, 2, 3, 4])
def test_lobatto_nodes_against_legendre_derivative_roots(oracle, q):
    from numpy.polynomial import legendre as Lg
    c = np.zeros(q + 1); c[q] = 1.0
    inner = np.sort(Lg.legroots(Lg.legder(c))) if q > 1 else np.array([])
    expect = np.concatenate([[0.0], 0.5 * (inner + 1.0), [1.0]])
    assert np.allclose(oracle.lobatto_nodes(q), expect, atol=1e-15)
    with pytest.raises(ValueError):
        oracle.lobatto_nodes(5)


def test_fe_profile_first_order_is_the_knot_profile(oracle):
    L, Ke = 37, 5
    p = oracle.level_pressures(L, 300.0, 1e-3)
    T_nodes = np.array([2500.0, 1900.0, 1500.0, 1300.0, 900.0, 600.0])
    a = oracle.temperature_profile_fe(p, Ke, 1, T_nodes, 300.0, 1e-3)
    b = oracle.temperature_profile(p, T_nodes, 300.0, 1e-3)
    assert np.allclose(a, b, rtol=1e-14)


@pytest.mark.parametrize("q", [2, 3, 4])
def test_fe_profile_reproduces_polynomials_and_is_continuous(oracle, q):
    L, Ke = 61, 3
    p_bot, p_top = 100.0, 1e-4
    p = oracle.level_pressures(L, p_bot, p_top)
    x = (np.log10(p) - np.log10(p_bot)) / (np.log10(p_top) - np.log10(p_bot))       # 0 (bottom) .. 1 (top)
    rng = np.random.default_rng(q)
    coef = rng.uniform(-1, 1, q + 1)
    poly = lambda s: 1500.0 + 400.0 * np.polyval(coef, s)                            # one global polynomial of degree q
    nodes = oracle.lobatto_nodes(q)
    dof_x = np.concatenate([[0.0]] + [(k + nodes[1:]) / Ke for k in range(Ke)])
    T = oracle.temperature_profile_fe(p, Ke, q, poly(dof_x), p_bot, p_top)
    assert np.allclose(T, poly(x), rtol=1e-12)
    # a constant stays constant (the Lagrange polynomials sum to one)
    assert np.allclose(oracle.temperature_profile_fe(p, Ke, q, np.full(Ke * q + 1, 777.0), p_bot, p_top), 777.0, rtol=1e-14)
    # continuity across element boundaries: evaluate just below / above the interface of elements 0 and 1
    dof = rng.uniform(500, 2500, Ke * q + 1)
    xb = 1.0 / Ke
    pp = p_bot * (p_top / p_bot) ** np.array([xb - 1e-9, xb, xb + 1e-9])
    Tb = oracle.temperature_profile_fe(pp, Ke, q, dof, p_bot, p_top)
    assert abs(Tb[0] - Tb[1]) < 1e-3 and abs(Tb[2] - Tb[1]) < 1e-3
    assert Tb[1] == pytest.approx(dof[q], rel=1e-12)                                  # the shared dof


def test_ratio_parametrisation(oracle):
    assert np.allclose(oracle.tp_dofs_from_ratios([1800.0, 1.0, 1.0, 1.0]), 1800.0)
    assert np.allclose(oracle.tp_dofs_from_ratios([2000.0, 0.5, 0.5, 0.5]), [2000.0, 1000.0, 500.0, 250.0])
    d = oracle.tp_dofs_from_ratios([1500.0, 0.9, 0.8, 1.1, 0.7])
    assert np.all(np.diff(d)[[0, 1, 3]] < 0) and d[3] > d[2]                          # b <= 1 monotone, b > 1 inversion


# ---------------------------------------------------------------------------- NEXT-3
def test_teff_of_a_black_body_is_its_temperature(oracle):
    T = 1350.0
    nu0, dnu, n = 1.0, 0.5, 120000                   # 1 .. 60000 cm^-1: x up to 64, the tail is < 1e-20
    nu = nu0 + dnu * np.arange(n)
    F = np.pi * planck(nu, T)
    assert oracle.teff(nu0, dnu, F, nu[0], nu[-1]) == pytest.approx(T, rel=2e-6)
    # constant flux over a window that cuts through grid cells
    Fc = np.full(n, 4.2e3)
    a, b = 1000.3, 2500.9
    assert oracle.teff(nu0, dnu, Fc, a, b) == pytest.approx((4.2e3 * (b - a) / SIGMA_SB) ** 0.25, rel=1e-10)   # 10-digit sigma_SB


# ---------------------------------------------------------------------------- NEXT-4
def test_cloud_optical_depth_distribution(oracle):
    p = oracle.level_pressures(40, 300.0, 1e-3)
    # fully inside the domain: the layer shares add up to tau_c, and vanish outside [p_top, p_bot]
    d = oracle.cloud_dtau(p, 3.7, 0.5, 1.0)          # 0.5 .. 1.0 bar
    assert d.sum() == pytest.approx(3.7, rel=1e-13) and np.all(d >= 0)
    lower, upper = p[:-1], p[1:]
    assert np.all(d[(upper >= 1.0) | (lower <= 0.5)] == 0.0)
    # uniform in pressure: a layer fully inside gets tau_c * dp / (p_bot - p_top)
    inside = (lower <= 1.0) & (upper >= 0.5)
    if inside.any():
        l = np.flatnonzero(inside)[0]
        assert d[l] == pytest.approx(3.7 * (lower[l] - upper[l]) / 0.5, rel=1e-12)
    # independent of the level grid
    assert oracle.cloud_dtau(oracle.level_pressures(173, 300.0, 1e-3), 3.7, 0.5, 1.0).sum() == pytest.approx(3.7, rel=1e-13)
    # half of the cloud below the bottom of the domain: half of the optical depth is dropped
    assert oracle.cloud_dtau(p, 2.0, 200.0, 1.0).sum() == pytest.approx(1.0, rel=1e-12)   # 200 .. 400 bar, domain ends at 300
    assert oracle.cloud_dtau(p, 2.0, 1e-5, 1.0).sum() == 0.0


def _tiny_setup():
    nNu, nT, nP = 64, 3, 3
    T_grid = np.array([300.0, 1500.0, 3000.0]); lp = np.array([-4.0, 0.0, 3.0])
    sigma = np.full((1, nT, nP, nNu), 1e-60, np.float32)           # gas opacity that never matters
    edges = np.linspace(5000.0, 5063.0, 9)
    return nNu, T_grid, lp, sigma, edges


def test_whole_path_grey_cloud_slab(oracle):
    """No gas opacity, a grey cloud of optical depth tau_c inside an isothermal stretch of the profile:
    I(mu) = B(T_0) e^{-tau_c/mu} + B(T_c) (1 - e^{-tau_c/mu}) exactly, whatever the level grid."""
    nNu, T_grid, lp, sigma, edges = _tiny_setup()
    Ke, A, L = 4, 4, 53
    T0, Tc = 2400.0, 900.0
    T_nodes = np.array([T0, 1600.0, Tc, Tc, Tc])                   # elements 2, 3 (p < 0.3 bar) are isothermal
    tau_c = 0.8
    params = np.concatenate([[5.0, 1.0], T_nodes, [-3.0], [np.log10(tau_c), np.log10(0.01), np.log10(2.0)]])
    r = oracle.forward(T_grid, lp, 5000.0, 1.0, sigma, None, L, 100.0, 1e-4, Ke + 1, A, 2.3, 0.17, 1.0,
                       edges, None, None, None, params[None, :], want_flux=True, want_spectra=False, want_logl=False,
                       tp_elements=Ke, tp_order=1, extras=oracle.EXTRA_GREY_CLOUD)
    mu, w = oracle.gauss_legendre_01(A)
    nu = 5000.0 + np.arange(nNu)
    I = planck(nu, T0)[None, :] * np.exp(-tau_c / mu)[:, None] + planck(nu, Tc)[None, :] * (-np.expm1(-tau_c / mu))[:, None]
    expect = 2 * np.pi * np.sum((w * mu)[:, None] * I, axis=0)
    assert np.allclose(r["flux_hr"][0], expect, rtol=2e-8)           # 10-digit c1, c2 in this test


def test_whole_path_distance_and_inflation(oracle):
    nNu, T_grid, lp, sigma, edges = _tiny_setup()
    sigma = sigma.copy(); sigma[:] = 3e-24
    base = np.array([4.5, 1.3, 2000.0, 700.0, -3.0])
    obs = np.full(8, 2.0e4); err = np.full(8, 5.0e2)
    kw = dict(want_flux=True)
    args = (T_grid, lp, 5000.0, 1.0, sigma, None, 30, 100.0, 1e-4, 2, 2, 2.3, 0.17, 9.0, edges, obs, err, None)
    r0 = oracle.forward(*args, base[None, :], **kw)
    # Eq. 9: F ~ 1/d^2
    r1 = oracle.forward(*args, np.concatenate([base, [3.0]])[None, :], extras=oracle.EXTRA_DISTANCE, **kw)
    assert np.allclose(r1["flux_hr"], r0["flux_hr"] / 9.0, rtol=1e-14)
    # both extras, in the documented order (d, eps); logL is Eq. 23 of the binned spectrum
    eps = 5.5
    r2 = oracle.forward(*args, np.concatenate([base, [3.0, eps]])[None, :],
                        extras=oracle.EXTRA_DISTANCE | oracle.EXTRA_ERROR_INFLATION, **kw)
    assert np.allclose(r2["spectra"], r1["spectra"], rtol=1e-15)
    assert r2["logl"][0] == pytest.approx(oracle.loglike_inflated(obs, err, r2["spectra"][0], eps), rel=1e-15)
    assert r2["logl"][0] > r1["logl"][0]                             # the model is far off: inflation helps
    # T_eff of an isothermal atmosphere over a window = the black-body value for that window
    riso = oracle.forward(*args[:6], 30, 100.0, 1e-4, 2, 8, 2.3, 0.17, 9.0, edges, obs, err, None,
                          np.array([[4.5, 1.3, 1100.0, 1100.0, -3.0]]), teff_range=(5000.0, 5063.0))
    nu = 5000.0 + np.arange(nNu)
    F = np.pi * planck(nu, 1100.0)
    expect = (np.sum(0.5 * (F[1:] + F[:-1])) / SIGMA_SB) ** 0.25
    assert riso["teff"][0] == pytest.approx(expect, rel=2e-9)        # 10-digit constants in this test
