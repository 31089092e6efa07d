"""Pins for the ORACLE (oracle/helios_oracle.c): closed forms, library routines,
brute-force quadrature of the paper's own continuous equations, invariants.

None of these retypes the oracle's formula and compares it with itself: each
compares with something the paper or the mathematics fixes independently
(DESIGN.md "Oracle pins" lists which plausible mistake each one catches).
Citations are to /root/reference/PAPER.md line numbers.
"""
import math
import os

import mpmath
import numpy as np
import pytest
from scipy import integrate, special

import workloads as W

H = 6.62607015e-27
C = 2.99792458e10
KB = 1.380649e-16
MU = 1.66053906660e-24
SIGMA_SB = 5.670374419e-5
C2 = H * C / KB


# --------------------------------------------------------------------------
# O0: grid, profile, mixing ratios
# --------------------------------------------------------------------------
def test_level_pressures_equidistant_in_log_p(oracle):
    # PAPER.md:55 "distributed equidistantly in log p-space"
    p = oracle.level_pressures(20, 300.0, 1e-3)
    assert p[0] == 300.0 and p[-1] == pytest.approx(1e-3, rel=1e-14)
    r = p[1:] / p[:-1]
    assert np.allclose(r, r[0], rtol=1e-13)
    assert np.all(np.diff(p) < 0)          # level 0 is the bottom


def test_temperature_profile_piecewise_linear_in_log_p(oracle):
    # PAPER.md:178-190 first-order elements: interpolant passes through the nodes,
    # is linear in log p inside an element, continuous across elements.
    K, L = 6, 101                            # 20 levels per element -> knots fall on levels
    knots = np.array([2500.0, 2100.0, 1500.0, 1400.0, 900.0, 600.0])
    p = oracle.level_pressures(L, 300.0, 1e-3)
    T = oracle.temperature_profile(p, knots, 300.0, 1e-3)
    assert np.allclose(T[::20], knots, rtol=1e-12)
    # second difference in log p vanishes inside each element
    for e in range(K - 1):
        seg = T[20 * e:20 * e + 21]
        assert np.allclose(np.diff(seg, 2), 0.0, atol=1e-9)
    # mid-element value is the mean of the two nodes
    assert T[10] == pytest.approx(0.5 * (knots[0] + knots[1]), rel=1e-12)
    # config 0's 2-knot case: 2000 K (bottom) -> 800 K (top)
    T2 = oracle.temperature_profile(oracle.level_pressures(20, 300.0, 1e-3), [2000.0, 800.0], 300.0, 1e-3)
    assert T2[0] == pytest.approx(2000.0) and T2[-1] == pytest.approx(800.0)
    assert np.allclose(np.diff(T2), np.diff(T2)[0])


def test_mixing_ratios_fill_with_h2_he(oracle):
    # PAPER.md:484
    x, h2, he = oracle.mixing_ratios([-3.0, -4.0, -2.5], 0.17)
    assert np.allclose(x, [1e-3, 1e-4, 10 ** -2.5])
    assert x.sum() + h2 + he == pytest.approx(1.0, rel=1e-15)
    assert he / h2 == pytest.approx(0.17, rel=1e-14)


# --------------------------------------------------------------------------
# O1: interpolation  (P1, P2, P3)
# --------------------------------------------------------------------------
def _rand_table(nT=4, nP=5, nNu=7, seed=0):
    rng = np.random.default_rng(seed)
    return (10.0 ** rng.uniform(-26, -20, (nT, nP, nNu))).astype(np.float32)


def test_interp_at_nodes_returns_node_values_exactly(oracle):
    T_grid = np.array([500.0, 1000.0, 1500.0, 2000.0])
    lp_grid = np.array([-3.0, -1.0, 0.0, 1.0, 2.5])
    tab = _rand_table()
    for iT, T in enumerate(T_grid):
        for ip, lp in enumerate(lp_grid):
            s, cl = oracle.interp_sigma(tab, T_grid, lp_grid, T, lp)
            assert not cl
            assert np.array_equal(s, tab[iT, ip].astype(np.float64))


def test_interp_reproduces_bilinear_function(oracle):
    # sigma = a + b T + c lp + d T lp is reproduced by a bilinear interpolant on
    # ANY rectilinear grid; fails for a transposed axis, swapped weights, or
    # interpolation in p instead of log10 p.
    T_grid = np.array([500.0, 1000.0, 1600.0, 2000.0])
    lp_grid = np.array([-3.0, -1.0, 1.0, 2.5])
    a, b, c, d = 8.0, 2e-3, 0.75, 5e-4
    nu_fac = np.array([1.0, 2.0, 4.0])
    TT, PP = np.meshgrid(T_grid, lp_grid, indexing="ij")
    tab = ((a + b * TT + c * PP + d * TT * PP)[:, :, None] * nu_fac).astype(np.float32)
    rng = np.random.default_rng(1)
    for _ in range(50):
        T = rng.uniform(500, 2000)
        lp = rng.uniform(-3, 2.5)
        s, cl = oracle.interp_sigma(tab, T_grid, lp_grid, T, lp)
        exact = (a + b * T + c * lp + d * T * lp) * nu_fac
        assert not cl
        assert np.allclose(s, exact, rtol=3e-7)   # fp32 storage of the nodes


def test_interp_clamps_outside_grid(oracle):
    T_grid = np.array([500.0, 1000.0, 1500.0, 2000.0])
    lp_grid = np.array([-3.0, -1.0, 0.0, 1.0, 2.5])
    tab = _rand_table()
    s, cl = oracle.interp_sigma(tab, T_grid, lp_grid, 3000.0, 5.0)
    assert cl and np.array_equal(s, tab[-1, -1].astype(np.float64))
    s, cl = oracle.interp_sigma(tab, T_grid, lp_grid, 100.0, -1.0)
    assert cl and np.array_equal(s, tab[0, 1].astype(np.float64))
    i, w, cl = oracle.cell(T_grid, 1000.0)
    assert (i, w, cl) == (1, 0.0, False)
    i, w, cl = oracle.cell(T_grid, 2000.0)
    assert (i, w, cl) == (2, 1.0, False)


def test_cia_interp_linear_in_T(oracle):
    T_grid = np.array([100.0, 400.0, 1000.0])
    tab = np.array([[1.0, 10.0], [4.0, 40.0], [10.0, 100.0]], dtype=np.float32)  # = T/100 * (1, 10)
    a = oracle.interp_cia(tab, T_grid, 700.0)
    assert np.allclose(a, [7.0, 70.0], rtol=1e-15)
    assert np.array_equal(oracle.interp_cia(tab, T_grid, 400.0), [4.0, 40.0])


# --------------------------------------------------------------------------
# O2/O3: absorption coefficient and optical depth  (P5, P6)
# --------------------------------------------------------------------------
def test_number_density_at_stp_is_loschmidt(oracle):
    # 1 atm, 0 C: n = n_L = 2.6867801118e19 cm^-3 (CODATA 2018, exact SI) -- pins k_B and the bar->cgs factor
    assert oracle.number_density(1.01325, 273.15) == pytest.approx(2.6867801118e19, rel=1e-10)


def test_chi_cia_at_one_amagat(oracle):
    # at n = n_L the CIA term is x_H2 (x_H2 a_HH + x_He a_HHe) exactly; line term n * sum x sigma
    n = oracle.number_density(1.01325, 273.15)
    chi = oracle.chi_level([0.0], [np.zeros(2)], 0.8, 0.1, [np.array([2.0, 4.0]), np.array([10.0, 20.0])], n)
    assert np.allclose(chi, [0.8 * (0.8 * 2 + 0.1 * 10), 0.8 * (0.8 * 4 + 0.1 * 20)], rtol=1e-7)
    chi2 = oracle.chi_level([0.0], [np.zeros(2)], 0.8, 0.1, [np.array([2.0, 4.0]), np.array([10.0, 20.0])], 3 * n)
    assert np.allclose(chi2, 9 * chi, rtol=1e-14)            # quadratic in density
    chi3 = oracle.chi_level([1e-3, 2e-3], [np.array([1e-20, 0.0]), np.array([0.0, 1e-21])], 0, 0, [], 1e18)
    assert np.allclose(chi3, [1e18 * 1e-23, 1e18 * 2e-24], rtol=1e-14)


def _column_tau(oracle, L, T_knots, sigma_x, g, mmw=2.3, p_bot=300.0, p_top=1e-3):
    p = oracle.level_pressures(L, p_bot, p_top)
    T = oracle.temperature_profile(p, T_knots, p_bot, p_top)
    chi = np.array([oracle.number_density(p[l], T[l]) * sigma_x for l in range(L)])
    tot = 0.0
    per_layer = []
    for l in range(L - 1):
        dz = oracle.layer_thickness(T[l], T[l + 1], p[l], p[l + 1], mmw, g)
        d = oracle.layer_dtau([chi[l]], [chi[l + 1]], dz)[0]
        per_layer.append(d)
        tot += d
    return p, T, np.array(per_layer), tot


def test_total_optical_depth_converges_to_hydrostatic_column(oracle):
    # Continuous problem: dtau = n sigma x dz and dp = -n mmw m_u g dz, so for
    # constant sigma*x the column is sigma x (p_bot - p_top)/(mmw m_u g) for ANY T(p).
    # The discretisation (R5) must converge to it, second order in d ln p.
    sigma_x, g, mmw = 2.5e-26, 1e5, 2.3
    exact = sigma_x * (300.0 - 1e-3) * 1e6 / (mmw * MU * g)
    errs = []
    for L in (50, 100, 200, 400):
        _, _, _, tot = _column_tau(oracle, L, [2400.0, 1900.0, 800.0, 700.0], sigma_x, g, mmw)
        errs.append(abs(tot / exact - 1.0))
    assert errs[-1] < 1e-4
    for a, b in zip(errs[:-1], errs[1:]):
        assert 3.0 < a / b < 5.0                               # second order


def test_isothermal_layer_dtau_closed_form(oracle):
    # T cancels for isothermal layers: dtau_l = sigma x (p_l + p_{l+1}) ln(p_l/p_{l+1}) / (2 mmw m_u g)
    sigma_x, g, mmw = 3e-25, 10 ** 4.5, 2.3
    for T0 in (700.0, 1900.0):
        p, T, per_layer, _ = _column_tau(oracle, 20, [T0, T0], sigma_x, g, mmw)
        pc = p * 1e6
        ref = sigma_x * (pc[:-1] + pc[1:]) * np.log(pc[:-1] / pc[1:]) / (2 * mmw * MU * g)
        assert np.allclose(per_layer, ref, rtol=1e-13)


# --------------------------------------------------------------------------
# O4: Planck, quadrature, short characteristics  (P7 - P13)
# --------------------------------------------------------------------------
def test_planck_limits_and_stefan_boltzmann(oracle):
    T = 1234.0
    # Wien limit x >> 1: B -> 2hc^2 nu^3 exp(-x);  Rayleigh-Jeans x << 1: B -> 2 c k T nu^2
    nu = 40.0 * T / C2
    assert oracle.planck(nu, T) == pytest.approx(2 * H * C * C * nu ** 3 * math.exp(-40.0), rel=1e-15)
    nu = 1e-6 * T / C2
    assert oracle.planck(nu, T) == pytest.approx(2 * C * KB * T * nu ** 2, rel=1e-6)
    # integral over wavenumber of pi B = sigma_SB T^4 (ties h, c, k_B together)
    val, _ = integrate.quad(lambda v: oracle.planck(v, T), 1e-9, 60 * T / C2, epsabs=0, epsrel=1e-12, limit=400)
    assert math.pi * val == pytest.approx(SIGMA_SB * T ** 4, rel=1e-9)
    # Wien displacement in wavenumber form: maximum at x = 2.821439...
    xs = np.linspace(2.7, 2.95, 2001)
    b = [oracle.planck(x * T / C2, T) for x in xs]
    assert xs[int(np.argmax(b))] == pytest.approx(2.821439, abs=2e-4)


def test_gauss_legendre_nodes(oracle):
    golden = np.loadtxt(os.path.join(W.golden_dir(), "gauss_legendre_n2.txt"), comments="#")
    mu, w = oracle.gauss_legendre_01(2)
    assert np.allclose(mu, golden[:, 0], atol=1e-10) and np.allclose(w, golden[:, 1], atol=1e-15)
    for n in (1, 2, 3, 4, 8, 16, 32):
        mu, w = oracle.gauss_legendre_01(n)
        x, ww = np.polynomial.legendre.leggauss(n)
        assert np.allclose(mu, 0.5 * (x + 1), atol=1e-15)
        assert np.allclose(w, 0.5 * ww, atol=1e-15)
        assert np.sum(w * mu) == pytest.approx(0.5, rel=1e-14)
        if n >= 2:
            assert np.sum(w * mu * mu) == pytest.approx(1.0 / 3.0, rel=1e-14)


def test_sc_coefficients_against_eq1_quadrature(oracle):
    # One layer of Eq. 1 with a source linear in optical depth:
    # contribution = int_0^D [S_i + (S_{i-1}-S_i) t/D] e^{-t} dt  (t = path optical depth from the
    # downwind level i towards the upwind level i-1) must equal beta S_i + gamma S_{i-1}.
    for D in (1e-6, 5e-4, 0.999e-3, 1.001e-3, 0.02, 0.7, 3.0, 40.0):
        e, beta, gamma = oracle.sc_coefficients(D)
        mp = mpmath.mpf
        mpmath.mp.dps = 40
        b_ref = mpmath.quad(lambda t: (1 - t / mp(D)) * mpmath.e ** (-t), [0, mp(D)])
        g_ref = mpmath.quad(lambda t: (t / mp(D)) * mpmath.e ** (-t), [0, mp(D)])
        assert beta == pytest.approx(float(b_ref), rel=1e-12)
        assert gamma == pytest.approx(float(g_ref), rel=1e-12)
        assert e == pytest.approx(float(mpmath.e ** (-mp(D))), rel=1e-15)
        assert beta + gamma == pytest.approx(-math.expm1(-D), rel=1e-12)   # reading R8
    assert oracle.sc_coefficients(0.0) == (1.0, 0.0, 0.0)


def test_rt_isothermal_gives_pi_B(oracle):
    # north_star closed form: isothermal atmosphere, any opacities -> F+ = pi B
    rng = np.random.default_rng(3)
    for A in (1, 2, 4, 8):
        mu, w = oracle.gauss_legendre_01(A)
        dtau = 10.0 ** rng.uniform(-6, 2, 49)
        S = np.full(50, 7.25)
        assert oracle.flux_one_nu(S, dtau, mu, w) == pytest.approx(math.pi * 7.25, rel=1e-13)


def test_rt_zero_opacity_gives_bottom_planck(oracle):
    # north_star closed form; also catches the Delta -> 0 cancellation bug
    mu, w = oracle.gauss_legendre_01(2)
    S = np.linspace(9.0, 1.0, 30)
    assert oracle.flux_one_nu(S, np.zeros(29), mu, w) == pytest.approx(math.pi * 9.0, rel=1e-14)
    assert oracle.flux_one_nu(S, np.full(29, 1e-12), mu, w) == pytest.approx(math.pi * 9.0, rel=1e-10)


def test_rt_linear_source_thick_bottom(oracle):
    # S = a + b tau, optically thick bottom: F+ = pi (a + 2b/3), exact for n >= 2 angles
    # (Eddington-Barbier); n = 1 gives pi (a + b/2).
    a, b = 1.3, 0.4
    tau = np.concatenate([[0.0], np.cumsum(10.0 ** np.linspace(-3, 1.2, 80))])   # top -> bottom
    S_top_down = a + b * tau
    S = S_top_down[::-1].copy()                 # level 0 = bottom
    dtau = np.diff(tau)[::-1].copy()            # dtau[l] between level l and l+1
    # thick bottom: the isothermal continuation below tau_max is invisible (e^{-tau_max/mu} ~ 0)
    for A in (2, 4, 8):
        mu, w = oracle.gauss_legendre_01(A)
        assert oracle.flux_one_nu(S, dtau, mu, w) == pytest.approx(math.pi * (a + 2 * b / 3), rel=1e-12)
    mu, w = oracle.gauss_legendre_01(1)
    assert oracle.flux_one_nu(S, dtau, mu, w) == pytest.approx(math.pi * (a + b / 2), rel=1e-12)


def _exact_flux_piecewise_linear(S, dtau):
    """Eq. 3 integrated exactly for a source piecewise linear in tau,
    isothermal below the bottom level: F = 2 pi int_0^inf S(t) E_2(t) dt."""
    L = len(S)
    tau = np.zeros(L)
    for l in range(L - 2, -1, -1):
        tau[l] = tau[l + 1] + dtau[l]
    F = S[0] * special.expn(3, tau[0])
    for l in range(L - 1):
        ta, tb, Sa, Sb = tau[l + 1], tau[l], S[l + 1], S[l]      # a = upper, b = lower
        if tb == ta:
            continue
        m = (Sb - Sa) / (tb - ta)
        F += Sa * special.expn(3, ta) - Sb * special.expn(3, tb) + m * (special.expn(4, ta) - special.expn(4, tb))
    return 2 * math.pi * F


def test_rt_converges_to_schwarzschild_milne(oracle):
    # The n-angle short-characteristics flux converges to the exact angular integral
    # (Eq. 3) of the same piecewise-linear source; 2 angles = "four-stream".
    rng = np.random.default_rng(5)
    L = 30
    S = np.sort(rng.uniform(1.0, 10.0, L))[::-1].copy()
    dtau = 10.0 ** rng.uniform(-2.5, 0.5, L - 1)
    exact = _exact_flux_piecewise_linear(S, dtau)
    # cross-check the closed form itself by brute-force quadrature of Eq. 3
    tau = np.concatenate([np.cumsum(dtau[::-1])[::-1], [0.0]])
    def Sfun(t):
        return np.interp(t, tau[::-1], S[::-1]) if t <= tau[0] else S[0]
    brute, _ = integrate.quad(lambda t: Sfun(t) * special.expn(2, t), 0, 60.0, points=sorted(tau), limit=2000,
                              epsabs=0, epsrel=1e-11)
    assert 2 * math.pi * brute == pytest.approx(exact, rel=1e-8)
    errs = {}
    for A in (2, 4, 8, 32):
        mu, w = oracle.gauss_legendre_01(A)
        errs[A] = abs(oracle.flux_one_nu(S, dtau, mu, w) / exact - 1.0)
    assert errs[2] < 3e-3 and errs[4] < 1e-4 and errs[8] < 3e-6 and errs[32] < 1e-10
    assert errs[2] > errs[4] > errs[8] > errs[32]


def test_rt_flux_bounded_by_source_extremes(oracle):
    rng = np.random.default_rng(7)
    mu, w = oracle.gauss_legendre_01(4)
    for _ in range(20):
        S = rng.uniform(0.1, 5.0, 40)
        dtau = 10.0 ** rng.uniform(-8, 3, 39)
        F = oracle.flux_one_nu(S, dtau, mu, w) / math.pi
        assert S.min() * (1 - 1e-12) <= F <= S.max() * (1 + 1e-12)


# --------------------------------------------------------------------------
# O5: instrument profile  (P14)
# --------------------------------------------------------------------------
def test_convolve_closed_forms(oracle):
    n, nu0, dnu = 400, 1000.0, 0.5
    nu = nu0 + dnu * np.arange(n)
    sig = np.full(n, 3.0)
    assert np.allclose(oracle.convolve(nu0, dnu, np.full(n, 2.5), sig), 2.5, rtol=1e-14)
    lin = 1.0 + 0.01 * (nu - nu0)
    out = oracle.convolve(nu0, dnu, lin, sig)
    inner = slice(40, n - 40)                                  # 5 sigma = 15 cm^-1 = 30 points
    assert np.allclose(out[inner], lin[inner], rtol=1e-13)
    # delta spike -> normalised, truncated Gaussian samples
    spike = np.zeros(n)
    spike[200] = 1.0
    out = oracle.convolve(nu0, dnu, spike, sig)
    d = nu - nu[200]
    g = np.exp(-d ** 2 / (2 * 9.0))
    g[np.abs(d) > 15.0] = 0.0
    assert np.allclose(out, g / g.sum(), rtol=1e-12, atol=1e-300)
    assert out[200 + 30] > 0.0 and out[200 + 31] == 0.0        # |x - nu| = 5 sigma is included
    # truncated mass is negligible: 2(1 - Phi(5)) = 5.7e-7
    assert abs(1.0 - g.sum() * dnu / (3.0 * math.sqrt(2 * math.pi))) < 1e-6
    # sigma = 0 / no profile -> identity
    rng = np.random.default_rng(0)
    F = rng.uniform(1, 2, n)
    assert np.array_equal(oracle.convolve(nu0, dnu, F, np.zeros(n)), F)
    assert np.array_equal(oracle.convolve(nu0, dnu, F, None), F)
    # sigma is taken at the OUTPUT point (wavelength-dependent sigma)
    sig2 = np.where(np.arange(n) < 200, 1.0, 4.0)
    out2 = oracle.convolve(nu0, dnu, spike, sig2)
    assert out2[190] == pytest.approx(math.exp(-25.0 / 2.0) / np.exp(-(dnu * np.arange(-10, 11)) ** 2 / 2.0).sum(), rel=1e-12)
    # ... probed right at the step, where a one-point shift of the sigma index changes the answer:
    # point 199 still has sigma = 1 (window +-10 points), point 200 is the first with sigma = 4 (+-40 points)
    assert out2[199] == pytest.approx(math.exp(-0.25 / 2.0) / np.exp(-(dnu * np.arange(-10, 11)) ** 2 / 2.0).sum(), rel=1e-12)
    assert out2[200] == pytest.approx(1.0 / np.exp(-(dnu * np.arange(-40, 41)) ** 2 / 32.0).sum(), rel=1e-12)
    assert out2[201] == pytest.approx(math.exp(-0.25 / 32.0) / np.exp(-(dnu * np.arange(-40, 41)) ** 2 / 32.0).sum(), rel=1e-12)


# --------------------------------------------------------------------------
# O6: binning  (P15)
# --------------------------------------------------------------------------
def test_bin_closed_forms(oracle):
    n, nu0, dnu = 101, 4000.0, 1.0
    nu = nu0 + dnu * np.arange(n)
    edges = np.array([4000.0, 4010.0, 4033.3, 4033.9, 4060.25, 4100.0])   # incl. a bin inside one cell
    assert np.allclose(oracle.bin_spectrum(nu0, dnu, np.full(n, 3.0), edges), 3.0, rtol=1e-14)
    lin = 2.0 + 0.05 * (nu - nu0)
    centres = 0.5 * (edges[:-1] + edges[1:])
    assert np.allclose(oracle.bin_spectrum(nu0, dnu, lin, edges), 2.0 + 0.05 * (centres - nu0), rtol=1e-13)
    rng = np.random.default_rng(2)
    F = rng.uniform(1.0, 2.0, n)
    M = oracle.bin_spectrum(nu0, dnu, F, edges)
    # conservation: sum M_j width_j = trapezoid integral over the whole grid
    assert np.sum(M * np.diff(edges)) == pytest.approx(np.trapezoid(F, nu), rel=1e-13)
    # brute force: integrate the piecewise-linear interpolant with a library quadrature
    for j in range(len(edges) - 1):
        xs = np.unique(np.concatenate([[edges[j], edges[j + 1]], nu[(nu > edges[j]) & (nu < edges[j + 1])]]))
        ref = np.trapezoid(np.interp(xs, nu, F), xs) / (edges[j + 1] - edges[j])
        assert M[j] == pytest.approx(ref, rel=1e-13)


# --------------------------------------------------------------------------
# O7: likelihood  (P16)
# --------------------------------------------------------------------------
def test_loglike_closed_forms(oracle):
    rng = np.random.default_rng(4)
    D = rng.uniform(1, 2, 30)
    err = rng.uniform(0.01, 0.1, 30)
    base = oracle.loglike(D, err, D)
    assert base == pytest.approx(-0.5 * np.sum(np.log(2 * math.pi * err ** 2)), rel=1e-14)
    M = D.copy()
    M[7] += 3.0 * err[7]
    assert oracle.loglike(D, err, M) == pytest.approx(base - 4.5, rel=1e-13)
    # it is the log of a product of normal densities (Eq. 19)
    from scipy.stats import norm
    M = D + rng.normal(0, 0.05, 30)
    assert oracle.loglike(D, err, M) == pytest.approx(np.sum(norm.logpdf(D, loc=M, scale=err)), rel=1e-13)


# --------------------------------------------------------------------------
# Whole path  (P17, P18, P19)
# --------------------------------------------------------------------------
def _grey_setup(nNu=3, nu0=2000.0, dnu=3500.0, sigma0=2.5e-23):
    T_grid = np.array([100.0, 1500.0, 3000.0])
    lp_grid = np.array([-4.0, 0.0, 3.0])
    sigma = np.full((1, 3, 3, nNu), sigma0, dtype=np.float32)
    return T_grid, lp_grid, sigma


def test_whole_path_isothermal(oracle):
    # Isothermal atmosphere through O0-O7: F = f * flux_const * pi * B_nu(T) whatever the opacity;
    # binned spectrum = conv+bin of that (stage functions pinned above).
    wl = W.make_workload(0)
    cfg = wl.cfg
    T0 = 1350.0
    params = np.array([[4.7, 1.7, T0, T0, -3.3]])
    edges, inst = W.observation_grid(cfg)
    r = oracle.forward(wl.T_grid, wl.log10p_grid, cfg.nu0, cfg.dnu, wl.sigma, None, cfg.n_levels,
                       cfg.p_bottom_bar, cfg.p_top_bar, 2, 2, 2.3, 0.17, 0.25, edges, None, None, inst,
                       params, want_flux=True, want_spectra=True, want_logl=False)
    nu = cfg.nu0 + cfg.dnu * np.arange(cfg.n_nu)
    x = C2 * nu / T0
    planck = 2 * H * C * C * nu ** 3 / np.expm1(x)
    ref = 1.7 * 0.25 * math.pi * planck
    assert np.allclose(r["flux_hr"][0], ref, rtol=1e-12)
    ref_binned = oracle.bin_spectrum(cfg.nu0, cfg.dnu, oracle.convolve(cfg.nu0, cfg.dnu, ref, inst), edges)
    assert np.allclose(r["spectra"][0], ref_binned, rtol=1e-12)


def test_whole_path_converges_to_continuous_solution(oracle):
    # Grey opacity sigma0*x: the continuous problem has tau(p) = sigma0 x (p - p_top)/(mmw m_u g)
    # (hydrostatic, any T(p)), S = B_nu(T(p)), semi-infinite isothermal below p_bot:
    #   F = 2 pi [ int_0^tau_b B(T(p(t))) E_2(t) dt + B(T_bot) E_3(tau_b) ]        (Eq. 3)
    # The discretised path (levels, trapezoid dtau, linear-source short characteristics,
    # Gauss angles) must converge to it.  Pins n, dz, dtau wiring, level order, Planck, RT.
    T_grid, lp_grid, sigma = _grey_setup()
    x_vmr, logg, mmw = 1e-3, 5.0, 2.3
    p_bot, p_top, T_bot, T_top = 300.0, 1e-3, 2200.0, 600.0
    kappa_m = 2.5e-23 * x_vmr / (mmw * MU * 10 ** logg)        # per dyn cm^-2
    tau_b = kappa_m * (p_bot - p_top) * 1e6
    nus = 2000.0 + 3500.0 * np.arange(3)

    def exact(nu):
        def S(t):
            p = p_top * 1e6 + t / kappa_m
            lp = math.log10(p / 1e6)
            T = T_bot + (T_top - T_bot) * (lp - math.log10(p_bot)) / (math.log10(p_top) - math.log10(p_bot))
            return 2 * H * C * C * nu ** 3 / math.expm1(C2 * nu / T)
        val, _ = integrate.quad(lambda t: S(t) * special.expn(2, t), 0.0, tau_b, limit=1000,
                                points=[1e-6, 1e-4, 1e-2, 1.0], epsabs=0, epsrel=1e-11)
        return 2 * math.pi * (val + S(tau_b) * special.expn(3, tau_b))

    ref = np.array([exact(nu) for nu in nus])
    params = np.array([[logg, 1.0, T_bot, T_top, math.log10(x_vmr)]])
    errs = []
    for L in (50, 100, 200, 400):
        r = oracle.forward(T_grid, lp_grid, 2000.0, 3500.0, sigma, None, L, p_bot, p_top, 2, 16,
                           mmw, 0.17, 1.0, np.array([2000.0, 9000.0]), None, None, None, params,
                           want_flux=True, want_spectra=False, want_logl=False)
        errs.append(np.max(np.abs(r["flux_hr"][0] / ref - 1.0)))
    assert errs[-1] < 1e-4
    for a, b in zip(errs[:-1], errs[1:]):
        assert a / b > 3.0                                       # ~second order


def test_whole_path_cia_only_grey(oracle):
    # CIA-only atmosphere, constant alpha, isothermal T -> flux pi B; and non-isothermal thin limit:
    # with alpha = 0 everywhere the flux is the bottom Planck flux (zero-opacity closed form via O0-O4).
    T_grid = np.array([100.0, 1500.0, 3000.0])
    lp_grid = np.array([-4.0, 0.0, 3.0])
    sigma = np.zeros((1, 3, 3, 2), dtype=np.float32)
    cia = np.zeros((2, 3, 2), dtype=np.float32)
    params = np.array([[4.5, 2.0, 1800.0, 700.0, -30.0]])
    r = oracle.forward(T_grid, lp_grid, 3000.0, 2000.0, sigma, cia, 40, 300.0, 1e-3, 2, 2, 2.3, 0.17, 1.0,
                       np.array([3000.0, 5000.0]), None, None, None, params, want_flux=True,
                       want_spectra=False, want_logl=False)
    nu = np.array([3000.0, 5000.0])
    ref = 2.0 * math.pi * 2 * H * C * C * nu ** 3 / np.expm1(C2 * nu / 1800.0)
    assert np.allclose(r["flux_hr"][0], ref, rtol=1e-13)


def test_batch_permutation_and_independence(oracle):
    wl = W.make_workload(0)
    cfg = wl.cfg
    rng = np.random.default_rng(11)
    params = np.column_stack([rng.uniform(4, 5.5, 5), rng.uniform(0.5, 2, 5),
                              rng.uniform(1500, 2000, 5), rng.uniform(500, 1000, 5), rng.uniform(-6, -2, 5)])
    obs = np.full(cfg.n_bins, 1e5)
    err = np.full(cfg.n_bins, 2e3)
    kw = dict(obs=obs, obs_err=err)
    full = oracle.forward_workload(wl, params=params, **kw)
    perm = np.array([3, 0, 4, 1, 2])
    shuf = oracle.forward_workload(wl, params=params[perm], **kw)
    assert np.array_equal(shuf["spectra"], full["spectra"][perm])
    assert np.array_equal(shuf["logl"], full["logl"][perm])
    single = oracle.forward_workload(wl, params=params[2:3], **kw)
    assert np.array_equal(single["spectra"][0], full["spectra"][2])
    one_thread = oracle.forward_workload(wl, params=params, n_threads=1, **kw)
    assert np.array_equal(one_thread["logl"], full["logl"])


def test_outputs_bounded_by_planck_extremes(oracle):
    # every I is a convex combination of level sources -> F/(pi f) in [B(T_min), B(T_max)]
    wl = W.make_workload(0)
    cfg = wl.cfg
    r = oracle.forward_workload(wl, want_flux=True, want_logl=False)
    nu = cfg.nu0 + cfg.dnu * np.arange(cfg.n_nu)
    b = lambda T: 2 * H * C * C * nu ** 3 / np.expm1(C2 * nu / T)
    F = r["flux_hr"][0] / math.pi
    assert np.all(F >= b(800.0) * (1 - 1e-12)) and np.all(F <= b(2000.0) * (1 + 1e-12))
    assert r["n_clamped"] == 0


def test_nonfinite_parameters(oracle):
    wl = W.make_workload(0)
    params = np.tile(wl.params[0], (3, 1))
    params[1, 2] = np.nan
    obs = np.full(wl.cfg.n_bins, 1e5)
    err = np.full(wl.cfg.n_bins, 2e3)
    r = oracle.forward_workload(wl, params=params, obs=obs, obs_err=err)
    assert np.isnan(r["spectra"][1]).all() and r["logl"][1] == -np.inf
    assert np.array_equal(r["spectra"][0], r["spectra"][2]) and np.isfinite(r["logl"][[0, 2]]).all()


def test_unphysical_parameters_are_rejected(oracle):
    # DESIGN.md R31 [paper silent]: finite but unphysical vectors are rejected like non-finite ones
    # (logL = -inf, NaN spectra) instead of producing NaN or finite garbage for the sampler.
    wl = W.make_workload(0)
    good = wl.params[0]
    cases = {"vmr_sum_gt_1": (4, 0.2), "negative_f": (1, -1.0), "g_overflow": (0, 400.0), "negative_T": (3, -10.0)}
    params = np.tile(good, (len(cases) + 1, 1))
    for i, (col, val) in enumerate(cases.values()):
        params[i + 1, col] = val
    obs = np.full(wl.cfg.n_bins, 1e5)
    err = np.full(wl.cfg.n_bins, 2e3)
    r = oracle.forward_workload(wl, params=params, obs=obs, obs_err=err, want_flux=True)
    assert np.isfinite(r["logl"][0]) and np.isfinite(r["spectra"][0]).all()
    for i, name in enumerate(cases):
        assert r["logl"][i + 1] == -np.inf, name
        assert np.isnan(r["spectra"][i + 1]).all() and np.isnan(r["flux_hr"][i + 1]).all(), name
    # f = 0 and VMRs summing to exactly <= 1 are legal
    edge = np.tile(good, (2, 1))
    edge[0, 1] = 0.0
    edge[1, 4] = math.log10(0.999)
    r = oracle.forward_workload(wl, params=edge, obs=obs, obs_err=err)
    assert np.isfinite(r["logl"]).all() and np.all(r["spectra"][0] == 0.0)
    # extras: d <= 0
    p = np.concatenate([good, [0.0]])[None, :]
    r = oracle.forward_workload(wl, params=p, obs=obs, obs_err=err, extras=1)
    assert r["logl"][0] == -np.inf


def test_clamp_count(oracle):
    wl = W.make_workload(0)
    params = wl.params.copy()
    params[0, 2] = 2600.0        # bottom knot above the 2000 K table edge
    r = oracle.forward_workload(wl, params=params, want_logl=False)
    p = oracle.level_pressures(wl.cfg.n_levels, 300.0, 1e-3)
    T = oracle.temperature_profile(p, params[0, 2:4], 300.0, 1e-3)
    assert r["n_clamped"] == int(np.sum(T > 2000.0))


@pytest.mark.parametrize("sanitizer", ["undefined", "address"])
def test_oracle_is_clean_under_sanitizers(tmp_path, sanitizer):
    """The oracle built with -fsanitize=undefined -fno-sanitize-recover (no signed overflow, bad shifts, misaligned
    accesses, NaN->int conversions ...) and with -fsanitize=address (no heap / stack / global out-of-bounds access,
    no use after free) runs the tiny workload, the NEXT rows and a finite-element case without tripping."""
    import os, subprocess, sys, textwrap
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    so = tmp_path / f"liboracle_{sanitizer}.so"
    flags = ["-fsanitize=undefined", "-fno-sanitize-recover=undefined"] if sanitizer == "undefined" else ["-fsanitize=address"]
    r = subprocess.run(["gcc", "-O1", "-g", "-std=c99", "-fopenmp", "-fPIC", "-shared"] + flags +
                       ["-o", str(so), os.path.join(root, "oracle", "helios_oracle.c"), "-lm"], capture_output=True, text=True)
    if r.returncode != 0:
        pytest.skip(f"gcc has no usable -fsanitize={sanitizer} runtime here: " + r.stderr[-200:])
    env = dict(os.environ)
    if sanitizer == "address":          # the runtime must be the first library of the (uninstrumented) interpreter
        rt = subprocess.run(["gcc", "-print-file-name=libasan.so"], capture_output=True, text=True).stdout.strip()
        if not os.path.isabs(rt) or not os.path.exists(rt):
            pytest.skip("libasan.so not found")
        env["LD_PRELOAD"] = rt
        env["ASAN_OPTIONS"] = "detect_leaks=0:abort_on_error=0:exitcode=66"      # the interpreter's own leaks are not ours
    code = textwrap.dedent(f"""
        import sys; sys.path.insert(0, {root!r})
        import numpy as np, oracle.binding as ob
        ob._SO = {str(so)!r}; ob.build = lambda force=False: ob._SO
        import oracle, workloads
        wl = workloads.make_workload(0)
        r = oracle.forward_workload(wl, want_flux=True, teff_range=(4000.0, 4999.0))
        p = np.concatenate([wl.params[0], [2.0, 4.0, -1.0, -1.0, 0.0]])[None, :]
        r2 = oracle.forward_workload(wl, params=p, extras=7)
        p3 = np.concatenate([wl.params[0, :2], [2000.0, 0.8, 0.9, 0.95, 0.7], wl.params[0, 4:]])[None, :]
        r3 = oracle.forward_workload(wl, params=p3, tp_elements=2, tp_order=2, tp_ratio=True)
        assert np.isfinite(r["logl"]).all() and np.isfinite(r2["logl"]).all() and np.isfinite(r3["logl"]).all()
        print("ok")
    """)
    out = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True, timeout=300, env=env)
    assert out.returncode == 0 and "ok" in out.stdout, out.stderr[-2000:]
    assert "runtime error" not in out.stderr and "AddressSanitizer" not in out.stderr


# --------------------------------------------------------------------------
# Whole path, brute force on a tiny NON-grey case  (P4 + P6, north_star's fifth closed form:
# "brute-force trapezoid tau on tiny inputs").  Everything between the parameter vector and the
# per-wavenumber (S, dtau) columns is recomputed here by hand in numpy from the paper's statements
# (PAPER.md:55 levels, :174-190 first-order elements, :484 H2/He fill, :241 interpolation to the level
# (T, p), :127/:133 species + H2-H2/H2-He CIA, :239 optical depths / DESIGN.md R5), with the table values
# taken from its ANALYTIC form and from scipy's RegularGridInterpolator, never from the oracle.  The
# table depends on species, T, p and nu, both CIA pairs are non-zero and differ, He/H2 != 1, the
# profile is not isothermal: every index the driver `oracle_forward_ext` passes along (species offset,
# CIA pair offset, level temperature, level pressure, wavenumber column, x_H2 / x_He) changes the result.
# Mutants of the driver this test kills are listed in DESIGN.md section 3.
# --------------------------------------------------------------------------
def _nongrey_tiny_case():
    T_grid = np.array([300.0, 900.0, 1400.0, 2600.0])
    lp_grid = np.array([-3.0, -0.5, 1.0, 2.5])
    nu0, dnu, nNu = 1500.0, 1750.0, 3
    # sigma_s(nu; T, lp) = a + b T + c lp + d T lp  (exactly bilinear; different per species and per nu)
    coef = np.array([  # [S][nNu][4]
        [[4.0e-23, 1.5e-26, 6.0e-24, 2.0e-27], [9.0e-24, 4.0e-27, -1.0e-24, 1.0e-27], [3.0e-22, -3.0e-26, 3.0e-23, 5.0e-27]],
        [[7.0e-22, -1.0e-25, 1.0e-22, -2.0e-26], [3.0e-23, 2.0e-26, 5.0e-24, -1.0e-27], [5.0e-24, 6.0e-27, 1.0e-24, 5.0e-28]],
    ])
    TT, PP = np.meshgrid(T_grid, lp_grid, indexing="ij")
    sigma = np.empty((2, 4, 4, nNu), np.float32)
    for s in range(2):
        for k in range(nNu):
            a, b, c, d = coef[s, k]
            sigma[s, :, :, k] = a + b * TT + c * PP + d * TT * PP
    assert sigma.min() > 0.0
    # alpha_c(nu; T) = a + b T, cm^-1 amagat^-2; pair 0 = H2-H2, pair 1 = H2-He
    ccoef = np.array([[[2.0e-6, 3.0e-9], [6.0e-7, -1.0e-10], [1.0e-6, 1.0e-9]],
                      [[9.0e-6, -2.0e-9], [2.0e-6, 4.0e-9], [4.0e-7, 2.0e-10]]])
    cia = np.empty((2, 4, nNu), np.float32)
    for c in range(2):
        for k in range(nNu):
            cia[c, :, k] = ccoef[c, k, 0] + ccoef[c, k, 1] * T_grid
    return dict(T_grid=T_grid, lp_grid=lp_grid, nu0=nu0, dnu=dnu, nNu=nNu, coef=coef, ccoef=ccoef,
                sigma=sigma, cia=cia)


def _by_hand_columns(case, L, p_bot, p_top, knots, logg, log_vmr, mmw, he_to_h2, analytic, T_levels=None):
    """(S_l(nu), dtau_l(nu)) from the paper's statements; `analytic` picks the analytic table or
    scipy's multilinear interpolation of the stored fp32 nodes.  T_levels: level temperatures worked out by the
    caller (higher-order elements) instead of the first-order profile through `knots`."""
    from scipy.interpolate import RegularGridInterpolator
    nu = case["nu0"] + case["dnu"] * np.arange(case["nNu"])
    lev = np.arange(L)
    lp = math.log10(p_bot) + (math.log10(p_top) - math.log10(p_bot)) * lev / (L - 1)
    p_cgs = 10.0 ** lp * 1e6
    K = len(knots)
    lp_knots = np.linspace(math.log10(p_bot), math.log10(p_top), max(K, 2))
    if K == 1:
        knots = [knots[0], knots[0]]
    T = np.interp(-lp, -lp_knots, knots)                       # linear in log p between the nodes (first-order elements)
    if T_levels is not None:
        T = np.asarray(T_levels, np.float64)
    x = 10.0 ** np.asarray(log_vmr)
    x_bg = 1.0 - x.sum()
    x_h2, x_he = x_bg / (1.0 + he_to_h2), x_bg * he_to_h2 / (1.0 + he_to_h2)
    n = p_cgs / (KB * T)
    amagat = n / (1.01325e6 / (KB * 273.15))
    chi = np.zeros((L, case["nNu"]))
    for l in range(L):
        for k in range(case["nNu"]):
            if analytic:
                sig = [c[0] + c[1] * T[l] + c[2] * lp[l] + c[3] * T[l] * lp[l] for c in case["coef"][:, k]]
                alp = [c[0] + c[1] * T[l] for c in case["ccoef"][:, k]]
            else:
                sig = [RegularGridInterpolator((case["T_grid"], case["lp_grid"]), case["sigma"][s, :, :, k].astype(np.float64))([[T[l], lp[l]]])[0]
                       for s in range(2)]
                alp = [np.interp(T[l], case["T_grid"], case["cia"][c, :, k].astype(np.float64)) for c in range(2)]
            chi[l, k] = n[l] * (x[0] * sig[0] + x[1] * sig[1]) \
                + amagat[l] ** 2 * x_h2 * (x_h2 * alp[0] + x_he * alp[1])           # PAPER.md:127, 133; R4
    g = 10.0 ** logg
    dz = KB * 0.5 * (T[:-1] + T[1:]) / (mmw * MU * g) * np.log(p_cgs[:-1] / p_cgs[1:])   # hydrostatic, R5
    dtau = 0.5 * (chi[:-1] + chi[1:]) * dz[:, None]                                 # trapezoid, R5
    S = 2 * H * C * C * nu[None, :] ** 3 / np.expm1(C2 * nu[None, :] / T[:, None])   # Eq. 2
    return T, S, dtau


def test_whole_path_brute_force_tiny_nongrey(oracle):
    case = _nongrey_tiny_case()
    L, p_bot, p_top, A = 4, 10.0, 1e-2, 3
    knots = [2100.0, 1300.0, 700.0]
    logg, f, flux_const, mmw, he = 5.3, 1.3, 0.7, 2.3, 0.4
    log_vmr = [-3.0, -3.7]
    params = np.array([[logg, f] + knots + log_vmr])
    edges = np.array([1500.0, 2800.0, 5000.0])
    obs = np.array([3.0e4, 2.0e4])
    err = np.array([2.0e3, 5.0e3])
    r = oracle.forward(case["T_grid"], case["lp_grid"], case["nu0"], case["dnu"], case["sigma"], case["cia"],
                       L, p_bot, p_top, len(knots), A, mmw, he, flux_const, edges, obs, err, None, params,
                       want_flux=True, want_spectra=True, want_logl=True)
    assert r["n_clamped"] == 0
    mu, w = np.polynomial.legendre.leggauss(A)
    mu, w = 0.5 * (mu + 1.0), 0.5 * w
    for analytic, rtol in ((False, 1e-12), (True, 2e-6)):          # fp32 storage of the nodes: 6e-8 per value
        T, S, dtau = _by_hand_columns(case, L, p_bot, p_top, knots, logg, log_vmr, mmw, he, analytic)
        assert len(set(np.searchsorted(case["T_grid"], T))) >= 3    # the levels sit in different T cells
        assert dtau.min() > 1e-3 and dtau.max() < 10.0              # neither transparent nor opaque everywhere
        F = np.array([f * flux_const * oracle.flux_one_nu(S[:, k], dtau[:, k], mu, w) for k in range(case["nNu"])])
        assert np.allclose(r["flux_hr"][0], F, rtol=rtol, atol=0.0)
    # each ingredient matters at this working point (so the comparison above is not vacuous)
    T, S, dtau = _by_hand_columns(case, L, p_bot, p_top, knots, logg, log_vmr, mmw, he, True)
    F = np.array([f * flux_const * oracle.flux_one_nu(S[:, k], dtau[:, k], mu, w) for k in range(case["nNu"])])
    for what in ("species0", "species1", "cia0", "cia1"):
        c2 = {k: (v.copy() if isinstance(v, np.ndarray) else v) for k, v in case.items()}
        if what.startswith("species"):
            c2["coef"][int(what[-1])] *= 0.0
        else:
            c2["ccoef"][int(what[-1])] *= 0.0
        _, S2, d2 = _by_hand_columns(c2, L, p_bot, p_top, knots, logg, log_vmr, mmw, he, True)
        F2 = np.array([f * flux_const * oracle.flux_one_nu(S2[:, k], d2[:, k], mu, w) for k in range(case["nNu"])])
        assert np.max(np.abs(F2 / F - 1.0)) > 1e-3, what
    # the rest of the driver: O5-O7 on that flux (no instrument profile here), Eq. 19
    from scipy.stats import norm
    nu = case["nu0"] + case["dnu"] * np.arange(case["nNu"])
    M = [np.trapezoid(np.interp(xs, nu, r["flux_hr"][0]), xs) / (xs[-1] - xs[0])
         for xs in (np.array([1500.0, 2800.0]), np.array([2800.0, 3250.0, 5000.0]))]
    assert np.allclose(r["spectra"][0], M, rtol=1e-13)
    assert r["logl"][0] == pytest.approx(np.sum(norm.logpdf(obs, loc=M, scale=err)), rel=1e-12)


def test_whole_path_brute_force_many_levels_and_batch(oracle):
    # same brute force with more levels than table nodes (several levels per cell, every cell of the
    # grid crossed), A = 2, and three models in one call (a model's columns must not leak into another's)
    case = _nongrey_tiny_case()
    L, p_bot, p_top, A = 9, 200.0, 2e-3, 2
    mmw, he = 2.5, 0.17
    models = [(5.0, 1.0, [2500.0, 1500.0, 1000.0, 400.0], [-2.5, -4.0]),
              (4.2, 0.6, [1200.0, 1100.0, 900.0, 850.0], [-5.0, -2.2]),
              (5.4, 1.9, [2000.0, 800.0, 700.0, 350.0], [-3.3, -3.1])]
    params = np.array([[m[0], m[1]] + m[2] + m[3] for m in models])
    r = oracle.forward(case["T_grid"], case["lp_grid"], case["nu0"], case["dnu"], case["sigma"], case["cia"],
                       L, p_bot, p_top, 4, A, mmw, he, 1.0, np.array([1500.0, 5000.0]), None, None, None, params,
                       want_flux=True, want_spectra=False, want_logl=False)
    mu, w = np.polynomial.legendre.leggauss(A)
    mu, w = 0.5 * (mu + 1.0), 0.5 * w
    for b, (logg, f, knots, log_vmr) in enumerate(models):
        T, S, dtau = _by_hand_columns(case, L, p_bot, p_top, knots, logg, log_vmr, mmw, he, False)
        F = np.array([f * oracle.flux_one_nu(S[:, k], dtau[:, k], mu, w) for k in range(case["nNu"])])
        assert np.allclose(r["flux_hr"][b], F, rtol=1e-12, atol=0.0)


# --------------------------------------------------------------------------
# Round-3 pins: the one-node (isothermal) branch of the profile and the wiring of the finite-element
# parametrisation in the driver (four one-token mutants survived; they are now in
# tests/test_oracle_mutants.py and die here).
# --------------------------------------------------------------------------
def test_single_node_profile_is_isothermal(oracle):
    # the profile is the interpolant through its nodes; with ONE node there is one value.
    p = oracle.level_pressures(17, 300.0, 1e-3)
    T = oracle.temperature_profile(p, [1234.5], 300.0, 1e-3)
    assert T.shape == (17,) and np.all(T == 1234.5)
    # whole path with n_knots = 1 on the non-grey tables: an isothermal atmosphere emits pi B_nu(T0) whatever the
    # opacity (north_star closed form), times f (R/d)^2 of Eq. 9
    case = _nongrey_tiny_case()
    T0, f, flux_const = 1700.0, 1.4, 0.6
    params = np.array([[5.0, f, T0, -3.0, -3.5]])
    r = oracle.forward(case["T_grid"], case["lp_grid"], case["nu0"], case["dnu"], case["sigma"], case["cia"],
                       7, 50.0, 1e-2, 1, 4, 2.3, 0.17, flux_const, np.array([1500.0, 5000.0]), None, None, None, params,
                       want_flux=True, want_spectra=False, want_logl=False)
    nu = case["nu0"] + case["dnu"] * np.arange(case["nNu"])
    B = 2 * H * C * C * nu ** 3 / np.expm1(C2 * nu / T0)
    assert np.allclose(r["flux_hr"][0], np.pi * f * flux_const * B, rtol=1e-12)


def _fe_levels_by_hand(L, p_bot, p_top, n_el, q, dof):
    """Eq. 12-14 written out: elements equidistant in log p, on each the Lagrange interpolant
    through its q + 1 Gauss-Lobatto points (end points + roots of P_q'), neighbouring elements sharing their end node."""
    from numpy.polynomial import legendre as leg
    inner = leg.legroots(leg.legder([0] * q + [1])) if q > 1 else np.array([])     # roots of P_q' on [-1, 1]
    nodes = np.concatenate([[0.0], 0.5 * (np.sort(inner) + 1.0), [1.0]])            # reference element [0, 1]
    assert len(nodes) == q + 1
    lp = math.log10(p_bot) + (math.log10(p_top) - math.log10(p_bot)) * np.arange(L) / (L - 1)
    s = (lp - math.log10(p_bot)) / (math.log10(p_top) - math.log10(p_bot)) * n_el
    T = np.empty(L)
    for l in range(L):
        k = min(int(math.floor(s[l])), n_el - 1)
        T[l] = np.polyval(np.polyfit(nodes, np.asarray(dof[k * q:k * q + q + 1]), q), s[l] - k)    # degree q through q + 1 points
    return T


@pytest.mark.parametrize("ratio_form", [False, True], ids=["nodal", "ratio"])
def test_whole_path_brute_force_finite_elements(oracle, ratio_form):
    # 2 second-order elements: N_T = 5 temperature parameters while n_knots = 3 is what the first-order call would
    # use -- the driver must take N_T (parameter offsets), the order and the ratio flag from the element settings
    case = _nongrey_tiny_case()
    L, p_bot, p_top, A, n_el, q = 9, 100.0, 1e-2, 3, 2, 2
    logg, f, flux_const, mmw, he = 5.1, 0.9, 1.2, 2.3, 0.3
    log_vmr = [-2.8, -3.9]
    dof = [2300.0, 2050.0, 1500.0, 1050.0, 800.0]          # mid-element nodes off the chords: order 1 would differ
    if ratio_form:                                          # T_1 and b_i = T_i / T_{i-1}
        t_par = [dof[0]] + [dof[i] / dof[i - 1] for i in range(1, 5)]
    else:
        t_par = dof
    params = np.array([[logg, f] + list(t_par) + log_vmr])
    r = oracle.forward(case["T_grid"], case["lp_grid"], case["nu0"], case["dnu"], case["sigma"], case["cia"],
                       L, p_bot, p_top, 3, A, mmw, he, flux_const, np.array([1500.0, 5000.0]), None, None, None, params,
                       want_flux=True, want_spectra=False, want_logl=False,
                       tp_elements=n_el, tp_order=q, tp_ratio=ratio_form)
    T = _fe_levels_by_hand(L, p_bot, p_top, n_el, q, dof)
    assert T[0] == pytest.approx(dof[0]) and T[-1] == pytest.approx(dof[-1]) and T[4] == pytest.approx(dof[2])
    chord = np.interp(np.arange(L), [0, 4, 8], [dof[0], dof[2], dof[4]])
    assert np.max(np.abs(T - chord)) > 50.0                 # a first-order profile through the element ends is far off
    mu, w = np.polynomial.legendre.leggauss(A)
    mu, w = 0.5 * (mu + 1.0), 0.5 * w
    _, S, dtau = _by_hand_columns(case, L, p_bot, p_top, [dof[0], dof[2], dof[4]], logg, log_vmr, mmw, he, False, T_levels=T)
    F = np.array([f * flux_const * oracle.flux_one_nu(S[:, k], dtau[:, k], mu, w) for k in range(case["nNu"])])
    assert np.allclose(r["flux_hr"][0], F, rtol=1e-11, atol=0.0)
