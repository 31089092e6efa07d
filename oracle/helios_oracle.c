/*
 * helios_oracle.c -- ORACLE: plain, slow, fp64 CPU statement of the Helios-r2
 * emission forward model + likelihood (Kitzmann et al. 2020, arXiv:1910.01070).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may build, load or call it.  It shares no code, header, table or constant
 * generator with the CUDA library (paper_1910_01070_b200/csrc) and neither
 * includes the other.  It follows the paper's algorithm step by step, in the
 * paper's order and notation, with no blocking, fusion or reordering; every
 * function cites the passage of /root/reference/PAPER.md (or the DESIGN.md
 * reading, where the paper is silent) that defines it.
 *
 * Pins (tests/test_oracle_pins.py, `-m "not gpu"`): every function below is
 * pinned to a closed form, a library routine or a brute-force value; see the
 * table in DESIGN.md "Oracle pins".  What CANNOT be pinned is agreement with
 * the ORIGINAL Helios-r2 code on the four points the paper never prints
 * (interpolant of sigma, optical-depth formula, convolution normalisation,
 * binning rule: DESIGN.md readings R1, R5, R15, R17) and, for the rows added
 * after the hot path (ratio form of the T-p parameters, grey-cloud geometry,
 * T_eff quadrature: R28, R29, R30) -- "parity unpinned" for those readings;
 * the arithmetic given the readings is pinned (tests/test_oracle_pins.py,
 * tests/test_oracle_next.py).
 *
 * Precision: all arithmetic in fp64; the cross-section tables are the same
 * fp32 values the GPU gets, promoted to double.
 *
 * Index convention: level 0 = bottom (highest pressure), level L-1 = top
 * ("T_1 ... bottom of the modeled atmosphere"; Eq. 4 marches
 * from i-1 outward to i).
 */
#include <math.h>
#include <stddef.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* CODATA 2018, cgs */
static const double H_PLANCK    = 6.62607015e-27;   /* erg s          */
static const double C_LIGHT     = 2.99792458e10;    /* cm s^-1        */
static const double K_BOLTZMANN = 1.380649e-16;     /* erg K^-1       */
static const double M_ATOMIC    = 1.66053906660e-24;/* g              */
static const double N_LOSCHMIDT = 2.686780111798444e19; /* cm^-3, 1 amagat = 101325 Pa/(k_B 273.15 K), CODATA 2018 */
static const double BAR_CGS     = 1.0e6;            /* dyn cm^-2      */
static const double PI          = 3.14159265358979323846;

/* ------------------------------------------------------------------------
 * O0  Atmosphere grid and temperature profile
 * ---------------------------------------------------------------------- */

/* PAPER.md:55 "levels/layers, distributed equidistantly in log p-space".
 * p_l = p_bot (p_top/p_bot)^(l/(L-1)), l = 0 (bottom) .. L-1 (top), in bar. */
void oracle_level_pressures(int L, double p_bot_bar, double p_top_bar, double *p_bar)
{
    for (int l = 0; l < L; ++l) {
        double frac = (L > 1) ? (double)l / (double)(L - 1) : 0.0;
        p_bar[l] = p_bot_bar * pow(p_top_bar / p_bot_bar, frac);
    }
}

/* PAPER.md:174-221 (Sect. 2.5.1), first-order elements (q = 1, Eq. 12-14):
 * K nodes equidistant in log p from p_bot (node 0) to p_top (node K-1); on
 * each element T is the Lagrange interpolant through its two nodes (Eq. 12-13
 * with N_p = 2), i.e. linear in log p; continuous across elements (Eq. 15).
 * The nodal temperatures themselves are the parameters (reading R23;
 * the (T_1, b_i) form of PAPER.md:219 is the NEXT-2 row). */
void oracle_temperature_profile(int L, const double *p_bar, int K, const double *T_knot,
                                double p_bot_bar, double p_top_bar, double *T)
{
    double x_bot = log10(p_bot_bar), x_top = log10(p_top_bar);
    for (int l = 0; l < L; ++l) {
        double x = log10(p_bar[l]);
        if (K == 1) { T[l] = T_knot[0]; continue; }
        double s = (x - x_bot) / (x_top - x_bot) * (double)(K - 1); /* element coordinate */
        int k = (int)floor(s);
        if (k < 0) k = 0;
        if (k > K - 2) k = K - 2;
        double xi = s - (double)k;                /* reference element [0,1] */
        double ell_1 = 1.0 - xi, ell_2 = xi;      /* Lagrange polynomials, Eq. 13, N_p = 2 */
        T[l] = T_knot[k] * ell_1 + T_knot[k + 1] * ell_2;   /* Eq. 12 */
    }
}

/* constant mixing ratios ("isoprofiles"); "H2 and He ... make up
 * the rest of the atmosphere, using the solar ratio of their elemental
 * abundances": x_bg = 1 - sum x_s, x_H2 = x_bg/(1+r), x_He = x_bg r/(1+r),
 * r = he_to_h2 (number ratio He/H2). */
void oracle_mixing_ratios(int S, const double *log10_vmr, double he_to_h2,
                          double *x, double *x_h2, double *x_he)
{
    double sum = 0.0;
    for (int s = 0; s < S; ++s) { x[s] = pow(10.0, log10_vmr[s]); sum += x[s]; }
    double x_bg = 1.0 - sum;
    *x_h2 = x_bg / (1.0 + he_to_h2);
    *x_he = x_bg * he_to_h2 / (1.0 + he_to_h2);
}

/* ------------------------------------------------------------------------
 * O1  Opacity interpolation ("interpolation of opacities to the
 *     corresponding atmospheric temperatures and pressures"; interpolant per
 *     BASELINE north_star / DESIGN.md R1: bilinear in (T, log10 p) on sigma).
 * ---------------------------------------------------------------------- */

/* Cell index and weight on one axis: i = largest index with grid[i] <= v,
 * clamped to [0, n-2]; w = clamp((v - grid[i])/(grid[i+1]-grid[i]), 0, 1).
 * Out-of-range values are clamped to the edge (R3); *clamped is set
 * to 1 when that happened. */
void oracle_cell(int n, const double *grid, double v, int *i_out, double *w_out, int *clamped)
{
    int i = 0;
    for (int k = 0; k < n; ++k) if (grid[k] <= v) i = k;
    if (i > n - 2) i = n - 2;
    double w = (v - grid[i]) / (grid[i + 1] - grid[i]);
    *clamped = 0;
    if (w < 0.0) { w = 0.0; *clamped = 1; }
    if (w > 1.0) { w = 1.0; *clamped = 1; }
    *i_out = i; *w_out = w;
}

/* sigma_s(nu; T, p) for ONE species at all wavenumbers.
 * table: fp32 [N_T][N_P][N_nu], nu contiguous.  Bilinear, 4 taps. */
void oracle_interp_sigma(const float *table, int nT, const double *T_grid,
                         int nP, const double *log10p_grid, int nNu,
                         double T, double log10p, double *sigma_out, int *clamped)
{
    int iT, iP, cT, cP; double t, u;
    oracle_cell(nT, T_grid, T, &iT, &t, &cT);
    oracle_cell(nP, log10p_grid, log10p, &iP, &u, &cP);
    if (clamped) *clamped = cT | cP;
    const float *s00 = table + ((size_t)iT * nP + iP) * nNu;
    const float *s01 = table + ((size_t)iT * nP + iP + 1) * nNu;
    const float *s10 = table + ((size_t)(iT + 1) * nP + iP) * nNu;
    const float *s11 = table + ((size_t)(iT + 1) * nP + iP + 1) * nNu;
    for (int k = 0; k < nNu; ++k)
        sigma_out[k] = (1.0 - t) * (1.0 - u) * (double)s00[k] + t * (1.0 - u) * (double)s10[k]
                     + (1.0 - t) * u * (double)s01[k] + t * u * (double)s11[k];
}

/* CIA coefficient alpha_c(nu; T): linear in T on the same T grid (R4).
 * table: fp32 [N_T][N_nu], cm^-1 amagat^-2. */
void oracle_interp_cia(const float *table, int nT, const double *T_grid, int nNu,
                       double T, double *alpha_out)
{
    int iT, cT; double t;
    oracle_cell(nT, T_grid, T, &iT, &t, &cT);
    const float *a0 = table + (size_t)iT * nNu, *a1 = table + (size_t)(iT + 1) * nNu;
    for (int k = 0; k < nNu; ++k)
        alpha_out[k] = (1.0 - t) * (double)a0[k] + t * (double)a1[k];
}

/* ------------------------------------------------------------------------
 * O2  Absorption coefficient chi_l(nu) [cm^-1]
 *     chi = n sum_s x_s sigma_s + (n/n_L)^2 x_H2 (x_H2 a_HH + x_He a_HHe),
 *     n = p/(k_B T).  CIA pair 0 = H2-H2, pair 1 = H2-He (R4).
 * ---------------------------------------------------------------------- */
double oracle_number_density(double p_bar, double T)
{
    return p_bar * BAR_CGS / (K_BOLTZMANN * T);
}

void oracle_chi_level(int S, const double *x, double *const *sigma_s, /* [S] -> [nNu] */
                      int C, double x_h2, double x_he, double *const *alpha_c, /* [C] -> [nNu] */
                      double n_cm3, int nNu, double *chi)
{
    double amagat = n_cm3 / N_LOSCHMIDT;
    for (int k = 0; k < nNu; ++k) {
        double sum = 0.0;
        for (int s = 0; s < S; ++s) sum += x[s] * sigma_s[s][k];
        double cia = 0.0;
        if (C >= 1) cia += x_h2 * alpha_c[0][k];
        if (C >= 2) cia += x_he * alpha_c[1][k];
        chi[k] = n_cm3 * sum + amagat * amagat * x_h2 * cia;
    }
}

/* ------------------------------------------------------------------------
 * O3  Layer optical depth ("calculation of the optical depths";
 *     formula not printed -> DESIGN.md R5): hydrostatic, ideal gas,
 *     dz_l = k_B (T_l+T_{l+1})/2 / (mmw m_u g) ln(p_l/p_{l+1}),
 *     dtau_l = (chi_l + chi_{l+1})/2 dz_l  (trapezoid),  l = 0 .. L-2.
 * ---------------------------------------------------------------------- */
double oracle_layer_thickness(double T_lo, double T_hi, double p_lo_bar, double p_hi_bar,
                              double mmw, double g_cgs)
{
    return K_BOLTZMANN * 0.5 * (T_lo + T_hi) / (mmw * M_ATOMIC * g_cgs) * log(p_lo_bar / p_hi_bar);
}

/* dtau(nu) of one layer from chi at its lower and upper level (trapezoid). */
void oracle_layer_dtau(int nNu, const double *chi_lo, const double *chi_hi, double dz, double *dtau)
{
    for (int k = 0; k < nNu; ++k) dtau[k] = 0.5 * (chi_lo[k] + chi_hi[k]) * dz;
}

/* ------------------------------------------------------------------------
 * O4  Source function, short characteristics, flux
 * ---------------------------------------------------------------------- */

/* Eq. 2: S_nu = B_nu(T).  Per-wavenumber Planck function (R13):
 * B = 2 h c^2 nu^3 / (exp(h c nu / k_B T) - 1)  [erg s^-1 cm^-2 sr^-1 (cm^-1)^-1]. */
double oracle_planck(double nu_cm1, double T)
{
    double c1 = 2.0 * H_PLANCK * C_LIGHT * C_LIGHT;
    double c2 = H_PLANCK * C_LIGHT / K_BOLTZMANN;
    return c1 * nu_cm1 * nu_cm1 * nu_cm1 / expm1(c2 * nu_cm1 / T);
}

/* PAPER.md:96 "a set of angles mu, distributed according to a Gauss quadrature
 * scheme": n-point Gauss-Legendre on [-1,1] (Newton iteration on P_n, the
 * textbook construction), mapped to mu in (0,1): mu = (x+1)/2, w = W/2 (R12). */
void oracle_gauss_legendre_01(int n, double *mu, double *w)
{
    for (int i = 0; i < n; ++i) {
        double x = cos(PI * ((double)i + 0.75) / ((double)n + 0.5));
        double dp = 1.0;
        for (int it = 0; it < 100; ++it) {
            double p0 = 1.0, p1 = x;
            for (int k = 2; k <= n; ++k) {
                double pk = ((2.0 * k - 1.0) * x * p1 - (k - 1.0) * p0) / (double)k;
                p0 = p1; p1 = pk;
            }
            if (n == 1) { p0 = 1.0; p1 = x; }
            dp = (double)n * (x * p1 - p0) / (x * x - 1.0);
            double dx = p1 / dp;
            x -= dx;
            if (fabs(dx) < 1e-16) break;
        }
        /* recompute derivative at the converged node */
        {
            double p0 = 1.0, p1 = x;
            for (int k = 2; k <= n; ++k) {
                double pk = ((2.0 * k - 1.0) * x * p1 - (k - 1.0) * p0) / (double)k;
                p0 = p1; p1 = pk;
            }
            dp = (double)n * (x * p1 - p0) / (x * x - 1.0);
        }
        double W = 2.0 / ((1.0 - x * x) * dp * dp);
        /* nodes come out descending in x; store ascending in mu */
        mu[n - 1 - i] = 0.5 * (x + 1.0);
        w[n - 1 - i]  = 0.5 * W;
    }
}

/* Eq. 6 with Delta from Eq. 7; linear source in the layer
 * (Olson & Kunasz 1987).  Readings R7-R10: exponent of Eq. 4 is -Delta; the
 * garbled "Lambda" is Delta; gamma's first term carries a minus sign so that
 * beta + gamma = 1 - e^-Delta.
 *   beta  = 1 + (e^-D - 1)/D            (weight of S_i, the downwind level)
 *   gamma = -e^-D - (e^-D - 1)/D        (weight of S_{i-1}, the upwind level)
 * D = 0: beta = gamma = 0.  D < 1e-3: Taylor series (R10); else expm1. */
void oracle_sc_coefficients(double D, double *e_out, double *beta, double *gamma)
{
    if (D == 0.0) { *e_out = 1.0; *beta = 0.0; *gamma = 0.0; return; }
    if (D < 1e-3) {
        double b = D / 2.0 - D * D / 6.0 + D * D * D / 24.0 - D * D * D * D / 120.0;
        double g = D / 2.0 - D * D / 3.0 + D * D * D / 8.0 - D * D * D * D / 30.0;
        *beta = b; *gamma = g; *e_out = 1.0 - (b + g);
        return;
    }
    double em1 = expm1(-D);          /* e^-D - 1 */
    double e = exp(-D);
    *e_out = e;
    *beta  = 1.0 + em1 / D;
    *gamma = -e - em1 / D;
}

/* Eq. 4, 5, 8 for ONE wavenumber.  S[l] = source at level l (0 = bottom),
 * dtau[l] = optical depth of the layer between level l and l+1.
 * Bottom boundary (R11, "semi-infinite atmosphere"):
 * I+(level 0, mu) = S_0.  Returns F+ = 2 pi sum_k w_k mu_k I_k (Eq. 8). */
double oracle_flux_one_nu(int L, const double *S, const double *dtau,
                          int A, const double *mu, const double *w)
{
    double flux = 0.0;
    for (int k = 0; k < A; ++k) {
        double I = S[0];
        for (int i = 1; i < L; ++i) {
            double D = dtau[i - 1] / mu[k];                    /* Eq. 7 */
            double e, beta, gamma;
            oracle_sc_coefficients(D, &e, &beta, &gamma);      /* Eq. 6 */
            double dI = beta * S[i] + gamma * S[i - 1];        /* Eq. 5, alpha = 0 */
            I = I * e + dI;                                    /* Eq. 4 */
        }
        flux += w[k] * mu[k] * I;
    }
    return 2.0 * PI * flux;
}

/* ------------------------------------------------------------------------
 * O5  Instrument profile (Eq. 17): Gaussian of standard
 *     deviation sigma evaluated at the output point, integration stopped at
 *     |x - nu| = 5 sigma; discrete sum on the grid, renormalised by the sum
 *     of the weights used (R15).  inst_sigma == NULL or sigma_k == 0: copy.
 * ---------------------------------------------------------------------- */
void oracle_convolve(int nNu, double nu0, double dnu, const double *F,
                     const double *inst_sigma, double *Fd)
{
    for (int k = 0; k < nNu; ++k) {
        double sg = inst_sigma ? inst_sigma[k] : 0.0;
        if (sg <= 0.0) { Fd[k] = F[k]; continue; }
        double nu_k = nu0 + dnu * k;
        double num = 0.0, den = 0.0;
        /* only grid points that can lie within 5 sigma are visited (the test
         * below still decides); this bounds the loop, it changes no value */
        int reach = (int)ceil(5.0 * sg / dnu) + 1;
        int j_lo = k - reach < 0 ? 0 : k - reach;
        int j_hi = k + reach > nNu - 1 ? nNu - 1 : k + reach;
        for (int j = j_lo; j <= j_hi; ++j) {
            double d = (nu0 + dnu * j) - nu_k;
            if (fabs(d) > 5.0 * sg) continue;
            double g = exp(-d * d / (2.0 * sg * sg));
            num += F[j] * g; den += g;
        }
        Fd[k] = num / den;
    }
}

/* ------------------------------------------------------------------------
 * O6  Binning ("integrate ... to a lower resolution";
 *     R17): bin mean of the piecewise-linear interpolant of Fd,
 *     M_j = 1/(e_{j+1}-e_j) int Fd dnu, trapezoid over {e_j, interior grid
 *     points, e_{j+1}} with linearly interpolated edge values.
 *     Edges must lie inside [nu_0, nu_{N-1}].
 * ---------------------------------------------------------------------- */
static double lin_interp_grid(int nNu, double nu0, double dnu, const double *Fd, double nu)
{
    double s = (nu - nu0) / dnu;
    int i = (int)floor(s);
    if (i < 0) i = 0;
    if (i > nNu - 2) i = nNu - 2;
    double a = s - (double)i;
    return (1.0 - a) * Fd[i] + a * Fd[i + 1];
}

void oracle_bin(int nNu, double nu0, double dnu, const double *Fd,
                int J, const double *edges, double *M)
{
    for (int j = 0; j < J; ++j) {
        double a = edges[j], b = edges[j + 1];
        double x_prev = a, y_prev = lin_interp_grid(nNu, nu0, dnu, Fd, a);
        double integral = 0.0;
        for (int i = 0; i < nNu; ++i) {
            double x = nu0 + dnu * i;
            if (x <= a || x >= b) continue;              /* interior grid points only */
            integral += 0.5 * (y_prev + Fd[i]) * (x - x_prev);
            x_prev = x; y_prev = Fd[i];
        }
        double y_b = lin_interp_grid(nNu, nu0, dnu, Fd, b);
        integral += 0.5 * (y_prev + y_b) * (b - x_prev);
        M[j] = integral / (b - a);
    }
}

/* ------------------------------------------------------------------------
 * O7  Likelihood, Eq. 19:
 *     ln L = sum_j ( -(D_j - M_j)^2/(2 sigma_j^2) - 1/2 ln(2 pi sigma_j^2) ).
 * ---------------------------------------------------------------------- */
double oracle_loglike(int J, const double *D, const double *err, const double *M)
{
    double lnL = 0.0;
    for (int j = 0; j < J; ++j) {
        double r = D[j] - M[j];
        lnL += -(r * r) / (2.0 * err[j] * err[j]) - 0.5 * log(2.0 * PI * err[j] * err[j]);
    }
    return lnL;
}

/* ========================================================================
 * Rows NEXT-1 .. NEXT-4 of SURVEY.md 8(f)
 * ====================================================================== */

/* NEXT-1.  Eq. 22-23: s_j^2 = sigma_j^2 + 10^eps,
 *   ln L = sum_j ( -(D_j - M_j)^2/(2 s_j^2) - 1/2 ln(2 pi s_j^2) )
 * (R20: the second term belongs inside the sum, as in Eq. 19). */
double oracle_loglike_inflated(int J, const double *D, const double *err, const double *M, double eps)
{
    double lnL = 0.0, add = pow(10.0, eps);
    for (int j = 0; j < J; ++j) {
        double s2 = err[j] * err[j] + add;                      /* Eq. 22 */
        double r = D[j] - M[j];
        lnL += -(r * r) / (2.0 * s2) - 0.5 * log(2.0 * PI * s2);  /* Eq. 23 */
    }
    return lnL;
}

/* NEXT-2.  Sect. 2.5.1.  Gauss-Lobatto points of the
 * reference element [0,1] for order q = 1..4 (N_p = q + 1, Eq. 14): the end
 * points plus the roots of P'_q mapped from [-1,1]. */
int oracle_lobatto_nodes(int q, double *xi)
{
    switch (q) {
        case 1: xi[0] = 0.0; xi[1] = 1.0; return 0;
        case 2: xi[0] = 0.0; xi[1] = 0.5; xi[2] = 1.0; return 0;
        case 3: { double a = 1.0 / sqrt(5.0);
                  xi[0] = 0.0; xi[1] = 0.5 * (1.0 - a); xi[2] = 0.5 * (1.0 + a); xi[3] = 1.0; return 0; }
        case 4: { double a = sqrt(3.0 / 7.0);
                  xi[0] = 0.0; xi[1] = 0.5 * (1.0 - a); xi[2] = 0.5; xi[3] = 0.5 * (1.0 + a); xi[4] = 1.0; return 0; }
        default: return -1;
    }
}

/* "The only, actually retrieved temperature is the one at the bottom ...  For all
 * other temperatures, we retrieve a parameter b, such that, e.g., T_2 = b_2 T_1"
 * (PAPER.md:219); b is "the slope between two adjacent temperature nodes", so each
 * ratio refers to the node below it (R28): T_i = b_i T_{i-1}.  theta = (T_1, b_2..b_N). */
void oracle_tp_dofs_from_ratios(int N, const double *theta, double *T_dof)
{
    T_dof[0] = theta[0];
    for (int i = 1; i < N; ++i) T_dof[i] = theta[i] * T_dof[i - 1];
}

/* Eq. 12-15: K_e elements equidistant in log p from p_bot (element 0) to p_top,
 * order q, continuous: element k owns the global dofs k q .. k q + q (N_T = K_e q + 1,
 * Eq. 16); inside an element T is the Lagrange interpolant (Eq. 13) through the
 * Gauss-Lobatto points of the reference element. */
int oracle_temperature_profile_fe(int L, const double *p_bar, int Ke, int q, const double *T_dof,
                                  double p_bot_bar, double p_top_bar, double *T)
{
    double xi_n[8];
    if (Ke < 1 || oracle_lobatto_nodes(q, xi_n)) return -1;
    double x_bot = log10(p_bot_bar), x_top = log10(p_top_bar);
    for (int l = 0; l < L; ++l) {
        double s = (log10(p_bar[l]) - x_bot) / (x_top - x_bot) * (double)Ke;
        int k = (int)floor(s);
        if (k < 0) k = 0;
        if (k > Ke - 1) k = Ke - 1;
        double xi = s - (double)k;                       /* reference element coordinate */
        double Tl = 0.0;
        for (int i = 0; i <= q; ++i) {
            double ell = 1.0;                            /* Eq. 13 */
            for (int j = 0; j <= q; ++j) if (j != i) ell *= (xi - xi_n[j]) / (xi_n[i] - xi_n[j]);
            Tl += T_dof[k * q + i] * ell;                /* Eq. 12 */
        }
        T[l] = Tl;
    }
    return 0;
}

/* NEXT-3.  Sect. 2.6: the outgoing flux F+ integrated over
 * [nu_a, nu_b] (the paper: 1-20 micron) "converted into an effective temperature by
 * using the Stefan-Boltzmann law".  Quadrature (R30): trapezoid on the grid with
 * linearly interpolated end points, i.e. the bin rule O6 times the width. */
void oracle_bin(int nNu, double nu0, double dnu, const double *Fd, int J, const double *edges, double *M);
double oracle_teff(int nNu, double nu0, double dnu, const double *Fplus, double nu_a, double nu_b)
{
    const double sigma_sb = 2.0 * pow(PI, 5) * pow(K_BOLTZMANN, 4) /
                            (15.0 * pow(H_PLANCK, 3) * C_LIGHT * C_LIGHT);
    double e[2] = {nu_a, nu_b}, mean;
    oracle_bin(nNu, nu0, dnu, Fplus, 1, e, &mean);
    return pow(mean * (nu_b - nu_a) / sigma_sb, 0.25);
}

/* NEXT-4.  App. B: a grey cloud with "three free parameters: the
 * cloud optical depth, the pressure of the cloud layer top, and the bottom of the cloud
 * layer, defined as the fraction of the top pressure".  Reading R29: p_bot = p_top (1 + phi);
 * the vertical optical depth tau_c is spread uniformly in pressure over [p_top, p_bot]; layer l
 * (levels l, l+1) receives the share of its pressure overlap; the part of the cloud outside the
 * modelled range is dropped.  dtau_cloud[l], l = 0 .. L-2, is added to dtau_l at every nu. */
void oracle_cloud_dtau(int L, const double *p_bar, double tau_c, double p_top_c, double phi, double *dtau_cloud)
{
    double p_bot_c = p_top_c * (1.0 + phi);
    for (int l = 0; l + 1 < L; ++l) {
        double hi = p_bar[l] < p_bot_c ? p_bar[l] : p_bot_c;            /* larger pressure end */
        double lo = p_bar[l + 1] > p_top_c ? p_bar[l + 1] : p_top_c;
        double overlap = hi - lo;
        dtau_cloud[l] = overlap > 0.0 ? tau_c * overlap / (p_bot_c - p_top_c) : 0.0;
    }
}

/* ------------------------------------------------------------------------
 * Whole path for B parameter vectors (OpenMP over models only).
 * params [B][P], P = 2 + K + S: log10 g (cgs), f, T_knot[0..K-1] (bottom->top),
 * log10 VMR[0..S-1].   Outputs (any may be NULL): flux_hr [B][nNu] (Eq. 9,
 * before the instrument profile), spectra [B][J], logl [B].
 * obs/err may be NULL when logl is NULL.  A model with a non-finite parameter,
 * or an unphysical one (R31, see below), gets NaN spectra and logl = -inf.
 * Returns the number of (model, level) pairs whose (T, p) was clamped.
 * ---------------------------------------------------------------------- */
#define ORACLE_EXTRA_DISTANCE        1u   /* + d:   F = F+ f flux_const / d^2 (Eq. 9, flux_const = R_*^2)   */
#define ORACLE_EXTRA_ERROR_INFLATION 2u   /* + eps: Eq. 22-23                                                */
#define ORACLE_EXTRA_GREY_CLOUD      4u   /* + log10 tau_c, log10 p_top [bar], log10 phi (App. B, R29)        */

/* Extended driver.  Temperature parameters: tp_elements = 0 -> K nodal temperatures, linear in
 * log p (the hot path); tp_elements = K_e > 0 -> K_e elements of order tp_order (N_T = K_e q + 1
 * values), nodal temperatures (tp_ratio = 0) or (T_1, b_2 .. b_N) (tp_ratio = 1).
 * params [B][P], P = 2 + N_T + S + extras: log10 g, f, temperature parameters, log10 VMR,
 * then the extras that are switched on, in the order of the flags above.
 * teff (or NULL): T_eff from F+ over [teff_nu_a, teff_nu_b] (NEXT-3). */
long oracle_forward_ext(int S, int nT, const double *T_grid, int nP, const double *log10p_grid,
                    int nNu, double nu0, double dnu,
                    const float *sigma,            /* [S][nT][nP][nNu] */
                    int C, const float *cia,       /* [C][nT][nNu]     */
                    int L, double p_bot_bar, double p_top_bar, int K, int A,
                    double mmw, double he_to_h2, double flux_const,
                    int J, const double *edges, const double *obs, const double *err,
                    const double *inst_sigma,      /* [nNu] or NULL    */
                    int B, const double *params,
                    double *flux_hr, double *spectra, double *logl, int n_threads,
                    int tp_elements, int tp_order, int tp_ratio, unsigned extras,
                    double teff_nu_a, double teff_nu_b, double *teff)
{
    int NT = tp_elements > 0 ? tp_elements * tp_order + 1 : K;
    int i_d = -1, i_eps = -1, i_cloud = -1, P = 2 + NT + S;
    if (extras & ORACLE_EXTRA_DISTANCE) i_d = P++;
    if (extras & ORACLE_EXTRA_ERROR_INFLATION) i_eps = P++;
    if (extras & ORACLE_EXTRA_GREY_CLOUD) { i_cloud = P; P += 3; }
    long n_clamped = 0;
    double *mu = (double *)malloc(sizeof(double) * A), *w = (double *)malloc(sizeof(double) * A);
    oracle_gauss_legendre_01(A, mu, w);
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
#pragma omp parallel for schedule(dynamic, 1) reduction(+ : n_clamped)
    for (int b = 0; b < B; ++b) {
        const double *th = params + (size_t)b * P;
        int finite = 1;
        for (int i = 0; i < P; ++i) if (!isfinite(th[i])) finite = 0;
        if (!finite) {
            if (flux_hr) for (int k = 0; k < nNu; ++k) flux_hr[(size_t)b * nNu + k] = NAN;
            if (spectra) for (int j = 0; j < J; ++j) spectra[(size_t)b * J + j] = NAN;
            if (logl) logl[b] = -INFINITY;
            if (teff) teff[b] = NAN;
            continue;
        }
        double g_cgs = pow(10.0, th[0]);
        double f = th[1];
        const double *T_par = th + 2;
        const double *log10_vmr = th + 2 + NT;
        double scale = f * flux_const;                                              /* Eq. 9 */
        if (i_d >= 0) scale /= th[i_d] * th[i_d];

        double *p_bar = (double *)malloc(sizeof(double) * L);
        double *T = (double *)malloc(sizeof(double) * L);
        double *x = (double *)malloc(sizeof(double) * (S > 0 ? S : 1));
        double x_h2, x_he;
        oracle_level_pressures(L, p_bot_bar, p_top_bar, p_bar);                     /* O0 */
        if (tp_elements > 0) {                                                       /* NEXT-2 */
            double *dof = (double *)malloc(sizeof(double) * NT);
            if (tp_ratio) oracle_tp_dofs_from_ratios(NT, T_par, dof);
            else for (int i = 0; i < NT; ++i) dof[i] = T_par[i];
            oracle_temperature_profile_fe(L, p_bar, tp_elements, tp_order, dof, p_bot_bar, p_top_bar, T);
            free(dof);
        } else
            oracle_temperature_profile(L, p_bar, K, T_par, p_bot_bar, p_top_bar, T);   /* O0 */
        oracle_mixing_ratios(S, log10_vmr, he_to_h2, x, &x_h2, &x_he);              /* O0 */

        /* Unphysical models are rejected like non-finite ones [paper silent; R31]: a level
         * temperature <= 0 (possible with elements of order >= 2 or ratio parameters), VMRs summing to
         * more than 1 (negative H2/He fill), f < 0, d <= 0, or g / 10^eps / a cloud parameter overflowing. */
        {
            int ok = isfinite(g_cgs) && f >= 0.0 && x_h2 + x_he >= 0.0;
            for (int l = 0; l < L; ++l) if (!(T[l] > 0.0) || !isfinite(T[l])) ok = 0;
            if (i_d >= 0 && !(th[i_d] > 0.0)) ok = 0;
            if (i_eps >= 0 && !isfinite(pow(10.0, th[i_eps]))) ok = 0;
            if (i_cloud >= 0 && (!isfinite(pow(10.0, th[i_cloud])) ||
                                 !isfinite(pow(10.0, th[i_cloud + 1]) * (1.0 + pow(10.0, th[i_cloud + 2]))))) ok = 0;
            if (!ok) {
                if (flux_hr) for (int k = 0; k < nNu; ++k) flux_hr[(size_t)b * nNu + k] = NAN;
                if (spectra) for (int j = 0; j < J; ++j) spectra[(size_t)b * J + j] = NAN;
                if (logl) logl[b] = -INFINITY;
                if (teff) teff[b] = NAN;
                free(p_bar); free(T); free(x);
                continue;
            }
        }

        /* chi[l][nu], then dtau[l][nu] */
        double *chi = (double *)malloc(sizeof(double) * (size_t)L * nNu);
        double **sig = (double **)malloc(sizeof(double *) * (S > 0 ? S : 1));
        double **alp = (double **)malloc(sizeof(double *) * (C > 0 ? C : 1));
        for (int s = 0; s < S; ++s) sig[s] = (double *)malloc(sizeof(double) * nNu);
        for (int c = 0; c < C; ++c) alp[c] = (double *)malloc(sizeof(double) * nNu);
        for (int l = 0; l < L; ++l) {
            int any_clamped = 0;
            for (int s = 0; s < S; ++s) {                                            /* O1 */
                int cl;
                oracle_interp_sigma(sigma + (size_t)s * nT * nP * nNu, nT, T_grid, nP, log10p_grid,
                                    nNu, T[l], log10(p_bar[l]), sig[s], &cl);
                any_clamped |= cl;
            }
            if (S == 0) {
                int iT, iP, cT, cP; double t, u;
                oracle_cell(nT, T_grid, T[l], &iT, &t, &cT);
                oracle_cell(nP, log10p_grid, log10(p_bar[l]), &iP, &u, &cP);
                any_clamped = cT | cP;
            }
            for (int c = 0; c < C; ++c)
                oracle_interp_cia(cia + (size_t)c * nT * nNu, nT, T_grid, nNu, T[l], alp[c]);
            n_clamped += any_clamped;
            oracle_chi_level(S, x, sig, C, x_h2, x_he, alp,                          /* O2 */
                             oracle_number_density(p_bar[l], T[l]), nNu, chi + (size_t)l * nNu);
        }
        double *dtau = (double *)malloc(sizeof(double) * (size_t)(L > 1 ? L - 1 : 1) * nNu);
        for (int l = 0; l + 1 < L; ++l) {                                            /* O3 */
            double dz = oracle_layer_thickness(T[l], T[l + 1], p_bar[l], p_bar[l + 1], mmw, g_cgs);
            oracle_layer_dtau(nNu, chi + (size_t)l * nNu, chi + (size_t)(l + 1) * nNu, dz,
                              dtau + (size_t)l * nNu);
        }

        if (i_cloud >= 0) {                                                          /* NEXT-4 */
            double *dc = (double *)malloc(sizeof(double) * (L > 1 ? L - 1 : 1));
            oracle_cloud_dtau(L, p_bar, pow(10.0, th[i_cloud]), pow(10.0, th[i_cloud + 1]),
                              pow(10.0, th[i_cloud + 2]), dc);
            for (int l = 0; l + 1 < L; ++l)
                for (int k = 0; k < nNu; ++k) dtau[(size_t)l * nNu + k] += dc[l];
            free(dc);
        }

        /* O4: RT per wavenumber, then Eq. 9 */
        double *F = (double *)malloc(sizeof(double) * nNu);
        double *Scol = (double *)malloc(sizeof(double) * L);
        double *dcol = (double *)malloc(sizeof(double) * (L > 1 ? L - 1 : 1));
        for (int k = 0; k < nNu; ++k) {
            double nu = nu0 + dnu * k;
            for (int l = 0; l < L; ++l) Scol[l] = oracle_planck(nu, T[l]);
            for (int l = 0; l + 1 < L; ++l) dcol[l] = dtau[(size_t)l * nNu + k];
            double Fplus = oracle_flux_one_nu(L, Scol, dcol, A, mu, w);
            F[k] = Fplus;
        }
        if (teff) teff[b] = oracle_teff(nNu, nu0, dnu, F, teff_nu_a, teff_nu_b);      /* NEXT-3 */
        for (int k = 0; k < nNu; ++k) F[k] *= scale;                                 /* Eq. 9 */
        if (flux_hr) for (int k = 0; k < nNu; ++k) flux_hr[(size_t)b * nNu + k] = F[k];

        if (spectra || logl) {
            double *Fd = (double *)malloc(sizeof(double) * nNu);
            double *M = (double *)malloc(sizeof(double) * J);
            oracle_convolve(nNu, nu0, dnu, F, inst_sigma, Fd);                       /* O5 */
            oracle_bin(nNu, nu0, dnu, Fd, J, edges, M);                              /* O6 */
            if (spectra) for (int j = 0; j < J; ++j) spectra[(size_t)b * J + j] = M[j];
            if (logl) logl[b] = i_eps >= 0 ? oracle_loglike_inflated(J, obs, err, M, th[i_eps])  /* NEXT-1 */
                                           : oracle_loglike(J, obs, err, M);                      /* O7 */
            free(Fd); free(M);
        }
        for (int s = 0; s < S; ++s) free(sig[s]);
        for (int c = 0; c < C; ++c) free(alp[c]);
        free(sig); free(alp); free(chi); free(dtau); free(F); free(Scol); free(dcol);
        free(p_bar); free(T); free(x);
    }
    free(mu); free(w);
    return n_clamped;
}

/* The hot path as BASELINE.json states it: K nodal temperatures, no extras. */
long oracle_forward(int S, int nT, const double *T_grid, int nP, const double *log10p_grid,
                    int nNu, double nu0, double dnu, const float *sigma, int C, const float *cia,
                    int L, double p_bot_bar, double p_top_bar, int K, int A,
                    double mmw, double he_to_h2, double flux_const,
                    int J, const double *edges, const double *obs, const double *err,
                    const double *inst_sigma, int B, const double *params,
                    double *flux_hr, double *spectra, double *logl, int n_threads)
{
    return oracle_forward_ext(S, nT, T_grid, nP, log10p_grid, nNu, nu0, dnu, sigma, C, cia, L, p_bot_bar,
                              p_top_bar, K, A, mmw, he_to_h2, flux_const, J, edges, obs, err, inst_sigma,
                              B, params, flux_hr, spectra, logl, n_threads, 0, 1, 0, 0u, 0.0, 0.0, NULL);
}

int oracle_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
