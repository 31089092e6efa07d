"""Derivations of the numerical constants compiled into the CUDA path (csrc/common.cuh), re-done here from
their definitions -- no GPU needed.  The logL tolerance leans on the small-optical-depth branch of the
short-characteristics update (R10), so its polynomial is re-derived and its error bound measured;
the compile-time Gauss-Legendre tables are checked against numpy's rule (R12)."""
import os
import re

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
COMMON = open(os.path.join(ROOT, "paper_1910_01070_b200", "csrc", "common.cuh")).read()


def _scalar(name):
    m = re.search(r"\b%s\s*=\s*(-?[0-9.eE+-]+)" % name, COMMON)
    assert m, name
    return float(m.group(1))


def _table(name):
    m = re.search(r"constexpr double %s\[8\]\[8\]\s*=\s*\{(.*?)\};" % name, COMMON, flags=re.S)
    assert m, name
    rows = re.findall(r"\{([^{}]*)\}", m.group(1))
    return np.array([[float(v) for v in r.split(",") if v.strip()] for r in rows])


def phi(D):
    return -np.expm1(-D) / D


def test_phi_polynomial_is_the_chebyshev_node_interpolant_and_stays_within_5e_9():
    """phi(D) = (1 - e^-D)/D on [0, 1/4] (kPhiSwitch): degree-4 interpolant at the 5 Chebyshev nodes of the
    interval, constant term then set to exactly 1 (so that a transparent layer is an exact no-op)."""
    shipped = np.array([_scalar("kPhiC%d" % i) for i in (1, 2, 3, 4)])
    assert _scalar("kPhiSwitch") == 0.25
    k = np.arange(5)
    nodes = 0.125 + 0.125 * np.cos((2 * k + 1) * np.pi / 10)
    coef = np.polyfit(nodes, phi(nodes), 4)[::-1]
    assert abs(coef[0] - 1.0) < 5e-9
    np.testing.assert_allclose(shipped, coef[1:], rtol=0, atol=1e-10)
    D = np.linspace(1e-12, 0.25, 2_000_001)
    p = 1.0 + D * (shipped[0] + D * (shipped[1] + D * (shipped[2] + D * shipped[3])))
    err = np.max(np.abs(p - phi(D)))
    assert err < 5e-9, err
    # the same Horner scheme in fp32, as the kernels evaluate it (phi_small in common.cuh; the staged kernels fold
    # 1/mu_k^(j+1) into the coefficients, which rescales the argument and nothing else)
    D32 = D.astype(np.float32)
    c32 = shipped.astype(np.float32)
    p32 = np.float32(1.0) + D32 * (c32[0] + D32 * (c32[1] + D32 * (c32[2] + D32 * c32[3])))
    assert np.max(np.abs(p32.astype(np.float64) - phi(D32.astype(np.float64)))) < 1.3e-7   # one fp32 ulp of 1


def test_thin_branch_identity_e_equals_one_minus_D_phi():
    """The thin branch never evaluates an exponential: e^-D = 1 - D phi(D) (exact identity), so
    J <- e^-D J + phi dS = J + phi (dS - D J).  With the polynomial in place of phi the implied e^-D is off by
    at most D * 5e-9 <= 1.25e-9."""
    c = np.array([_scalar("kPhiC%d" % i) for i in (1, 2, 3, 4)])
    D = np.linspace(0.0, 0.25, 100_001)
    p = 1.0 + D * (c[0] + D * (c[1] + D * (c[2] + D * c[3])))
    assert np.max(np.abs((1.0 - D * p) - np.exp(-D))) < 1.25e-9


def test_compile_time_gauss_legendre_tables():
    mu, w = _table("kGLmu"), _table("kGLw")
    for n in range(1, 9):
        x, W = np.polynomial.legendre.leggauss(n)
        np.testing.assert_allclose(mu[n - 1, :n], 0.5 * (x + 1.0), rtol=0, atol=2e-16)
        np.testing.assert_allclose(w[n - 1, :n], 0.5 * W, rtol=0, atol=2e-16)
        assert abs(np.sum(w[n - 1, :n] * mu[n - 1, :n]) - 0.5) < 1e-15     # the rule integrates mu exactly


def test_physical_constants_are_codata_2018():
    assert _scalar("kPlanckH") == 6.62607015e-27 and _scalar("kLightC") == 2.99792458e10
    assert _scalar("kBoltzmann") == 1.380649e-16 and _scalar("kAtomicMass") == 1.66053906660e-24
