"""ctypes access to oracle/helios_oracle.c (marshalling only; no arithmetic).

ORACLE = test infrastructure.  See the header of helios_oracle.c.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "helios_oracle.c")
_SO = os.path.join(_HERE, "libhelios_oracle.so")
_lock = threading.Lock()
_lib = None

_dp = C.POINTER(C.c_double)
_fp = C.POINTER(C.c_float)
_ip = C.POINTER(C.c_int)


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp -shared; rebuilt when the source is newer than the .so."""
    with _lock:
        stale = (not os.path.exists(_SO)) or os.path.getmtime(_SO) < os.path.getmtime(_SRC)
        if force or stale:
            tmp = _SO + f".tmp{os.getpid()}"
            cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-Wall",
                   "-o", tmp, _SRC, "-lm"]
            subprocess.run(cmd, check=True)
            os.replace(tmp, _SO)
    return _SO


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_SO)
        L.oracle_level_pressures.argtypes = [C.c_int, C.c_double, C.c_double, _dp]
        L.oracle_level_pressures.restype = None
        L.oracle_temperature_profile.argtypes = [C.c_int, _dp, C.c_int, _dp, C.c_double, C.c_double, _dp]
        L.oracle_temperature_profile.restype = None
        L.oracle_mixing_ratios.argtypes = [C.c_int, _dp, C.c_double, _dp, _dp, _dp]
        L.oracle_mixing_ratios.restype = None
        L.oracle_cell.argtypes = [C.c_int, _dp, C.c_double, _ip, _dp, _ip]
        L.oracle_cell.restype = None
        L.oracle_interp_sigma.argtypes = [_fp, C.c_int, _dp, C.c_int, _dp, C.c_int, C.c_double,
                                          C.c_double, _dp, _ip]
        L.oracle_interp_sigma.restype = None
        L.oracle_interp_cia.argtypes = [_fp, C.c_int, _dp, C.c_int, C.c_double, _dp]
        L.oracle_interp_cia.restype = None
        L.oracle_number_density.argtypes = [C.c_double, C.c_double]
        L.oracle_number_density.restype = C.c_double
        L.oracle_chi_level.argtypes = [C.c_int, _dp, C.POINTER(_dp), C.c_int, C.c_double, C.c_double,
                                       C.POINTER(_dp), C.c_double, C.c_int, _dp]
        L.oracle_chi_level.restype = None
        L.oracle_layer_thickness.argtypes = [C.c_double] * 6
        L.oracle_layer_thickness.restype = C.c_double
        L.oracle_layer_dtau.argtypes = [C.c_int, _dp, _dp, C.c_double, _dp]
        L.oracle_layer_dtau.restype = None
        L.oracle_planck.argtypes = [C.c_double, C.c_double]
        L.oracle_planck.restype = C.c_double
        L.oracle_gauss_legendre_01.argtypes = [C.c_int, _dp, _dp]
        L.oracle_gauss_legendre_01.restype = None
        L.oracle_sc_coefficients.argtypes = [C.c_double, _dp, _dp, _dp]
        L.oracle_sc_coefficients.restype = None
        L.oracle_flux_one_nu.argtypes = [C.c_int, _dp, _dp, C.c_int, _dp, _dp]
        L.oracle_flux_one_nu.restype = C.c_double
        L.oracle_convolve.argtypes = [C.c_int, C.c_double, C.c_double, _dp, _dp, _dp]
        L.oracle_convolve.restype = None
        L.oracle_bin.argtypes = [C.c_int, C.c_double, C.c_double, _dp, C.c_int, _dp, _dp]
        L.oracle_bin.restype = None
        L.oracle_loglike.argtypes = [C.c_int, _dp, _dp, _dp]
        L.oracle_loglike.restype = C.c_double
        L.oracle_forward.argtypes = [
            C.c_int, C.c_int, _dp, C.c_int, _dp, C.c_int, C.c_double, C.c_double, _fp,
            C.c_int, _fp,
            C.c_int, C.c_double, C.c_double, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double,
            C.c_int, _dp, _dp, _dp, _dp,
            C.c_int, _dp, _dp, _dp, _dp, C.c_int]
        L.oracle_forward.restype = C.c_long
        L.oracle_forward_ext.argtypes = [
            C.c_int, C.c_int, _dp, C.c_int, _dp, C.c_int, C.c_double, C.c_double, _fp,
            C.c_int, _fp,
            C.c_int, C.c_double, C.c_double, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double,
            C.c_int, _dp, _dp, _dp, _dp,
            C.c_int, _dp, _dp, _dp, _dp, C.c_int, C.c_int, C.c_int, C.c_int, C.c_uint, C.c_double, C.c_double, _dp]
        L.oracle_forward_ext.restype = C.c_long
        L.oracle_loglike_inflated.argtypes = [C.c_int, _dp, _dp, _dp, C.c_double]
        L.oracle_loglike_inflated.restype = C.c_double
        L.oracle_lobatto_nodes.argtypes = [C.c_int, _dp]
        L.oracle_lobatto_nodes.restype = C.c_int
        L.oracle_tp_dofs_from_ratios.argtypes = [C.c_int, _dp, _dp]
        L.oracle_tp_dofs_from_ratios.restype = None
        L.oracle_temperature_profile_fe.argtypes = [C.c_int, _dp, C.c_int, C.c_int, _dp, C.c_double, C.c_double, _dp]
        L.oracle_temperature_profile_fe.restype = C.c_int
        L.oracle_teff.argtypes = [C.c_int, C.c_double, C.c_double, _dp, C.c_double, C.c_double]
        L.oracle_teff.restype = C.c_double
        L.oracle_cloud_dtau.argtypes = [C.c_int, _dp, C.c_double, C.c_double, C.c_double, _dp]
        L.oracle_cloud_dtau.restype = None
        L.oracle_max_threads.argtypes = []
        L.oracle_max_threads.restype = C.c_int
        _lib = L
    return _lib


def _d(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(_dp)


def _f(a):
    a = np.ascontiguousarray(a, dtype=np.float32)
    return a, a.ctypes.data_as(_fp)


def max_threads() -> int:
    return int(lib().oracle_max_threads())


def level_pressures(L, p_bot_bar, p_top_bar):
    out = np.empty(L, np.float64)
    lib().oracle_level_pressures(L, p_bot_bar, p_top_bar, out.ctypes.data_as(_dp))
    return out


def temperature_profile(p_bar, T_knot, p_bot_bar, p_top_bar):
    p, pp = _d(p_bar)
    k, kp = _d(T_knot)
    out = np.empty(len(p), np.float64)
    lib().oracle_temperature_profile(len(p), pp, len(k), kp, p_bot_bar, p_top_bar, out.ctypes.data_as(_dp))
    return out


def mixing_ratios(log10_vmr, he_to_h2):
    v, vp = _d(log10_vmr)
    x = np.empty(max(len(v), 1), np.float64)
    h2 = C.c_double()
    he = C.c_double()
    lib().oracle_mixing_ratios(len(v), vp, he_to_h2, x.ctypes.data_as(_dp), C.byref(h2), C.byref(he))
    return x[:len(v)], h2.value, he.value


def cell(grid, v):
    g, gp = _d(grid)
    i = C.c_int()
    w = C.c_double()
    cl = C.c_int()
    lib().oracle_cell(len(g), gp, float(v), C.byref(i), C.byref(w), C.byref(cl))
    return i.value, w.value, bool(cl.value)


def interp_sigma(table, T_grid, log10p_grid, T, log10p):
    """table float32 [N_T][N_P][N_nu] -> (sigma float64 [N_nu], clamped)."""
    t, tp = _f(table)
    tg, tgp = _d(T_grid)
    pg, pgp = _d(log10p_grid)
    nT, nP, nNu = t.shape
    out = np.empty(nNu, np.float64)
    cl = C.c_int()
    lib().oracle_interp_sigma(tp, nT, tgp, nP, pgp, nNu, float(T), float(log10p),
                              out.ctypes.data_as(_dp), C.byref(cl))
    return out, bool(cl.value)


def interp_cia(table, T_grid, T):
    t, tp = _f(table)
    tg, tgp = _d(T_grid)
    nT, nNu = t.shape
    out = np.empty(nNu, np.float64)
    lib().oracle_interp_cia(tp, nT, tgp, nNu, float(T), out.ctypes.data_as(_dp))
    return out


def number_density(p_bar, T):
    return float(lib().oracle_number_density(float(p_bar), float(T)))


def chi_level(x, sigma_s, x_h2, x_he, alpha_c, n_cm3):
    """sigma_s [S][N_nu], alpha_c [C][N_nu] float64 -> chi [N_nu]."""
    xs, xp = _d(x)
    sig = [np.ascontiguousarray(s, dtype=np.float64) for s in sigma_s]
    alp = [np.ascontiguousarray(a, dtype=np.float64) for a in alpha_c]
    nNu = len(sig[0]) if sig else len(alp[0])
    S, Cn = len(sig), len(alp)
    sp = (_dp * max(S, 1))(*[s.ctypes.data_as(_dp) for s in sig])
    ap = (_dp * max(Cn, 1))(*[a.ctypes.data_as(_dp) for a in alp])
    out = np.empty(nNu, np.float64)
    lib().oracle_chi_level(S, xp, sp, Cn, float(x_h2), float(x_he), ap, float(n_cm3), nNu,
                           out.ctypes.data_as(_dp))
    return out


def layer_thickness(T_lo, T_hi, p_lo_bar, p_hi_bar, mmw, g_cgs):
    return float(lib().oracle_layer_thickness(T_lo, T_hi, p_lo_bar, p_hi_bar, mmw, g_cgs))


def layer_dtau(chi_lo, chi_hi, dz):
    a, ap = _d(chi_lo)
    b, bp = _d(chi_hi)
    out = np.empty(len(a), np.float64)
    lib().oracle_layer_dtau(len(a), ap, bp, float(dz), out.ctypes.data_as(_dp))
    return out


def planck(nu_cm1, T):
    return float(lib().oracle_planck(float(nu_cm1), float(T)))


def gauss_legendre_01(n):
    mu = np.empty(n, np.float64)
    w = np.empty(n, np.float64)
    lib().oracle_gauss_legendre_01(n, mu.ctypes.data_as(_dp), w.ctypes.data_as(_dp))
    return mu, w


def sc_coefficients(D):
    e = C.c_double()
    b = C.c_double()
    g = C.c_double()
    lib().oracle_sc_coefficients(float(D), C.byref(e), C.byref(b), C.byref(g))
    return e.value, b.value, g.value


def flux_one_nu(S_levels, dtau_layers, mu, w):
    s, sp = _d(S_levels)
    d, dpp = _d(dtau_layers if len(dtau_layers) else [0.0])
    m, mp = _d(mu)
    ww, wp = _d(w)
    return float(lib().oracle_flux_one_nu(len(s), sp, dpp, len(m), mp, wp))


def convolve(nu0, dnu, F, inst_sigma):
    f, fp = _d(F)
    out = np.empty(len(f), np.float64)
    if inst_sigma is None:
        sp = None
    else:
        sg, sp = _d(inst_sigma)
    lib().oracle_convolve(len(f), nu0, dnu, fp, sp, out.ctypes.data_as(_dp))
    return out


def bin_spectrum(nu0, dnu, Fd, edges):
    f, fp = _d(Fd)
    e, ep = _d(edges)
    out = np.empty(len(e) - 1, np.float64)
    lib().oracle_bin(len(f), nu0, dnu, fp, len(e) - 1, ep, out.ctypes.data_as(_dp))
    return out


def loglike(D, err, M):
    d, dpp = _d(D)
    e, ep = _d(err)
    m, mp = _d(M)
    return float(lib().oracle_loglike(len(d), dpp, ep, mp))


EXTRA_DISTANCE, EXTRA_ERROR_INFLATION, EXTRA_GREY_CLOUD = 1, 2, 4


def loglike_inflated(D, err, M, eps):
    d, dpp = _d(D)
    e, ep = _d(err)
    m, mp = _d(M)
    return float(lib().oracle_loglike_inflated(len(d), dpp, ep, mp, float(eps)))


def lobatto_nodes(q):
    out = np.empty(q + 1, np.float64)
    if lib().oracle_lobatto_nodes(int(q), out.ctypes.data_as(_dp)):
        raise ValueError("order must be 1..4")
    return out


def tp_dofs_from_ratios(theta):
    t, tp = _d(theta)
    out = np.empty(len(t), np.float64)
    lib().oracle_tp_dofs_from_ratios(len(t), tp, out.ctypes.data_as(_dp))
    return out


def temperature_profile_fe(p_bar, n_elements, order, T_dof, p_bottom_bar, p_top_bar):
    p, pp = _d(p_bar)
    t, tp = _d(T_dof)
    assert len(t) == n_elements * order + 1
    out = np.empty(len(p), np.float64)
    if lib().oracle_temperature_profile_fe(len(p), pp, int(n_elements), int(order), tp, float(p_bottom_bar),
                                           float(p_top_bar), out.ctypes.data_as(_dp)):
        raise ValueError("bad element count / order")
    return out


def teff(nu0, dnu, F_plus, nu_a, nu_b):
    f, fp = _d(F_plus)
    return float(lib().oracle_teff(len(f), float(nu0), float(dnu), fp, float(nu_a), float(nu_b)))


def cloud_dtau(p_bar, tau_c, p_top_c, phi):
    p, pp = _d(p_bar)
    out = np.zeros(max(len(p) - 1, 1), np.float64)
    lib().oracle_cloud_dtau(len(p), pp, float(tau_c), float(p_top_c), float(phi), out.ctypes.data_as(_dp))
    return out[:len(p) - 1]


def forward(T_grid, log10p_grid, nu0, dnu, sigma, cia, n_levels, p_bottom_bar, p_top_bar,
            n_knots, n_angles, mean_mol_weight, he_to_h2, flux_const,
            bin_edges, obs, obs_err, inst_sigma, params,
            want_flux=False, want_spectra=True, want_logl=True, n_threads=0,
            tp_elements=0, tp_order=1, tp_ratio=False, extras=0, teff_range=None):
    """Whole path.  Returns dict(flux_hr, spectra, logl, n_clamped[, teff]).
    tp_elements/tp_order/tp_ratio, extras (EXTRA_* flags) and teff_range = (nu_a, nu_b)
    switch on the NEXT rows (oracle_forward_ext)."""
    sg, sgp = _f(sigma)
    S, nT, nP, nNu = sg.shape
    if cia is None or len(cia) == 0:
        Cn, cp = 0, None
    else:
        ca, cp = _f(cia)
        Cn = ca.shape[0]
    tg, tgp = _d(T_grid)
    pg, pgp = _d(log10p_grid)
    ed, edp = _d(bin_edges)
    J = len(ed) - 1
    par, parp = _d(params)
    n_t = tp_elements * tp_order + 1 if tp_elements > 0 else n_knots
    n_extra = (1 if extras & EXTRA_DISTANCE else 0) + (1 if extras & EXTRA_ERROR_INFLATION else 0) + \
              (3 if extras & EXTRA_GREY_CLOUD else 0)
    par = par.reshape(-1, 2 + n_t + S + n_extra)
    B = par.shape[0]
    if want_logl:
        ob, obp = _d(obs)
        er, erp = _d(obs_err)
    else:
        obp = erp = None
    if inst_sigma is None:
        isp = None
    else:
        isg, isp = _d(inst_sigma)
    flux = np.empty((B, nNu), np.float64) if want_flux else None
    spec = np.empty((B, J), np.float64) if want_spectra else None
    logl = np.empty(B, np.float64) if want_logl else None
    teff = np.empty(B, np.float64) if teff_range is not None else None
    ncl = lib().oracle_forward_ext(
        S, nT, tgp, nP, pgp, nNu, float(nu0), float(dnu), sgp, Cn, cp,
        int(n_levels), float(p_bottom_bar), float(p_top_bar), int(n_knots), int(n_angles),
        float(mean_mol_weight), float(he_to_h2), float(flux_const),
        J, edp, obp, erp, isp, B, parp,
        flux.ctypes.data_as(_dp) if want_flux else None,
        spec.ctypes.data_as(_dp) if want_spectra else None,
        logl.ctypes.data_as(_dp) if want_logl else None, int(n_threads),
        int(tp_elements), int(tp_order), int(bool(tp_ratio)), int(extras),
        float(teff_range[0]) if teff_range is not None else 0.0,
        float(teff_range[1]) if teff_range is not None else 0.0,
        teff.ctypes.data_as(_dp) if teff is not None else None)
    return dict(flux_hr=flux, spectra=spec, logl=logl, n_clamped=int(ncl), teff=teff)


def forward_workload(wl, params=None, want_flux=False, want_spectra=True, want_logl=True,
                     n_threads=0, obs=None, obs_err=None, **ext):
    """Convenience: run the oracle on a workloads.Workload."""
    cfg = wl.cfg
    obs = wl.obs if obs is None else obs
    obs_err = wl.obs_err if obs_err is None else obs_err
    if obs is None:
        want_logl = False
    return forward(wl.T_grid, wl.log10p_grid, cfg.nu0, cfg.dnu, wl.sigma, wl.cia,
                   cfg.n_levels, cfg.p_bottom_bar, cfg.p_top_bar, cfg.n_knots, cfg.n_angles,
                   cfg.mean_mol_weight, cfg.he_to_h2, cfg.flux_const,
                   wl.bin_edges, obs, obs_err, wl.inst_sigma,
                   wl.params if params is None else params,
                   want_flux=want_flux, want_spectra=want_spectra, want_logl=want_logl,
                   n_threads=n_threads, **ext)
