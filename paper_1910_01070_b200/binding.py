"""Thin Python binding of include/helios.h (argument marshalling only).

Every step of the hot path runs in the CUDA kernels of libhelios_b200.so;
PyTorch supplies device memory and the CUDA stream.  There is no CPU fallback:
if the shared library is missing and cannot be built, or no CUDA device is
present, the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np

from . import build as _build

HELIOS_OK = 0
HELIOS_EINVAL, HELIOS_ENOMEM, HELIOS_ECUDA, HELIOS_ESTATE = -1, -2, -3, -4
HELIOS_PTRS_ON_DEVICE = 1
HELIOS_OPT_KERNEL = 1
HELIOS_OPT_MODELS_PER_CTA = 2
HELIOS_OPT_TIMING = 3
HELIOS_OPT_NU_ORDER = 4
HELIOS_OPT_FUSED_OBS = 5
HELIOS_OPT_GRAPHS = 6
NU_ORDER_GRID, NU_ORDER_OPACITY = 0, 1
KERNEL_AUTO, KERNEL_DIRECT, KERNEL_SLAB, KERNEL_LEVEL_PARALLEL = 0, 1, 2, 3
HELIOS_EXTRA_DISTANCE, HELIOS_EXTRA_ERROR_INFLATION, HELIOS_EXTRA_GREY_CLOUD = 1, 2, 4

_dp = C.POINTER(C.c_double)
_fp = C.POINTER(C.c_float)
_vp = C.c_void_p


class HeliosError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"helios error {code}: {msg}")
        self.code = code


class helios_stats(C.Structure):
    _fields_ = [("n_clamped", C.c_ulonglong), ("n_nonfinite", C.c_ulonglong),
                ("n_models", C.c_ulonglong), ("n_launches", C.c_ulonglong), ("n_graph_launches", C.c_ulonglong)]


class helios_peaks(C.Structure):
    _fields_ = [("sm_clock_mhz", C.c_double), ("ffma_per_clk_sm", C.c_double), ("ffma2_per_clk_sm", C.c_double),
                ("mufu_per_clk_sm", C.c_double), ("ffma2_cycles", C.c_double * 3), ("alu_extra_cycles", C.c_double),
                ("fsel_extra_cycles", C.c_double), ("ffma_3reg_cycles", C.c_double), ("mufu_extra_cycles", C.c_double),
                ("n_sms", C.c_int)]


_lib = None


def lib() -> C.CDLL:
    """Loads (building it in-tree if the sources are newer) libhelios_b200.so."""
    global _lib
    if _lib is None:
        if _build.is_stale():
            _build.build_library()
        if not os.path.exists(_build.LIB_PATH):
            raise RuntimeError("libhelios_b200.so is missing; run __graft_entry__.build()")
        L = C.CDLL(_build.LIB_PATH)
        L.helios_create.argtypes = [C.POINTER(_vp), C.c_int, _vp]
        L.helios_destroy.argtypes = [_vp]
        L.helios_destroy.restype = None
        L.helios_set_stream.argtypes = [_vp, _vp]
        L.helios_last_error.argtypes = [_vp]
        L.helios_last_error.restype = C.c_char_p
        L.helios_set_option.argtypes = [_vp, C.c_int, C.c_int]
        L.helios_load_opacity.argtypes = [_vp, C.c_int, C.c_int, _dp, C.c_int, _dp, C.c_int, C.c_double,
                                          C.c_double, C.POINTER(_vp), C.c_int, C.POINTER(_vp), C.c_uint]
        L.helios_set_atmosphere.argtypes = [_vp, C.c_int, C.c_double, C.c_double, C.c_int, C.c_int,
                                            C.c_double, C.c_double, C.c_double]
        L.helios_set_observation.argtypes = [_vp, C.c_int, _dp, _dp, _dp, _dp]
        L.helios_reserve.argtypes = [_vp, C.c_int]
        L.helios_forward_batch.argtypes = [_vp, C.c_int, C.c_int, _vp, _vp, _vp]
        L.helios_loglike_batch.argtypes = [_vp, C.c_int, C.c_int, _vp, _vp]
        L.helios_forward_highres.argtypes = [_vp, C.c_int, C.c_int, _vp, _vp]
        L.helios_forward_batch_host.argtypes = [_vp, C.c_int, C.c_int, _vp, _vp, _vp]
        L.helios_get_stats.argtypes = [_vp, C.POINTER(helios_stats), C.c_int]
        L.helios_get_angles.argtypes = [_vp, _dp, _dp]
        L.helios_get_stage_ms.argtypes = [_vp, _dp, C.POINTER(C.c_int)]
        L.helios_set_tp_elements.argtypes = [_vp, C.c_int, C.c_int, C.c_int]
        L.helios_set_extras.argtypes = [_vp, C.c_uint]
        L.helios_get_n_params.argtypes = [_vp, C.POINTER(C.c_int)]
        L.helios_teff_batch.argtypes = [_vp, C.c_int, C.c_int, _vp, C.c_double, C.c_double, _vp]
        L.helios_measure_peaks.argtypes = [_vp, C.POINTER(helios_peaks)]
        L.helios_teff_batch_host.argtypes = [_vp, C.c_int, C.c_int, _vp, C.c_double, C.c_double, _vp]
        L.helios_observe_noalloc.argtypes = [_vp, C.c_int, _vp, _vp, _vp]
        for name in ("helios_create", "helios_set_stream", "helios_set_option", "helios_load_opacity",
                     "helios_set_atmosphere", "helios_set_observation", "helios_reserve",
                     "helios_forward_batch", "helios_loglike_batch", "helios_forward_highres",
                     "helios_forward_batch_host", "helios_get_stats", "helios_get_angles",
                     "helios_get_stage_ms", "helios_set_tp_elements", "helios_set_extras", "helios_get_n_params",
                     "helios_teff_batch", "helios_measure_peaks", "helios_teff_batch_host",
                     "helios_observe_noalloc"):
            getattr(L, name).restype = C.c_int
        _lib = L
    return _lib


def _check(ctx, rc: int):
    if rc != HELIOS_OK:
        msg = lib().helios_last_error(ctx)
        raise HeliosError(rc, msg.decode() if msg else "")


def _f64(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(_dp)


# ---------------------------------------------------------------------------
# functions with the names of the C ABI
# ---------------------------------------------------------------------------
def helios_create(device: int = 0, cuda_stream: int = 0) -> int:
    h = _vp()
    rc = lib().helios_create(C.byref(h), int(device), _vp(cuda_stream))
    _check(None, rc)
    return h.value


def helios_destroy(ctx: int) -> None:
    lib().helios_destroy(_vp(ctx))


def helios_set_stream(ctx: int, cuda_stream: int) -> None:
    _check(ctx, lib().helios_set_stream(_vp(ctx), _vp(cuda_stream)))


def helios_set_option(ctx: int, key: int, value: int) -> None:
    _check(ctx, lib().helios_set_option(_vp(ctx), int(key), int(value)))


def helios_load_opacity(ctx: int, T_grid, log10p_grid, nu0: float, dnu: float, sigma, cia=None) -> None:
    """sigma: numpy float32 [S][nT][nP][nNu] or a CUDA torch tensor of that shape;
    cia: float32 [C][nT][nNu] (numpy or CUDA tensor) or None."""
    tg, tgp = _f64(T_grid)
    pg, pgp = _f64(log10p_grid)
    on_dev = hasattr(sigma, "is_cuda") and sigma.is_cuda
    keep = []

    def ptrs(arr, ndim):
        if arr is None or len(arr) == 0:
            return 0, None
        if on_dev:
            arr = arr.contiguous().float()
            keep.append(arr)
            base, step = arr.data_ptr(), arr[0].numel() * 4
        else:
            arr = np.ascontiguousarray(arr, dtype=np.float32)
            keep.append(arr)
            base, step = arr.ctypes.data, arr[0].size * 4
        assert arr.ndim == ndim
        n = arr.shape[0]
        return n, (_vp * n)(*[base + i * step for i in range(n)])

    S, sp = ptrs(sigma, 4)
    Cn, cp = ptrs(cia, 3)
    shape = tuple(sigma.shape)
    nT, nP, nNu = shape[1], shape[2], shape[3]
    assert nT == len(tg) and nP == len(pg)
    _check(ctx, lib().helios_load_opacity(_vp(ctx), S, nT, tgp, nP, pgp, nNu, float(nu0), float(dnu), sp, Cn, cp,
                                          HELIOS_PTRS_ON_DEVICE if on_dev else 0))


def helios_set_atmosphere(ctx: int, n_levels: int, p_bottom_bar: float, p_top_bar: float, n_knots: int,
                          n_angles: int, mean_mol_weight: float, he_to_h2: float, flux_const: float) -> None:
    _check(ctx, lib().helios_set_atmosphere(_vp(ctx), n_levels, p_bottom_bar, p_top_bar, n_knots, n_angles,
                                            mean_mol_weight, he_to_h2, flux_const))


def helios_set_observation(ctx: int, bin_edges, obs=None, obs_err=None, inst_sigma=None) -> None:
    e, ep = _f64(bin_edges)
    o = op = r = rp = s = sp = None
    if obs is not None:
        o, op = _f64(obs)
        r, rp = _f64(obs_err)
    if inst_sigma is not None:
        s, sp = _f64(inst_sigma)
    _check(ctx, lib().helios_set_observation(_vp(ctx), len(e) - 1, ep, op, rp, sp))


def helios_set_tp_elements(ctx: int, n_elements: int, order: int, ratio_form: bool = False) -> None:
    _check(ctx, lib().helios_set_tp_elements(_vp(ctx), int(n_elements), int(order), int(bool(ratio_form))))


def helios_set_extras(ctx: int, flags: int) -> None:
    _check(ctx, lib().helios_set_extras(_vp(ctx), int(flags)))


def helios_get_n_params(ctx: int) -> int:
    n = C.c_int()
    _check(ctx, lib().helios_get_n_params(_vp(ctx), C.byref(n)))
    return n.value


def _rows(params):
    """(B, P) of a 2-D parameter block; the C side checks P against the context."""
    if params.ndim != 2:
        raise ValueError("params must be 2-D [B][n_params]")
    return int(params.shape[0]), int(params.shape[1])


def helios_teff_batch(ctx: int, params, nu_a_cm1: float, nu_b_cm1: float, teff_out) -> None:
    """params: CUDA float64 [B][P]; teff_out: CUDA float64 [B]."""
    B, P = _rows(params)
    _check(ctx, lib().helios_teff_batch(_vp(ctx), B, P, _dev_ptr(params, "float64"), float(nu_a_cm1),
                                        float(nu_b_cm1), _dev_ptr(teff_out, "float64", (B,))))


def helios_reserve(ctx: int, max_batch: int) -> None:
    _check(ctx, lib().helios_reserve(_vp(ctx), int(max_batch)))


def _dev_ptr(t, dtype_name: str, shape=None):
    if t is None:
        return _vp(0)
    import torch
    want = getattr(torch, dtype_name)
    if not (t.is_cuda and t.dtype == want and t.is_contiguous()):
        raise ValueError(f"expected a contiguous CUDA tensor of dtype {dtype_name}")
    if shape is not None and tuple(t.shape) != tuple(shape):
        raise ValueError(f"expected an output tensor of shape {tuple(shape)}, got {tuple(t.shape)}")
    return _vp(t.data_ptr())


def helios_forward_batch(ctx: int, params, spectra_out=None, logl_out=None) -> None:
    """params: CUDA float64 [B][P]; spectra_out: CUDA float32 [B][J] or None; logl_out: CUDA float64 [B] or None."""
    B, P = _rows(params)
    if spectra_out is not None and (spectra_out.ndim != 2 or spectra_out.shape[0] != B):
        raise ValueError("spectra_out must be [B][n_bins]")
    _check(ctx, lib().helios_forward_batch(_vp(ctx), B, P, _dev_ptr(params, "float64"),
                                           _dev_ptr(spectra_out, "float32"), _dev_ptr(logl_out, "float64", (B,))))


def helios_loglike_batch(ctx: int, params, logl_out) -> None:
    B, P = _rows(params)
    _check(ctx, lib().helios_loglike_batch(_vp(ctx), B, P, _dev_ptr(params, "float64"),
                                           _dev_ptr(logl_out, "float64", (B,))))


def helios_forward_highres(ctx: int, params, flux_out) -> None:
    B, P = _rows(params)
    if flux_out is None or flux_out.ndim != 2 or flux_out.shape[0] != B:
        raise ValueError("flux_out must be [B][n_nu]")
    _check(ctx, lib().helios_forward_highres(_vp(ctx), B, P, _dev_ptr(params, "float64"),
                                             _dev_ptr(flux_out, "float32")))


def helios_observe_noalloc(ctx: int, flux, spectra_out=None, logl_out=None) -> None:
    """Instrument profile + binning + chi-square of a flux the caller already holds, without any device allocation
    inside the call (include/helios.h: for callers that run under someone else's stream capture, or whose GPU memory is
    all spoken for).  flux: CUDA float32 [B][n_nu], contiguous; spectra_out: CUDA float32 [B][n_bins] or None;
    logl_out: CUDA float64 [B] or None.  The outputs are the caller's: this wrapper allocates nothing either.
    B <= 4096 and B * ceil(n_bins / 8) <= 65536, else HeliosError(HELIOS_EINVAL)."""
    if flux is None or flux.ndim != 2:
        raise ValueError("flux must be [B][n_nu]")
    B = int(flux.shape[0])
    if spectra_out is not None and (spectra_out.ndim != 2 or spectra_out.shape[0] != B):
        raise ValueError("spectra_out must be [B][n_bins]")
    _check(ctx, lib().helios_observe_noalloc(_vp(ctx), B, _dev_ptr(flux, "float32"), _dev_ptr(spectra_out, "float32"),
                                             _dev_ptr(logl_out, "float64", (B,))))


def _host_ptr(a, dtype):
    if a is None:
        return _vp(0)
    if hasattr(a, "data_ptr"):           # (pinned) CPU torch tensor
        import torch
        want = {np.float64: torch.float64, np.float32: torch.float32}[dtype]
        if a.is_cuda or not a.is_contiguous() or a.dtype != want:
            raise ValueError(f"expected a contiguous HOST tensor of dtype {want}")
        return _vp(a.data_ptr())
    if a.dtype != dtype or not a.flags["C_CONTIGUOUS"]:
        raise ValueError(f"expected a C-contiguous numpy array of dtype {dtype}")
    return _vp(a.ctypes.data)


def helios_forward_batch_host(ctx: int, params_host, spectra_out_host=None, logl_out_host=None) -> None:
    """HOST buffers (numpy or pinned CPU tensors): H2D copy, hot path, D2H copy, stream sync."""
    B, P = _rows(params_host)
    for out, n in ((spectra_out_host, None), (logl_out_host, 1)):
        if out is not None and (out.shape[0] != B or (n == 1 and out.ndim != 1)):
            raise ValueError("output buffers must have B rows")
    _check(ctx, lib().helios_forward_batch_host(_vp(ctx), B, P, _host_ptr(params_host, np.float64),
                                                _host_ptr(spectra_out_host, np.float32),
                                                _host_ptr(logl_out_host, np.float64)))


def helios_teff_batch_host(ctx: int, params_host, nu_a_cm1: float, nu_b_cm1: float, teff_out_host) -> None:
    B, P = _rows(params_host)
    if teff_out_host is None or teff_out_host.ndim != 1 or teff_out_host.shape[0] != B:
        raise ValueError("teff_out_host must be [B]")
    _check(ctx, lib().helios_teff_batch_host(_vp(ctx), B, P, _host_ptr(params_host, np.float64), float(nu_a_cm1),
                                             float(nu_b_cm1), _host_ptr(teff_out_host, np.float64)))


def helios_get_stats(ctx: int, reset: bool = False) -> dict:
    st = helios_stats()
    _check(ctx, lib().helios_get_stats(_vp(ctx), C.byref(st), int(reset)))
    return {k: int(getattr(st, k)) for k, _ in helios_stats._fields_}


def helios_get_stage_ms(ctx: int) -> dict:
    ms = (C.c_double * 3)()
    n = C.c_int()
    _check(ctx, lib().helios_get_stage_ms(_vp(ctx), ms, C.byref(n)))
    return {"prep_ms": ms[0], "rt_ms": ms[1], "obs_ms": ms[2], "n_calls": n.value}


def helios_measure_peaks(ctx: int) -> dict:
    pk = helios_peaks()
    _check(ctx, lib().helios_measure_peaks(_vp(ctx), C.byref(pk)))
    out = {k: getattr(pk, k) for k, _ in helios_peaks._fields_ if k != "ffma2_cycles"}
    out["ffma2_cycles"] = list(pk.ffma2_cycles)
    return out


def helios_get_angles(ctx: int, n_angles: int):
    mu = np.empty(n_angles, np.float64)
    w = np.empty(n_angles, np.float64)
    _check(ctx, lib().helios_get_angles(_vp(ctx), mu.ctypes.data_as(_dp), w.ctypes.data_as(_dp)))
    return mu, w


# ---------------------------------------------------------------------------
# convenience wrapper (still marshalling only)
# ---------------------------------------------------------------------------
class Helios:
    """Owns one helios_ctx bound to torch's current CUDA stream."""

    def __init__(self, device: int = 0, stream: Optional[int] = None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1910_01070_b200 needs a CUDA device (no CPU fallback)")
        self.device = device
        if stream is None:
            stream = torch.cuda.current_stream(device).cuda_stream
        self.ctx = helios_create(device, stream)
        self.n_bins = 0
        self.n_nu = 0
        self.n_params = 0
        self._n_species = 0

    def close(self):
        if getattr(self, "ctx", None):
            helios_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def load_opacity(self, T_grid, log10p_grid, nu0, dnu, sigma, cia=None):
        helios_load_opacity(self.ctx, T_grid, log10p_grid, nu0, dnu, sigma, cia)
        self.n_nu = int(sigma.shape[3])
        self._n_species = int(sigma.shape[0])

    def set_atmosphere(self, n_levels, p_bottom_bar, p_top_bar, n_knots, n_angles, mean_mol_weight,
                       he_to_h2, flux_const=1.0):
        helios_set_atmosphere(self.ctx, n_levels, p_bottom_bar, p_top_bar, n_knots, n_angles,
                              mean_mol_weight, he_to_h2, flux_const)
        self.n_params = helios_get_n_params(self.ctx)     # extras survive this call; the context knows P

    def set_observation(self, bin_edges, obs=None, obs_err=None, inst_sigma=None):
        helios_set_observation(self.ctx, bin_edges, obs, obs_err, inst_sigma)
        self.n_bins = len(bin_edges) - 1

    def set_nu_order(self, order: int):
        """Column order of the resident tables for the NEXT load_opacity (NU_ORDER_OPACITY is the default)."""
        helios_set_option(self.ctx, HELIOS_OPT_NU_ORDER, order)

    def set_graphs(self, on: bool):
        helios_set_option(self.ctx, HELIOS_OPT_GRAPHS, 1 if on else 0)

    def set_fused_obs(self, on: bool):
        helios_set_option(self.ctx, HELIOS_OPT_FUSED_OBS, 1 if on else 0)

    def set_kernel(self, which: int, models_per_cta: int = 0):
        helios_set_option(self.ctx, HELIOS_OPT_KERNEL, which)
        helios_set_option(self.ctx, HELIOS_OPT_MODELS_PER_CTA, models_per_cta)

    def setup_workload(self, wl, with_data: bool = True):
        """wl: any object with the fields of workloads.Workload (duck-typed; no import)."""
        cfg = wl.cfg
        self.load_opacity(wl.T_grid, wl.log10p_grid, cfg.nu0, cfg.dnu, wl.sigma, wl.cia)
        self.set_atmosphere(cfg.n_levels, cfg.p_bottom_bar, cfg.p_top_bar, cfg.n_knots, cfg.n_angles,
                            cfg.mean_mol_weight, cfg.he_to_h2, cfg.flux_const)
        have = with_data and wl.obs is not None
        self.set_observation(wl.bin_edges, wl.obs if have else None, wl.obs_err if have else None, wl.inst_sigma)

    def forward_batch(self, params, want_spectra=True, want_logl=True):
        import torch
        B = params.shape[0]
        spec = torch.empty((B, self.n_bins), dtype=torch.float32, device=params.device) if want_spectra else None
        logl = torch.empty((B,), dtype=torch.float64, device=params.device) if want_logl else None
        helios_forward_batch(self.ctx, params, spec, logl)
        return spec, logl

    def loglike_batch(self, params, out=None):
        import torch
        if out is None:
            out = torch.empty((params.shape[0],), dtype=torch.float64, device=params.device)
        helios_loglike_batch(self.ctx, params, out)
        return out

    def forward_highres(self, params):
        import torch
        flux = torch.empty((params.shape[0], self.n_nu), dtype=torch.float32, device=params.device)
        helios_forward_highres(self.ctx, params, flux)
        return flux

    def forward_batch_host(self, params_host, spectra_out_host=None, logl_out_host=None):
        helios_forward_batch_host(self.ctx, params_host, spectra_out_host, logl_out_host)

    def observe_noalloc(self, flux, spectra_out=None, logl_out=None):
        if flux.shape[1] != self.n_nu or (spectra_out is not None and spectra_out.shape[1] != self.n_bins):
            raise ValueError("flux must be [B][n_nu], spectra_out [B][n_bins]")
        helios_observe_noalloc(self.ctx, flux, spectra_out, logl_out)

    def set_tp_elements(self, n_elements, order, ratio_form=False):
        helios_set_tp_elements(self.ctx, n_elements, order, ratio_form)
        self.n_params = helios_get_n_params(self.ctx)

    def set_extras(self, flags):
        helios_set_extras(self.ctx, flags)
        self.n_params = helios_get_n_params(self.ctx)

    def teff_batch(self, params, nu_a_cm1, nu_b_cm1):
        import torch
        out = torch.empty((params.shape[0],), dtype=torch.float64, device=params.device)
        helios_teff_batch(self.ctx, params, nu_a_cm1, nu_b_cm1, out)
        return out

    def set_timing(self, on: bool):
        helios_set_option(self.ctx, HELIOS_OPT_TIMING, 1 if on else 0)

    def stage_ms(self) -> dict:
        return helios_get_stage_ms(self.ctx)

    def stats(self, reset=False):
        return helios_get_stats(self.ctx, reset)

    def measure_peaks(self) -> dict:
        return helios_measure_peaks(self.ctx)
