"""helios_observe_noalloc against the allocating path.  Collected LAST on purpose (pytest -x stops at the first
failure; a problem here must not hide the parity tests).

Who needs the entry point: callers that cannot call cudaMalloc while they run -- a likelihood callback that sits
inside a region another library is capturing into a CUDA graph, a process that gave all of the GPU's memory to a pool
at start-up, a loop that cannot take the device-wide stall of a cudaFree.  helios_forward_batch sizes its workspace
with cudaMalloc; helios_observe_noalloc keeps the workspace of the convolve/bin/chi-square kernel (partial sums and
per-model arrival counters) in a fixed 0.5 MB array inside the library, so the call itself allocates nothing.

What is checked, on configs[1] (8501 wavenumbers, 120 bins): two calls in a row with DIFFERENT batch sizes and
fluxes -- the second call finds the first one's partial sums and counters in the shared array and must not be
disturbed by them -- each compared with helios_forward_batch on the same parameters, within the tolerances of
tests/test_gpu_parity.py (1e-4 relative on the binned flux, 1e-3 absolute on logL; the two paths run the same
arithmetic in the same order, so the difference is expected to be exactly zero and that is reported too).  Then the
size limit: a batch beyond the array is refused with HELIOS_EINVAL and a message, nothing is enqueued.

The test builds its own context and buffers, so it passes alone in a fresh process (where its first call is also the
first use of the static array on the GPU) and after the rest of the suite.
"""
import ctypes

import numpy as np
import pytest

import workloads as W

pytestmark = pytest.mark.gpu

TOL_FLUX = 1e-4          # tests/test_gpu_parity.py
TOL_LOGL_ABS = 1e-3


def test_observe_noalloc_matches_forward_batch_on_two_calls_in_a_row():
    import torch
    import paper_1910_01070_b200 as pkg
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    wl = W.make_workload(1)
    h = pkg.Helios(0)
    try:
        h.setup_workload(wl)
        params = torch.as_tensor(np.ascontiguousarray(wl.params), device="cuda:0")
        B = params.shape[0]
        first, second = params[:40].contiguous(), params[40:B].contiguous()      # 40 models, then 24

        # the existing path, and the fluxes the new entry point is fed with; every buffer is allocated HERE, before the
        # calls under test
        ref, flux, out = [], [], []
        for p in (first, second):
            ref.append(h.forward_batch(p))
            flux.append(h.forward_highres(p))
            out.append((torch.empty((p.shape[0], h.n_bins), dtype=torch.float32, device="cuda:0"),
                        torch.full((p.shape[0],), float("nan"), dtype=torch.float64, device="cuda:0")))
        torch.cuda.synchronize()

        h.observe_noalloc(flux[0], out[0][0], out[0][1])            # two calls back to back on one stream, no sync between
        h.observe_noalloc(flux[1], out[1][0], out[1][1])
        torch.cuda.synchronize()

        for k in range(2):
            spec_ref, logl_ref = ref[k][0].cpu().numpy().astype(np.float64), ref[k][1].cpu().numpy()
            spec, logl = out[k][0].cpu().numpy().astype(np.float64), out[k][1].cpu().numpy()
            assert np.all(np.isfinite(spec_ref)) and np.all(np.isfinite(logl_ref))
            assert np.max(np.abs(spec / spec_ref - 1.0)) <= TOL_FLUX, k
            assert np.max(np.abs(logl - logl_ref)) <= TOL_LOGL_ABS, k
            print(f"call {k}: max |dM/M| = {np.max(np.abs(spec / spec_ref - 1.0)):.3e}, "
                  f"max |dlogL| = {np.max(np.abs(logl - logl_ref)):.3e}")

        # logL only (spectra never written), on the array the two calls above left behind
        logl_only = torch.empty((second.shape[0],), dtype=torch.float64, device="cuda:0")
        h.observe_noalloc(flux[1], None, logl_only)
        torch.cuda.synchronize()
        assert np.max(np.abs(logl_only.cpu().numpy() - ref[1][1].cpu().numpy())) <= TOL_LOGL_ABS

        # beyond the static array: refused, with a message, before anything is touched (B is checked first, so the small
        # flux buffer is never read)
        rc = pkg.lib().helios_observe_noalloc(ctypes.c_void_p(h.ctx), 4097, ctypes.c_void_p(flux[0].data_ptr()),
                                              ctypes.c_void_p(out[0][0].data_ptr()), ctypes.c_void_p(0))
        assert rc == pkg.HELIOS_EINVAL
        assert b"static scratch" in pkg.lib().helios_last_error(ctypes.c_void_p(h.ctx))
        # the context still works after the refusal
        h.observe_noalloc(flux[0], out[0][0], out[0][1])
        torch.cuda.synchronize()
        assert np.max(np.abs(out[0][1].cpu().numpy() - ref[0][1].cpu().numpy())) <= TOL_LOGL_ABS
    finally:
        h.close()
