"""bench.py -- throughput of the batched Helios-r2 forward model on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config I] [--impl reference]

A "step" is one pass of the whole hot path (profile prep -> interpolate ->
optical depth -> RT -> convolve/bin/chi-square) over one batch of synthetic
input, through the C ABI (helios_forward_batch; spectra and logL written).
Default workload: BASELINE.json configs[3] (high-resolution opacity sampling,
85 001 wavenumbers x 150 levels x 8 angles, 1.66 GB of tables, B = 1024), the
largest single-GPU configuration; --config 4 is the likelihood-only stream
(16 x 256), --config 0..2 the smaller ones, --workload teff the T_eff
post-processing workload.
Prints ONE JSON line.
"""
import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

import workloads  # noqa: E402

# Fallback only (used when helios_measure_peaks is unavailable): 148 SMs x 128 FP32 lanes x 1.965 GHz
# (guide unit counts, clocks.max.sm), 1 FMA = 2 flop; 16 MUFU results per clock per SM.
NOMINAL_FMA_PER_CLK_SM, NOMINAL_MUFU_PER_CLK_SM, NOMINAL_SM_MHZ = 128.0, 16.0, 1965.0
HBM_NOMINAL_GBS = 8000.0
# dram__bytes_read.sum + dram__bytes_write.sum of the dominant kernel, per launch, from the
# ncu --set full captures summarised in profiles/ (None until captured for this workload).
NCU_TRAFFIC_BYTES = {2: 220606720 + 8583680,        # profiles/r02_k_rt_slab_cfg2_ncu_full.txt
                     3: 3734714000 + 2687789000}    # profiles/r02_k_rt_slab_cfg3_ncu_full.txt (flux: scattered 4-byte writes)


def algorithmic_ops(cfg):
    """FMA-class fp32 ops and MUFU ops per (model, nu) point, as the METHOD defines them
    (4-tap bilinear per species, 2-tap per CIA pair)."""
    L, S, C, A = cfg.n_levels, cfg.n_species, cfg.n_cia, cfg.n_angles
    fma = L * (4 * S + 2 * C) + 2 * (L - 1) + 4 * L + 6 * (L - 1) * A
    mufu = 2 * L + (L - 1) * (A + 1)
    return fma, mufu


def must_move_bytes(cfg, B):
    """BASELINE.json's HBM roofline numerator: table bytes + parameter and output bytes."""
    table = 4 * cfg.n_nu * len(cfg.T_grid) * (cfg.n_species * len(cfg.log10p_grid) + cfg.n_cia)
    P = 2 + cfg.n_knots + cfg.n_species
    return table + B * P * 8 + B * cfg.n_bins * 4 + B * 8


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            return json.load(open(path)), "measured"
        except Exception:
            pass
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.proc = None
        self.tmp = None

    def start(self):
        try:
            self.tmp = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=self.tmp, stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        self.tmp.flush()
        rows = [r.strip().split(",") for r in open(self.tmp.name) if r.strip()]
        os.unlink(self.tmp.name)
        sm, reasons = [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            try:
                sm.append(float(r[0]))
                out["sm_max_mhz"] = float(r[1])
                for n, v in zip(names, r[3:7]):
                    if v.strip().lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                continue
        if sm:
            out["sm_mhz"] = float(np.median(sm))
        out["reasons"] = sorted(reasons)
        out["samples"] = len(sm)
        return out


def oracle_sample_size(wl, cfg, cores, target_s=15.0):
    """Bounded sample: about `target_s` seconds of wall time on all cores.  One model per core is
    timed first (a fraction of a second to a few seconds) and the count scaled from that."""
    probe = min(cores, cfg.batch)
    dt, _ = time_oracle(wl, probe)
    per_model_core_s = dt * min(cores, probe) / probe
    n = int(target_s * cores / max(per_model_core_s, 1e-4))
    n = max(probe, (n // cores) * cores if n >= cores else n)
    return max(1, min(n, cfg.batch))


def time_oracle(wl, n_models, repeats=1, min_wall_s=0.0, n_threads=0):
    """The oracle as it stands (never tuned), all host cores (n_threads = 0) or n_threads, table generation excluded.
    Returns (mean wall seconds of one pass over n_models models, threads).  Passes are repeated
    until `min_wall_s` of work has been timed, so a whole-batch sample that takes only a second
    or two (configs[1], [2]) is still a 10 s measurement."""
    import oracle
    params = np.ascontiguousarray(wl.params[:n_models])
    total, passes = 0.0, 0
    while passes < repeats or total < min_wall_s:
        t0 = time.perf_counter()
        oracle.forward_workload(wl, params=params, want_spectra=True, want_logl=wl.obs is not None, n_threads=n_threads)
        total += time.perf_counter() - t0
        passes += 1
        if passes >= 200:
            break
    return total / passes, (n_threads if n_threads > 0 else oracle.max_threads())


def workload_for(args):
    """(cfg, workload name).  --workload teff: the T_eff post-processing workload (Sect. 2.6, PAPER.md:223-227;
    SURVEY.md 8(f) NEXT-3) = helios_teff_batch over 500-10 000 cm^-1 (1-20 micron) on the configs[2] tables and grid."""
    index = 2 if args.workload == "teff" and args.config < 0 else (3 if args.config < 0 else args.config)
    cfg = workloads.get_config(index)
    if args.batch > 0:
        import dataclasses
        cfg = dataclasses.replace(cfg, batch=args.batch * cfg.n_calls)
    name = f"configs[{cfg.index}] {cfg.name}"
    if args.workload == "teff":
        name = f"teff: T_eff over 500-10000 cm^-1 on {name}"
    return cfg, name


def run_reference(args):
    """--impl reference: the fp64 CPU oracle on this box's host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    cfg, name = workload_for(args)
    # the opacity tables (1.6 GB at configs[3]) are synthesised with torch on the GPU when there is one -- input
    # preparation, cached under /tmp and never timed; the oracle itself runs on the host cores only
    try:
        import torch
        gen_device = "cuda" if torch.cuda.is_available() else "cpu"
    except Exception:
        gen_device = "cpu"
    wl = workloads.make_workload(cfg.index, batch=cfg.batch if cfg.n_calls == 1 else cfg.batch // cfg.n_calls, device=gen_device)
    import oracle
    cores = oracle.max_threads()
    # keep the whole --steps K --warmup W run within a few minutes: ~60 s of oracle time in total
    n = oracle_sample_size(wl, cfg, cores, target_s=min(15.0, 60.0 / max(1, args.steps)))
    for _ in range(args.warmup):
        time_oracle(wl, min(n, cores), n_threads=cores)
    t = [time_oracle(wl, n, n_threads=cores)[0] for _ in range(args.steps)]
    dt = float(np.mean(t))
    value = n / dt
    sample = f"{n} of {cfg.batch} models of configs[{cfg.index}] per step, all nu/levels/bins"
    line = {
        "impl": "reference", "metric": "forward_models_per_s", "value": value, "unit": "models/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": name, "batch_per_step": n, "n_nu": cfg.n_nu,
                   "n_levels": cfg.n_levels, "n_species": cfg.n_species, "n_cia": cfg.n_cia,
                   "n_angles": cfg.n_angles, "n_bins": cfg.n_bins},
        "points_per_s": value * cfg.n_nu,
        "cpu_baseline": {"value": value, "unit": "models/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": "models/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def other_workloads(h3, wl3, pk, local, dev):
    """The other workloads north_star names, each under its own clock sample, appended to the default line so that they
    are measured by whoever runs `python bench.py`: configs[2] at B = 256 (the batch the
    target is quoted on), configs[4] (16 back-to-back logL-only calls on one stream, ONE event pair around the 16
    enqueues: SURVEY.md 8(d)), and B = 1 / 8 on the configs[2] tables (the paper's own usage).
    Inputs resident in HBM, tables larger than L2 (no flush), >= 3 warm-up steps, CUDA events, device pointers."""
    import torch
    from paper_1910_01070_b200 import Helios, helios_forward_batch, helios_loglike_batch
    peaks, _ = measured_peaks()
    n_sms = pk.get("n_sms", 148)
    fma_clk = max(pk["ffma_per_clk_sm"], pk["ffma2_per_clk_sm"])
    out = []

    def measure(name, cfg, h, params, n_calls, want_spec, min_s):
        B = params.shape[0]
        B_call = B // n_calls
        p = torch.as_tensor(params, device=dev)
        spec = torch.empty((B, cfg.n_bins), dtype=torch.float32, device=dev) if want_spec else None
        logl = torch.empty((B,), dtype=torch.float64, device=dev)

        def step():
            for c in range(n_calls):
                sl = slice(c * B_call, (c + 1) * B_call)
                if want_spec:
                    helios_forward_batch(h.ctx, p[sl], spec[sl], logl[sl])
                else:
                    helios_loglike_batch(h.ctx, p[sl], logl[sl])

        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        for _ in range(3):
            step()
        e0.record(); step(); e1.record(); torch.cuda.synchronize()
        steps = int(min(5000, max(5, min_s * 1e3 / max(e0.elapsed_time(e1), 1e-3))))
        sampler = ClockSampler(local)
        torch.cuda.synchronize()
        sampler.start()
        e0.record()
        for _ in range(steps):
            step()
        e1.record()
        torch.cuda.synchronize()
        clocks = sampler.stop()
        ms_step = e0.elapsed_time(e1) / steps
        fma, _ = algorithmic_ops(cfg)
        sm_mhz = clocks.get("sm_mhz") or pk["sm_clock_mhz"]
        alu_peak = fma_clk * n_sms * 2.0 * sm_mhz * 1e6 / 1e12
        ach = 2.0 * fma * B * cfg.n_nu / (ms_step * 1e-3) / 1e12        # whole step (prep + RT + observation) in the denominator
        bytes_move = must_move_bytes(cfg, B_call)
        gbs = bytes_move / (ms_step / n_calls * 1e-3) / 1e9
        out.append({"workload": name, "batch": B, "calls_per_step": n_calls, "spectra_written": bool(want_spec),
                    "steps": steps, "warmup": 4, "ms_per_step": ms_step, "value": B / (ms_step * 1e-3), "unit": "models/s",
                    "points_per_s": B * cfg.n_nu / (ms_step * 1e-3),
                    "roofline": {"bound": "alu", "achieved": ach, "peak": alu_peak, "unit": "TFLOP/s", "frac": ach / alu_peak,
                                 "note": "algorithmic FMAs x 2 / WHOLE-STEP time (all three kernels), so a lower bound on "
                                         "the RT kernel's own fraction"},
                    "hbm_roofline": {"must_move_bytes_per_call": bytes_move, "achieved_gbs": gbs,
                                     "frac_of_8TBs": gbs / HBM_NOMINAL_GBS, "frac_of_measured": gbs / peaks["hbm_gbs"],
                                     "note": "BASELINE's definition counts the WHOLE table; a call of a few models fetches "
                                             "only the table cells those models cross, so the fraction can exceed 1 at B = 1"},
                    "clocks": clocks})

    # configs[4] on the context that already holds the configs[3] tables, atmosphere and observation
    cfg4 = workloads.get_config(4)
    measure(f"configs[4] {cfg4.name}", cfg4, h3, workloads.draw_params(cfg4, cfg4.batch), cfg4.n_calls, False, 0.9)
    cfg2 = workloads.get_config(2)
    wl2 = workloads.make_workload(2, device="cuda")
    h2 = Helios(local)
    h2.setup_workload(wl2)
    measure(f"configs[2] {cfg2.name}", cfg2, h2, wl2.params, 1, True, 0.5)
    for b in (1, 8):
        measure(f"configs[2] tables, B = {b} (one sampler point per call: PAPER.md:245)", cfg2, h2, wl2.params[:b], 1, True, 0.3)
    h2.close()
    return out



def run_gpu(args):
    import torch
    import torch.distributed as dist
    from paper_1910_01070_b200 import Helios

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)

    cfg, wl_name = workload_for(args)
    teff = args.workload == "teff"
    n_calls = cfg.n_calls                       # configs[4]: 16 back-to-back calls per step
    B_call = cfg.batch // n_calls
    wl = workloads.make_workload(cfg.index, batch=cfg.batch, device="cuda")
    # replicas: every rank evaluates its own cfg.batch models against replicated tables, no data-path
    # collective; rank r draws different parameter vectors.
    if rank > 0:
        rng = np.random.default_rng([cfg.seed, rank])
        wl.params = wl.params[rng.permutation(cfg.batch)]
    want_spec = cfg.spectra_out and not teff

    h = Helios(local)
    h.setup_workload(wl)
    h.set_kernel(args.kernel, args.models_per_cta)
    h.set_fused_obs(args.fused_obs)
    # measured FP32-FMA / MUFU rates of THIS GPU, before the timed region (the roofline denominators)
    try:
        pk = h.measure_peaks()
        peak_src = "measured by helios_measure_peaks on this GPU just before the timed region"
    except Exception as exc:          # keep the bench alive; say that the peak is nominal
        pk = {"ffma_per_clk_sm": NOMINAL_FMA_PER_CLK_SM, "ffma2_per_clk_sm": NOMINAL_FMA_PER_CLK_SM,
              "mufu_per_clk_sm": NOMINAL_MUFU_PER_CLK_SM, "sm_clock_mhz": NOMINAL_SM_MHZ, "n_sms": 148}
        peak_src = f"nominal fallback ({exc})"
    P = wl.params.shape[1]
    p_dev = torch.as_tensor(wl.params, device=dev)
    spec = torch.empty((cfg.batch, cfg.n_bins), dtype=torch.float32, device=dev) if want_spec else None
    logl = torch.empty((cfg.batch,), dtype=torch.float64, device=dev)
    p_host = torch.as_tensor(wl.params).pin_memory()
    spec_host = torch.empty((cfg.batch, cfg.n_bins), dtype=torch.float32).pin_memory() if want_spec else None
    logl_host = torch.empty((cfg.batch,), dtype=torch.float64).pin_memory()
    NU_A, NU_B = 500.0, 10000.0

    from paper_1910_01070_b200 import (helios_forward_batch, helios_forward_batch_host, helios_teff_batch,
                                       helios_teff_batch_host)

    def step_device():
        for c in range(n_calls):
            s = slice(c * B_call, (c + 1) * B_call)
            if teff:
                helios_teff_batch(h.ctx, p_dev[s], NU_A, NU_B, logl[s])
            else:
                helios_forward_batch(h.ctx, p_dev[s], spec[s] if want_spec else None, logl[s])

    def step_host():
        for c in range(n_calls):
            s = slice(c * B_call, (c + 1) * B_call)
            if teff:
                helios_teff_batch_host(h.ctx, p_host[s], NU_A, NU_B, logl_host[s])
            else:
                helios_forward_batch_host(h.ctx, p_host[s], spec_host[s] if want_spec else None, logl_host[s])

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # Timing hygiene: the tables of configs[2..4] (244 MB .. 1.6 GB) exceed the 126 MB L2, so every step
    # re-reads them from HBM.  Smaller tables (configs[0], [1]) would stay L2-resident from one step to
    # the next: then 256 MiB are written between steps to flush L2 and only the steps themselves are summed.
    table_bytes = wl.sigma.nbytes + wl.cia.nbytes
    flush_l2 = table_bytes < 1.5 * 126e6 and not os.environ.get("HELIOS_BENCH_NOFLUSH")
    scratch = torch.empty(256 << 20, dtype=torch.uint8, device=dev) if flush_l2 else None

    def timed(fn, steps, sampler=None):
        """K steps between a barrier + synchronize on both sides.  Total = first event to last event
        (flush time subtracted when L2 is flushed between steps); every step also has its own event
        pair, for the median and the minimum."""
        barrier()
        if sampler:
            sampler.start()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        for e0, e1 in ev:
            if flush_l2:
                scratch.zero_()
            e0.record()
            fn()
            e1.record()
        barrier()
        per_step = [e0.elapsed_time(e1) for e0, e1 in ev]
        ms = float(sum(per_step)) if flush_l2 else ev[0][0].elapsed_time(ev[-1][1])
        clocks = sampler.stop() if sampler else None
        if world > 1:
            t = torch.tensor([ms], device=dev, dtype=torch.float64)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            ms = float(t.item())
        return ms, clocks, per_step

    for _ in range(max(args.warmup, 3)):
        step_device()
    h.stats(reset=True)
    ms, clocks, per_step = timed(step_device, args.steps, ClockSampler(local) if rank == 0 else None)
    st = h.stats(reset=True)
    # per-stage device times: a separate, untimed pass with the library's own CUDA events between the kernels (those
    # events serialise the kernels, which the timed region above launches as programmatic dependents)
    h.set_timing(True)
    for _ in range(max(3, min(args.steps, 64 // n_calls))):
        step_device()
    stage = h.stage_ms()
    h.set_timing(False)
    h.stats(reset=True)
    for _ in range(2):
        step_host()
    ms_host, _, per_step_host = timed(step_host, args.steps)

    ms_step = ms / args.steps
    total_models = cfg.batch * world
    value = total_models / (ms_step * 1e-3)
    e2e_value = total_models / (ms_host / args.steps * 1e-3)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    peaks, hbm_src = measured_peaks()
    fma, mufu = algorithmic_ops(cfg)
    rt_ms = stage["rt_ms"]                                    # per call, CUDA events on the ctx stream
    n_sms = pk.get("n_sms", 148)
    # peak of the binding pipe: measured FMAs per clock per SM (the better of FFMA and FFMA2) x SMs x the SM clock
    # sampled DURING the timed region (nvidia-smi), 1 FMA = 2 flop
    sm_mhz = (clocks or {}).get("sm_mhz") or pk["sm_clock_mhz"]
    fma_clk = max(pk["ffma_per_clk_sm"], pk["ffma2_per_clk_sm"])
    alu_peak = fma_clk * n_sms * 2.0 * sm_mhz * 1e6 / 1e12
    mufu_peak = pk["mufu_per_clk_sm"] * n_sms * sm_mhz * 1e6          # results / s
    points = B_call * cfg.n_nu
    ach_tflops = 2.0 * fma * points / (rt_ms * 1e-3) / 1e12
    ach_mufu = mufu * points / (rt_ms * 1e-3)
    bytes_move = must_move_bytes(cfg, B_call)
    line = {
        "metric": "forward_models_per_s", "value": value, "unit": "models/s", "n_gpus": world,
        "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms_step,
        "ms_per_step_median": float(np.median(per_step)), "ms_per_step_min": float(np.min(per_step)),
        "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": wl_name, "batch": cfg.batch, "calls_per_step": n_calls,
                   "n_nu": cfg.n_nu, "n_levels": cfg.n_levels, "n_species": cfg.n_species, "n_cia": cfg.n_cia,
                   "n_angles": cfg.n_angles, "n_bins": cfg.n_bins, "spectra_written": bool(want_spec),
                   "parallelism": f"replicas x{world}: batch per rank, tables replicated, no collective",
                   "l2": ("opacity table (%.0f MB) fits L2: 256 MiB written between timed steps, only the steps summed"
                          if flush_l2 else "opacity table (%.0f MB) exceeds the 126 MB L2; no flush")
                         % (table_bytes / 1e6),
                   "kernel": {0: "auto", 1: "direct", 2: "slab", 3: "level-parallel"}[args.kernel],
                   "fused_obs": bool(args.fused_obs)},
        "points_per_s": value * cfg.n_nu,
        "stage_ms_per_call": stage,
        "roofline": {"bound": "alu", "kernel": "fused interpolate+tau+RT (k_rt_slab / k_rt_seg)", "achieved": ach_tflops,
                     "achieved_is": "algorithmic FMAs of the method (4-tap bilinear per species and level) x 2 flop / kernel time: "
                                    "useful work per second, not pipe utilisation (ncu pipe counters: profiles/r02_*)",
                     "algorithmic_bytes": must_move_bytes(cfg, B_call),
                     "peak": alu_peak, "unit": "TFLOP/s", "frac": ach_tflops / alu_peak,
                     "traffic": NCU_TRAFFIC_BYTES.get(cfg.index) if args.batch <= 0 and not teff and not args.fused_obs else None,
                     "peak_source": peak_src, "peak_fma_per_clk_sm": fma_clk, "peak_sm_mhz": sm_mhz,
                     "algorithmic_fma_per_point": fma, "algorithmic_mufu_per_point": mufu,
                     "mufu_frac": ach_mufu / mufu_peak, "mufu_peak_per_clk_sm": pk["mufu_per_clk_sm"],
                     "nominal_frac": ach_tflops / (NOMINAL_FMA_PER_CLK_SM * 148 * 2 * NOMINAL_SM_MHZ * 1e6 / 1e12)},
        "measured_peaks": pk,
        "hbm_roofline": {"must_move_bytes_per_call": bytes_move,
                         "achieved_gbs": bytes_move / (ms_step / n_calls * 1e-3) / 1e9,
                         "frac_of_8TBs": bytes_move / (ms_step / n_calls * 1e-3) / 1e9 / HBM_NOMINAL_GBS,
                         "frac_of_measured": bytes_move / (ms_step / n_calls * 1e-3) / 1e9 / peaks["hbm_gbs"],
                         "measured_peak_gbs": peaks["hbm_gbs"], "peak_source": hbm_src,
                         "note": "north_star's target (>= 0.6 at batch >= 256) is out of reach for this method: the path "
                                 "is FP32/MUFU-bound there (SURVEY.md 8(d)); HBM binds only for B <= 8"},
        "e2e": {"value": e2e_value, "unit": "models/s", "h2d_bytes_per_step": cfg.batch * P * 8,
                "d2h_bytes_per_step": cfg.batch * ((cfg.n_bins * 4 if want_spec else 0) + 8),
                "ms_per_step_median": float(np.median(per_step_host)), "ms_per_step_min": float(np.min(per_step_host))},
        "gpu_launches": st["n_launches"],
        "clocks": clocks,
    }
    if world == 1 and not args.no_cpu_baseline:
        import oracle
        cores = oracle.max_threads()
        n = oracle_sample_size(wl, cfg, cores)
        dt, _ = time_oracle(wl, n, min_wall_s=10.0, n_threads=cores)
        line["cpu_baseline"] = {"value": n / dt, "unit": "models/s", "cores": cores, "kind": "oracle",
                                "sample": f"first {n} of {cfg.batch} models of configs[{cfg.index}], "
                                          f"all nu/levels/bins, {dt:.1f} s wall per pass, passes repeated for >= 10 s"}
        n1 = max(1, min(n, int(round(5.0 * (n / dt) / cores))))       # about 5 s on one thread
        dt1, _ = time_oracle(wl, n1, n_threads=1)
        line["cpu_baseline_1thread"] = {"value": n1 / dt1, "unit": "models/s", "cores": 1, "kind": "oracle",
                                        "sample": f"first {n1} models, one pass of {dt1:.1f} s"}
    if world == 1 and cfg.index == 3 and args.batch <= 0 and not teff and not args.no_other_workloads:
        line["other_workloads"] = other_workloads(h, wl, pk, local, dev)
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1,
                    help="ranks of the run; this script does NOT start them: launch it under torchrun "
                         "(python -m torch.distributed.run --nproc-per-node N ... bench.py --gpus N), it reads "
                         "RANK / LOCAL_RANK / WORLD_SIZE from the environment")
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=-1, help="BASELINE.json configs index (default 3; 2 for --workload teff)")
    ap.add_argument("--workload", default="forward", choices=["forward", "teff"])
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--kernel", type=int, default=0, help="0 auto, 1 direct, 2 slab, 3 level-parallel")
    ap.add_argument("--models-per-cta", type=int, default=0)
    ap.add_argument("--fused-obs", action="store_true",
                    help="HELIOS_OPT_FUSED_OBS = 1: convolve + bin in the RT kernel's epilogue, no flux buffer (DESIGN.md section 6)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-other-workloads", action="store_true",
                    help="skip the configs[2] / configs[4] / B = 1, 8 records the default configs[3] run appends")
    ap.add_argument("--batch", type=int, default=0, help="override the workload's batch size (sweeps only)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()
