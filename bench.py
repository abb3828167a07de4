#!/usr/bin/env python
"""bench.py -- throughput of the FEW interpolated mode-summation hot path on B200 (one process per GPU).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1] [--impl ours|reference]

A step is ONE pass of the whole hot path (S0 harmonics, S2 mode selection, S1 spline fits, S3 summation; DESIGN.md
section 1) over one synthetic workload: by default BASELINE.json configs[1], the one-year single-source waveform with
eps = 1e-5 that the metric "ms per 1-yr FP64 waveform; sample*mode evals/s; % of FP64 roofline" is quoted on.
After the headline measurement the default run (N = 1, no flag) also times, for a few steps each, the other BASELINE
configurations the perf targets are stated on and reports them under `also`: config 2 (all modes: the FP64 roofline
probe), config 3 (64-source batch: spline fit and selection against HBM, host-buffer call), config 4 at eps = 1e-2 and 0.

With N > 1 the path shards with no data-path collective:
  --config 1 (default), 2   every rank runs its own copy of the workload (independent waveforms of an MCMC): "replicas", weak
  --config 3                rank r takes sources shard_sources(64, r, N): strong scaling by source
  --config 4                rank r takes samples shard_samples(N_samples, r, N) and repeats S0-S2-S1: strong scaling by time range
value = total sample*mode evaluations of all ranks / max-over-ranks time.

Prints ONE JSON line (see the keys at the bottom).  `--impl reference` times the CPU oracle instead (rank 0 only).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

FLOP_PER_EVAL = 20.0          # WORK-EQUIVALENT, per-mode form of SURVEY 8(d): complex cubic Horner (6 DFMA) + complex MAC (4 DFMA) per sample*mode
FLOP_PER_PAIR = 38.0          # WORK-EQUIVALENT, round 1's scalar (m,n)-pair form: 18 DFMA + 2 DMUL per sample*pair.  Neither is what the DMMA
                              # kernel executes (the l-merge and the +-n sharing remove work), so fractions built on them may exceed 1.
# What few_sum_kernel EXECUTES on the FP64 pipe, per sample:
#   DMMA.8x8x4: 4 per step and 8 samples (2 when m = 0), 256 FMA each -> 256 (128) flop per sample and step, zero padding included;
#   scalar DFMA/DMUL/DADD (phases, rho^nu table, run closes, output): 258 + 20 per (m, k) run thread-instructions per sample, each
#   holding one FMA slot of the pipe (counted as 2 flop).  From smsp__sass_thread_inst_executed_op_{dfma,dmul,dadd}_pred_on of the two
#   captures in profiles/r02_sum_kernel.md: 358.0 per sample at 5 runs (config 1), 477.9 at 11 runs (config 2); the SASS count of the
#   source page gives the same slope (16 per close + 4 per new P) and 267 for the constant (lanes predicated off make up the rest).
DMMA_FLOP_PER_SAMPLE_STEP = 256.0
SCALAR_FP64_PER_SAMPLE = 258.0
SCALAR_FP64_PER_SAMPLE_RUN = 20.0
DFMA_PER_CLK_PER_SM = 64      # B200 FP64 pipe: 16 lanes x 4 sub-partitions (public 37 TFLOP/s at 148 SM, 1.965 GHz)
# dram__bytes_read.sum + dram__bytes_write.sum of ONE few_sum_kernel launch: static figures from `ncu --set full` captures (the
# run itself does not measure them); the coefficient stream and h stay in the 126 MB L2 while the kernel runs
SUM_KERNEL_DRAM_TRAFFIC = {"config1_1yr_eps1e-5": 8.14e6, "config2_1yr_allmodes": 13.46e6}
SUM_KERNEL_DRAM_TRAFFIC_SOURCE = "profiles/r02_sum_kernel.md (ncu --set full, dram__bytes_read.sum + dram__bytes_write.sum; static, not measured by this run)"


def config_dict(w, **extra):
    """The `config` object: the same keys in the repo arm and in the reference arm."""
    d = {"workload": w.name, "n_src": int(w.n_src), "n_t": int(w.n_t), "n_modes": int(w.n_modes), "n_samples": int(w.n_samples),
         "dt": float(w.dt), "eps": float(w.eps)}
    d.update(extra)
    return d


def cpu_model() -> str:
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d.get("hbm_gbs", 6650.0)), float(d.get("sm_max_mhz", 1965.0)), "measured"
    return 6650.0, 1965.0, "fallback"


class ClockSampler:
    """Samples nvidia-smi clocks and throttle reasons while the timed region runs (B200_PROFILING.md clocks line)."""
    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index: int):
        self.rows, self.stop_evt, self.index = [], threading.Event(), index
        self.thread = threading.Thread(target=self._run, daemon=True)

    def _run(self):
        try:
            proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                     "-lms", "20"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            return
        try:
            while not self.stop_evt.is_set():
                line = proc.stdout.readline()
                if not line:
                    break
                self.rows.append((time.perf_counter(), [x.strip() for x in line.split(",")]))
        finally:
            proc.terminate()

    def start(self): self.thread.start()

    def stop(self, t_begin: float, t_end: float):
        self.stop_evt.set(); self.thread.join(timeout=3)
        rows = [r for (ts, r) in self.rows if t_begin <= ts <= t_end + 0.15] or [r for (_, r) in self.rows[-3:]]
        sm = [float(r[0]) for r in rows if r and r[0].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({n for r in rows for n, v in zip(names, r[3:7]) if v.lower().startswith("active")})
        mx = [float(r[1]) for r in rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        pw = [float(r[2]) for r in rows if len(r) > 2 and r[2].replace(".", "").isdigit()]
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "reasons": reasons, "samples": len(rows)}


def oracle_sample(w, target_s: float, threads: int | None = None, max_samples: int = 1 << 22):
    """Times the CPU oracle, as it stands, on a bounded contiguous slice of the workload (whole path: harmonics,
    selection, spline fits, summation).  threads = None: all host cores.  Returns (evals/s, description, cores, seconds, n, K)."""
    import oracle
    from paper_2104_04582_b200 import synth
    oracle.build()
    all_cores = oracle.num_threads()
    if threads is not None:
        oracle.set_threads(threads)
    cores = oracle.num_threads()
    mid = (w.n_samples // 2) // 256 * 256
    per_step = {}

    def run(n):
        ws = synth.Workload(w.name, w.t[:1], w.phase[:1], w.amp[:1], w.l, w.m, w.n, w.theta[:1], w.phi[:1],
                            w.t0 + mid * w.dt, w.dt, n, w.eps)
        # oracle.waveform's own chain (same calls, same order: PAPER.md:192), with a clock between the steps
        c = [time.perf_counter()]
        yp, ym = oracle.ylm_modes(ws.l, ws.m, float(ws.theta[0]), float(ws.phi[0])); c.append(time.perf_counter())
        keep, _ = oracle.select_modes(ws.amp[0], ws.m, yp, ym, ws.eps); c.append(time.perf_counter())
        ca = oracle.spline_fit(ws.t[0], np.ascontiguousarray(ws.amp[0]).view(np.float64))
        cp = oracle.spline_fit_ext(ws.t[0], ws.phase[0]); c.append(time.perf_counter())
        oracle.sum_waveform(ws.t[0], ca, cp, ws.l, ws.m, ws.n, keep, yp, ym, ws.t0, ws.dt, n); c.append(time.perf_counter())
        per_step.clear()
        per_step.update({"O2_harmonics_s": c[1] - c[0], "O3_selection_s": c[2] - c[1], "O1_spline_fits_s": c[3] - c[2],
                         "O4_summation_s": c[4] - c[3], "O4_samples": int(n), "O3_rows": int(ws.n_t), "O1_systems": int(2 * ws.n_modes + 2)})
        return c[4] - c[0], len(keep)

    try:
        # two calibration sizes separate the fixed cost (harmonics, selection, fits) from the per-sample cost
        n1, n2 = (2048, 16384) if threads is None else (256, 2048)
        t1, K = run(n1)
        t2, K = run(n2)
        per_sample = max((t2 - t1) / (n2 - n1), 1e-9)
        fixed = max(t1 - per_sample * n1, 0.0)
        n = int(min(max((target_s - fixed) / per_sample, n2), w.n_samples - mid, max_samples))
        t_run, K = run(n)
    finally:
        if threads is not None:
            oracle.set_threads(all_cores)
    oracle_sample.per_step = dict(per_step)          # seconds of each oracle step in the last (timed) run
    return n * K / t_run, f"{n} contiguous samples of source 0 from sample {mid}, whole path, K={K}", cores, t_run, n, K


def kept_structure(w, keep_h, nk_h):
    """Bookkeeping for the roofline, summed over the sources: kept modes; (m, n) pairs (all l of a pair are summed into one
    pair of splines before the sample loop); STEPS of the summation kernel = kept (m, |n| >> 2) blocks (one step = 4 DMMA.8x8x4
    per 8 samples, 2 when m = 0: DESIGN.md section 5) as (steps, steps with m = 0), and the number of (m) RUNS (the scalar close + new P per run)."""
    K = int(nk_h.sum())
    pairs = steps = single = runs = 0
    for s in range(w.n_src):
        kept = keep_h[s, : nk_h[s]]
        pairs += len({(int(w.m[j]), int(w.n[j])) for j in kept})
        blocks = {(int(w.m[j]), abs(int(w.n[j])) >> 2) for j in kept}
        steps += len(blocks)
        single += sum(1 for (mm, _) in blocks if mm == 0)
        runs += len({mm for (mm, _) in blocks})          # a run = the kept modes of one m (Schwarzschild lists: k = 0)
    return K, pairs, steps, single, runs


class Bench:
    """One workload resident on the device, and the timed step over it."""

    def __init__(self, api, torch, w, dev):
        self.api, self.torch, self.w, self.dev = api, torch, w, dev
        host = dict(t=w.t, phase=w.phase, amp=w.amp, l=w.l, m=w.m, n=w.n, theta=w.theta, phi=w.phi)
        self.pinned = {k: torch.as_tensor(np.ascontiguousarray(v)).pin_memory() for k, v in host.items()}
        self.g = {k: v.to(dev) for k, v in self.pinned.items()}
        self.h = torch.empty((w.n_src, w.n_samples), dtype=torch.complex128, device=dev)
        self.keep = torch.empty((w.n_src, w.n_modes), dtype=torch.int32, device=dev)
        self.nk = torch.empty((w.n_src,), dtype=torch.int32, device=dev)
        # the summation's workspace is laid out for the steps this mode list can produce at most (88 on the paper's grid) instead of
        # the default capacity (few.h, few_set_max_steps): same kernels, same bits, a fraction of the device memory
        self.step_bound = api.few_max_steps_for_modes(self.pinned["m"], self.pinned["n"])
        api.few_set_max_steps(self.step_bound)
        self.ws_default_bytes = api.few_waveform_workspace(w.n_src, w.n_t, w.n_modes, w.n_samples, max_steps=0)
        self.ws = torch.empty(api.few_waveform_workspace(w.n_src, w.n_t, w.n_modes, w.n_samples), dtype=torch.uint8, device=dev)

    def step(self):
        g, w = self.g, self.w
        self.api.few_waveform(g["t"], g["phase"], g["amp"], g["l"], g["m"], g["n"], g["theta"], g["phi"], w.eps, w.t0, w.dt,
                              w.n_samples, out=self.h, keep_idx=self.keep, n_keep=self.nk, workspace=self.ws)

    def warm(self, n, flush):
        for _ in range(n):
            flush.fill_(1); self.step()
        self.api.few_device_status()
        self.K, self.pairs, self.steps, self.single, self.runs = kept_structure(self.w, self.keep.cpu().numpy(), self.nk.cpu().numpy())

    def timed(self, steps, flush, barrier=None):
        """steps timed steps, L2 flushed before each (outside the event pair), CUDA events on the launch stream; the library's
        own event pair around the hot kernel gives its duration.  Returns (step ms list, hot-kernel ms list, launches)."""
        torch, api = self.torch, self.api
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        sum_ms = []
        if barrier:
            barrier()
        n0 = api.few_launch_count()
        for a, b in ev:
            flush.fill_(1)
            a.record(); self.step(); b.record()
            sum_ms.append(api.few_profile_sum_ms())       # waits for this step's hot kernel
        launches = api.few_launch_count() - n0
        if barrier:
            barrier()
        else:
            torch.cuda.synchronize()
        return [a.elapsed_time(b) for a, b in ev], sum_ms, launches

    def graph_replay(self, steps, flush):
        """The same step captured once into a CUDA graph (few_waveform is capturable: one stream, two forked and joined side
        streams, no host synchronisation, no allocation) and replayed: what is left of the CPU's share of the 12 launches."""
        torch, api = self.torch, self.api
        api.few_profile_enable(False)                   # the profiling events are not part of the captured work
        try:
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph):
                self.step()
            for _ in range(3):
                flush.fill_(1); graph.replay()
            torch.cuda.synchronize()
            ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
            for a, b in ev:
                flush.fill_(1)
                a.record(); graph.replay(); b.record()
            torch.cuda.synchronize()
            del graph
            return float(np.mean([a.elapsed_time(b) for a, b in ev]))
        finally:
            api.few_profile_enable(True)

    def e2e(self, reps, device_index):
        """The same step through few_waveform_host (C ABI, HOST pointers): H2D + kernels + D2H inside the call."""
        torch, api, w, p = self.torch, self.api, self.w, self.pinned
        h_host = torch.empty((w.n_src, w.n_samples), dtype=torch.complex128).pin_memory()
        call = lambda: api.few_waveform_host(p["t"], p["phase"], p["amp"], p["l"], p["m"], p["n"], p["theta"], p["phi"], w.eps, w.t0,
                                             w.dt, w.n_samples, out=h_host, device=device_index)
        call()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(reps):
            call()                           # synchronous: returns after the D2H copy completed
        sec = (time.perf_counter() - t0) / reps
        h2d = sum(v.numel() * v.element_size() for v in p.values())
        return sec, int(h2d), int(h_host.numel() * 16)


def sum_kernel_roofline(w, pairs, kernel_ms, sm_max_mhz, steps, single, runs, n_src=1):
    """FP64 ALU roofline of the summation kernel (table instantiation) from what it EXECUTES on the FP64 pipe (SURVEY 8(d)(i),
    H6): DMMA flop, zero padding included (256 per sample and step, 128 when m = 0) + 2 flop per scalar FP64 thread-instruction
    ((258 + 20 per run) per sample, measured: see the constants), divided by the kernel's event time and by the nominal pipe
    (148 SM x 64 FMA/clk x 2 x sm_max_mhz).  `steps`, `single`, `runs` are summed over the `n_src` sources of the launch.
    The two work-equivalents (38 flop per sample*(m,n) pair, 20 per sample*mode) are returned beside it; they count work the
    kernel no longer does and may exceed the peak."""
    peak = 148 * DFMA_PER_CLK_PER_SM * 2 * sm_max_mhz * 1e6 / 1e12
    per_s = float(w.n_samples) / (kernel_ms * 1e-3) / 1e12
    dmma = per_s * (DMMA_FLOP_PER_SAMPLE_STEP * (steps - single) + 0.5 * DMMA_FLOP_PER_SAMPLE_STEP * single)
    scalar = per_s * 2.0 * (SCALAR_FP64_PER_SAMPLE * n_src + SCALAR_FP64_PER_SAMPLE_RUN * runs)
    return {"peak": peak, "executed": dmma + scalar, "dmma": dmma, "scalar": scalar, "pair_equivalent": per_s * pairs * FLOP_PER_PAIR}


def time_stages(api, torch, w, g, flush, reps: int = 10):
    """Each C-ABI stage timed alone with CUDA events (L2 flushed before every launch); GB/s = algorithmic bytes / time:
    S1 reads 8 B and writes 32 B per knot and system; S2 reads the 16 B complex amplitude of every mode at every step."""
    yp, ym = api.few_ylm_modes(g["theta"], g["phi"], g["l"], g["m"])
    keep, nk = api.few_select_modes(g["amp"], g["m"], yp, ym, w.eps)       # eps <= 0: the identity list (all modes)
    y_amp = torch.view_as_real(g["amp"]).reshape(w.n_src, w.n_t, -1)
    coef = api.few_spline_fit(g["t"], y_amp)
    cdd = api.few_spline_fit_dd(g["t"], g["phase"])
    spl_ws = torch.empty(max(api._lib.few_spline_fit_workspace(w.n_src, w.n_t), 256), dtype=torch.uint8, device=coef.device)
    sel_ws = torch.empty(api._lib.few_select_modes_workspace(w.n_src, w.n_t, w.n_modes), dtype=torch.uint8, device=coef.device)
    sum_ws = torch.empty(api.few_sum_waveform_workspace(w.n_src, w.n_t, w.n_modes, w.n_samples), dtype=torch.uint8, device=coef.device)
    h = torch.empty((w.n_src, w.n_samples), dtype=torch.complex128, device=coef.device)
    calls = {
        "S0_ylm_modes": lambda: api.few_ylm_modes(g["theta"], g["phi"], g["l"], g["m"]),
        "S1_spline_fit": lambda: api.few_spline_fit(g["t"], y_amp, out=coef, workspace=spl_ws),
        "S1_spline_fit_dd": lambda: api.few_spline_fit_dd(g["t"], g["phase"], out=cdd),
        "S2_select_modes": lambda: api.few_select_modes(g["amp"], g["m"], yp, ym, max(w.eps, 1e-5), workspace=sel_ws),
        "S3_sum_waveform": lambda: api.few_sum_waveform(g["t"], coef, cdd, g["l"], g["m"], g["n"], keep, nk, yp, ym, w.t0, w.dt,
                                                        w.n_samples, out=h, workspace=sum_ws),
    }
    nbytes = {"S1_spline_fit": 40.0 * w.n_src * w.n_t * 2 * w.n_modes, "S2_select_modes": 16.0 * w.n_src * w.n_t * w.n_modes}
    out = {}
    for name, fn in calls.items():
        fn(); torch.cuda.synchronize()
        ts = []
        for _ in range(reps):
            flush.fill_(1)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); fn(); b.record(); torch.cuda.synchronize()
            ts.append(a.elapsed_time(b))
        out[name] = {"ms_avg": float(np.mean(ts)), "ms_min": float(min(ts))}
        if name in nbytes:
            out[name]["algorithmic_bytes"] = nbytes[name]
            out[name]["gbs"] = nbytes[name] / (float(np.mean(ts)) * 1e-3) / 1e9
    return out


def time_next(api, torch, w, g, flush, hbm_gbs, reps: int = 5, direct_samples: int = 1 << 18):
    """SURVEY.md 8(f) rows, each timed with CUDA events after an L2 flush: the detector-frame whole path (NEXT-1) against the
    source-frame one and against the separate rotation pass; the likelihood step with the inner products fused and h never
    written (NEXT-2) against the separate reduction; the direct summation (NEXT-3) against the HBM roofline."""
    from paper_2104_04582_b200 import synth
    dev = g["t"].device
    sky_h, mu_h = synth.sky_angles(w.n_src)
    sky, mu = torch.as_tensor(sky_h).to(dev), torch.as_tensor(mu_h).to(dev)
    h = torch.empty((w.n_src, w.n_samples), dtype=torch.complex128, device=dev)
    d = torch.randn((w.n_src, w.n_samples), dtype=torch.complex128, device=dev)
    ws = torch.empty(api.few_waveform_workspace(w.n_src, w.n_t, w.n_modes, w.n_samples), dtype=torch.uint8, device=dev)
    ipws = torch.empty(max(api._lib.few_inner_products_workspace(w.n_src, w.n_samples), 256), dtype=torch.uint8, device=dev)
    th, ph, fac = api.few_frame_constants(sky, mu)
    args_ = (g["t"], g["phase"], g["amp"], g["l"], g["m"], g["n"])

    def timed(fn):
        fn(); torch.cuda.synchronize()
        ts = []
        for _ in range(reps):
            flush.fill_(1)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); fn(); b.record(); torch.cuda.synchronize()
            ts.append(a.elapsed_time(b))
        return float(np.mean(ts))

    out = {}
    out["source_frame_step_ms"] = timed(lambda: api.few_waveform(*args_, th, ph, w.eps, w.t0, w.dt, w.n_samples, out=h, workspace=ws))
    out["ssb_step_ms_fused"] = timed(lambda: api.few_waveform_ssb(*args_, sky, w.eps, w.t0, w.dt, w.n_samples, mu_over_dl=mu, out=h,
                                                                  workspace=ws))
    ms = timed(lambda: api.few_frame_rotate(h, fac, out=h))
    nb = 32.0 * w.n_src * w.n_samples
    out["frame_rotate_pass"] = {"ms": ms, "algorithmic_bytes": nb, "gbs": nb / ms / 1e6, "hbm_frac": nb / ms / 1e6 / hbm_gbs}
    out["likelihood_step_ms_fused_no_h"] = timed(lambda: api.few_waveform_ssb(*args_, sky, w.eps, w.t0, w.dt, w.n_samples, mu_over_dl=mu,
                                                                              d=d, want_h=False, workspace=ws))
    out["likelihood_step_ms_fused_with_h"] = timed(lambda: api.few_waveform_ssb(*args_, sky, w.eps, w.t0, w.dt, w.n_samples,
                                                                                mu_over_dl=mu, d=d, out=h, workspace=ws))
    ms = timed(lambda: api.few_inner_products(d, h, w.dt, workspace=ipws))
    out["inner_products_pass"] = {"ms": ms, "algorithmic_bytes": nb, "gbs": nb / ms / 1e6, "hbm_frac": nb / ms / 1e6 / hbm_gbs}
    del h, d, ws
    # direct summation: the full 3843-mode grid at every sample (the slow model's summation); amplitudes are
    # device-generated noise of the workload's shape (the kernel has no data-dependent path), phases ramp to ~2e5 rad
    l_h, m_h, n_h = synth.mode_grid()
    K, N = len(l_h), int(direct_samples)
    amp = torch.empty((1, N, K), dtype=torch.complex128, device=dev)
    ar = torch.view_as_real(amp)
    for c0 in range(0, N, 1 << 14):
        ar[0, c0:c0 + (1 << 14)].normal_()
    tt = torch.arange(N, dtype=torch.float64, device=dev) * 10.0
    phase = torch.stack([tt * 6.9e-3, tt * 3.8e-3], dim=1)[None].contiguous()
    l_d, m_d, n_d = (torch.as_tensor(x).to(dev) for x in (l_h, m_h, n_h))
    yp, ym = api.few_ylm_modes(g["theta"][:1], g["phi"][:1], l_d, m_d)
    hd = torch.empty((1, N), dtype=torch.complex128, device=dev)
    dws = torch.empty(max(api._lib.few_sum_direct_workspace(1, K), 256), dtype=torch.uint8, device=dev)
    ms = timed(lambda: api.few_sum_direct(amp, phase, l_d, m_d, n_d, yp, ym, out=hd, workspace=dws))
    nb = 16.0 * N * K
    out["direct_sum"] = {"ms": ms, "n_samples": N, "n_modes": K, "algorithmic_bytes": nb, "gbs": nb / ms / 1e6,
                         "hbm_frac": nb / ms / 1e6 / hbm_gbs, "evals_per_s": N * K / (ms * 1e-3),
                         "note": "16 B per sample*mode evaluation; L2 flushed; inputs 16 GB >> L2"}
    del amp, hd, phase
    # Kerr-shaped list (NEXT-4, summation part): 42 273 modes = 7381 (m, k, n) triples, third phase, one year at dt = 10 s;
    # all modes, then the 4000 strongest at mid-trajectory (a kept list of the size selection would hand over)
    wk = synth.make_kerr()
    main_bound = api.few_max_steps_for_modes(torch.as_tensor(w.m), torch.as_tensor(w.n))
    api.few_set_max_steps(api.few_max_steps_for_modes(torch.as_tensor(wk.m), torch.as_tensor(wk.n), torch.as_tensor(wk.k)))   # 11 m x 11 k x 8 blocks
    tk = torch.as_tensor(wk.t).to(dev)
    coef = api.few_spline_fit(tk, torch.as_tensor(wk.amp).to(dev))
    cdd = api.few_spline_fit_dd(tk, torch.as_tensor(wk.phase).to(dev))
    lk, mk, kk, nk_ = (torch.as_tensor(x).to(dev) for x in (wk.l, wk.m, wk.k, wk.n))
    ypk, ymk = api.few_ylm_modes(g["theta"][:1], g["phi"][:1], lk, mk)
    hk = torch.empty((1, wk.n_samples), dtype=torch.complex128, device=dev)
    kws = torch.empty(api.few_sum_waveform_workspace(1, wk.n_t, wk.n_modes, wk.n_samples), dtype=torch.uint8, device=dev)
    out["kerr_shaped_sum"] = {}
    for label, n_keep in (("all_modes", None), ("kept_4000", 4000)):
        keep = nkeep = None
        triples = len({(int(a), int(b), int(c)) for a, b, c in zip(wk.m, wk.k, wk.n)})
        if n_keep is not None:
            idx = np.sort(np.argsort(-np.abs(wk.amp[0, wk.n_t // 2]))[:n_keep]).astype(np.int32)
            pad = np.full((1, wk.n_modes), -1, np.int32); pad[0, :n_keep] = idx
            keep, nkeep = torch.as_tensor(pad).to(dev), torch.as_tensor(np.array([n_keep], np.int32)).to(dev)
            triples = len({(int(wk.m[j]), int(wk.k[j]), int(wk.n[j])) for j in idx})
        api.few_profile_enable(True)
        ms = timed(lambda: api.few_sum_waveform_kerr(tk, coef, cdd, lk, mk, kk, nk_, keep, nkeep, ypk, ymk, wk.t0, wk.dt, wk.n_samples,
                                                     out=hk, workspace=kws))
        kern_ms = api.few_profile_sum_ms()
        K = wk.n_modes if n_keep is None else n_keep
        fl = FLOP_PER_PAIR * wk.n_samples * triples
        out["kerr_shaped_sum"][label] = {"ms": ms, "sum_kernel_ms": kern_ms, "kept_modes": K, "mkn_triples": triples,
                                         "evals_per_s": wk.n_samples * K / (ms * 1e-3), "tflops_pair_equivalent": fl / (kern_ms * 1e-3) / 1e12}
    # the Kerr-shaped chain on the device: S2 on 100 rows of 78 507 entries (streamed keys), S1 on 84 546 systems, S3 on the kept list
    amp_k = torch.as_tensor(wk.amp).to(dev)
    ph_k = torch.as_tensor(wk.phase).to(dev)
    sel_ws = torch.empty(api._lib.few_select_modes_workspace(1, wk.n_t, wk.n_modes), dtype=torch.uint8, device=dev)
    keep_k = torch.empty((1, wk.n_modes), dtype=torch.int32, device=dev)
    nkeep_k = torch.empty((1,), dtype=torch.int32, device=dev)
    ms_sel = timed(lambda: api.few_select_modes(amp_k, mk, ypk, ymk, wk.eps, keep_idx=keep_k, n_keep=nkeep_k, workspace=sel_ws))
    ms_fit = timed(lambda: api.few_spline_fit(tk, amp_k, out=coef))
    nb_sel, nb_fit = 16.0 * wk.n_t * wk.n_modes, 40.0 * wk.n_t * 2 * wk.n_modes

    def chain():
        api.few_select_modes(amp_k, mk, ypk, ymk, wk.eps, keep_idx=keep_k, n_keep=nkeep_k, workspace=sel_ws)
        api.few_spline_fit(tk, amp_k, out=coef)
        api.few_spline_fit_dd(tk, ph_k, out=cdd)
        api.few_sum_waveform_kerr(tk, coef, cdd, lk, mk, kk, nk_, keep_k, nkeep_k, ypk, ymk, wk.t0, wk.dt, wk.n_samples, out=hk, workspace=kws)
    ms_chain = timed(chain)
    Kk = int(nkeep_k.item())
    out["kerr_shaped_chain"] = {"eps": wk.eps, "kept_modes": Kk, "step_ms": ms_chain, "evals_per_s": wk.n_samples * Kk / (ms_chain * 1e-3),
                                "select": {"ms": ms_sel, "rows": wk.n_t, "entries_per_row": int(wk.n_modes + np.count_nonzero(wk.m > 0)),
                                           "algorithmic_bytes": nb_sel, "gbs": nb_sel / ms_sel / 1e6},
                                "spline_fit": {"ms": ms_fit, "algorithmic_bytes": nb_fit, "gbs": nb_fit / ms_fit / 1e6,
                                               "hbm_frac": nb_fit / ms_fit / 1e6 / hbm_gbs}}
    api.few_set_max_steps(main_bound)
    return out


def reference_arm(args):
    """--impl reference: the CPU oracle on the host cores, each step a bounded sample of the same workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from paper_2104_04582_b200 import synth
    w = synth.make_config(args.config, eps=args.eps)
    per_step = max(6.0, min(30.0, 120.0 / max(args.steps + args.warmup, 1)))
    vals, times = [], []
    desc = cores = None
    for i in range(args.warmup + args.steps):
        v, desc, cores, t_run, n, K = oracle_sample(w, per_step if i >= args.warmup else 2.0)
        if i >= args.warmup:
            vals.append(v); times.append(t_run)
    value = float(np.mean(vals))
    out = {"impl": "reference", "metric": METRIC, "value": value,
           "unit": "evals/s", "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": 1e3 * float(np.mean(times)), "higher_is_better": True, "scaling": parallelism_label(w, args.config, args.gpus)[1], "vs_baseline": None,
           "dtype": "f64", "data": "synthetic", "config": config_dict(w, parallelism=parallelism_label(w, args.config, args.gpus)[0]),
           "cpu_baseline": {"value": value, "unit": "evals/s", "cores": cores, "kind": "oracle", "sample": desc, "cpu_model": cpu_model()},
           "e2e": {"value": value, "unit": "evals/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(out), flush=True)
    return 0


METRIC = "sample*mode evaluations per second (1-yr FP64 waveform, whole hot path)"


def parallelism_label(w, config: int, world: int):
    """(label, scaling) of the split `--gpus world --config config` runs; the same in both arms."""
    if world == 1:
        return "single GPU", "weak"
    if config == 3:
        return f"by source, {world} x {w.n_src // world} sources, no collective", "strong"
    if config == 4:
        return f"by contiguous time range, {world} x ~{w.n_samples // world} samples, S0-S2-S1 repeated per rank, no collective", "strong"
    return f"{world} independent replicas (one waveform per GPU, an MCMC's walkers), no collective", "weak"


def shard_workload(w, config: int, rank: int, world: int):
    """The rank's share of the workload.  No data-path collective."""
    from paper_2104_04582_b200 import synth
    from paper_2104_04582_b200.shard import shard_samples, shard_sources, shard_t0
    if world > 1 and config == 3:
        s0, sc = shard_sources(w.n_src, rank, world)
        return synth.Workload(w.name, w.t[s0:s0 + sc], w.phase[s0:s0 + sc], w.amp[s0:s0 + sc], w.l, w.m, w.n, w.theta[s0:s0 + sc],
                              w.phi[s0:s0 + sc], w.t0, w.dt, w.n_samples, w.eps)
    if world > 1 and config == 4:
        i0, cnt = shard_samples(w.n_samples, rank, world)
        return synth.Workload(w.name, w.t, w.phase, w.amp, w.l, w.m, w.n, w.theta, w.phi, shard_t0(w.t0, w.dt, i0), w.dt, cnt, w.eps)
    return w


def also_configs(api, torch, dev, flush, hbm_gbs, sm_max_mhz, local):
    """The other BASELINE configurations the perf targets are stated on, a few steps each (N = 1 default run only)."""
    from paper_2104_04582_b200 import synth
    out = {}

    def short(w, steps=4, warm=3):
        b = Bench(api, torch, w, dev)
        b.warm(warm, flush)
        step_ms, sum_ms, launches = b.timed(steps, flush)
        kms = float(np.mean(sum_ms))
        rf = sum_kernel_roofline(w, b.pairs, kms, sm_max_mhz, b.steps, b.single, b.runs, w.n_src)
        r = {"workload": w.name, "eps": float(w.eps), "kept_modes": b.K, "mn_pairs": b.pairs, "kernel_steps": b.steps,
             "steps_m0": b.single, "runs": b.runs, "steps": steps, "workspace_bytes": int(b.ws.numel()), "workspace_default_bytes": int(b.ws_default_bytes),
             "ms_per_step": float(np.mean(step_ms)), "kernel_ms": kms, "tflops": rf["executed"], "frac": rf["executed"] / rf["peak"],
             "dmma_tflops_executed": rf["dmma"], "dmma_share_of_pipe": rf["dmma"] / rf["peak"],
             "scalar_fp64_share_of_pipe": rf["scalar"] / rf["peak"],
             "pair_equivalent_frac": rf["pair_equivalent"] / rf["peak"],
             "evals_per_s": float(w.n_samples) * b.K / (float(np.mean(step_ms)) * 1e-3), "gpu_launches_per_step": launches / steps}
        return b, r

    b, out["config2"] = short(synth.make_config(2))
    del b
    for eps, key in ((1e-2, "config4_eps1e-2"), (0.0, "config4_eps0")):
        b, out[key] = short(synth.make_config(4, eps=eps), steps=3)
        del b
    torch.cuda.empty_cache()
    w3 = synth.make_config(3)
    b, r = short(w3, steps=3)
    st = time_stages(api, torch, w3, b.g, flush, reps=20)
    for name, key in (("S1_spline_fit", "S1"), ("S2_select_modes", "S2")):
        r[key] = {"ms": st[name]["ms_avg"], "gbs": st[name]["gbs"], "hbm_frac": st[name]["gbs"] / hbm_gbs,
                  "algorithmic_bytes": st[name]["algorithmic_bytes"]}
    r["output_bytes"] = 16.0 * w3.n_src * w3.n_samples
    del b.h
    sec, h2d, d2h = b.e2e(2, local)
    r["e2e_ms"] = 1e3 * sec
    r["e2e_h2d_bytes"], r["e2e_d2h_bytes"] = h2d, d2h
    out["config3"] = r
    del b
    torch.cuda.empty_cache()
    return out


def self_launch(args) -> int:
    """`python bench.py --gpus N` without torchrun: start N copies of this command, one rank per GPU (RANK, LOCAL_RANK, WORLD_SIZE,
    MASTER_ADDR = 127.0.0.1, a free MASTER_PORT), exactly what `python -m torch.distributed.run --nproc-per-node N` would set up.
    Rank 0 prints the one JSON line.  Fails loudly when the node has fewer than N GPUs: never a silent 1-GPU run labelled N."""
    import socket
    n = args.gpus
    if not args.dry_shard:
        import torch
        have = torch.cuda.device_count() if torch.cuda.is_available() else 0
        if have < n:
            sys.exit(f"bench.py: --gpus {n} needs {n} CUDA devices on this node, found {have}")
    sock = socket.socket(); sock.bind(("127.0.0.1", 0)); port = sock.getsockname()[1]; sock.close()
    procs = []
    for r in range(n):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE=str(n), LOCAL_WORLD_SIZE=str(n), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, os.path.abspath(__file__), *sys.argv[1:]], env=env))
    rcs = [p.wait() for p in procs]
    bad = [(r, rc) for r, rc in enumerate(rcs) if rc != 0]
    if bad:
        print(f"bench.py: ranks failed (rank, exit code): {bad}", file=sys.stderr)
        return 1
    return 0


def dry_shard(args) -> int:
    """--dry-shard: the host side of a --gpus N run with no GPU in it (gloo): rendezvous from the environment, the rank's share of
    the workload (shard_workload), barrier, max-over-ranks and sum-over-ranks reductions as the timed run does them; rank 0 prints
    one line.  Workload shapes only: nothing is computed."""
    import torch
    import torch.distributed as dist
    from paper_2104_04582_b200 import synth
    world, rank = int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("RANK", "0"))
    if world > 1:
        dist.init_process_group("gloo")
    w_full = synth.make_config(0) if args.config == 4 else synth.random_problem(9, n_src=7, n_modes=5, n_samples=96)
    w = shard_workload(w_full, args.config, rank, world)
    parallelism, scaling = parallelism_label(w_full, args.config, world)
    share = torch.tensor([float(w.n_src) * float(w.n_samples)], dtype=torch.float64)
    t = torch.tensor([float(rank + 1)], dtype=torch.float64)
    if world > 1:
        dist.barrier()
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        allsh = [torch.zeros(1, dtype=torch.float64) for _ in range(world)]
        dist.all_gather(allsh, share)
    else:
        allsh = [share]
    if rank == 0:
        print(json.dumps({"dry_shard": True, "n_gpus": world, "ranks_seen": len(allsh), "max_over_ranks": float(t.item()),
                          "scaling": scaling, "parallelism": parallelism, "source_samples_per_rank": [float(x.item()) for x in allsh],
                          "source_samples_total": float(w_full.n_src) * float(w_full.n_samples)}), flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=1, help="BASELINE.json config index (1 = headline; 2, 3, 4 for profiling and sharded scaling)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-also", action="store_true", help="skip the short runs of configs 2, 3, 4 that the default run appends")
    ap.add_argument("--eps", type=float, default=None)
    ap.add_argument("--stages", action="store_true", help="also time every C-ABI stage on its own (S0, S1, S2, S3) and report GB/s")
    ap.add_argument("--next", action="store_true", help="also time the SURVEY 8(f) rows: detector frame, fused inner products, direct sum")
    ap.add_argument("--dry-shard", action="store_true",
                    help="no GPU work: go through the launch, rendezvous (gloo), sharding and max-over-ranks reduction of a --gpus N run and "
                         "print one line with each rank's share (what the CPU test of the multi-GPU entry point runs)")
    args = ap.parse_args()
    if args.impl == "reference":
        return reference_arm(args)
    if args.gpus < 1:
        ap.error("--gpus must be >= 1")
    if "WORLD_SIZE" not in os.environ and args.gpus > 1:
        return self_launch(args)                  # plain `python bench.py --gpus N`: start the N ranks ourselves
    if int(os.environ.get("WORLD_SIZE", "1")) != args.gpus:
        sys.exit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={os.environ.get('WORLD_SIZE')}: launch with --nproc-per-node {args.gpus} "
                 f"(or without torchrun: bench.py starts its own ranks)")
    if args.dry_shard:
        return dry_shard(args)
    args.warmup = max(args.warmup, 3)

    import torch
    import torch.distributed as dist
    from paper_2104_04582_b200 import api, synth

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a GPU (no CPU fallback)"
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.device("cuda", local)

    w_full = synth.make_config(args.config, eps=args.eps)
    w = shard_workload(w_full, args.config, rank, world)
    parallelism, scaling = parallelism_label(w_full, args.config, world)
    bench = Bench(api, torch, w, dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)            # > 126 MB L2
    api.few_profile_enable(True)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    bench.warm(args.warmup, flush)
    K_kept, pairs, bench_steps, bench_single, bench_runs = bench.K, bench.pairs, bench.steps, bench.single, bench.runs
    bench_ws = (bench.ws.numel(), bench.ws_default_bytes, bench.step_bound)
    evals_per_step = float(w.n_samples) * K_kept

    # FP64 peak probe (register-resident DFMA chains), timed alone: the measured denominator beside the nominal one
    sink = torch.empty(148 * 8 * 256, dtype=torch.float64, device=dev)
    api.few_fp64_peak_probe(148 * 8, 256, 2000, sink)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize(); e0.record()
    probe_flops = api.few_fp64_peak_probe(148 * 8, 256, 20000, sink)
    e1.record(); torch.cuda.synchronize()
    fp64_measured_tflops = probe_flops / (e0.elapsed_time(e1) * 1e-3) / 1e12

    sampler = ClockSampler(local) if rank == 0 else None
    if sampler:
        sampler.start(); time.sleep(0.3)
    t_begin = time.perf_counter()
    step_ms, sum_ms, launches = bench.timed(args.steps, flush, barrier)
    t_end = time.perf_counter()
    total_ms = torch.tensor([sum(step_ms)], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(total_ms, op=dist.ReduceOp.MAX)
        ev_all = torch.tensor([evals_per_step, float(K_kept), float(pairs)], dtype=torch.float64, device=dev)
        dist.all_reduce(ev_all, op=dist.ReduceOp.SUM)
        evals_all = float(ev_all[0].item())
    else:
        evals_all = evals_per_step
    clocks = sampler.stop(t_begin, t_end) if sampler else None
    ms_per_step = float(total_ms.item()) / args.steps
    value = evals_all / (ms_per_step * 1e-3)

    # e2e: the same metric through the C-ABI call with HOST buffers (H2D of the inputs and D2H of h inside the timed region)
    e2e = None
    if not args.no_e2e:
        barrier()
        sec, h2d, d2h = bench.e2e(max(3, min(args.steps, 10)), local)
        t_e2e = torch.tensor([sec], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(t_e2e, op=dist.ReduceOp.MAX)
        e2e = {"value": evals_all / float(t_e2e.item()), "unit": "evals/s", "ms_per_step": 1e3 * float(t_e2e.item()),
               "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
               "note": "few_waveform_host (C ABI, host pointers): H2D of the sparse inputs + kernels + D2H of h, pinned host buffers"}

    graph_ms = None
    if world == 1 and not args.no_e2e:
        try:
            graph_ms = bench.graph_replay(args.steps, flush)
        except Exception as exc:                      # a measurement aid: the line stays valid without it
            graph_ms = f"unavailable: {exc}"

    hbm_gbs, sm_max_mhz, peak_kind = load_peaks()
    stages = None
    if args.stages and rank == 0:
        stages = time_stages(api, torch, w, bench.g, flush)
    nxt = None
    default_run = world == 1 and args.config == 1 and args.eps is None and not args.no_also
    if (args.next or default_run) and rank == 0:
        # in full with --next; the default N = 1 line carries a compact block (3 timed calls per row)
        del bench.h
        nxt = time_next(api, torch, w, bench.g, flush, hbm_gbs, reps=5 if args.next else 3)
        if not args.next:
            nxt = {"source_frame_step_ms": nxt["source_frame_step_ms"], "ssb_step_ms_fused": nxt["ssb_step_ms_fused"],
                   "likelihood_step_ms_fused_no_h": nxt["likelihood_step_ms_fused_no_h"],
                   "inner_products_pass_ms": nxt["inner_products_pass"]["ms"],
                   "direct_sum": {k: nxt["direct_sum"][k] for k in ("ms", "gbs", "hbm_frac")},
                   "kerr_shaped_chain": {k: nxt["kerr_shaped_chain"][k] for k in ("step_ms", "kept_modes", "evals_per_s")},
                   "note": "SURVEY 8(f) rows on this workload, 3 timed calls each after an L2 flush; `--next` prints the full block"}
    also = None
    if default_run:
        del bench
        torch.cuda.empty_cache()
        also = also_configs(api, torch, dev, flush, hbm_gbs, sm_max_mhz, local)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    sum_ms_avg = float(np.mean(sum_ms))
    rf = sum_kernel_roofline(w, pairs, sum_ms_avg, sm_max_mhz, bench_steps, bench_single, bench_runs, w.n_src)
    achieved_tflops, peak_tflops = rf["executed"], rf["peak"]
    nominal_tflops = evals_per_step * FLOP_PER_EVAL / (sum_ms_avg * 1e-3) / 1e12
    traffic = SUM_KERNEL_DRAM_TRAFFIC.get(w.name) if (args.eps is None and world == 1) else None
    roofline = {"bound": "alu", "kernel": "few_sum_kernel (table instantiation; the recurrence instantiation is launched too and returns at once unless a source needs it)", "achieved": achieved_tflops, "peak": peak_tflops, "unit": "TFLOP/s",
                "frac": achieved_tflops / peak_tflops, "traffic": traffic,
                "traffic_source": SUM_KERNEL_DRAM_TRAFFIC_SOURCE if traffic is not None else None,
                "peak_kind": f"nominal FP64 pipe: 148 SM x 64 DFMA/clk x 2 x {sm_max_mhz:.0f} MHz (sm_max_mhz {peak_kind})",
                "achieved_kind": "EXECUTED FP64 flop per launch on this rank / kernel event time: n_samples x [256 x (kernel_steps - steps_m0) + 128 x steps_m0 "
                                 f"(DMMA.8x8x4, zero padding included) + 2 x ({SCALAR_FP64_PER_SAMPLE:.0f} x n_src + {SCALAR_FP64_PER_SAMPLE_RUN:.0f} x runs) (scalar DFMA/DMUL/DADD "
                                 "thread-instructions, one FMA slot each; counts from profiles/r02_sum_kernel.md)]",
                "peak_measured_dfma_probe": fp64_measured_tflops, "frac_of_measured_probe": achieved_tflops / fp64_measured_tflops,
                "kernel_ms": sum_ms_avg, "kernel_share_of_step": sum_ms_avg / float(np.mean(step_ms)),
                "kernel_steps": bench_steps, "steps_m0": bench_single, "runs": bench_runs,
                "executed_dmma": {"tflops": rf["dmma"], "share_of_pipe": rf["dmma"] / peak_tflops},
                "executed_scalar_fp64": {"tflops": rf["scalar"], "share_of_pipe": rf["scalar"] / peak_tflops,
                                         "thread_instructions_per_sample": SCALAR_FP64_PER_SAMPLE + SCALAR_FP64_PER_SAMPLE_RUN * bench_runs / max(w.n_src, 1)},
                "pair_equivalent": {"achieved": rf["pair_equivalent"], "frac": rf["pair_equivalent"] / peak_tflops,
                                    "note": f"WORK-EQUIVALENT, may exceed 1: {FLOP_PER_PAIR:.0f} flop (round 1's scalar (m,n)-pair form) per sample*(m,n)-pair x "
                                            f"{float(w.n_samples) * pairs:.4g} pair evaluations per launch on this rank ({pairs} pairs from {K_kept} kept modes); the DMMA form "
                                            "executes 32 FMA per unit where two pairs were counted as 2 x 19"},
                "nominal_per_mode": {"achieved": nominal_tflops, "frac": nominal_tflops / peak_tflops,
                                     "note": "WORK-EQUIVALENT, may exceed 1: 20 flop per sample*mode evaluation (per-mode form, SURVEY 8(d)); all l of an "
                                             "(m,n) pair are summed into one spline before the sample loop, so the kernel does less"}}
    cpu = None
    if not args.no_cpu_baseline:
        v, desc, cores, t_run, n, K = oracle_sample(w, 12.0)
        cpu = {"value": v, "unit": "evals/s", "cores": cores, "kind": "oracle", "sample": desc, "seconds": t_run, "cpu_model": cpu_model(),
               "per_step": dict(oracle_sample.per_step, note="seconds of the oracle's steps inside the timed sample (PAPER.md:342, 350 quote "
                                "CPU/GPU ratios per step): O3 selection on every sparse row, O1 fits of all systems, O4 summation of the slice")}
        v1, desc1, cores1, t1, n1, K1 = oracle_sample(w, 8.0, threads=1, max_samples=1 << 18)
        cpu["one_core"] = {"value": v1, "unit": "evals/s", "cores": cores1, "sample": desc1, "seconds": t1,
                           "note": "the paper's CPU convention is one core (PAPER.md:332, 378)"}
    out = {"metric": METRIC, "value": value, "unit": "evals/s",
           "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True,
           "scaling": scaling, "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": config_dict(w_full, parallelism=parallelism),
           "kept_modes": K_kept, "mn_pairs": pairs, "timing": "L2 flushed between timed steps (256 MiB write); CUDA events on the launch stream; max over ranks",
           "ms_per_waveform": ms_per_step / w_full.n_src, "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e,
           "workspace": {"bytes": int(bench_ws[0]), "default_bytes": int(bench_ws[1]), "max_steps": int(bench_ws[2]),
                         "note": "few_waveform workspace of this rank with the step bound few_max_steps_for_modes gives for the mode list "
                                 "(few_set_max_steps), against the default capacity"},
           "gpu_launches": int(launches), "gpu_launches_note": "counted by the library at its launch sites (few_launch_count) over the timed steps of this rank",
           "clocks": clocks, "step_ms_min": min(step_ms), "step_ms_max": max(step_ms)}
    if graph_ms is not None:
        out["graph_replay"] = {"ms_per_step": graph_ms,
                               "note": "the same few_waveform call captured once into a CUDA graph and replayed (L2 flushed, CUDA events): "
                                       "the step without the host's share of its launches; `value` and `ms_per_step` are the plain call"}
    if stages is not None:
        for v in stages.values():
            if "gbs" in v:
                v["hbm_frac"] = v["gbs"] / hbm_gbs
        out["stages"] = stages
        out["stages_hbm_peak_gbs"] = hbm_gbs
    if nxt is not None:
        out["next"] = nxt
    if also is not None:
        out["also"] = also
        out["also_hbm_peak_gbs"] = hbm_gbs
    print(json.dumps(out), flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
