#!/usr/bin/env python
"""bench.py -- pyramid-WFS frames/s, effective FFT GFLOP/s and roofline fraction on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--impl ours|reference]

A *step* is one pass of the whole hot path (field build -> separable FFT-mask-IFFT passes ->
sum_k |.|^2 -> rebin -> slopes) = one ``pyr_compute`` call on one batch of synthetic input;
a *frame* is one source at one time step (all modulation points).  Default workload: C5, the
ELT-scale config the metric's target is quoted on (BASELINE.json).  One JSON line on stdout.

  value       frames/s with inputs resident in HBM; L2 flushed between timed steps; every step
              timed with CUDA events on the launching stream; max over ranks.
  e2e         the same metric through ``pyr_compute_host`` with pinned HOST buffers (H2D of amp
              and phase, D2H of intensity and slopes inside the timed region).
  roofline    dominant kernel (k_rows) against the FP32 ALU peak, see DESIGN.md "Measurement".
  chain       north_star's whole-chain figure: nominal 2*M*B 2-D FFTs x 5 N^2 log2 N^2 flops
              per step over the step time, as a fraction of the FP32 peak.
  cpu_baseline the oracle (oracle/) timed on this box's host cores on a bounded sample.

Multi-GPU: the path does not shard (north_star: one GPU, no collectives) -> "replicas only":
under torchrun every rank runs the same workload on its own GPU, no data-path collective.
``--impl reference`` times the CPU oracle as it stands (rank 0 only).
"""
from __future__ import annotations

import argparse
import json
import math
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "pyramid_wfs_frames_per_s"
UNIT = "frames/s"
FP32_LANES_PER_SM = 128
N_SM = 148


def fp32_peak_tflops(sm_mhz: float) -> float:
    """148 SMs x 128 FP32 lanes x 2 flop (FMA) x clock."""
    return N_SM * FP32_LANES_PER_SM * 2 * sm_mhz * 1e6 / 1e12


def load_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f), "measured"
    except Exception:
        return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


# --------------------------------------------------------------------------- clocks
class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""
    REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown",
               0x40: "hw_thermal_slowdown", 0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting",
               0x10: "sync_boost"}

    def __init__(self, device_index: int, period_s: float = 0.005):
        super().__init__(daemon=True)
        self.period = period_s
        self.samples, self.reasons, self.power = [], set(), []
        self.sm_max = None
        self.ok = False
        self._stop_evt = threading.Event()
        try:
            import pynvml
            self.nv = pynvml
            pynvml.nvmlInit()
            import torch
            h = None
            try:
                uuid = str(torch.cuda.get_device_properties(device_index).uuid)
                h = pynvml.nvmlDeviceGetHandleByUUID(("GPU-" + uuid) if not uuid.startswith("GPU-") else uuid)
            except Exception:
                vis = os.environ.get("CUDA_VISIBLE_DEVICES")
                idx = device_index
                if vis:
                    try:
                        idx = int(vis.split(",")[device_index])
                    except Exception:
                        pass
                h = pynvml.nvmlDeviceGetHandleByIndex(idx)
            self.h = h
            self.sm_max = float(pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception as e:  # pragma: no cover
            self.err = repr(e)

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        while not self._stop_evt.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                try:
                    bits = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    bits = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in self.REASONS.items():
                    if bits & bit:
                        self.reasons.add(name)
                self.power.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0)
            except Exception:
                pass
            time.sleep(self.period)

    def stop(self):
        self._stop_evt.set()
        if self.is_alive():
            self.join(timeout=2.0)

    def summary(self):
        if not self.ok or not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.sm_max, "reasons": ["unavailable"], "samples": 0}
        return {"sm_mhz": statistics.median(self.samples), "sm_max_mhz": self.sm_max,
                "reasons": sorted(self.reasons), "samples": len(self.samples),
                "power_w_max": max(self.power) if self.power else None}


# --------------------------------------------------------------------------- the oracle legs
def oracle_sample(c, cores: int, budget_core_s: float = 32.0):
    """Time the oracle, as it stands, on a bounded sample of config ``c``: source 0 only and
    M' <= M modulation points (each (source, k) task costs the same: two full N x N double FFTs),
    scaled to frames/s by M'/M.  Returns (frames_per_s, description, seconds)."""
    import numpy as np
    from oracle import pyr_oracle
    from paper_2602_06688_b200 import synth
    amp, phase = synth.make_inputs(c, 0)
    per_task_s = 5e-9 * c.N * c.N * math.log2(c.N * c.N) + 1e-4   # ~0.45 core-s at N = 2048 (measured), for sizing only
    m_sub = c.M
    while m_sub > 4 and m_sub * per_task_s > budget_core_s:
        m_sub //= 2
    m_sub = max(1, min(c.M, m_sub))
    threads = max(1, min(cores, m_sub))
    t0 = time.perf_counter()
    pyr_oracle.compute(c.P, c.N, m_sub, c.r, c.b, amp[:1], phase[:1], nthreads=threads)
    dt = time.perf_counter() - t0
    frames = m_sub / c.M     # fraction of one frame's work
    desc = "config C%d: source 0, %d of %d modulation points (same N, P; all other steps whole), %d threads" % (
        c.cfg, m_sub, c.M, threads)
    return frames / dt, desc, dt, threads


def run_reference(args, c):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    cores = os.cpu_count() or 1
    use = min(cores, 32)
    vals = []
    desc, threads = "", use
    for i in range(args.warmup + args.steps):
        fps, desc, dt, threads = oracle_sample(c, use)
        if i >= args.warmup:
            vals.append((fps, dt))
    fps = len(vals) / sum(1.0 / v[0] for v in vals)
    ms = 1e3 * sum(v[1] for v in vals) / len(vals)
    line = {
        "impl": "reference", "metric": METRIC, "value": fps, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(c, "none (CPU)"),
        "cpu_baseline": {"value": fps, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": desc},
        "e2e": {"value": fps, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


def workload_config(c, l2):
    return {"workload": "C%d %s: N_pup=%d N_fft=%d n_mod=%d r_mod=%g lambda/D binning=%d batch=%d, %d%% obstruction, "
                        "Kolmogorov phase %g rad rms" % (c.cfg, c.name, c.P, c.N, c.M, c.r, c.b, c.B, c.eps_pct, c.sigma),
            "N_pup": c.P, "N_fft": c.N, "n_mod": c.M, "r_mod_lambda_over_D": c.r, "binning": c.b, "batch": c.B,
            "frames_per_step": c.B, "l2": l2, "parallelism": "replicas only (no sharding, no collectives)"}


# --------------------------------------------------------------------------- our arm
def field_stop_mask(N):
    """The built-in pyramid with a circular field stop of radius 0.3 N: a non-separable mask."""
    import numpy as np
    u = np.arange(N)
    f = np.where(u < N // 2, u, u - N).astype(np.float64)
    pyramid = np.exp(-2j * np.pi * (N / 4) * (np.abs(f)[:, None] + np.abs(f)[None, :]) / N)
    return (pyramid * ((f[:, None] ** 2 + f[None, :] ** 2) <= (0.3 * N) ** 2)).astype(np.complex64)


def cufft_side_reference(torch, synth, c, flush, reps=3):
    """Time the plain chain with torch.fft (cuFFT) and element-wise torch ops on config c: field build,
    zero-padding, fft2, mask, ifft2, |.|^2 summed over k -- what a CuPy-style implementation does.  A
    side reference point for the reader, not a baseline arm and not used by the library."""
    import numpy as np
    amp, phase = synth.make_inputs(c, 0)
    P, N, M = c.P, c.N, c.M
    a = torch.from_numpy(amp).cuda()
    ph = torch.from_numpy(phase).cuda()
    n = torch.arange(N, device="cuda")
    f = torch.where(n < N // 2, n, n - N).abs()
    e = (f[:, None] + f[None, :]) % 4
    mask = torch.polar(torch.ones_like(e, dtype=torch.float32), -0.5 * math.pi * e.to(torch.float32))
    th = 2 * math.pi * torch.arange(M, device="cuda", dtype=torch.float32) / M
    xs = torch.arange(P, device="cuda", dtype=torch.float32) - 0.5 * (P - 1)
    tilt = (2 * math.pi / P) * (c.r * torch.cos(th)[:, None, None] * xs[None, None, :]
                                + c.r * torch.sin(th)[:, None, None] * xs[None, :, None])      # [M][P][P]
    o = (N - P) // 2
    kb = max(1, min(M, int(2e9 // (N * N * 8))))          # points per batch of transforms (<= ~2 GB of fields)

    def run():
        out = []
        for s in range(c.B):
            I = torch.zeros((N, N), device="cuda")
            for k0 in range(0, M, kb):
                t = tilt[k0:k0 + kb]
                E = torch.zeros((t.shape[0], N, N), dtype=torch.complex64, device="cuda")
                E[:, o:o + P, o:o + P] = torch.polar(a[s].expand_as(t), ph[s][None] + t)
                O = torch.fft.ifft2(torch.fft.fft2(E) * mask)
                I += (O.real ** 2 + O.imag ** 2).sum(0)
            out.append(I.reshape(N // c.b, c.b, N // c.b, c.b).sum((1, 3)))
        return torch.stack(out)

    run()
    torch.cuda.synchronize()
    ts = []
    for _ in range(reps):
        flush.zero_()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        D = run()
        e1.record()
        e1.synchronize()
        ts.append(e0.elapsed_time(e1))
    ms = statistics.median(ts)
    return {"ms_per_call": ms, "frames_per_s": c.B / (ms * 1e-3), "what": "torch.fft (cuFFT) fft2/ifft2 of %d padded "
            "%dx%d fields per call + element-wise torch kernels; intensities only (no slopes)" % (2 * M * c.B, N, N),
            "checksum_rel_to_flux": float(D.sum() / (M * float((amp.astype(np.float64) ** 2).sum())))}


def time_sh(torch, synth, name, flush, reps=10, with_cpu=True):
    """Shack-Hartmann path on one of synth.SH_SHAPES: median device time of one
    sh_compute call (slopes + flux + detector pixels), sub-apertures/s, effective FFT GFLOP/s with the
    nominal 5 F^2 log2 F^2 per sub-aperture, executed flops (those of the pruned transforms the kernel in use
    has to do; modulus, moments and pixel sums not counted) and a bounded oracle sample on the host."""
    from paper_2602_06688_b200 import sh
    P, n_sub, F, bs, B, sigma = synth.SH_SHAPES[name]
    amp, phase = synth.make_sh_inputs(P, B, sigma)
    a, ph = torch.from_numpy(amp).cuda(), torch.from_numpy(phase).cuda()
    p = P // n_sub
    with sh.Plan(P, n_sub, F, bs, B) as plan:
        s, f, sp = plan.empty_outputs(spots=True)
        st = torch.cuda.Stream()
        with torch.cuda.stream(st):
            for _ in range(3):
                plan.compute(a, ph, s, f, sp)
            st.synchronize()
            ts = []
            for _ in range(reps):
                if flush is not None:
                    flush.zero_()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(st)
                plan.compute(a, ph, s, f, sp)
                e1.record(st)
                e1.synchronize()
                ts.append(e0.elapsed_time(e1))
    ms = statistics.median(ts)
    nsub = B * n_sub * n_sub
    nominal = nsub * 5.0 * F * F * math.log2(F * F)
    if p in (4, 8, 16) and F % p == 0 and (F // p) % bs == 0 and bs <= 32:
        # k_shp: (p + F) lines per sub-aperture, each F/p twisted p-point DFTs (p - 1 complex multiplies + a radix-p butterfly)
        executed = nsub * (p + F) * (F / p) * ((p - 1) * 6.0 + 5.0 * p * math.log2(p))
    else:                                               # k_sh: skinny direct contractions, 8 flops per complex FMA
        executed = nsub * 8.0 * (p * F * p + F * F * p)
    out = {"ms_per_call": ms, "subapertures_per_s": nsub / (ms * 1e-3), "effective_fft_gflops": nominal / (ms * 1e-3) / 1e9,
           "executed_tflops": executed / (ms * 1e-3) / 1e12,
           "workload": "N_pup=%d n_sub=%d (p=%d) F=%d spot_binning=%d batch=%d" % (P, n_sub, p, F, bs, B)}
    if with_cpu:
        from oracle import sh_oracle
        rows = max(1, min(n_sub, int(2.0e9 / (2.0 * F ** 3 * n_sub)) or 1))     # whole lenslet rows, ~1-2 core-s
        t0 = time.perf_counter()
        sh_oracle.compute(rows * p, rows, F, bs, amp[:1, :rows * p, :rows * p], phase[:1, :rows * p, :rows * p])
        dt = time.perf_counter() - t0
        out["cpu_oracle_subapertures_per_s"] = rows * rows / dt
        out["cpu_sample"] = "%d x %d sub-apertures of source 0, 1 thread, %.2f s" % (rows, rows, dt)
    return out


def time_chain(torch, pyr, synth, c, flush, peaks, reps=10, n_modes=4096, with_cpu=True):
    """The sensor chain resident on the device: atmo_propagate -> pyr_compute -> ccd_integrate ->
    pyr_slopes_from_pixels -> modalrec_compute on config c; per step the host sends 64 bytes of layer shifts and reads
    back only the reconstructed modes.  Reports the step time (CUDA events on the launching stream, L2 flushed), the
    end-to-end time including the D2H of the modes, and every kernel of f3 against the HBM roofline (algorithmic
    bytes of DESIGN.md section 14 over its own event-timed duration)."""
    import numpy as np
    from paper_2602_06688_b200 import chain
    L, S = 4, 1024
    rng = np.random.Generator(np.random.PCG64(99))
    f = np.fft.fftfreq(S) * S
    ff = np.hypot(f[:, None], f[None, :]); ff[0, 0] = 1.0
    filt = ff ** (-11.0 / 6.0); filt[0, 0] = 0.0
    scr = np.stack([np.real(np.fft.ifft2(np.fft.fft2(rng.standard_normal((S, S))) * filt)) for _ in range(L)])
    scr = (scr * (c.sigma / np.sqrt(L) / scr.std())).astype(np.float32)
    amp = np.stack([synth.pupil_amplitude(c.P, c.eps_pct)] * c.B)
    valid = synth.valid_from_amplitude(amp[0], c.N, c.b)
    nsv = 2 * int(valid.sum())
    R = (rng.standard_normal((n_modes, nsv)) / np.sqrt(nsv)).astype(np.float32)
    wind = np.array([[0.31, 0.07], [0.52, -0.44], [-0.9, 0.2], [3.1, 2.9]])        # pixels per step and layer
    a, d_scr = torch.from_numpy(amp).cuda(), torch.from_numpy(scr).cuda()
    out = {}
    with pyr.Plan(c.P, c.N, c.M, c.r, c.b, c.B) as plan, chain.Atmo(L, S, c.P, c.B) as atmo, \
            chain.CCD((c.B, c.N_det, c.N_det), 1, True, True, 0.4, 0.0, 16, 7) as ccd, chain.Modalrec(R, valid, c.B) as rec:
        plan.set_valid(valid)
        phase = torch.empty((c.B, c.P, c.P), device="cuda")
        I, s = plan.empty_outputs()
        px = torch.empty_like(I)
        modes = torch.empty((c.B, n_modes), device="cuda")
        modes_h = torch.empty((c.B, n_modes), dtype=torch.float32).pin_memory()
        st = torch.cuda.Stream()
        gain = 1.0e6 / (c.M * float((amp[0] ** 2).sum()))         # 1e6 photo-electrons per frame and source
        names = ["atmo_propagate", "pyr_compute", "ccd_integrate", "pyr_slopes_from_pixels", "modalrec_compute"]

        def step(i, ev=None):
            sh = np.stack([wind * i + 17.0 * b for b in range(c.B)])
            mark = (lambda k: ev[k].record(st)) if ev else (lambda k: None)
            mark(0); atmo.propagate(d_scr, sh, phase, stream=st)
            mark(1); plan.compute(a, phase, I, None, stream=st)
            mark(2); ccd.integrate(I, gain, px, stream=st)
            mark(3); plan.slopes_from_pixels(px, s, stream=st)
            mark(4); rec.compute(s, modes, stream=st)
            mark(5)

        with torch.cuda.stream(st):
            for i in range(3):
                step(i)
            st.synchronize()
            tot, per = [], {n: [] for n in names}
            for i in range(reps):
                if flush is not None:
                    flush.zero_()
                ev = [torch.cuda.Event(enable_timing=True) for _ in range(6)]
                step(3 + i, ev)
                ev[5].synchronize()
                tot.append(ev[0].elapsed_time(ev[5]))
                for k, n in enumerate(names):
                    per[n].append(ev[k].elapsed_time(ev[k + 1]))
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(st)
            for i in range(reps):
                step(100 + i)
                modes_h.copy_(modes, non_blocking=True)
                st.synchronize()
            e1.record(st)
            e1.synchronize()
            e2e_ms = e0.elapsed_time(e1) / reps
        ms = statistics.median(tot)
        kms = {n: statistics.median(v) for n, v in per.items()}
        npx = c.B * c.N_det * c.N_det
        alg_bytes = {"atmo_propagate": c.B * c.P * c.P * 4 * (L + 1),            # every layer's footprint read once + phase written
                     "ccd_integrate": npx * 4 * 4,                                 # D read, acc read + written, pixels written
                     "pyr_slopes_from_pixels": npx * 4 * 2 + c.B * 2 * c.N_q ** 2 * 4,
                     "modalrec_compute": n_modes * nsv * 4 + c.B * (nsv + n_modes) * 4}
        hbm = peaks["hbm_gbs"]
        out = {"ms_per_step": ms, "frames_per_s": c.B / (ms * 1e-3), "kernel_ms": kms,
               "e2e_ms_per_step_modes_d2h": e2e_ms, "e2e_frames_per_s": c.B / (e2e_ms * 1e-3),
               "h2d_bytes_per_step": int(c.B * L * 2 * 8), "d2h_bytes_per_step": int(c.B * n_modes * 4),
               "workload": "C%d sensor + %d layers of %dx%d screens, CCD photon + readout noise, %d modes from %d slopes"
                           % (c.cfg, L, S, S, n_modes, nsv),
               "roofline_hbm": {n: {"algorithmic_bytes": int(bts), "achieved_gbs": bts / (kms[n] * 1e-3) / 1e9,
                                    "frac_of_hbm": bts / (kms[n] * 1e-3) / 1e9 / hbm} for n, bts in alg_bytes.items()}}
        if with_cpu:
            from oracle import chain_oracle
            t0 = time.perf_counter()
            chain_oracle.atmo(scr, np.stack([wind * 3.0] * c.B)[:1], c.P)
            t_atmo = time.perf_counter() - t0
            D = I.cpu().numpy()
            det = chain_oracle.CCD(D[:1].shape, 1, True, True, 0.4, 0.0, 16, 7)
            t0 = time.perf_counter()
            det.integrate(D[:1], gain)
            t_ccd = time.perf_counter() - t0
            rows = min(n_modes, 512)
            t0 = time.perf_counter()
            chain_oracle.modalrec(R[:rows], valid, s.cpu().numpy()[:1])
            t_rec = (time.perf_counter() - t0) * n_modes / rows
            out["cpu_oracle_s_per_frame"] = {"atmo": t_atmo, "ccd": t_ccd, "modalrec": t_rec, "cores": 1,
                                             "sample": "source 0; modalrec on %d of %d rows, scaled" % (rows, n_modes)}
    return out


def time_config(pyr, synth, torch, c, reps, flush, use_graph=False, general_mask=False, l2_schedule=None):
    """Median device time (ms) of one pyr_compute call for config c (inputs resident)."""
    amp, phase = synth.make_inputs(c, 0)
    a, p = torch.from_numpy(amp).cuda(), torch.from_numpy(phase).cuda()
    with pyr.Plan(c.P, c.N, c.M, c.r, c.b, c.B) as plan:
        plan.set_valid(synth.valid_from_amplitude(amp[0], c.N, c.b))
        if general_mask:
            plan.set_mask(field_stop_mask(c.N))
        if l2_schedule is not None:
            plan.set_schedule(True, l2_schedule)
        I, s = plan.empty_outputs()
        st = torch.cuda.Stream()
        with torch.cuda.stream(st):
            for _ in range(3):
                plan.compute(a, p, I, s)
            st.synchronize()
            g = None
            if use_graph:
                g = torch.cuda.CUDAGraph()
                with torch.cuda.graph(g, stream=st):
                    plan.compute(a, p, I, s)
                g.replay()
                st.synchronize()
            ts = []
            for _ in range(reps):
                if flush is not None:
                    flush.zero_()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(st)
                if g is not None:
                    g.replay()
                else:
                    plan.compute(a, p, I, s)
                e1.record(st)
                e1.synchronize()
                ts.append(e0.elapsed_time(e1))
        return statistics.median(ts)


def run_ours(args, c):
    import numpy as np
    import torch

    from paper_2602_06688_b200 import pyr, synth   # raises if libpyr.so is missing: no fallback
    from paper_2602_06688_b200.replicas import Replicas

    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    rep = Replicas(backend="nccl", device=torch.device("cuda", local))
    rank, world = rep.rank, rep.world
    barrier, max_over_ranks = rep.barrier, rep.max_over_ranks

    peaks, peaks_kind = load_peaks()
    K, W = args.steps, args.warmup
    # every rank: its own seeded inputs (different sources per rank), resident on its device
    amp, phase = synth.make_inputs(c, 0)
    if rank:
        phase = np.stack([synth.kolmogorov_phase(c.P, amp[0], c.sigma, synth.seed_for(c.cfg, s, 0) + rep.seed_offset())
                          for s in range(c.B)])
    a, p = torch.from_numpy(amp).cuda(), torch.from_numpy(phase).cuda()
    plan = pyr.Plan(c.P, c.N, c.M, c.r, c.b, c.B)
    plan.set_valid(synth.valid_from_amplitude(amp[0], c.N, c.b))
    if args.l2_schedule:
        plan.set_schedule(True, args.l2_schedule)
    I, s = plan.empty_outputs()
    flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")   # > 126 MB L2
    st = torch.cuda.Stream()
    sampler = ClockSampler(local)

    with torch.cuda.stream(st):
        for _ in range(W):
            flush.zero_()
            plan.compute(a, p, I, s)
        st.synchronize()
        plan.set_profiling(True)
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
        kern_ms = {}
        barrier()
        torch.cuda.synchronize()
        sampler.start()
        t_wall0 = time.perf_counter()
        for i in range(K):
            flush.zero_()
            ev[i][0].record(st)
            plan.compute(a, p, I, s)
            ev[i][1].record(st)
            if not args.l2_schedule:
                for k, v in plan.last_kernel_ms().items():     # waits for this step (outside its event window)
                    kern_ms.setdefault(k, []).append(v)
        torch.cuda.synchronize()
        barrier()
        t_wall = time.perf_counter() - t_wall0
        sampler.stop()
        plan.set_profiling(False)
        step_ms = [e0.elapsed_time(e1) for e0, e1 in ev]
        total_ms = max_over_ranks(sum(step_ms))
        ms_per_step = total_ms / K
        frames = c.B * world * K
        value = frames / (total_ms * 1e-3)

        # ---- e2e: host buffers through the C ABI, every step: H2D of amp and phase from pinned memory, the kernels, D2H
        # of intensity and slopes.  (a) pyr_compute_host: synchronous, one step after the other; (b) the headline:
        # pyr_compute_host_async on two staging slots, the copies of step i + 1 overlapping the kernels of step i.
        ah = torch.from_numpy(amp).pin_memory()
        ph2 = [torch.from_numpy(phase).clone().pin_memory() for _ in range(2)]
        Ih2 = [torch.empty(I.shape, dtype=torch.float32).pin_memory() for _ in range(2)]
        sh2 = [torch.empty(s.shape, dtype=torch.float32).pin_memory() for _ in range(2)]
        ph, Ih, sh = ph2[0], Ih2[0], sh2[0]
        for _ in range(max(1, W)):
            plan.compute_host(ah, ph, Ih, sh, stream=st)
        barrier()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(st)
        for i in range(K):
            ph[0, 0, 0] = float(i) * 1e-3          # the host input changes every step
            plan.compute_host(ah, ph, Ih, sh, stream=st)
        e1.record(st)
        e1.synchronize()
        barrier()
        e2e_sync_ms = max_over_ranks(e0.elapsed_time(e1))
        for i in range(max(2, W)):
            plan.compute_host_async(ah, ph2[i % 2], Ih2[i % 2], sh2[i % 2], slot=i % 2)
            plan.host_wait(i % 2)
        barrier()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        checks = 0.0
        for i in range(K):
            k = i % 2
            ph2[k][0, 0, 0] = float(i) * 1e-3      # slot k was waited for in iteration i - 1
            plan.compute_host_async(ah, ph2[k], Ih2[k], sh2[k], slot=k)
            if i:
                plan.host_wait(1 - k)
                checks += float(sh2[1 - k][0, 0, 0, 0])      # the step's result is read on the host
        plan.host_wait((K - 1) % 2)
        checks += float(sh2[(K - 1) % 2][0, 0, 0, 0])
        e2e_ms = max_over_ranks((time.perf_counter() - t0) * 1e3)    # host clock: the copies run on the library's streams
        barrier()
        e2e_value = frames / (e2e_ms * 1e-3)
        h2d = ah.numel() * 4 + ph.numel() * 4
        d2h = Ih.numel() * 4 + sh.numel() * 4

    clocks = sampler.summary()
    if rank != 0:
        rep.close()
        return 0

    if args.l2_schedule:      # whole-step numbers of the optional schedule only
        print(json.dumps({"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
                          "ms_per_step": ms_per_step, "higher_is_better": True, "schedule": "l2_resident",
                          "j_per_chunk": args.l2_schedule, "gpu_launches": K * plan.launches_per_compute,
                          "config": workload_config(c, "flushed between timed steps"), "clocks": clocks,
                          "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h}}), flush=True)
        plan.destroy()
        rep.close()
        return 0

    # ---- roofline of the dominant kernel and of the chain
    sm_max = float(clocks.get("sm_max_mhz") or peaks.get("sm_max_mhz", 1965.0))
    peak_tf = fp32_peak_tflops(sm_max)
    kern_avg = {k: sum(v) / len(v) for k, v in kern_ms.items()}
    dom = max(kern_avg, key=kern_avg.get)
    # nominal (north_star / SURVEY 8(d)) count: forward + inverse N-point FFT per line, 5 N log2 N each
    line_flops = 2 * 5.0 * c.N * math.log2(c.N)
    lines = {"k_rows": c.B * c.N * c.M, "k_cols": c.B * (c.M // 2 + 1 if c.M % 2 == 0 else c.M) * c.P}
    alg_flops = lines.get(dom, 0) * line_flops
    achieved_tf = alg_flops / (kern_avg[dom] * 1e-3) / 1e12
    # what the half-band form actually has to execute: two N/2-point FFTs per line (N >= 32)
    # (and only N/2 + P of the N rows need a line of their own: out-of-band rows y', y' + N/2 share one)
    h = c.N // 2 if c.N >= 32 else c.N
    lines_exec = dict(lines)
    if c.N >= 32:
        lines_exec["k_rows"] = c.B * (h + c.P) * c.M
    exec_flops = lines_exec.get(dom, 0) * 2 * 5.0 * h * math.log2(h)
    exec_tf = exec_flops / (kern_avg[dom] * 1e-3) / 1e12
    traffic = None     # DRAM bytes per launch of the dominant kernel from the committed ncu capture
    try:
        import csv
        with open(os.path.join(ROOT, "profiles", "traffic.csv")) as f:
            for row in csv.DictReader(f):
                if row["config"] == "C%d" % c.cfg and row["kernel"] == dom:
                    traffic = int(row["dram_bytes_per_launch"])
    except Exception:
        pass
    try:
        peak_meas_tf, peak_meas_mhz = pyr.measure_fp32_peak()     # packed-FMA chains on every SM
    except Exception:
        peak_meas_tf, peak_meas_mhz = None, None
    nominal = c.B * c.nominal_flops_per_frame
    eff_tf = nominal / (ms_per_step * 1e-3) / 1e12
    compulsory_bytes = 2 * c.B * c.P * c.P * 4 + c.B * (c.N_det ** 2 + 2 * c.N_q ** 2) * 4
    t_roof_us = max(nominal / (peak_tf * 1e12), compulsory_bytes / (peaks["hbm_gbs"] * 1e9)) * 1e6

    # ---- the other configs (reported, not the headline) and the CPU baseline
    per_config = {}
    if world == 1 and not args.no_extras:
        for cfg in (1, 2, 3, 4, 5):
            cc = synth.CONFIGS[cfg]
            ms = time_config(pyr, synth, torch, cc, 20, flush)
            ent = {"ms_per_call": ms, "frames_per_s": cc.B / (ms * 1e-3),
                   "effective_tflops": cc.B * cc.nominal_flops_per_frame / (ms * 1e-3) / 1e12}
            ent["frac_of_fp32_peak"] = ent["effective_tflops"] / peak_tf
            if cfg <= 3:
                msg = time_config(pyr, synth, torch, cc, 20, None, use_graph=True)
                ent["graph_replay_ms_per_call_l2_warm"] = msg
            per_config["C%d" % cfg] = ent
        # side reference point only (never on the product path; north_star: "cuFFT may be timed only as a
        # side reference point"): the chain as the paper runs it -- padded fields, library 2-D FFTs and
        # element-wise kernels (torch.fft = cuFFT), all M points of one source per batch of transforms
        try:
            per_config["C%d_cufft_side_reference" % c.cfg] = cufft_side_reference(torch, synth, c, flush)
        except Exception as e:      # e.g. out of memory on a smaller device: the reference point is optional
            per_config["C%d_cufft_side_reference" % c.cfg] = {"unavailable": repr(e)[:200]}
        # the paper's own FFT sizes (not powers of two: embedded table-mask path), for context
        for name, cc in synth.PAPER_SHAPES.items():
            ms = time_config(pyr, synth, torch, cc, 10, flush)
            per_config[name] = {"ms_per_call": ms, "frames_per_s": cc.B / (ms * 1e-3),
                                "effective_tflops": cc.B * cc.nominal_flops_per_frame / (ms * 1e-3) / 1e12,
                                "frac_of_fp32_peak": cc.B * cc.nominal_flops_per_frame / (ms * 1e-3) / 1e12 / peak_tf,
                                "workload": "N_pup=%d N_fft=%d n_mod=%d binning=%d" % (cc.P, cc.N, cc.M, cc.b)}
        # second workload: Shack-Hartmann spots and centroids
        for name in synth.SH_SHAPES:
            per_config[name] = time_sh(torch, synth, name, flush)
            per_config[name]["executed_frac_of_fp32_peak"] = per_config[name]["executed_tflops"] / peak_tf
        # the L2-resident launch schedule (pyr_plan_set_schedule): the two passes per chunk of 4 y-tilts, R a 92 MB ring
        if c.N == 2048:
            msl = time_config(pyr, synth, torch, c, 10, flush, l2_schedule=4)
            per_config["C%d_l2_resident_schedule" % c.cfg] = {
                "ms_per_call": msl, "frames_per_s": c.B / (msl * 1e-3), "j_per_chunk": 4,
                "note": "R never leaves L2 (DRAM traffic in profiles/README.md r2) at the price of 2 x 9 launches whose "
                        "row grids are 2.5 waves each and 9 epilogues per row: slower, not the default"}
        # the steps either side of the sensor, resident on the device
        per_config["C%d_sensor_chain_on_device" % c.cfg] = time_chain(torch, pyr, synth, c, flush, peaks,
                                                                      with_cpu=not args.no_cpu_baseline)
        # the general (non-separable mask) three-pass path on the same workload, for reference
        msg = time_config(pyr, synth, torch, c, 5, flush, general_mask=True)
        per_config["C%d_general_mask" % c.cfg] = {
            "ms_per_call": msg, "frames_per_s": c.B / (msg * 1e-3),
            "effective_tflops": c.B * c.nominal_flops_per_frame / (msg * 1e-3) / 1e12,
            "frac_of_fp32_peak": c.B * c.nominal_flops_per_frame / (msg * 1e-3) / 1e12 / peak_tf,
            "mask": "pyramid with a circular field stop (pyr_plan_set_mask)"}
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        cores = min(os.cpu_count() or 1, 32)
        fps, desc, dt, threads = oracle_sample(c, cores)
        cpu = {"value": fps, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": desc, "seconds": dt}
        fps1, desc1, dt1, _ = oracle_sample(c, 1, budget_core_s=3.0)      # also single-threaded
        cpu["single_thread"] = {"value": fps1, "sample": desc1, "seconds": dt1}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": workload_config(c, "flushed between timed steps (512 MiB memset), per-step CUDA events"),
        "effective_fft_gflops": eff_tf * 1e3,
        # achieved = the flops the implemented (exact) form of the method has to execute per launch
        # over the kernel's measured time; `nominal` = the same with north_star's count (N-point FFTs
        # on all N rows), which the half-band identities undercut -- hence a nominal fraction > 1.
        "roofline": {"bound": "alu", "kernel": dom, "achieved": exec_tf, "peak": peak_tf, "unit": "TFLOP/s",
                     "frac": exec_tf / peak_tf, "traffic": traffic,
                     "peak_measured": peak_meas_tf, "peak_measured_sm_mhz": peak_meas_mhz,
                     "frac_of_peak_measured": (exec_tf / peak_meas_tf) if peak_meas_tf else None,
                     "peak_source": "148 SM x 128 FP32 lanes x 2 x %.0f MHz (clocks.max.sm); HBM %s %.0f GB/s"
                                    % (sm_max, peaks_kind, peaks["hbm_gbs"]),
                     "dram_gbs": (traffic / (kern_avg[dom] * 1e-3) / 1e9) if traffic else None,
                     "dram_frac_of_hbm": (traffic / (kern_avg[dom] * 1e-3) / 1e9 / peaks["hbm_gbs"]) if traffic else None,
                     "kernel_ms": kern_avg, "algorithmic_flops_per_launch": exec_flops,
                     "algorithmic_flops": "lines x 2 FFTs x 5 L log2 L, L = N/2 (half-band form), "
                                          "lines = B (N/2 + P) M for k_rows, B J P for k_cols (DESIGN.md 6.3, 6.4, 7)",
                     "nominal": {"flops_per_launch": alg_flops, "achieved": achieved_tf, "frac": achieved_tf / peak_tf,
                                 "note": "north_star / SURVEY 8(d) count: B N M (k_rows) lines x 2 x 5 N log2 N"}},
        "chain": {"nominal_flops_per_step": nominal, "effective_tflops": eff_tf, "frac_of_fp32_peak": eff_tf / peak_tf,
                  "roofline_us_per_step": t_roof_us, "frac_of_roofline": t_roof_us / (ms_per_step * 1e3),
                  "frac_at_sustained_clock": (eff_tf / fp32_peak_tflops(clocks["sm_mhz"])) if clocks.get("sm_mhz") else None},
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "ms_per_step": e2e_ms / K,
                "how": "pyr_compute_host_async on two staging slots (H2D, kernels, D2H of consecutive steps overlap); "
                       "host wall clock over all steps, every step's slopes read on the host",
                "synchronous": {"value": frames / (e2e_sync_ms * 1e-3), "ms_per_step": e2e_sync_ms / K,
                                "how": "pyr_compute_host, one step after the other, CUDA events"}},
        "gpu_launches": K * plan.launches_per_compute,
        "clocks": clocks,
        "wall_s_timed_region": t_wall,
        "per_config": per_config,
        "cpu_baseline": cpu,
    }
    print(json.dumps(line), flush=True)
    plan.destroy()
    rep.close()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=None)
    ap.add_argument("--config", type=int, default=5, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-extras", action="store_true", help="skip the per-config table")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--l2-schedule", type=int, default=0, metavar="JC",
                    help="time the L2-resident launch schedule (JC y-tilts per chunk) instead of the default single pass; "
                         "whole-step numbers only (used for the DRAM-traffic capture)")
    ap.add_argument("--sh", default=None, help="time only the Shack-Hartmann path on this synth.SH_SHAPES workload "
                                               "(one JSON line; used for the ncu capture of k_sh)")
    ap.add_argument("--paper", default=None, help="time only this synth.PAPER_SHAPES pyramid workload, e.g. "
                                                  "ANDES_24x1600x1600 (one JSON line; used for ncu captures)")
    args = ap.parse_args()
    from paper_2602_06688_b200 import synth
    if args.paper:
        import torch
        torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
        from paper_2602_06688_b200 import build, pyr
        build.build()
        flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")
        cc = synth.PAPER_SHAPES[args.paper]
        ms = time_config(pyr, synth, torch, cc, args.steps or 10, flush)
        print(json.dumps({"workload": args.paper, "ms_per_call": ms, "frames_per_s": cc.B / (ms * 1e-3),
                          "effective_tflops": cc.B * cc.nominal_flops_per_frame / (ms * 1e-3) / 1e12}), flush=True)
        return 0
    if args.sh:
        import torch
        torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
        flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")
        print(json.dumps({"workload": args.sh, **time_sh(torch, synth, args.sh, flush, reps=args.steps or 10,
                                                         with_cpu=not args.no_cpu_baseline)}), flush=True)
        return 0
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and args.impl != "reference":
        # `python bench.py --gpus N` without torchrun: start the N replica ranks ourselves (one process per GPU)
        import socket
        import subprocess
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
               "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        return subprocess.call(cmd)
    c = synth.CONFIGS[args.config]
    if args.impl == "reference":
        args.steps = 3 if args.steps is None else args.steps
        args.warmup = 1 if args.warmup is None else args.warmup
        return run_reference(args, c)
    args.steps = 40 if args.steps is None else args.steps
    args.warmup = max(3, 5 if args.warmup is None else args.warmup)
    return run_ours(args, c)


if __name__ == "__main__":
    sys.exit(main())
