#!/usr/bin/env python
"""bench.py -- throughput of the optical forward model on workload c4 (BASELINE.json configs[4]).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]

A "step" is one simulation time step of the whole hot path: ray-trace + Shack-Hartmann images +
centre-of-gravity slopes for 6 LGS (80x80 subapertures, FFT M) and 3 NGS (2x2 subapertures,
FFT 1024), plus the science PSF (FFT 2048) accumulated into the long exposure, on 35 seeded
von Karman screens of 8192^2.  Prints ONE JSON line (see DESIGN.md section 7 for every key).
`--impl reference` times the FP64 CPU oracle on a bounded sample of the same workload.
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

METRIC = "sh_subaperture_frames_per_sec"
UNIT = "subaperture-frames/s"
FP32_LANES_PER_SM = 128
REPS = 20                      # median of >= 20 repetitions after the warm-up
# ncu-derived fields of the roofline line are NOT measured in this run: they are read from the committed raw metric
# table of the latest `ncu --set full` capture of the fused kernel (profiles/, see the .md beside it) and labelled so.
NCU_RAW_CSV = os.path.join(ROOT, "profiles", "r2_k_fused_raw.csv")


# ------------------------------------------------------------------------------ work model
def flops_per_subap_frame(n: int, M: int, n_layers: int) -> float:
    """Algorithmic FLOPs of one valid subaperture frame, exactly SURVEY.md section 8(d): trace 12 flop per sample and
    layer; pruned FFT = (n + M) 1-D transforms of 5M(log2 M - 1) + 3M; 4 flop per FFT point for |.|^2 + binning."""
    fft1d = 5.0 * M * (math.log2(M) - 1.0) + 3.0 * M
    return 12.0 * n * n * n_layers + (n + M) * fft1d + 4.0 * M * M


def ncu_static(steps_per_launch_here: int):
    """dram bytes per launch and shared-memory pipe utilisation from the committed ncu capture (None if absent)."""
    out = {"traffic": None, "smem_wavefront_frac": None, "source": None}
    try:
        import csv
        rows = list(csv.reader(open(NCU_RAW_CSV)))
        head = rows[0]
        data = [r for r in rows[1:] if len(r) == len(head) and "k_fused" in r[head.index("Kernel Name")]]
        units = rows[1] if rows[1][head.index("Kernel Name")] == "" else None
        r = data[0]

        def col(name):
            return float(r[head.index(name)].replace(",", ""))

        def scale(name):
            u = units[head.index(name)] if units else "byte"
            return {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}.get(u, 1.0)
        dram = col("dram__bytes_read.sum") * scale("dram__bytes_read.sum") + col("dram__bytes_write.sum") * scale("dram__bytes_write.sum")
        grid = r[head.index("Grid Size")] if "Grid Size" in head else ""
        steps_cap = None
        meta = NCU_RAW_CSV[:-4] + ".md"
        if os.path.exists(meta):
            import re
            m = re.search(r"steps per launch:\s*(\d+)", open(meta).read())
            steps_cap = int(m.group(1)) if m else None
        out["traffic"] = dram / steps_cap * steps_per_launch_here if steps_cap else dram
        name = "l1tex__data_pipe_lsu_wavefronts_mem_shared.sum.pct_of_peak_sustained_elapsed"
        if name in head:
            out["smem_wavefront_frac"] = col(name) / 100.0
        out["source"] = ("from_profile: " + os.path.relpath(NCU_RAW_CSV, ROOT) + " (one ncu --set full capture, grid " + grid +
                         (f", {steps_cap} steps per launch, scaled to {steps_per_launch_here}" if steps_cap else "") + "); not measured in this run")
    except Exception as ex:        # no capture committed yet, or an unexpected layout: report nothing rather than a stale constant
        out["source"] = f"unavailable ({type(ex).__name__})"
    return out


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    p = {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "source": "fallback (B200_PROFILING.md)"}
    if os.path.exists(path):
        try:
            m = json.load(open(path))
            p.update({"hbm_gbs": float(m["hbm_gbs"]), "sm_max_mhz": float(m.get("sm_max_mhz", 1965.0)),
                      "source": "measured (MEASURED_PEAKS.json)"})
        except Exception:
            pass
    return p


# ------------------------------------------------------------------------------ clocks
class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int):
        self.index, self.samples, self.reasons, self.max_mhz = index, [], set(), None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def _loop(self):
        nv = self.nv
        names = {"hw_slowdown": getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8),
                 "hw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40),
                 "sw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20),
                 "sw_power_cap": getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4)}
        while not self._stop.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            self._stop.wait(0.002)

    def start(self):
        if self.nv is not None:
            self._thr = threading.Thread(target=self._loop, daemon=True)
            self._thr.start()

    def stop(self):
        self._stop.set()
        if self._thr:
            self._thr.join()
        med = statistics.median(self.samples) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


# ------------------------------------------------------------------------------ oracle leg
def _oracle_cfg(cfg_full, host_screens, n_sub=None):
    """The workload for the oracle: the full config with host screens, or a reduced-pupil copy of it."""
    from paper_1608_00386_b200 import inputs
    M = cfg_full.wfs[0].fft
    cfg = inputs.make_config(4, n_sub=n_sub, lgs_fft=M, n_layers=len(cfg_full.layers),
                             screen_n=cfg_full.layers[0].n, with_screens=False)
    for lay, full, scr in zip(cfg.layers, cfg_full.layers, host_screens):
        lay.wind_x_mps, lay.wind_y_mps, lay.height_m, lay.weight = \
            full.wind_x_mps, full.wind_y_mps, full.height_m, full.weight
        lay.screen = scr
    return cfg


def _valid_frames(cfg, res):
    return sum(int(res["valid"][w].sum()) * len(cfg.sources_of_wfs(w)) for w in range(len(cfg.wfs)))


def oracle_sample(cfg_full, host_screens, *, n_sub=None, steps=None, warmup=0, budget_s=12.0, threads=None):
    """Time oracle.forward() (as it stands) on whole steps of the workload: every LGS and NGS sensor and the science
    PSF.  n_sub = None: the full pupil (one full c4 step per oracle step); otherwise a
    reduced-pupil copy.  steps = None: as many steps as fit the time budget (at least one)."""
    import oracle
    cfg = _oracle_cfg(cfg_full, host_screens, n_sub)
    all_threads = oracle.num_threads()
    if threads:
        oracle.set_num_threads(threads)
    try:
        t0 = time.perf_counter()
        r = oracle.forward(cfg, 0, 1, want_phase=False)                  # calibration / warm-up
        per = time.perf_counter() - t0
        frames = _valid_frames(cfg, r)
        for k in range(max(0, warmup - 1)):
            oracle.forward(cfg, k + 1, 1, want_phase=False)
        if steps is None:
            steps = max(1, min(200, int(budget_s / max(per, 1e-3))))
        t0 = time.perf_counter()
        oracle.forward(cfg, 1000, steps, want_phase=False)
        dt = time.perf_counter() - t0
        used = oracle.num_threads()
    finally:
        oracle.set_num_threads(all_threads)
    M = cfg.wfs[0].fft
    pupil = "the full pupil" if n_sub is None else f"a REDUCED pupil ({n_sub}x{n_sub} subapertures per LGS)"
    sample = (f"{steps} whole step(s) of c4 at M={M} on {pupil}: {cfg.wfs[0].n_sub}x{cfg.wfs[0].n_sub} subapertures x "
              f"{len(cfg.sources_of_wfs(0))} LGS, {len(cfg.sources_of_wfs(1))} NGS FFT {cfg.wfs[1].fft}, PSF FFT {cfg.psf_fft}, "
              f"all {len(cfg.layers)} layers of {cfg.layers[0].n}^2 screens, {frames} valid subaperture frames per step")
    return {"value": frames * steps / dt, "unit": UNIT, "cores": used, "kind": "oracle", "sample": sample,
            "seconds": dt, "steps": steps, "ms_per_step": 1e3 * dt / steps, "same_config": n_sub is None}


def host_screens_of(cfg):
    from paper_1608_00386_b200 import inputs
    inputs.screens_to_host(cfg)
    return [l.screen for l in cfg.layers]


# ------------------------------------------------------------------------------ reference arm
def run_reference(args):
    """The oracle as it stands on the host cores: each step is one whole c4 step on the full pupil when the run stays
    within a few minutes (K + W <= 60 steps), else on a reduced pupil (stated in the line)."""
    from paper_1608_00386_b200 import inputs, sharding
    rank, _, world = sharding.env_world()
    if rank != 0:
        return 0
    import torch
    dev = "cuda:0" if torch.cuda.is_available() else "cpu"
    screen_n = args.screen_n if dev != "cpu" else min(args.screen_n, 2048)
    cfg = inputs.make_config(4, lgs_fft=args.lgs_fft, screen_n=screen_n, n_layers=args.layers,
                             device=dev, keep_on_device=(dev != "cpu"))
    K, Wm = args.steps, args.warmup
    n_sub = None if K + Wm <= 60 else (20 if K + Wm <= 400 else 10)
    res = oracle_sample(cfg, host_screens_of(cfg), n_sub=n_sub, steps=K, warmup=Wm)
    line = {"impl": "reference", "metric": METRIC, "value": res["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": K, "warmup": Wm, "ms_per_step": res["ms_per_step"], "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"c4_throughput_M{args.lgs_fft}" + ("" if n_sub is None else " (bounded sample: reduced pupil)"),
                       "sample": res["sample"], "screen_n": screen_n, "same_config": res["same_config"]},
            "cpu_baseline": {"value": res["value"], "unit": UNIT, "cores": res["cores"], "kind": "oracle",
                             "sample": res["sample"], "same_config": res["same_config"]},
            "e2e": {"value": res["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------ GPU arm
def run_gpu(args):
    import numpy as np
    import torch
    from paper_1608_00386_b200 import binding, inputs, sharding
    rank, local_rank, world = sharding.init("nccl")
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device; the product has no CPU fallback")
    dev = f"cuda:{local_rank}"
    torch.cuda.set_device(local_rank)
    K, Wm, batch, R = args.steps, max(args.warmup, 3), args.batch, max(1, args.reps)   # timing rule: >= 3 warm-up steps
    t_setup = time.perf_counter()
    cfg = inputs.make_config(4, lgs_fft=args.lgs_fft, screen_n=args.screen_n, n_layers=args.layers,
                             device=dev, keep_on_device=True)
    torch.cuda.synchronize()
    t_screens = time.perf_counter() - t_setup
    geo = binding.Geometry(cfg, device=dev, workspace_steps=batch)
    if args.phase_maps:      # NEXT-1: a static aberration map on every source, synthetic smooth field
        gen = torch.Generator(device=dev); gen.manual_seed(1608)
        for si in range(len(cfg.sources)):
            n_s = cfg.grid_n(si)
            coarse = torch.randn((1, 1, 8, 8), generator=gen, device=dev)
            geo.set_phase_map(si, torch.nn.functional.interpolate(coarse, size=(n_s, n_s), mode="bilinear",
                                                                  align_corners=True)[0, 0].contiguous())
    torch.cuda.synchronize()
    t_setup = time.perf_counter() - t_setup
    lgs, ngs = cfg.wfs[0], cfg.wfs[1]
    n_lgs, n_ngs, n_sci = len(cfg.sources_of_wfs(0)), len(cfg.sources_of_wfs(1)), len(cfg.science_sources())
    valid_lgs = int(geo.wfs_valid(0).sum()) * n_lgs
    valid_ngs = int(geo.wfs_valid(1).sum()) * n_ngs
    frames_per_step = valid_lgs + valid_ngs
    nmax = max(K, Wm, 1)
    sl_lgs = torch.empty((nmax, n_lgs, 2, lgs.n_sub ** 2), dtype=torch.float32, device=dev)
    sl_ngs = torch.empty((nmax, n_ngs, 2, ngs.n_sub ** 2), dtype=torch.float32, device=dev)
    psf = torch.zeros((n_sci, cfg.psf_fft, cfg.psf_fft), dtype=torch.float32, device=dev)
    first, _ = sharding.step_range(rank, world, K)

    def run_lgs(g, f0, count):
        for b0 in range(0, count, batch):
            ks = min(batch, count - b0)
            g.sh_images(0, None, f0 + b0, ks, cfg.dt_s, want_images=False, slopes=sl_lgs[b0:b0 + ks])

    def run_steps(f0, count):
        for b0 in range(0, count, batch):
            ks = min(batch, count - b0)
            if args.serial:
                geo.sh_images(0, None, f0 + b0, ks, cfg.dt_s, want_images=False, slopes=sl_lgs[b0:b0 + ks])
                geo.sh_images(1, None, f0 + b0, ks, cfg.dt_s, want_images=False, slopes=sl_ngs[b0:b0 + ks])
                geo.psf(None, f0 + b0, ks, cfg.dt_s, psf=psf, accumulate=True)
            else:       # ao_forward: the same three legs, the workspace users on the library's side stream
                geo.forward(f0 + b0, ks, cfg.dt_s, [sl_lgs[b0:b0 + ks], sl_ngs[b0:b0 + ks]], psf=psf, accumulate=True)

    def timed(fn, reps, g=geo):
        """`reps` back-to-back repetitions of fn(), each bracketed by its own CUDA events on the launching stream, with
        a barrier + synchronize on both sides of the whole region.  Returns (seconds per repetition, launches)."""
        stream = torch.cuda.current_stream()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(reps)]
        torch.cuda.synchronize(); sharding.barrier()
        l0 = g.launch_count()
        for e0, e1 in ev:
            e0.record(stream); fn(); e1.record(stream)
        torch.cuda.synchronize(); sharding.barrier()
        return [e0.elapsed_time(e1) * 1e-3 for e0, e1 in ev], (g.launch_count() - l0) // reps

    # ---- warm-up, then R repetitions of the K timed full steps ----
    run_steps(first, Wm)
    torch.cuda.synchronize()
    psf.zero_()
    sampler = ClockSampler(local_rank)
    sampler.start()

    def full_job():
        run_steps(first, K)
        if world > 1:
            sharding.sum_over_ranks_(psf)          # the one exchange: long-exposure PSF all-reduce

    t_reps, launches = timed(full_job, R)
    clocks = sampler.stop()
    t_reps = [sharding.max_over_ranks(t, device=dev) for t in t_reps]       # each repetition: max over ranks
    t_full = statistics.median(t_reps)
    value = frames_per_step * K * world / t_full

    # ---- dominant kernel: the LGS WFS forward model (trace + SH + CoG), timed alone, median of R repetitions ----
    pk = peaks()
    fp32_peak = geo_sm_count(dev) * FP32_LANES_PER_SM * 2 * pk["sm_max_mhz"] * 1e6 / 1e12     # TFLOP/s, nominal

    def lgs_leg(g, wfs, steps):
        run_lgs(g, first, min(Wm, steps) or 1)
        sc = ClockSampler(local_rank); sc.start()
        ts, nl = timed(lambda: run_lgs(g, first, steps), R, g)
        ck = sc.stop()
        t = statistics.median(ts)
        fl = flops_per_subap_frame(wfs.n_samp, wfs.fft, len(cfg.layers))
        ach = fl * valid_lgs * steps / t / 1e12
        return {"us_per_step": 1e6 * t / steps, "us_per_step_min": 1e6 * min(ts) / steps, "us_per_step_max": 1e6 * max(ts) / steps,
                "achieved": ach, "frac": ach / fp32_peak, "flop_per_subaperture_frame": fl, "launches": nl,
                "steps": steps, "repetitions": R, "sm_mhz_during": ck["sm_mhz"]}

    leg = lgs_leg(geo, lgs, K)
    probe = {"ffma": geo.probe_fp32(False), "ffma2": geo.probe_fp32(True)}
    static = ncu_static(min(batch, K))
    roofline = {"bound": "alu", "kernel": "LGS WFS forward model (ray-trace + SH image + CoG; ao_sh_images, phase_dev=NULL)",
                "achieved": leg["achieved"], "peak": fp32_peak, "unit": "TFLOP/s", "frac": leg["frac"],
                "traffic": static["traffic"], "traffic_source": static["source"],
                "smem_wavefront_frac": static["smem_wavefront_frac"],
                "peak_source": f"148 SMs x 128 FP32 lanes x 2 x {pk['sm_max_mhz']:.0f} MHz (nominal; DESIGN.md section 6)",
                "peak_measured": max(probe.values()), "peak_measured_source": "ao_probe_fp32 in this run (FMA-chain micro-kernel, CUDA events): "
                f"FFMA {probe['ffma']:.1f}, FFMA2 {probe['ffma2']:.1f} TFLOP/s",
                "frac_of_measured_peak": leg["achieved"] / max(probe.values()) if max(probe.values()) > 0 else None,
                "flop_model": "SURVEY.md section 8(d): 12 n^2 L + (n + M)(5 M (log2 M - 1) + 3 M) + 4 M^2 per VALID subaperture frame",
                "flop_per_subaperture_frame": leg["flop_per_subaperture_frame"],
                "us_per_step": leg["us_per_step"], "us_per_step_min": leg["us_per_step_min"], "us_per_step_max": leg["us_per_step_max"],
                "repetitions": R, "launches": leg["launches"], "sm_mhz_during": leg["sm_mhz_during"],
                "lgs_frames_per_sec": valid_lgs * 1e6 / leg["us_per_step"],
                "lgs_grid_slot_frames_per_sec": n_lgs * lgs.n_sub ** 2 * 1e6 / leg["us_per_step"],
                "frac_counting_grid_slots": leg["frac"] * n_lgs * lgs.n_sub ** 2 / valid_lgs,
                "hbm_peak_gbs": pk["hbm_gbs"], "hbm_peak_source": pk["source"]}

    # ---- the rest of the c4 sweep (LGS FFT 16 / 32 / 64): LGS leg of each size in the same run ----
    sweep = {str(lgs.fft): {k: leg[k] for k in ("us_per_step", "frac", "achieved", "flop_per_subaperture_frame", "steps")}}
    if not args.skip_sweep:
        for M in (16, 32, 64):
            if M == lgs.fft:
                continue
            c2 = inputs.make_config(4, lgs_fft=M, screen_n=args.screen_n, n_layers=args.layers, with_screens=False)
            g2 = binding.Geometry(c2, device=dev, workspace_steps=batch, screens=geo.screens)
            r2 = lgs_leg(g2, c2.wfs[0], min(K, 100))
            sweep[str(M)] = {k: r2[k] for k in ("us_per_step", "frac", "achieved", "flop_per_subaperture_frame", "steps")}
            g2.close()

    # ---- the widened rows, timed in the same run: NEXT-3 (extended sodium layer) and NEXT-4 (polychromatic PSF) ----
    widened = {}
    if not args.skip_sweep:
        ks = min(K, 50)
        geo.set_sodium(inputs.sodium_profile(cfg, n_z=5, n_t=8, launch="side"))
        r3 = lgs_leg(geo, lgs, ks)
        geo.set_sodium(None)
        widened["next3_lgs_elongation"] = {"scatterers": 5, "us_per_step": r3["us_per_step"], "steps": ks,
                                           "note": "LGS leg (ao_sh_images, phase_dev = NULL) with ao_set_sodium: 5 scatterers, side launch"}
        band = ([2.0e-6, 2.2e-6, 2.4e-6], [0.3, 0.4, 0.3])
        geo.set_psf_band(*band)
        kp = min(K, 8)
        p4 = torch.zeros_like(psf)
        geo.psf_poly(None, first, kp, cfg.dt_s, psf=p4)
        ts, _ = timed(lambda: geo.psf_poly(None, first, kp, cfg.dt_s, psf=p4, accumulate=True), R)
        t_mono, _ = timed(lambda: geo.psf(None, first, kp, cfg.dt_s, psf=p4, accumulate=True), R)
        geo.set_psf_band(None)
        widened["next4_psf_poly"] = {"wavelengths": len(band[0]), "us_per_step": 1e6 * statistics.median(ts) / kp,
                                     "us_per_step_monochromatic": 1e6 * statistics.median(t_mono) / kp, "steps": kp,
                                     "note": f"ao_psf_poly (ray-trace + chirp-z, FFT 4096) against ao_psf, {cfg.psf_fft}^2 pixels, on-axis direction"}
        del p4

    # ---- the other workloads of BASELINE.json (c0 .. c3) at their stated sizes: full-step time of each ----
    others = {}
    if not args.skip_sweep:
        for ci in (0, 1, 2, 3):
            cc = inputs.make_config(ci, device=dev, keep_on_device=True)
            nst = cc.n_steps
            gc = binding.Geometry(cc, device=dev, workspace_steps=min(nst, batch))
            slc = [torch.empty((nst, len(cc.sources_of_wfs(w)), 2, W.n_sub ** 2), dtype=torch.float32, device=dev)
                   for w, W in enumerate(cc.wfs)]
            pc = (torch.zeros((len(cc.science_sources()), cc.psf_fft, cc.psf_fft), dtype=torch.float32, device=dev)
                  if cc.psf_fft else None)

            def job():
                for b0 in range(0, nst, batch):
                    ksb = min(batch, nst - b0)
                    gc.forward(b0, ksb, cc.dt_s, [t[b0:b0 + ksb] for t in slc], psf=pc, accumulate=True, noise=cc.noise)
            job()
            ts, nl = timed(job, max(3, R // 4), gc)
            t = statistics.median(ts)
            vf = sum(int(gc.wfs_valid(w).sum()) * len(cc.sources_of_wfs(w)) for w in range(len(cc.wfs)))
            others[cc.name] = {"steps": nst, "ms_per_step": 1e3 * t / nst, "valid_subaperture_frames_per_step": vf,
                               "subaperture_frames_per_sec": vf * nst / t, "launches": nl,
                               "noise": cc.noise is not None, "science_psfs": len(cc.science_sources())}
            gc.close()
            del gc, slc, pc, cc

    # ---- optional: the residual-phase entry (NEXT-2), HBM-bound: every mode array is read once ----
    dm = None
    if args.dm_modes > 0:
        n_el = lgs.n_sub * lgs.n_samp
        n_el *= n_el
        modes = torch.randn((args.dm_modes, n_el), dtype=torch.float32, device=dev)
        coeffs = torch.randn((args.dm_modes,), dtype=torch.float32, device=dev)
        dmap = torch.empty((n_el,), dtype=torch.float32, device=dev)
        geo.modes_to_map(modes, coeffs, -1.0, dmap)
        ts, _ = timed(lambda: geo.modes_to_map(modes, coeffs, -1.0, dmap), R)
        t_dm = statistics.median(ts)
        nbytes = (args.dm_modes + 1) * n_el * 4.0
        dm = {"modes": args.dm_modes, "elems": n_el, "us_per_call": 1e6 * t_dm, "bound": "hbm",
              "achieved": nbytes / t_dm / 1e9, "peak": pk["hbm_gbs"], "unit": "GB/s",
              "frac": nbytes / t_dm / 1e9 / pk["hbm_gbs"]}
        del modes

    # ---- end to end through the host-buffer entry point ----
    e2e = None
    if not args.skip_e2e:
        scr_host = [torch.empty((l.n, l.n), dtype=torch.float32).pin_memory() for l in cfg.layers]
        for h, d in zip(scr_host, geo.screens):
            h.copy_(d)
        slh = [torch.empty((K, n_lgs, 2, lgs.n_sub ** 2), dtype=torch.float32).pin_memory(),
               torch.empty((K, n_ngs, 2, ngs.n_sub ** 2), dtype=torch.float32).pin_memory()]
        psfh = torch.empty((n_sci, cfg.psf_fft, cfg.psf_fft), dtype=torch.float32).pin_memory()

        def host_call(screens):
            torch.cuda.synchronize(); sharding.barrier()
            t0 = time.perf_counter()
            geo.forward_host(first, K, cfg.dt_s, slh, psfh, screens_host=screens)     # synchronises inside
            return sharding.max_over_ranks(time.perf_counter() - t0, device=dev)

        t_e2e = statistics.median([host_call(scr_host) for _ in range(3)])
        h2d = geo.last_h2d_bytes()                 # what the call uploaded: the part of every screen the K steps read
        t_res = statistics.median([host_call(None) for _ in range(5)])
        d2h = sum(t.numel() * 4 for t in slh) + psfh.numel() * 4
        e2e = {"value": frames_per_step * K * world / t_e2e, "unit": UNIT,
               "h2d_bytes_per_step": h2d / K, "d2h_bytes_per_step": d2h / K, "seconds": t_e2e,
               "value_screens_resident": frames_per_step * K * world / t_res, "seconds_screens_resident": t_res,
               "h2d_bytes_per_call": h2d, "host_screen_bytes": sum(h.numel() * 4 for h in scr_host),
               "note": "ao_forward_host, pinned host buffers (all 35 screens of 8192^2 live in host memory), host clock around the "
                       "call (it synchronises), median of 3: H2D of the part of every screen the K steps read (bounding box of all "
                       "footprints + margin; counted by the library, ao_last_h2d_bytes), K steps, D2H of all slopes and the "
                       "long-exposure PSF; value_screens_resident: the same call with the screens already on the device (D2H only, median of 5)"}
        del scr_host

    # ---- parity spot check against the oracle + the oracle timed on the host cores (rank 0, N = 1) ----
    cpu = spot = None
    if rank == 0 and world == 1 and not args.skip_cpu:
        import oracle
        from tests.parity_util import per_subap_max_rel_l2, rel_l2
        hs = host_screens_of(cfg)
        img, slp = geo.sh_images(0, None, first, 2, cfg.dt_s)
        torch.cuda.synchronize()
        ref = oracle.forward(cfg, first, 1, want_phase=False, want_psf=False, sources=[cfg.sources_of_wfs(0)[0]])
        s0 = cfg.sources_of_wfs(0)[0]
        spot = {"what": f"LGS source {s0}, step {first}: all {int(ref['valid'][0].sum())} valid subapertures against the FP64 oracle",
                "slopes_max_abs_px": float(np.abs(slp[0, 0].cpu().numpy().astype(np.float64) - ref["slopes"][s0][0]).max()),
                "images_rel_l2": rel_l2(img[0, 0].cpu().numpy(), ref["images"][s0][0]),
                "per_subaperture_max_rel_l2": per_subap_max_rel_l2(img[0, 0].cpu().numpy(), ref["images"][s0][0], ref["valid"][0]),
                "bars": {"slopes_max_abs_px": 1e-4, "images_rel_l2": 1e-5}}
        full = oracle_sample(cfg, hs, budget_s=10.0)
        cpu = {k: full[k] for k in ("value", "unit", "cores", "kind", "sample", "ms_per_step", "same_config")}
        if full["ms_per_step"] * 1e-3 * full["cores"] <= 90.0:       # one thread: one whole step if it stays near a minute
            one = oracle_sample(cfg, hs, steps=1, threads=1)
        else:
            one = oracle_sample(cfg, hs, n_sub=20, steps=1, threads=1)
        cpu["single_thread"] = {k: one[k] for k in ("value", "cores", "sample", "ms_per_step", "same_config")}

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
                "ms_per_step": 1e3 * t_full / K, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": cfg.name, "lgs": f"{n_lgs} LGS x {lgs.n_sub}x{lgs.n_sub} subaps, n={lgs.n_samp}, FFT {lgs.fft}, {lgs.n_pix}x{lgs.n_pix} px",
                           "ngs": f"{n_ngs} NGS x 2x2 subaps, n={ngs.n_samp}, FFT {ngs.fft}",
                           "psf": f"{n_sci} science PSF, FFT {cfg.psf_fft}", "layers": len(cfg.layers),
                           "screen_n": cfg.layers[0].n, "steps_per_call": batch, "phase_maps": bool(args.phase_maps),
                           "valid_subaperture_frames_per_step": frames_per_step,
                           "grid_slot_frames_per_step": n_lgs * lgs.n_sub ** 2 + n_ngs * ngs.n_sub ** 2,
                           "l2_policy": "inputs larger than L2: 9.4 GB of screens, ~211 MB touched per step",
                           "parallelism": f"steps split over {world} GPU(s), screens replicated"},
                "timing": {"repetitions": R, "statistic": "median over repetitions of the K-step region, CUDA events, max over ranks",
                           "ms_per_step_min": 1e3 * min(t_reps) / K, "ms_per_step_max": 1e3 * max(t_reps) / K},
                "clocks": clocks, "gpu_launches": launches, "roofline": roofline, "e2e": e2e,
                "cpu_baseline": cpu, "parity_spot_check": spot, "extra": {"sweep_lgs_leg": sweep, "widened": widened, "other_configs_full_step": others},
                "setup_seconds": t_setup,
                "setup_note": f"{t_screens:.1f} s of it is the harness generating the 35 screens of 8192^2 (torch.fft), not the library"}
        if dm is not None:
            line["dm_modes"] = dm
        print(json.dumps(line))
    geo.close()
    return 0


def geo_sm_count(dev) -> int:
    import torch
    return torch.cuda.get_device_properties(dev).multi_processor_count


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=1000)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--lgs-fft", type=int, default=32, choices=[16, 32, 64])
    ap.add_argument("--screen-n", type=int, default=8192)
    ap.add_argument("--layers", type=int, default=35)
    ap.add_argument("--batch", type=int, default=50, help="time steps per C-ABI call")
    ap.add_argument("--reps", type=int, default=REPS, help="repetitions of every timed region (the median is reported)")
    ap.add_argument("--serial", action="store_true", help="one C-ABI call per leg on one stream instead of ao_forward")
    ap.add_argument("--phase-maps", action="store_true", help="set a static additive phase map on every source (ao_set_phase_map)")
    ap.add_argument("--dm-modes", type=int, default=0, help="also time ao_modes_to_map with this many modes on the LGS grid")
    ap.add_argument("--skip-e2e", action="store_true")
    ap.add_argument("--skip-cpu", action="store_true")
    ap.add_argument("--skip-sweep", action="store_true")
    args = ap.parse_args()
    if args.steps < 1:
        args.steps = 1
    if args.impl == "reference":
        if args.steps > 1 and args.steps == ap.get_default("steps"):
            args.steps, args.warmup = 10, 2          # no flags: a run of whole oracle steps that ends within minutes
        return run_reference(args)
    return run_gpu(args)


if __name__ == "__main__":
    sys.exit(main())
