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
# From the committed ncu --set full capture of k_fused<32,0> (profiles/r1_v4_k_fused.md): DRAM bytes read + written per
# simulated step (506.2 MB per 10-step launch) and the shared-memory data-pipe utilisation, the unit that binds.
NCU_DRAM_BYTES_PER_STEP = 50.62e6
NCU_SMEM_WAVEFRONT_FRAC = 0.735
NCU_SOURCE = ("profiles/r1_v4_k_fused.md: dram__bytes_read.sum + dram__bytes_write.sum of one ncu --set full capture, "
              "scaled from its 10-step launch to the steps of one launch here")


# ------------------------------------------------------------------------------ work model
def flops_per_subap_frame(n: int, M: int, n_layers: int) -> float:
    """Algorithmic FLOPs of one valid subaperture frame:
    trace 12 flop/sample/layer; pruned FFT = (n + M) 1-D transforms of 5M(log2 M - 1) + 3M;
    4 flop per FFT point for |.|^2 + binning; 8 flop per sample for A exp(i phi)."""
    fft1d = 5.0 * M * (math.log2(M) - 1.0) + 3.0 * M
    return 12.0 * n * n * n_layers + (n + M) * fft1d + 4.0 * M * M + 8.0 * n * n


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
            self._stop.wait(0.02)

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
def oracle_sample(cfg_full, n_sub: int, host_screens, budget_s: float, steps=None, warmup: int = 0):
    """Time oracle.forward() on a reduced-pupil copy of the workload (same layers, screens, sources,
    samples per subaperture and FFT sizes; pupil scaled to n_sub subapertures per side)."""
    import oracle
    from paper_1608_00386_b200 import inputs
    M = cfg_full.wfs[0].fft
    cfg = inputs.make_config(4, n_sub=n_sub, lgs_fft=M, n_layers=len(cfg_full.layers),
                             screen_n=cfg_full.layers[0].n, with_screens=False)
    for lay, full, scr in zip(cfg.layers, cfg_full.layers, host_screens):
        lay.wind_x_mps, lay.wind_y_mps, lay.height_m, lay.weight = \
            full.wind_x_mps, full.wind_y_mps, full.height_m, full.weight
        lay.screen = scr
    valid_per_step = 0
    r = oracle.forward(cfg, 0, 1, want_phase=False)                      # calibration / warm-up
    for w, W in enumerate(cfg.wfs):
        valid_per_step += int(r["valid"][w].sum()) * len(cfg.sources_of_wfs(w))
    for k in range(warmup):
        oracle.forward(cfg, k, 1, want_phase=False)
    if steps is None:
        t0 = time.perf_counter()
        oracle.forward(cfg, 0, 1, want_phase=False)
        per = time.perf_counter() - t0
        steps = max(1, min(200, int(budget_s / max(per, 1e-3))))
    t0 = time.perf_counter()
    oracle.forward(cfg, 1000, steps, want_phase=False)
    dt = time.perf_counter() - t0
    sample = (f"{steps} full steps of c4 at M={M} on a reduced pupil: {n_sub}x{n_sub} subapertures per LGS "
              f"({cfg.pupil.n}^2 pupil, NGS FFT {cfg.wfs[1].fft}, PSF FFT {cfg.psf_fft}), all {len(cfg.layers)} "
              f"layers of {cfg.layers[0].n}^2 screens, {valid_per_step} valid subaperture frames per step")
    return {"value": valid_per_step * steps / dt, "unit": UNIT, "cores": oracle.num_threads(),
            "kind": "oracle", "sample": sample, "seconds": dt, "steps": steps,
            "ms_per_step": 1e3 * dt / steps}


def host_screens_of(cfg):
    from paper_1608_00386_b200 import inputs
    inputs.screens_to_host(cfg)
    return [l.screen for l in cfg.layers]


# ------------------------------------------------------------------------------ reference arm
def run_reference(args):
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
    n_sub = 40 if K + Wm <= 12 else (20 if K + Wm <= 120 else 10)
    res = oracle_sample(cfg, n_sub, host_screens_of(cfg), 0.0, steps=K, warmup=Wm)
    line = {"impl": "reference", "metric": METRIC, "value": res["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": K, "warmup": Wm, "ms_per_step": res["ms_per_step"], "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"c4_throughput_M{args.lgs_fft} (bounded sample)", "sample": res["sample"],
                       "screen_n": screen_n},
            "cpu_baseline": {"value": res["value"], "unit": UNIT, "cores": res["cores"], "kind": "oracle",
                             "sample": res["sample"]},
            "e2e": {"value": res["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------ GPU arm
def run_gpu(args):
    import torch
    from paper_1608_00386_b200 import binding, inputs, sharding
    rank, local_rank, world = sharding.init("nccl")
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device; the product has no CPU fallback")
    dev = f"cuda:{local_rank}"
    torch.cuda.set_device(local_rank)
    K, Wm, batch = args.steps, max(args.warmup, 3), args.batch     # timing rule: at least 3 warm-up steps
    t_setup = time.perf_counter()
    cfg = inputs.make_config(4, lgs_fft=args.lgs_fft, screen_n=args.screen_n, n_layers=args.layers,
                             device=dev, keep_on_device=True)
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

    def run_lgs(f0, count):
        for b0 in range(0, count, batch):
            ks = min(batch, count - b0)
            geo.sh_images(0, None, f0 + b0, ks, cfg.dt_s, want_images=False, slopes=sl_lgs[b0:b0 + ks])

    def run_steps(f0, count):
        for b0 in range(0, count, batch):
            ks = min(batch, count - b0)
            if args.serial:
                geo.sh_images(0, None, f0 + b0, ks, cfg.dt_s, want_images=False, slopes=sl_lgs[b0:b0 + ks])
                geo.sh_images(1, None, f0 + b0, ks, cfg.dt_s, want_images=False, slopes=sl_ngs[b0:b0 + ks])
                geo.psf(None, f0 + b0, ks, cfg.dt_s, psf=psf, accumulate=True)
            else:       # ao_forward: the same three legs, the workspace-free LGS leg on the library's side stream
                geo.forward(f0 + b0, ks, cfg.dt_s, [sl_lgs[b0:b0 + ks], sl_ngs[b0:b0 + ks]], psf=psf, accumulate=True)

    def timed(fn, *a):
        stream = torch.cuda.current_stream()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize(); sharding.barrier()
        l0 = geo.launch_count()
        e0.record(stream); fn(*a); e1.record(stream)
        torch.cuda.synchronize(); sharding.barrier()
        return e0.elapsed_time(e1) * 1e-3, geo.launch_count() - l0

    # ---- warm-up, then the timed full steps ----
    if Wm:
        run_steps(first, Wm)
    torch.cuda.synchronize()
    psf.zero_()
    sampler = ClockSampler(local_rank)
    sampler.start()

    def full_job():
        run_steps(first, K)
        if world > 1:
            sharding.sum_over_ranks_(psf)          # the one exchange: long-exposure PSF all-reduce

    t_full, launches = timed(full_job)
    clocks = sampler.stop()
    t_full = sharding.max_over_ranks(t_full, device=dev)
    value = frames_per_step * K * world / t_full

    # ---- dominant kernel: the LGS WFS forward model (trace + SH + CoG), timed alone ----
    run_lgs(first, min(Wm, K) or 1)
    s2 = ClockSampler(local_rank); s2.start()
    t_wfs, launches_wfs = timed(run_lgs, first, K)
    clocks_wfs = s2.stop()
    pk = peaks()
    fp32_peak = geo_sm_count(dev) * FP32_LANES_PER_SM * 2 * pk["sm_max_mhz"] * 1e6 / 1e12     # TFLOP/s
    flop = flops_per_subap_frame(lgs.n_samp, lgs.fft, len(cfg.layers)) * valid_lgs * K
    achieved = flop / t_wfs / 1e12
    roofline = {"bound": "alu", "kernel": "LGS WFS forward model (ray-trace + SH image + CoG; ao_sh_images, phase_dev=NULL)",
                "achieved": achieved, "peak": fp32_peak, "unit": "TFLOP/s", "frac": achieved / fp32_peak,
                "traffic": NCU_DRAM_BYTES_PER_STEP * min(batch, K), "traffic_source": NCU_SOURCE,
                "smem_wavefront_frac": NCU_SMEM_WAVEFRONT_FRAC, "peak_source": f"148 SMs x 128 FP32 lanes x 2 x {pk['sm_max_mhz']:.0f} MHz (nominal; DESIGN.md section 6)",
                "flop_per_subaperture_frame": flops_per_subap_frame(lgs.n_samp, lgs.fft, len(cfg.layers)),
                "us_per_step": 1e6 * t_wfs / K, "launches": launches_wfs,
                "sm_mhz_during": clocks_wfs["sm_mhz"],
                "lgs_frames_per_sec": valid_lgs * K / t_wfs,
                "lgs_grid_slot_frames_per_sec": n_lgs * lgs.n_sub ** 2 * K / t_wfs,
                "hbm_peak_gbs": pk["hbm_gbs"], "hbm_peak_source": pk["source"]}

    # ---- optional: the residual-phase entry (NEXT-2), HBM-bound: every mode array is read once ----
    dm = None
    if args.dm_modes > 0:
        n_el = lgs.n_sub * lgs.n_samp
        n_el *= n_el
        modes = torch.randn((args.dm_modes, n_el), dtype=torch.float32, device=dev)
        coeffs = torch.randn((args.dm_modes,), dtype=torch.float32, device=dev)
        dmap = torch.empty((n_el,), dtype=torch.float32, device=dev)
        reps = 10
        geo.modes_to_map(modes, coeffs, -1.0, dmap)
        t_dm, _ = timed(lambda: [geo.modes_to_map(modes, coeffs, -1.0, dmap) for _ in range(reps)])
        nbytes = (args.dm_modes + 1) * n_el * 4.0
        dm = {"modes": args.dm_modes, "elems": n_el, "us_per_call": 1e6 * t_dm / reps, "bound": "hbm",
              "achieved": nbytes * reps / t_dm / 1e9, "peak": pk["hbm_gbs"], "unit": "GB/s",
              "frac": nbytes * reps / t_dm / 1e9 / pk["hbm_gbs"]}
        del modes

    # ---- end to end through the host-buffer entry point (screens uploaded inside the region) ----
    e2e = None
    if not args.skip_e2e:
        scr_host = [torch.empty((l.n, l.n), dtype=torch.float32).pin_memory() for l in cfg.layers]
        for h, d in zip(scr_host, geo.screens):
            h.copy_(d)
        slh = [torch.empty((K, n_lgs, 2, lgs.n_sub ** 2), dtype=torch.float32).pin_memory(),
               torch.empty((K, n_ngs, 2, ngs.n_sub ** 2), dtype=torch.float32).pin_memory()]
        psfh = torch.empty((n_sci, cfg.psf_fft, cfg.psf_fft), dtype=torch.float32).pin_memory()
        torch.cuda.synchronize(); sharding.barrier()
        t0 = time.perf_counter()
        geo.forward_host(first, K, cfg.dt_s, slh, psfh, screens_host=scr_host)     # synchronises inside
        t_e2e = time.perf_counter() - t0
        t_e2e = sharding.max_over_ranks(t_e2e, device=dev)
        h2d = sum(h.numel() * 4 for h in scr_host)
        d2h = sum(t.numel() * 4 for t in slh) + psfh.numel() * 4
        e2e = {"value": frames_per_step * K * world / t_e2e, "unit": UNIT,
               "h2d_bytes_per_step": h2d / K, "d2h_bytes_per_step": d2h / K, "seconds": t_e2e,
               "note": "ao_forward_host: H2D of all screens (once per run, amortised over the K steps), "
                       "K steps, D2H of all slopes and the long-exposure PSF; pinned host buffers"}
        del scr_host

    cpu = None
    if rank == 0 and world == 1 and not args.skip_cpu:
        cpu = oracle_sample(cfg, 20, host_screens_of(cfg), 15.0)
        cpu = {k: cpu[k] for k in ("value", "unit", "cores", "kind", "sample")}

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
                "clocks": clocks, "gpu_launches": launches, "roofline": roofline, "e2e": e2e,
                "cpu_baseline": cpu, "setup_seconds": t_setup}
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
    ap.add_argument("--serial", action="store_true", help="one C-ABI call per leg on one stream instead of ao_forward")
    ap.add_argument("--phase-maps", action="store_true", help="set a static additive phase map on every source (ao_set_phase_map)")
    ap.add_argument("--dm-modes", type=int, default=0, help="also time ao_modes_to_map with this many modes on the LGS grid")
    ap.add_argument("--skip-e2e", action="store_true")
    ap.add_argument("--skip-cpu", action="store_true")
    args = ap.parse_args()
    if args.steps < 1:
        args.steps = 1
    if args.impl == "reference":
        return run_reference(args)
    return run_gpu(args)


if __name__ == "__main__":
    sys.exit(main())
