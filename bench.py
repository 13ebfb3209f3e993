#!/usr/bin/env python
"""bench.py — one JSON line for the driver.

A step = one pass of the whole hot path (mk_run = begin + niter Neumann steps + finals,
niter + 2 = 18 syntheses) over one batch of seeded synthetic input of BASELINE.json config 1 (601 x 601 x 2048,
one focal point, 16 iterations; the bandwidth-bound regime the metric is quoted on).  R^ (1.30 GB) is resident in
HBM and far larger than the 126 MB L2, so no cache flush is needed between steps.

  value      synthesis GB/s of R^ streamed  = passes over R^ * bytes(R^ unpadded) / device time   (inputs resident in HBM;
             with 1, 2 or 4 focal points the two final syntheses share one pass: 17 passes per step; value_algorithmic
             counts the 18 syntheses of Algorithm 1)
  secondary  the large-batch regimes, measured in the same invocation (N = 1): config 2 (tcgen05 3xTF32 and FP32-FFMA),
             config 3, config 4 — each with its own ms_per_step, clocks and roofline
  e2e        same metric through mk_run_host: pinned HOST G_d / t_d in, six HOST output fields out, copies timed
  roofline   the streaming contraction kernel (k_syn_gemv): algorithmic bytes of R^ per launch / its CUDA-event time
  cpu_baseline  the fp64 oracle timed on this box's host cores on a bounded sample (one full synthesis R N_0)

`--impl reference` times the oracle itself (a deliberately slow, plain CPU program) on the same workload.
`--workload K` benches another BASELINE.json config (2 = the 601-focal-point GEMM regime) for DESIGN.md's tables.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

from paper_2106_04649_b200 import configs, gen, shard  # noqa: E402

METRIC = "synthesis_GBps_of_R_streamed"
UNIT = "GB/s"


def dist_env():
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return rank, world, local


def measured_peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        d = json.loads(p.read_text())
        return {"hbm_gbs": float(d["hbm_gbs"]), "bf16_tflops": float(d.get("bf16_tflops", 1590.0)),
                "bf16_tflops_sustained": float(d.get("bf16_tflops_sustained", 1400.0)), "source": "measured"}
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "source": "fallback"}


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons DURING the timed region (pynvml; nvidia-smi would show the same)."""
    REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
               0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting", 0x10: "sync_boost"}

    def __init__(self, index, period=0.05):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.samples, self.reasons, self.power = [], set(), []
        self.max_mhz = None
        self._stop_evt = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception:
            self.ok = False

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        while not self._stop_evt.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                try:
                    mask = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, nm in self.REASONS.items():
                    if mask & bit:
                        self.reasons.add(nm)
                self.power.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0)
            except Exception:
                pass
            time.sleep(self.period)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=2)
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "samples": 0}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples), "power_w_max": max(self.power) if self.power else None}


def workload_arrays(cfg):
    base = gen.base_traces(cfg)
    R = gen.R_full(cfg, base)
    Gd, td = gen.first_arrivals(cfg)
    return R, Gd, td


def nsyn_per_step(cfg):
    return cfg.niter + 2        # niter Neumann steps + one extra synthesis each for G^- and G^+ 


def rhat_bytes(cfg):
    import math
    df = 1.0 / (cfg.nt * cfg.dt)
    klo = max(int(math.ceil(cfg.fmin / df - 1e-6)), 0)
    khi = min(int(math.floor(cfg.fmax / df + 1e-6)), cfg.nt // 2)
    return 8.0 * cfg.n * cfg.n * (khi - klo + 1), khi - klo + 1


# ------------------------------------------------------------------------------------------------ oracle legs
def oracle_sample(cfg, R, Gd, td, budget_s, full_first=True, repeat=True):
    """Times the oracle (as it stands) on a bounded sample: one synthesis R N_0 over `nrec_s` receivers of the same
    workload, N_0 being the first windowed iterate (computed by the oracle, untimed).  Returns (seconds, nrec_s)."""
    import oracle
    w = oracle.weights(cfg.n, cfg.dx)
    klo, khi, _ = oracle.band(cfg.nt, cfg.dt, cfg.fmin, cfg.fmax)
    f = [0] if Gd.shape[0] > 1 else slice(None)
    # N_0 = the oracle's own first iterate (untimed; N_{-1} = T G_d is sparse, so this pass is cheap)
    N0 = oracle.marchenko(R, Gd[f], td[f], cfg.dt, cfg.dx, cfg.fmin, cfg.fmax, 1, cfg.eps, want=())["N_iters"][0]
    # size the sample from a 4-receiver probe
    probe = np.linspace(0, cfg.n - 1, 4).round().astype(int)
    t0 = time.perf_counter()
    oracle.synthesis(np.ascontiguousarray(R[:, probe]), N0, cfg.dt, w, klo, khi)
    per_rec = (time.perf_counter() - t0) / 4 * max(1, min(4, oracle.num_threads())) / max(1, oracle.num_threads())
    nrec_s = int(min(cfg.n, max(oracle.num_threads(), budget_s / max(per_rec, 1e-6))))
    recs = np.linspace(0, cfg.n - 1, nrec_s).round().astype(int)
    Rs = np.ascontiguousarray(R[:, recs])
    # when the whole problem is cheaper than the budget, repeat it: about `budget_s` seconds of CPU work in all
    reps, t_total = 0, 0.0
    while reps == 0 or (repeat and nrec_s == cfg.n and t_total < 0.8 * budget_s and reps < 64):
        t0 = time.perf_counter()
        oracle.synthesis(Rs, N0, cfg.dt, w, klo, khi)
        t_total += time.perf_counter() - t0
        reps += 1
    oracle_sample.reps = reps
    return t_total / reps, nrec_s, N0, (w, klo, khi)


def run_reference(args):
    """--impl reference: the oracle is the reference arm.  Each step = one synthesis on a bounded receiver sample."""
    rank, world, _ = dist_env()
    if rank != 0:
        return 0
    import oracle
    cfg = configs.get(args.workload)
    R, Gd, td = workload_arrays(cfg) if cfg.nfoc == 1 else (gen.R_full(cfg), *gen.first_arrivals(cfg, focs=[cfg.nfoc // 2]))
    nbytes, nb = rhat_bytes(cfg)
    total_budget = 150.0
    per_step = total_budget / (args.steps + args.warmup)
    _, _, N0, (w, klo, khi) = oracle_sample(cfg, R, Gd, td, budget_s=per_step, repeat=False)
    # pick the sample so that one step fits per_step seconds
    probe = np.linspace(0, cfg.n - 1, 4).round().astype(int)
    t0 = time.perf_counter()
    oracle.synthesis(np.ascontiguousarray(R[:, probe]), N0, cfg.dt, w, klo, khi)
    t_probe = time.perf_counter() - t0
    nrec_s = int(min(cfg.n, max(1, 4 * per_step / max(t_probe, 1e-6))))
    recs = np.linspace(0, cfg.n - 1, nrec_s).round().astype(int)
    Rs = np.ascontiguousarray(R[:, recs])
    for _ in range(args.warmup):
        oracle.synthesis(Rs, N0, cfg.dt, w, klo, khi)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.synthesis(Rs, N0, cfg.dt, w, klo, khi)
    dt_s = time.perf_counter() - t0
    val = (nbytes * nrec_s / cfg.n) * args.steps / dt_s / 1e9
    sample = f"per step: one oracle synthesis R N_0 on {nrec_s} of {cfg.n} receivers x 1 focal point of config {cfg.k}"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * dt_s / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"config{cfg.k}:{cfg.name}", "n": cfg.n, "nt": cfg.nt, "nfoc": 1, "nb": nb, "sample": sample},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


# ------------------------------------------------------------------------------------------------ our arm
FIELDS = ("N_last", "f1plus", "f1min", "G", "Gplus", "Gminus")


def traffic_entry(cfg_k, regime):
    """DRAM bytes per launch of the contraction kernel from the last committed `ncu --set full` capture (profiles/traffic.json;
    it names the commit the captures were taken at, so a stale figure can be told from a current one)."""
    tp = ROOT / "profiles" / "traffic.json"
    if not tp.exists():
        return None, None
    d = json.loads(tp.read_text())
    return d.get("entries", d).get(f"config{cfg_k}_regime{regime}"), d.get("source")


def roofline_of(cfg, nb, nbytes, regime_used, syn_n, syn_ms, ms_total, clocks, share=1.0, syn_total=None):
    """Roofline of the dominant kernel (the contraction) from the CUDA events the library records on its own stream."""
    peaks = measured_peaks()
    avg_ms = syn_ms / max(syn_n, 1)
    traffic, traffic_src = traffic_entry(cfg.k, regime_used)
    syn_total = syn_n if syn_total is None else syn_total     # launches in the timed region; syn_n of them carried events
    common = {"traffic": traffic, "traffic_source": traffic_src, "launches_timed": int(syn_n), "launches": int(syn_total),
              "avg_launch_ms": avg_ms, "share_of_step": avg_ms * syn_total / ms_total}
    if regime_used == 1:
        ach = share * nbytes / (avg_ms * 1e-3) / 1e9
        return {"bound": "hbm", "kernel": "k_syn_gemv", "achieved": ach, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                "frac": ach / peaks["hbm_gbs"], "peak_source": peaks["source"] + " copy bandwidth (MEASURED_PEAKS.json)",
                "frac_of_nominal_8TBps": ach / 8000.0, **common}
    flops = share * 8.0 * cfg.nfoc * cfg.n * cfg.n * nb        # algorithmic: one complex MAC (8 flops) per element of R^ and focal point
    ach = flops / (avg_ms * 1e-3) / 1e12
    sm_max = clocks.get("sm_max_mhz") or 1965.0
    ffma_peak = 2 * 128 * 148 * sm_max * 1e6 / 1e12            # FFMA lanes x SMs x max clock
    if regime_used == 2:
        return {"bound": "alu", "kernel": "k_syn_gemm_ffma", "achieved": ach, "peak": ffma_peak, "unit": "TFLOP/s",
                "frac": ach / ffma_peak, "peak_source": "2 x 128 FFMA lanes x 148 SMs x clocks.max.sm (guide unit counts)", **common}
    # 3xTF32: every algorithmic flop costs three tf32 tensor flops.  Peak for this dtype = measured bf16 peak (sustained
    # figure: the kernel is timed inside a long step) x 1/2 (nominal tf32 : bf16), / 3 for the split.
    tf32_peak = 0.5 * peaks["bf16_tflops_sustained"]
    return {"bound": "tensor", "kernel": "k_syn_gemm_tf32x3", "achieved": ach, "peak": tf32_peak / 3.0, "unit": "TFLOP/s",
            "frac": ach / (tf32_peak / 3.0),
            "peak_source": peaks["source"] + " bf16 sustained x 0.5 (nominal tf32:bf16) / 3 (3xTF32 split); "
                           "achieved counts algorithmic fp32 flops (8 per complex MAC)",
            "tensor_tflops_issued": 3.0 * ach, "tf32_peak": tf32_peak, "frac_of_fp32_ffma_roofline": ach / ffma_peak, **common}


def ingest_device(mk, cfg, dev):
    """33 GB / 250 GB of time-domain R never exist at once: generated on the device in 64-shot chunks (BASELINE.json config 4)."""
    import torch
    gR = gen.DeviceR(cfg, dev)
    for s0 in range(0, cfg.n, 64):
        mk.load_R(gR.take(np.arange(s0, min(s0 + 64, cfg.n))), s0)
    torch.cuda.synchronize()
    del gR
    torch.cuda.empty_cache()


def device_fields(cfg, dev):
    """Output fields of one run.  180 GB of HBM do not hold six distinct fields of config 4 next to R^ and the operands:
    f1plus and f1min (the accumulators of the run) get their own, the other four outputs are written one after the
    other into ONE shared field there (same kernels, same traffic; include/mk.h allows it)."""
    import torch

    def field():
        return torch.empty((cfg.nfoc, cfg.n, cfg.nt), dtype=torch.float32, device=dev)
    shared = field() if cfg.k == 4 else None
    return {nm: (field() if (shared is None or nm in ("f1plus", "f1min")) else shared) for nm in FIELDS}


def timed_steps(mk, run_step, steps, warmup, local, dist=None, barrier=None, stride=1):
    """W untimed warm-up steps, then exactly K steps between CUDA events (device time, max over ranks), clocks sampled
    during the timed region, contraction launches timed by the library's own events (every `stride`-th launch: an event
    record between two kernels costs ~3 us and keeps them from overlapping, which a step of 40 launches of 3 .. 190 us feels)."""
    import torch
    from paper_2106_04649_b200 import binding as B
    if barrier is None:
        barrier = torch.cuda.synchronize
    for _ in range(warmup):
        run_step()
    mk.set_option(B.MK_OPT_TIMING, stride)
    mk.get_info(B.MK_INFO_SYN_RESET)
    l0 = mk.get_info(B.MK_INFO_KERNEL_LAUNCHES)
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        run_step()
    e1.record()
    barrier()
    clocks = sampler.stop()
    ms_total = shard.max_over_ranks(e0.elapsed_time(e1), dist)
    res = {"ms_total": ms_total, "clocks": clocks, "launches": int(mk.get_info(B.MK_INFO_KERNEL_LAUNCHES) - l0),
           "syn_n": mk.get_info(B.MK_INFO_SYN_LAUNCHES), "syn_ms": mk.get_info(B.MK_INFO_SYN_MS_TOTAL),
           "syn_total": mk.get_info(B.MK_INFO_SYN_COUNT),
           "regime_used": int(mk.get_info(B.MK_INFO_REGIME_USED))}
    mk.set_option(B.MK_OPT_TIMING, 0)
    return res


def secondary_entry(mk, cfg, regime, steps, warmup, local, dev, image=False):
    """One large-batch configuration for the `secondary` list of the JSON line: same protocol as the headline (mk_run steps
    between CUDA events, inputs resident in HBM), its own clocks and roofline."""
    import torch
    from paper_2106_04649_b200 import binding as B
    nbytes, nb = rhat_bytes(cfg)
    mk.set_option(B.MK_OPT_REGIME, regime)
    dGd, dtd = gen.first_arrivals_torch(cfg, dev)
    douts = device_fields(cfg, dev)
    r = timed_steps(mk, lambda: mk.run(dGd, dtd, cfg.niter, douts), steps, warmup, local)
    ms = r["ms_total"] / steps
    nsyn = nsyn_per_step(cfg)
    entry = {"workload": f"config{cfg.k}:{cfg.name}", "n": cfg.n, "nt": cfg.nt, "nfoc": cfg.nfoc, "niter": cfg.niter, "nb": nb,
             "regime": r["regime_used"], "steps": steps, "warmup": warmup, "ms_per_step": ms,
             "value": nsyn * nbytes / (ms * 1e-3) / 1e9, "unit": UNIT,
             "focal_point_iterations_per_s": cfg.nfoc * cfg.niter / (ms * 1e-3),
             "contraction_launches_per_step": r["syn_n"] / steps, "gpu_launches": r["launches"], "clocks": r["clocks"],
             "roofline": roofline_of(cfg, nb, nbytes, r["regime_used"], r["syn_n"], r["syn_ms"], r["ms_total"], r["clocks"]),
             "rhat_layout": "tiled (16 KB boxes of 128 receivers x 16 shots)" if mk.get_info(B.MK_INFO_RHAT_LAYOUT) else "row-major [rec][bin][shot]",
             "input_source": "device generator" + (", R in 64-shot chunks" if cfg.k >= 3 else " for G_d / t_d; R from the host generator")}
    if image:   # NEXT-1: the double-focusing image of the run just made, timed alone ("about 2% of the total processing time")
        img = torch.empty(cfg.nfoc, dtype=torch.float32, device=dev)
        mk.image(douts["Gminus"], img)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(5):
            mk.image(douts["Gminus"], img)
        e1.record()
        torch.cuda.synchronize()
        entry["image_ms"] = e0.elapsed_time(e1) / 5
        entry["image_share_of_step"] = entry["image_ms"] / ms
    del dGd, dtd, douts
    torch.cuda.empty_cache()
    return entry


def h2d_peak_gbs(dev, nbytes=1 << 28, reps=4):
    """Pinned host -> device copy rate of this box, measured live: the roofline of the out-of-core contraction."""
    import torch
    h = torch.empty(nbytes, dtype=torch.uint8).pin_memory()
    d = torch.empty(nbytes, dtype=torch.uint8, device=dev)
    d.copy_(h, non_blocking=True)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        d.copy_(h, non_blocking=True)
    e1.record()
    torch.cuda.synchronize()
    return reps * nbytes / (e0.elapsed_time(e1) * 1e-3) / 1e9


def variant_entry(cfg, R, Gd, td, steps, warmup, local, dev, rhat_format=0, resident_frac=None):
    """Config 1 again on a context of its own, with (a) R^ stored as q16 block floats (MK_OPT_RHAT_FORMAT = 1: the
    bandwidth-bound regime with 4.25 instead of 8 bytes per element; its own tolerance) or (b) R^ out
    of core (mk_create_streamed: a fraction of the rows resident, the rest streamed from pinned host memory through two
    windows in HBM every contraction; bit-identical results; bound by the host link)."""
    import torch
    from paper_2106_04649_b200 import binding as B
    nbytes, nb = rhat_bytes(cfg)
    streamed = None
    if resident_frac is not None:
        streamed = (int(round(resident_frac * cfg.n)), 0)
    mk = B.Marchenko(cfg.n, cfg.n, cfg.nt, cfg.dt, cfg.dx, cfg.fmin, cfg.fmax, streamed=streamed)
    mk.set_option(B.MK_OPT_EPS_SAMPLES, cfg.eps)
    mk.set_option(B.MK_OPT_RHAT_FORMAT, rhat_format)
    dR = torch.empty((64, cfg.n, cfg.nt), dtype=torch.float32, device=dev)
    for s0 in range(0, cfg.n, 64):
        s1 = min(s0 + 64, cfg.n)
        dR[:s1 - s0].copy_(torch.from_numpy(R[s0:s1]))
        mk.load_R(dR[:s1 - s0], s0)
    torch.cuda.synchronize()
    del dR
    dGd, dtd = torch.from_numpy(Gd).to(dev), torch.from_numpy(td).to(dev)
    douts = {nm: torch.empty((cfg.nfoc, cfg.n, cfg.nt), dtype=torch.float32, device=dev) for nm in FIELDS}
    h0 = mk.get_info(B.MK_INFO_H2D_BYTES)
    r = timed_steps(mk, lambda: mk.run(dGd, dtd, cfg.niter, douts), steps, warmup, local, stride=5 if rhat_format == 1 else 1)
    ms = r["ms_total"] / steps
    passes = r["syn_total"] / steps
    avg_ms = r["syn_ms"] / max(r["syn_n"], 1)
    stored = mk.get_info(B.MK_INFO_RHAT_BYTES_STORED) * cfg.n / mk.get_info(B.MK_INFO_LD_SHOT)     # unpadded bytes as stored
    entry = {"workload": f"config{cfg.k}:{cfg.name}", "n": cfg.n, "nt": cfg.nt, "nfoc": cfg.nfoc, "niter": cfg.niter, "nb": nb,
             "regime": r["regime_used"], "steps": steps, "warmup": warmup, "ms_per_step": ms, "unit": UNIT,
             "contraction_launches_per_step": passes, "gpu_launches": r["launches"], "clocks": r["clocks"],
             "focal_point_iterations_per_s": cfg.nfoc * cfg.niter / (ms * 1e-3)}
    peaks = measured_peaks()
    if rhat_format == 1:
        ach = stored / (avg_ms * 1e-3) / 1e9
        entry.update({"variant": "R^ stored as q16 block floats (4.25 B per complex element; lossy: tolerance 5e-4 per iteration / 1e-3 finals)",
                      "value": passes * stored / (ms * 1e-3) / 1e9, "value_fp32_equivalent": passes * nbytes / (ms * 1e-3) / 1e9,
                      "rhat_bytes_stored": stored,
                      "roofline": {"bound": "hbm", "kernel": "k_syn_gemv_q16", "achieved": ach, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                                   "frac": ach / peaks["hbm_gbs"], "peak_source": peaks["source"] + " copy bandwidth (MEASURED_PEAKS.json)",
                                   "fp32_equivalent_GBps": nbytes / (avg_ms * 1e-3) / 1e9, "traffic": None,
                                   "launches_timed": int(r["syn_n"]), "launches": int(r["syn_total"]), "avg_launch_ms": avg_ms,
                                   "share_of_step": avg_ms * r["syn_total"] / r["ms_total"]}})
    else:
        h2d = (mk.get_info(B.MK_INFO_H2D_BYTES) - h0) / (steps + warmup)       # bytes of R^ over the host link per step
        link = h2d_peak_gbs(dev)
        ach = h2d / (ms * 1e-3) / 1e9
        entry.update({"variant": f"R^ out of core: {streamed[0]} of {cfg.n} rows resident, window {int(mk.get_info(B.MK_INFO_WINDOW_ROWS))} rows "
                                 "(mk_create_streamed; results bit-identical to the resident context)",
                      "value": passes * nbytes / (ms * 1e-3) / 1e9, "h2d_bytes_per_step": h2d,
                      "roofline": {"bound": "host_link", "kernel": "H2D copies of R^ row blocks overlapped with k_syn_gemv", "achieved": ach,
                                   "peak": link, "unit": "GB/s", "frac": ach / link,
                                   "peak_source": "pinned host -> device cudaMemcpyAsync rate measured in this run (256 MiB copies)",
                                   "floor_ms_per_step": h2d / link / 1e6, "traffic": None,
                                   "launches_timed": int(r["syn_n"]), "avg_launch_ms": avg_ms, "share_of_step": r["syn_ms"] / r["ms_total"]}})
    mk.close()
    del dGd, dtd, douts
    torch.cuda.empty_cache()
    return entry


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2106_04649_b200 import binding as B

    rank, world, local = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.device("cuda", local)

    rows_mode = args.parallel in ("rows", "rows_fused")
    # weak scaling: replicas, no collective;  --parallel rows: ONE job, R^ split by receiver rows over the ranks
    cfg = configs.get(args.workload) if rows_mode else shard.replica_config(configs.get(args.workload), rank, world)
    my_rows = shard.row_slice(cfg.n, rank, world) if rows_mode else range(cfg.n)
    nbytes, nb = rhat_bytes(cfg)
    nfoc, niter, nsyn = cfg.nfoc, cfg.niter, nsyn_per_step(cfg)
    big = cfg.k >= 3            # 33 GB / 250 GB of time-domain R: generated on the device in 64-shot chunks, never on the host

    mk = B.Marchenko(cfg.n, cfg.n, cfg.nt, cfg.dt, cfg.dx, cfg.fmin, cfg.fmax, rows=(my_rows.start, len(my_rows)))
    mk.set_option(B.MK_OPT_EPS_SAMPLES, cfg.eps)
    mk.set_option(B.MK_OPT_REGIME, args.regime)
    if args.rhat_layout and cfg.nfoc > 8 and not rows_mode and args.regime in (0, 3):
        mk.set_option(B.MK_OPT_RHAT_LAYOUT, 1)
    if args.tune:
        mk.set_option(B.MK_OPT_TUNE, args.tune)
    ipc_ptrs = []
    if args.parallel == "rows_fused":
        if world > 1:
            ipc_ptrs = shard.attach_ipc(mk, cfg.nfoc, dist)
            ipc_ptrs += shard.sync_attach_ipc(mk, dist)
            torch.cuda.synchronize()
            dist.barrier()              # every rank's flags exist before anyone writes
        else:
            mk.sync_create(0, 1)

        def run_step():                 # the barriers between the ranks are stream-ordered flag writes / waits (mk_sync_barrier)
            shard.run_row_sharded_fused(mk, dGd, dtd, niter, douts, mk.sync_barrier)
    elif rows_mode:
        if world > 1:
            exchange = shard.distributed_exchange(mk, dist)
        else:
            exchange = mk.operand_exchanged                 # one rank owns every row: nothing to move

        def run_step():
            shard.run_row_sharded(mk, dGd, dtd, niter, douts, exchange)
    else:
        def run_step():
            mk.run(dGd, dtd, niter, douts)
    if big:
        ingest_device(mk, cfg, dev)
        dGd, dtd = gen.first_arrivals_torch(cfg, dev)
        R = Gd = td = None
        douts = device_fields(cfg, dev)
    else:
        R, Gd, td = workload_arrays(cfg)
        mk.load_R_host(R)
        dGd = torch.from_numpy(Gd).to(dev)
        dtd = torch.from_numpy(td).to(dev)
        douts = {nm: torch.empty((nfoc, cfg.n, cfg.nt), dtype=torch.float32, device=dev) for nm in FIELDS}

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-timed region: inputs resident in HBM
    r = timed_steps(mk, run_step, args.steps, args.warmup, local, dist, barrier, stride=args.timing_stride)
    ms_total, clocks, launches, syn_n, syn_ms, regime_used = (r[k] for k in ("ms_total", "clocks", "launches", "syn_n", "syn_ms", "regime_used"))
    syn_total = r["syn_total"]
    jobs = 1 if rows_mode else world        # rows: the ranks share ONE job (strong scaling)
    passes = syn_total / max(args.steps, 1)  # contraction launches = passes over R^ per step (17 with the fused finals, else 18)
    value = jobs * passes * nbytes * args.steps / (ms_total * 1e-3) / 1e9          # bytes of R^ actually streamed
    value_alg = jobs * nsyn * nbytes * args.steps / (ms_total * 1e-3) / 1e9        # one R^ per synthesis of Algorithm 1

    # ---- end-to-end through the public host API: pinned host inputs, host outputs, copies inside the timed region
    e2e = None
    if not big and not rows_mode:
        hGd = torch.from_numpy(Gd).pin_memory()
        htd = torch.from_numpy(td).pin_memory()
        houts = {nm: torch.empty((nfoc, cfg.n, cfg.nt), dtype=torch.float32).pin_memory() for nm in FIELDS}
        e2e_steps = max(1, min(args.steps, args.e2e_steps))
        for _ in range(min(3, args.warmup)):
            mk.run_host(hGd, htd, niter, houts)
        barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            mk.run_host(hGd, htd, niter, houts)          # returns after the results are in host memory
        torch.cuda.synchronize()
        e2e_s = shard.max_over_ranks(time.perf_counter() - t0, dist)
        barrier()
        e2e = {"value": world * passes * nbytes * e2e_steps / e2e_s / 1e9, "unit": UNIT,
               "value_algorithmic": world * nsyn * nbytes * e2e_steps / e2e_s / 1e9,
               "h2d_bytes_per_step": int(hGd.numel() * 4 + htd.numel() * 4),
               "d2h_bytes_per_step": int(sum(t.numel() * 4 for t in houts.values())), "steps": e2e_steps,
               "ms_per_step": 1e3 * e2e_s / e2e_steps, "api": "mk_run_host (pinned host G_d, t_d in; 6 host fields out)"}
        del hGd, htd, houts

    for ptr in ipc_ptrs:            # peers' operand mappings: closed on every rank before any context goes away
        B.ipc_close(ptr)
    barrier()
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    share = len(my_rows) / cfg.n            # rows mode: this rank's launches contract its own rows of R^ only
    roof = roofline_of(cfg, nb, nbytes, regime_used, syn_n, syn_ms, ms_total, clocks, share, syn_total)

    # ---- the oracle as it stands, on this box's host cores, bounded sample (rank 0, N = 1 only)
    cpu = None
    if world == 1 and not args.no_cpu_baseline and not big:
        import oracle
        f = [0] if nfoc > 1 else None
        t_s, nrec_s, _, _ = oracle_sample(cfg, R, Gd if f is None else Gd[f], td if f is None else td[f], budget_s=args.cpu_budget)
        cpu = {"value": (nbytes * nrec_s / cfg.n) / t_s / 1e9, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
               "sample": f"one oracle synthesis R N_0 (direct time-domain convolution, fp64) on {nrec_s} of {cfg.n} receivers x 1 focal "
                         f"point of config {cfg.k}: {t_s:.2f} s per synthesis, {getattr(oracle_sample, 'reps', 1)} repetitions"}

    # ---- the large-batch regimes in the same invocation (N = 1, default workload only): configs 2 (tcgen05 and FFMA), 3, 4
    secondary = []
    if world == 1 and args.workload == 1 and not rows_mode and not args.no_secondary:
        # config 1 with compressed R^ (NEXT-4) and with R^ out of core (NEXT-3): contexts of their own
        secondary.append(variant_entry(cfg, R, Gd, td, 100, 5, local, dev, rhat_format=1))
        secondary.append(variant_entry(cfg, R, Gd, td, 5, 3, local, dev, resident_frac=0.25))
        del dGd, dtd, douts, R, Gd, td
        torch.cuda.empty_cache()
        mk.close()
        c2 = configs.get(2)          # same R as config 1 (BASELINE.json), ingested again in the layout of the tensor regime
        mk = B.Marchenko(c2.n, c2.n, c2.nt, c2.dt, c2.dx, c2.fmin, c2.fmax)
        mk.set_option(B.MK_OPT_EPS_SAMPLES, c2.eps)
        mk.set_option(B.MK_OPT_RHAT_LAYOUT, args.rhat_layout)
        mk.load_R_host(gen.R_full(c2))
        # the paper's middle case, 29 focal points, on config 1's R^: the narrow end of the tensor regime
        c29 = configs.scaled(2, nfoc=29, focal="fan:600", name="3GB_29foc")
        secondary.append(secondary_entry(mk, c29, 0, 20, 3, local, dev))
        secondary.append(secondary_entry(mk, c2, 0, args.secondary_steps, 3, local, dev, image=True))
        mk.close()
        if args.rhat_layout:         # the FFMA kernel reads the row-major layout
            mk = B.Marchenko(c2.n, c2.n, c2.nt, c2.dt, c2.dx, c2.fmin, c2.fmax)
            mk.set_option(B.MK_OPT_EPS_SAMPLES, c2.eps)
            mk.load_R_host(gen.R_full(c2))
        secondary.append(secondary_entry(mk, c2, 2, args.secondary_steps, 3, local, dev))
        mk.close()
        for k in (3, 4):
            ck = configs.get(k)
            free, _ = torch.cuda.mem_get_info()
            need = 8.0 * ck.n * nb * (ck.n + 16) + 4.0 * ck.nfoc * ck.n * ck.nt * 4.2 + 8.0 * ck.n * nb * ck.nfoc * 6 + 6e9
            if free < need:
                secondary.append({"workload": f"config{k}:{ck.name}", "skipped": f"needs about {need / 1e9:.0f} GB of device memory, {free / 1e9:.0f} GB free"})
                continue
            mkk = B.Marchenko(ck.n, ck.n, ck.nt, ck.dt, ck.dx, ck.fmin, ck.fmax)
            mkk.set_option(B.MK_OPT_EPS_SAMPLES, ck.eps)
            mkk.set_option(B.MK_OPT_RHAT_LAYOUT, args.rhat_layout)
            t0 = time.perf_counter()
            ingest_device(mkk, ck, dev)
            t_ing = time.perf_counter() - t0
            e = secondary_entry(mkk, ck, 0, args.secondary_steps, 3, local, dev)
            e["ingest_s"] = t_ing
            secondary.append(e)
            mkk.close()
            torch.cuda.empty_cache()
    else:
        mk.close()

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "strong" if rows_mode else "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "value_algorithmic": value_alg,
            "config": {"workload": f"config{cfg.k}:{cfg.name}", "n": cfg.n, "nt": cfg.nt, "nfoc": nfoc, "niter": niter, "nb": nb,
                       "syntheses_per_step": nsyn, "contraction_launches_per_step": passes,
                       "note": ("value = bytes of R^ actually streamed per second (contraction launches x bytes of R^ / time); "
                                "value_algorithmic counts one R^ per synthesis of Algorithm 1 (niter + 2): with 1, 2 or 4 focal points the two "
                                "syntheses of the finals share ONE pass over R^ (2 nfoc right-hand sides), so a step makes niter + 1 passes"
                                if passes < nsyn else "one pass over R^ per synthesis"),
                       "rhat_bytes": nbytes, "regime": regime_used,
                       "kernel_timing": f"every {args.timing_stride}-th contraction launch of the timed region carries CUDA events "
                                        f"({int(syn_n)} of {int(syn_total)}; MK_OPT_TIMING = {args.timing_stride})",
                       "l2": f"inputs_larger_than_L2 (R^ {nbytes / 1e9:.2f} GB vs 126 MB L2; no flush needed)",
                       "input_source": "device generator, 64-shot chunks (no e2e / cpu_baseline legs)" if big else "host arrays",
                       "parallelism": "1 GPU" if world == 1 and not rows_mode else
                                      (f"{world} ranks, receiver rows sharded, " + ("operand rows stored into the peers' operands by the producing kernels"
                                                                                if args.parallel == "rows_fused" else
                                                                                "all-gather of the operand rows per synthesis") if rows_mode
                                       else f"{world} independent replicas (no collective)")},
            "focal_point_iterations_per_s": jobs * nfoc * niter * args.steps / (ms_total * 1e-3),
            "clocks": clocks,
            "e2e": e2e,
            "gpu_launches": launches, "roofline": roof, "cpu_baseline": cpu, "secondary": secondary}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=400)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", type=int, default=1, help="BASELINE.json config index (default 1)")
    ap.add_argument("--regime", type=int, default=0)
    ap.add_argument("--parallel", default="replicas", choices=["replicas", "rows", "rows_fused"],
                    help="N > 1: independent replicas (default, weak scaling) or receiver-row sharding with one all-gather of the "
                         "operand rows per synthesis (strong scaling; SURVEY.md section 8(e) / NEXT-3); rows_fused: the same with the "
                         "all-gather fused into the producing kernels as peer stores over CUDA IPC mappings; the two barriers per synthesis are "
                         "stream memory operations (mk_sync_barrier), no host synchronisation inside a step")
    ap.add_argument("--rhat-layout", type=int, default=1, help="layout of R^ for the tensor-regime workloads (MK_OPT_RHAT_LAYOUT): "
                    "1 tiled in 16 KB boxes (default), 0 row-major")
    ap.add_argument("--timing-stride", type=int, default=5,
                    help="headline run: every N-th contraction launch of the timed region carries CUDA events (MK_OPT_TIMING = N; 17 "
                         "launches per config-1 step, so 5 walks through every position of the step)")
    ap.add_argument("--tune", type=int, default=0, help="MK_OPT_TUNE bit mask (measurement switches of the kernels; include/mk.h)")
    ap.add_argument("--e2e-steps", type=int, default=50)
    ap.add_argument("--cpu-budget", type=float, default=15.0, help="seconds of oracle work for cpu_baseline")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-secondary", action="store_true", help="skip the large-batch configurations (2, 2 with --regime 2, 3, 4) of the default run")
    ap.add_argument("--secondary-steps", type=int, default=10)
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3
    return run_reference(args) if args.impl == "reference" else run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
