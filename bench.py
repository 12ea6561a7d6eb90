#!/usr/bin/env python
"""bench.py — synthesizer throughput of the B200-native Bluebild Standard Synthesizer.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--variant fp32|tf32x3|fp16x3]
                    [--impl ours|reference] [--probe]

A "step" is one pass of the whole hot path over one batch of synthetic input: all collects of
the config (config 4: 20 epochs of the 512-station, N_eig = 64, 8-level, 1024^2 wide-field case)
through collect_eig (prep kernel: centring + phase fold + cast; fused synthesizer kernel: phase
generation, contraction, level epilogue, multi-epoch accumulation). B = W V, the eigenvalues
and hence D come from the library's own device glue (bb_eig), run before the timed region and
timed separately ("glue" in the JSON line), as BASELINE.json's north_star prescribes.
Metric: synthesizer terms/s, a term being one (antenna, eigenpair, pixel) complex MAC.
Prints ONE JSON line on rank 0. See DESIGN.md "Measurement".
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "synthesizer_terms_per_s"
UNIT = "terms/s"
SM_COUNT, FP32_LANES, SM_MAX_MHZ = 148, 128, 1965.0
FP32_PEAK_TFLOPS = SM_COUNT * FP32_LANES * 2 * SM_MAX_MHZ * 1e6 / 1e12        # 74.45, DESIGN.md "Roofline"


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        d["_source"] = "measured"
        return d
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "_source": "fallback"}


# ------------------------------------------------------------------------------------ clocks
class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index=0, period=0.002):
        super().__init__(daemon=True)
        self.index, self.period, self.samples, self.reasons, self.max_mhz = index, period, [], set(), None
        self._stop_ev = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception:
            self.nv = None

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {"hw_slowdown": getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8),
                 "hw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40),
                 "sw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20),
                 "sw_power_cap": getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4),
                 "hw_power_brake": getattr(nv, "nvmlClocksEventReasonHwPowerBrakeSlowdown", 0x80)}
        while not self._stop_ev.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                try:
                    mask = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if mask & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(self.period)

    def finish(self):
        self._stop_ev.set()
        if self.is_alive():
            self.join(timeout=2)
        med = float(np.median(self.samples)) if self.samples else None
        lo = float(np.min(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_min_mhz": lo, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


# ------------------------------------------------------------------------------------ workload
def prepare_inputs(cfg_idx, ctx, binding, workloads):
    """Per-collect (B, D, xyz, wavelength) from the library's own glue; level edges per DESIGN.md."""
    w = workloads.make_workload(cfg_idx)
    c = w.cfg
    mid = w.collect_inputs(w.mid_collect())
    t0 = time.time()
    mu, _ = ctx.eig(mid["S"], mid["W"], mid["xyz"], mid["wavelength"], c.n_eig, want_B=False)
    items, lo, hi = [], mu[-1], mu[0]
    for n in range(c.n_collects):
        ci = w.collect_inputs(n)
        lam, B = ctx.eig(ci["S"], ci["W"], ci["xyz"], ci["wavelength"], c.n_eig)
        lo, hi = min(lo, lam[-1]), max(hi, lam[0])
        items.append(dict(B=B, lam=lam, xyz=ci["xyz"], wavelength=ci["wavelength"]))
    iv = workloads.choose_intervals(mu, c.n_levels, lam_max=hi, lam_min=lo)
    for it in items:
        lam = it["lam"]
        inside = (lam[None, :] >= iv[:, :1]) & (lam[None, :] <= iv[:, 1:])
        it["D"] = np.asfortranarray(np.where(inside, lam[None, :], 0.0).astype(np.float32))
    return w, items, iv, time.time() - t0


# ------------------------------------------------------------------------------------ ranks
def dist_env():
    return int(os.environ.get("RANK", 0)), int(os.environ.get("WORLD_SIZE", 1)), int(os.environ.get("LOCAL_RANK", 0))


def init_dist(backend):
    import torch.distributed as dist
    rank, world, _ = dist_env()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29511")
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, world


def aggregate_over_ranks(local_ms: float, local_units: float, device=None):
    """Replicas only: every rank processes its own units; the job time is the
    MAX over ranks, the job's units the SUM. No data-path collective exists; these two scalars are
    the only thing reduced. Returns (max_ms, total_units)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(local_ms), float(local_units)
    t = torch.tensor([local_ms], dtype=torch.float64, device=device)
    u = torch.tensor([local_units], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


# ------------------------------------------------------------------------------------ oracle leg
def oracle_sample_run(oracle, w, items, n_levels, target_s, reps=1):
    """Times the oracle, as it stands, on a bounded pixel sample of the same workload (all collects)."""
    cores = oracle.hardware_threads()
    sub_all = w.sample_pixels(4)
    terms_per_pix = sum(it["B"].shape[0] * it["B"].shape[1] for it in items)
    probe = w.pixels(sub_all[:4 * cores])
    t0 = time.perf_counter()
    oracle.synth(items[0]["B"], items[0]["D"], items[0]["xyz"], probe, items[0]["wavelength"])
    rate = items[0]["B"].size * probe.shape[0] / max(time.perf_counter() - t0, 1e-6)
    n_s = int(max(cores, min(sub_all.size, target_s * rate / terms_per_pix)))
    n_s = max(cores, n_s // cores * cores)
    pix = w.pixels(sub_all[:n_s])
    times = []
    for _ in range(reps):
        img = np.zeros((n_levels, pix.shape[0]))
        t0 = time.perf_counter()
        for it in items:
            oracle.synth(it["B"], it["D"], it["xyz"], pix, it["wavelength"], img=img)
        times.append(time.perf_counter() - t0)
    terms = terms_per_pix * pix.shape[0]
    sample = "%d of %d pixels (every 4th row/column subset), all %d collects" % (pix.shape[0], w.cfg.n_pix, len(items))
    return terms, times, cores, sample


def run_reference(args):
    rank, world, _ = dist_env()
    if rank != 0:
        return
    from oracle import bluebild_oracle as oracle
    from paper_2310_09200_b200 import workloads
    oracle.build()
    w = workloads.make_workload(args.config)
    c = w.cfg
    items = []
    mid = w.collect_inputs(w.mid_collect())
    mu, _ = oracle.eig_stage(mid["S"], mid["W"], mid["xyz"], mid["wavelength"], c.n_eig)
    iv = workloads.choose_intervals(mu, c.n_levels, lam_max=4 * mu[0], lam_min=mu[-1] / 4)
    for n in range(c.n_collects):
        ci = w.collect_inputs(n)
        lam, B = oracle.eig_stage(ci["S"], ci["W"], ci["xyz"], ci["wavelength"], c.n_eig)
        items.append(dict(B=np.asfortranarray(B.astype(np.complex64)), D=oracle.level_weights(lam, iv).astype(np.float32),
                          xyz=ci["xyz"], wavelength=ci["wavelength"]))
    terms, times, cores, sample = oracle_sample_run(oracle, w, items, c.n_levels, args.ref_step_seconds,
                                                    reps=args.warmup + args.steps)
    timed = times[args.warmup:]
    ms = 1e3 * float(np.mean(timed))
    value = terms / (ms * 1e-3)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": "config %d: %s" % (c.idx, c.name), "n_ant": c.n_ant, "n_eig": c.n_eig,
                       "n_levels": c.n_levels, "n_pix": c.n_pix, "n_collects": c.n_collects, "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# ------------------------------------------------------------------------------------ our arm
def run_ours(args):
    import torch
    from paper_2310_09200_b200 import binding, workloads
    rank, world, local_rank = dist_env()
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU fallback)"
    torch.cuda.set_device(local_rank)
    init_dist("nccl")
    binding.load_library()
    ctx = binding.Context(local_rank)
    dev = "cuda:%d" % local_rank
    w, items, iv, glue_wall_s = prepare_inputs(args.config, ctx, binding, workloads)
    c = w.cfg
    L = c.n_levels
    pix = w.pixels()

    # ---- device-resident arm ------------------------------------------------------------------
    DM = binding.DeviceMatrix
    dev_items = [dict(B=DM.from_numpy(it["B"], np.complex64, dev), D=DM.from_numpy(it["D"], np.float32, dev),
                      xyz=DM.from_numpy(it["xyz"], np.float64, dev), wavelength=it["wavelength"]) for it in items]
    s = binding.StandardSynthesis(ctx, DM.from_numpy(pix, np.float64, dev), L, args.variant)
    flush_buf = torch.empty(256 << 20, dtype=torch.uint8, device=dev)

    def step_device():
        for it in dev_items:
            s.collect_eig(it["B"], it["D"], it["xyz"], it["wavelength"])
        s.flush()

    for _ in range(args.warmup):
        step_device()
        flush_buf.zero_()
    torch.cuda.synchronize()
    t_before, l_before = s.timings(), s.launches()
    sampler = ClockSampler(local_rank)
    sampler.start()
    barrier()
    torch.cuda.synchronize()
    evs = []
    for _ in range(args.steps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        step_device()
        e1.record()
        evs.append((e0, e1))
        flush_buf.zero_()                           # L2 flush between steps, outside the event pairs
    torch.cuda.synchronize()
    barrier()
    clocks = sampler.finish()
    local_ms = sum(a.elapsed_time(b) for a, b in evs)
    t_after, l_after = s.timings(), s.launches()
    terms_step = float(c.total_terms)
    max_ms, total_terms = aggregate_over_ranks(local_ms, terms_step * args.steps, dev)
    ms_per_step = max_ms / args.steps
    value = total_terms / (max_ms * 1e-3)
    synth_ms = t_after["synth_ms"] - t_before["synth_ms"]
    prep_ms = t_after["prep_ms"] - t_before["prep_ms"]
    launches = l_after - l_before
    # synthesizer launches: one per queue flush (and per eigen slab) — everything else is a prep launch
    synth_launches = launches - args.steps * len(items)
    avg_launch_ms = synth_ms / max(synth_launches, 1)
    flops_per_launch = 8.0 * terms_step * args.steps / max(synth_launches, 1)
    achieved_tflops = flops_per_launch / (avg_launch_ms * 1e-3) / 1e12

    # ---- end-to-end arm: host buffers in, host images out, through the C ABI --------------------
    s2 = binding.StandardSynthesis(ctx, pix, L, args.variant)
    out = torch.empty((L, c.n_pix), dtype=torch.float32, pin_memory=True).numpy()    # page-locked result buffer

    def step_e2e():
        for it in items:
            s2.collect_eig(it["B"], it["D"], it["xyz"], it["wavelength"])
        for l in range(L):
            s2.get(l, out[l])

    e2e_steps = max(1, min(args.steps, 5))
    step_e2e()
    torch.cuda.synchronize()
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        step_e2e()
    torch.cuda.synchronize()
    e2e_local_ms = 1e3 * (time.perf_counter() - t0)
    barrier()
    e2e_ms, e2e_terms = aggregate_over_ranks(e2e_local_ms, terms_step * e2e_steps, dev)
    h2d = sum(it["B"].nbytes + it["D"].nbytes + it["xyz"].nbytes for it in items)
    d2h = out.nbytes

    # ---- glue, timed separately: whole collect (Gram + eigensolve + select + prep) on one handle ----
    glue = None
    if rank == 0:
        s3 = binding.StandardSynthesis(ctx, pix[:1024], L, args.variant)
        ncol = min(len(items), 8)
        for n in range(ncol):
            ci = w.collect_inputs(n)
            s3.collect(ci["S"], ci["W"], ci["xyz"], ci["wavelength"], c.n_eig, iv)
        t3 = s3.timings()
        glue = {"gram_ms_per_collect": t3["gram_ms"] / ncol, "eig_ms_per_collect": t3["eig_ms"] / ncol,
                "collects_timed": ncol, "precision": "f64", "solver": "cusolverDnZhegvd"}
        # the same through bb_synth_collect_batch: one potrfBatched / trsmBatched / XsyevBatched per 16 collects
        nb = min(len(items), 16)
        raws = [w.collect_inputs(n) for n in range(nb)]
        Sb, Xb = np.stack([r["S"] for r in raws]), np.stack([r["xyz"] for r in raws])
        Wb = None if raws[0]["W"] is None else np.stack([r["W"] for r in raws])
        s4 = binding.StandardSynthesis(ctx, pix[:1024], L, args.variant)
        for rep in range(2):                                      # first pass pays the library's one-time setup
            tb4 = s4.timings()
            s4.collect_batch(Sb, Wb, Xb, [r["wavelength"] for r in raws], c.n_eig, iv)
        t4 = s4.timings()
        glue["batched"] = {"gram_ms_per_collect": (t4["gram_ms"] - tb4["gram_ms"]) / nb,
                           "eig_ms_per_collect": (t4["eig_ms"] - tb4["eig_ms"]) / nb, "collects_per_batch": nb,
                           "solver": "cusolverDnZpotrfBatched + cublasZtrsmBatched + cusolverDnXsyevBatched"}

    # ---- the other kernel variants on the same device-resident inputs (north_star: compare them) ----
    others = {}
    if rank == 0 and not args.no_compare:
        for v in ("fp32", "tf32x3", "fp16x3"):
            if v == args.variant:
                continue
            sv = binding.StandardSynthesis(ctx, DM.from_numpy(pix, np.float64, dev), L, v)
            for rep in range(3):                                  # 2 warm-up passes, 1 timed
                if rep == 2:
                    tb = sv.timings()
                for it in dev_items:
                    sv.collect_eig(it["B"], it["D"], it["xyz"], it["wavelength"])
                sv.flush()
                flush_buf.zero_()
            ms = sv.timings()["synth_ms"] - tb["synth_ms"]
            others[v] = {"synth_ms_per_step": ms, "terms_per_s": terms_step / (ms * 1e-3)}
            del sv

    if rank != 0:
        return
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": {"fp32": "f32", "tf32x3": "tf32x3", "fp16x3": "fp16x3"}[args.variant], "data": "synthetic",
        "config": {"workload": "config %d: %s" % (c.idx, c.name), "n_ant": c.n_ant, "n_beam": c.n_beam, "n_eig": c.n_eig,
                   "n_levels": L, "n_pix": c.n_pix, "n_collects": c.n_collects, "variant": args.variant,
                   "parallelism": "replicas x%d (no collective)" % world,
                   "l2": "flushed between steps (256 MiB memset, outside the per-step event pairs)",
                   "timing": "sum of per-step CUDA-event pairs on the library's stream, max over ranks"},
        "clocks": clocks,
        "e2e": {"value": e2e_terms / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "ms_per_step": e2e_ms / e2e_steps, "steps": e2e_steps,
                "what": "collect_eig from host numpy buffers + bb_synth_get of every level image to host"},
        "gpu_launches": int(launches),
        "images_per_s": {"image_sets": 1e3 / ms_per_step * world, "collect_images": c.n_collects * 1e3 / ms_per_step * world},
        "kernel_ms": {"synth_ms_per_step": synth_ms / args.steps, "prep_ms_per_step": prep_ms / args.steps,
                      "synth_launches": int(synth_launches)},
        "glue": glue,
        "other_variants": others,
    }
    peak = FP32_PEAK_TFLOPS
    bound = "alu"
    if args.variant != "fp32":
        mp = measured_peaks()
        # dense FP16 = dense bf16; dense TF32 = 1/2 of it (guide's nominal ratio)
        peak = mp["bf16_tflops"] * (1.0 if args.variant == "fp16x3" else 0.5)
        bound = "tensor"
    line["roofline"] = {"bound": bound, "achieved": achieved_tflops, "peak": peak, "unit": "TFLOP/s",
                        "frac": achieved_tflops / peak, "traffic": None,
                        "kernel": "synth_fp32_kernel" if args.variant == "fp32" else "synth_tc_kernel",
                        "flops_per_launch": flops_per_launch, "avg_launch_ms": avg_launch_ms,
                        "peak_basis": ("148 SM x 128 FP32 lanes x 2 x 1.965 GHz (derived, DESIGN.md)" if bound == "alu" else
                                       ("1.0" if args.variant == "fp16x3" else "0.5") + " x measured bf16 burst (MEASURED_PEAKS.json); useful flops = 8/term, issued = 24/term")}
    # DRAM traffic of one launch of this kernel, from the committed `ncu --set full` capture of the same command
    prof = os.path.join(ROOT, "profiles", "r01_%s_ncu_full.csv" % args.variant)
    if args.config == 4 and os.path.exists(prof):
        try:
            import csv
            mb = {r[0]: float(r[2]) for r in csv.reader(open(prof)) if len(r) >= 3 and r[0].startswith("dram__bytes_") and r[1] == "Mbyte"}
            if "dram__bytes_read.sum" in mb and "dram__bytes_write.sum" in mb:
                line["roofline"]["traffic"] = (mb["dram__bytes_read.sum"] + mb["dram__bytes_write.sum"]) * 1e6
                line["roofline"]["traffic_source"] = "profiles/" + os.path.basename(prof)
        except Exception:
            pass
    if bound == "tensor":
        # the split-precision scheme issues 3 tensor passes per useful one: 24 flops per term on the pipe
        line["roofline"]["issued_tflops"] = 3.0 * achieved_tflops
        line["roofline"]["issued_frac"] = 3.0 * achieved_tflops / peak
        sus = mp.get("bf16_tflops_sustained")
        if sus:                                              # the power-capped figure (cuBLAS bf16 back to back for seconds)
            line["roofline"]["issued_frac_of_sustained_peak"] = 3.0 * achieved_tflops / (sus * (1.0 if args.variant == "fp16x3" else 0.5))
    if clocks.get("sm_mhz"):
        line["roofline"]["frac_at_observed_clock"] = achieved_tflops / (peak * clocks["sm_mhz"] / SM_MAX_MHZ) if bound == "alu" else None
    if args.probe:
        line["probe"] = {k: ctx.probe_peak(i)[0] for i, k in enumerate(
            ["ffma_per_s", "ffma2_fma_per_s", "mufu_per_s", "dfma_per_s", "dfma_chains_alone_per_s", "dfma_chains_under_mma_per_s",
             "imad_chains_alone_per_s", "imad_chains_under_mma_per_s"])}
    if world == 1 and not args.no_cpu_baseline:
        from oracle import bluebild_oracle as oracle      # cpu_baseline leg: the one place bench.py runs the oracle
        oracle.build()
        terms, times, cores, sample = oracle_sample_run(oracle, w, items, L, args.cpu_seconds)
        line["cpu_baseline"] = {"value": terms / times[0], "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample}
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--variant", default=os.environ.get("BB_VARIANT", "fp16x3"), choices=["fp32", "tf32x3", "fp16x3"])
    ap.add_argument("--no-compare", action="store_true", help="skip the short timing of the other two variants")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--probe", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    ap.add_argument("--ref-step-seconds", type=float, default=10.0)
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
