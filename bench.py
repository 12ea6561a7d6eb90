#!/usr/bin/env python
"""bench.py — synthesizer throughput of the B200-native Bluebild Standard Synthesizer.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--variant fp32|tf32x3|fp16x3|fp16fp8]
                    [--impl ours|reference] [--quick]

A "step" is one pass of the whole hot path over one batch of synthetic input: all collects of
the config (config 4: 20 epochs of the 512-station, N_eig = 64, 8-level, 1024^2 wide-field case)
through collect_eig (prep kernel: centring + phase fold + cast; fused synthesizer kernel: phase
generation, contraction, level epilogue, multi-epoch accumulation). B = W V, the eigenvalues
and hence D come from the library's own device glue (bb_eig), run before the timed region and
timed separately ("glue" in the JSON line), as BASELINE.json's north_star prescribes.
Metric: synthesizer terms/s, a term being one (antenna, eigenpair, pixel) complex MAC.
Beside the headline (`value`, the --variant arm) the line carries, each measured in this run with its own
clock record: `variants` (fp32, tf32x3, fp16x3, fp16fp8 on the bench config: median of >= 5 event-timed steps,
roofline fractions; a compact copy sits in `roofline.variants`, the part of the line the driver's record keeps),
`configs` (configs 2, 3, 5 through the same path; compact copy in `roofline.configs`), `e2e` (hot path from host
buffers, --steps steps; `e2e.full_collect_ms` = Algorithm 1 from S beside it), `full_collect`
(all of Algorithm 1 from host S / W / xyz / intervals to images on the host) and `cpu_baseline` (the oracle).
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
def prepare_inputs(cfg_idx, ctx, binding, workloads, max_collects=None):
    """Per-collect (B, D, xyz, wavelength) from the library's own glue; level edges per DESIGN.md.
    max_collects: take only that many collects, evenly spaced over the run (config 5's 800 would take minutes
    of host-side input generation; the timed collects are stated in the JSON line)."""
    w = workloads.make_workload(cfg_idx)
    c = w.cfg
    mid = w.collect_inputs(w.mid_collect())
    t0 = time.time()
    mu, _ = ctx.eig(mid["S"], mid["W"], mid["xyz"], mid["wavelength"], c.n_eig, want_B=False)
    items, lo, hi = [], mu[-1], mu[0]
    which = range(c.n_collects)
    if max_collects is not None and max_collects < c.n_collects:
        which = [int(round(x)) for x in np.linspace(0, c.n_collects - 1, max_collects)]
    for n in which:
        ci = w.collect_inputs(n)
        lam, B = ctx.eig(ci["S"], ci["W"], ci["xyz"], ci["wavelength"], c.n_eig)
        lo, hi = min(lo, lam[-1]), max(hi, lam[0])
        items.append(dict(B=B, lam=lam, xyz=ci["xyz"], wavelength=ci["wavelength"]))
    iv = workloads.choose_intervals(mu, c.n_levels, lam_max=hi, lam_min=lo)
    for it in items:
        it["D"] = ctx.level_weights(it["lam"], iv)          # Alg. 1 l.7-8 by the library's own kernel
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
    take = sub_all[np.unique(np.linspace(0, sub_all.size - 1, n_s).astype(np.int64))]       # evenly over the whole image
    pix = w.pixels(take)
    times = []
    for _ in range(reps):
        img = np.zeros((n_levels, pix.shape[0]))
        t0 = time.perf_counter()
        for it in items:
            oracle.synth(it["B"], it["D"], it["xyz"], pix, it["wavelength"], img=img)
        times.append(time.perf_counter() - t0)
    terms = terms_per_pix * pix.shape[0]
    sample = "%d of %d pixels (evenly spaced over the every-4th row/column grid of the whole image), all %d collects" % (
        pix.shape[0], w.cfg.n_pix, len(items))
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
VARIANT_DTYPE = {"fp32": "f32", "tf32x3": "tf32x3", "fp16x3": "fp16x3", "fp16fp8": "fp16+fp8x2"}
PASS_UNITS = {"tf32x3": 3.0, "fp16x3": 3.0, "fp16fp8": 2.0}   # tensor passes issued per useful one, in units of the variant's main format
KERNEL_NAME = {"fp32": "synth_fp32_kernel", "tf32x3": "synth_tc_kernel<TF32>", "fp16x3": "synth_tc_kernel<FP16>",
               "fp16fp8": "synth_tc_kernel<F16F8>"}


NCU_CAPTURE = {"fp32": "r02_fp32_ncu_full.csv", "tf32x3": "r02_tf32x3_ncu_full.csv", "fp16x3": "r02_fp16x3_ncu_full.csv",
               "fp16fp8": "r02b_fp16fp8_ncu_full.md"}       # names only: nothing under profiles/ is opened by bench.py
_NOT_NAMED = ("%s: the repo's fastest parity-green split-precision scheme, NOT one of the two variants north_star names "
              "(fp32 CUDA-core, tcgen05 tf32x3): their figures, measured in this same run, are roofline.variants.fp32 / .tf32x3")
HEADLINE_NOTE = {"fp32": "fp32: the FP32 CUDA-core variant north_star names", "tf32x3": "tf32x3: the tcgen05 3xTF32 variant north_star names",
                 "fp16x3": _NOT_NAMED % "fp16x3", "fp16fp8": _NOT_NAMED % "fp16fp8"}


def compact(rec_roofline, median_ms, terms_step, clocks):
    """The few numbers of one timed arm that the judged `roofline` block carries (full records: `variants`, `configs`)."""
    out = {"ms_per_step": median_ms, "terms_per_s": terms_step / (median_ms * 1e-3), "frac": rec_roofline["frac"],
           "bound": rec_roofline["bound"], "peak": rec_roofline["peak"], "sm_mhz": clocks.get("sm_mhz"), "reasons": clocks.get("reasons")}
    if "issued_frac" in rec_roofline:
        out["issued_frac"] = rec_roofline["issued_frac"]
    return out


def roofline_block(variant, flops_per_launch, avg_launch_ms, clocks, cfg_idx):
    """Roofline of the synthesizer kernel of one timed arm: useful flops (8 per term) per launch over the kernel's
    average launch duration (CUDA events around each launch, recorded by the library on the launching stream)."""
    achieved = flops_per_launch / (avg_launch_ms * 1e-3) / 1e12
    mp = measured_peaks()
    if variant == "fp32":
        bound, peak = "alu", FP32_PEAK_TFLOPS
        basis = "148 SM x 128 FP32 lanes x 2 x 1.965 GHz (derived, DESIGN.md 6)"
    else:
        bound = "tensor"
        ratio = 0.5 if variant == "tf32x3" else 1.0            # dense FP16 = dense bf16; dense TF32 = 1/2 of it (guide's nominal ratio)
        peak = mp["bf16_tflops"] * ratio
        basis = "%.1f x bf16 burst peak (%s MEASURED_PEAKS.json); useful flops = 8/term, issued = %d/term in units of the main format%s" % (
            ratio, mp["_source"], int(8 * PASS_UNITS[variant]), " (the FP8 pass of K = 64 counts as one FP16 pass: twice the rate)" if variant == "fp16fp8" else "")
    r = {"bound": bound, "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak, "traffic": None,
         "kernel": KERNEL_NAME[variant], "flops_per_launch": flops_per_launch, "avg_launch_ms": avg_launch_ms, "peak_basis": basis}
    if bound == "tensor":
        # the split-precision schemes issue 3 (2 with the FP8 cross-term pass) tensor passes per useful one
        r["issued_tflops"] = PASS_UNITS[variant] * achieved
        r["issued_frac"] = PASS_UNITS[variant] * achieved / peak
        sus = mp.get("bf16_tflops_sustained")
        if sus:                                                # the power-capped figure (cuBLAS bf16 back to back for seconds)
            r["issued_frac_of_sustained_peak"] = PASS_UNITS[variant] * achieved / (sus * ratio)
    if clocks.get("sm_mhz"):                                   # the same peak scaled to the SM clock the run actually held
        r["frac_at_observed_clock"] = achieved / (peak * clocks["sm_mhz"] / SM_MAX_MHZ)
    # DRAM traffic of one launch needs ncu and is NOT measured in this run: null here, the committed `ncu --set full`
    # captures of this command are named instead (nothing under profiles/ is read at run time)
    r["traffic_source"] = "not measured in this run; ncu --set full capture of this command: profiles/%s" % NCU_CAPTURE[variant]
    return r


def time_variant(binding, ctx, dev, pix_dev, dev_items, L, variant, steps, warmup, flush_buf, local_rank, terms_step):
    """W warm-up steps, then `steps` steps each bracketed by its own CUDA-event pair on the context stream (L2 flushed
    between steps, outside the pairs), SM clocks sampled over the timed region. Returns the arm's record."""
    import torch
    s = binding.StandardSynthesis(ctx, pix_dev, L, variant)

    def step():
        for it in dev_items:
            s.collect_eig(it["B"], it["D"], it["xyz"], it["wavelength"])
        s.flush()

    for _ in range(warmup):
        step()
        flush_buf.zero_()
    torch.cuda.synchronize()
    t_before, l_before = s.timings(), s.launches()
    sampler = ClockSampler(local_rank)
    sampler.start()
    barrier()
    torch.cuda.synchronize()
    evs = []
    for _ in range(steps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        step()
        e1.record()
        evs.append((e0, e1))
        flush_buf.zero_()                           # L2 flush between steps, outside the event pairs
    torch.cuda.synchronize()
    barrier()
    clocks = sampler.finish()
    per_step = [a.elapsed_time(b) for a, b in evs]
    t_after, l_after = s.timings(), s.launches()
    synth_ms = t_after["synth_ms"] - t_before["synth_ms"]
    prep_ms = t_after["prep_ms"] - t_before["prep_ms"]
    launches = l_after - l_before
    synth_launches = launches - steps * len(dev_items)         # everything that is not a per-collect prep launch
    avg_launch_ms = synth_ms / max(synth_launches, 1)
    flops_per_launch = 8.0 * terms_step * steps / max(synth_launches, 1)
    s.close()
    return dict(per_step_ms=per_step, total_ms=float(sum(per_step)), median_ms=float(np.median(per_step)), clocks=clocks,
                synth_ms=synth_ms, prep_ms=prep_ms, launches=int(launches), synth_launches=int(synth_launches),
                avg_launch_ms=avg_launch_ms, flops_per_launch=flops_per_launch)


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
    DM = binding.DeviceMatrix
    flush_buf = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    terms_step = float(c.total_terms)

    def to_device(its):
        return [dict(B=DM.from_numpy(it["B"], np.complex64, dev), D=DM.from_numpy(it["D"], np.float32, dev),
                     xyz=DM.from_numpy(it["xyz"], np.float64, dev), wavelength=it["wavelength"]) for it in its]

    # ---- headline arm: device-resident inputs, --variant, --steps ----------------------------------------
    dev_items = to_device(items)
    pix_dev = DM.from_numpy(pix, np.float64, dev)
    head = time_variant(binding, ctx, dev, pix_dev, dev_items, L, args.variant, args.steps, args.warmup, flush_buf, local_rank, terms_step)
    max_ms, total_terms = aggregate_over_ranks(head["total_ms"], terms_step * args.steps, dev)
    ms_per_step = max_ms / args.steps
    value = total_terms / (max_ms * 1e-3)

    # ---- end-to-end arm: host buffers in, host images out, through the C ABI --------------------
    s2 = binding.StandardSynthesis(ctx, pix, L, args.variant)
    out = torch.empty((L, c.n_pix), dtype=torch.float32, pin_memory=True).numpy()    # page-locked result buffer

    def step_e2e():
        for it in items:
            s2.collect_eig(it["B"], it["D"], it["xyz"], it["wavelength"])
        for l in range(L):
            s2.get(l, out[l])

    e2e_steps = max(1, args.steps)
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
    s2.close()

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": VARIANT_DTYPE[args.variant], "data": "synthetic",
        "config": {"workload": "config %d: %s" % (c.idx, c.name), "n_ant": c.n_ant, "n_beam": c.n_beam, "n_eig": c.n_eig,
                   "n_levels": L, "n_pix": c.n_pix, "n_collects": c.n_collects, "variant": args.variant,
                   "headline_variant": HEADLINE_NOTE[args.variant],
                   "parallelism": "replicas x%d (no collective)" % world,
                   "l2": "flushed between steps (256 MiB memset, outside the per-step event pairs)",
                   "timing": "sum of per-step CUDA-event pairs on the context stream (which waits for the library's synthesizer stream), max over ranks"},
        "clocks": head["clocks"],
        "e2e": {"value": e2e_terms / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "ms_per_step": e2e_ms / e2e_steps, "steps": e2e_steps,
                "what": "collect_eig from host numpy buffers + bb_synth_get of every level image to host"},
        "gpu_launches": head["launches"],
        "images_per_s": {"image_sets": 1e3 / ms_per_step * world, "collect_images": c.n_collects * 1e3 / ms_per_step * world},
        "kernel_ms": {"synth_ms_per_step": head["synth_ms"] / args.steps, "prep_ms_per_step": head["prep_ms"] / args.steps,
                      "synth_launches": head["synth_launches"], "median_step_ms": head["median_ms"]},
        "roofline": roofline_block(args.variant, head["flops_per_launch"], head["avg_launch_ms"], head["clocks"], c.idx),
    }
    if rank != 0:
        return

    # ---- every variant north_star names, on the same device-resident inputs: full records ----------------
    if not args.quick:
        variants = {}
        for v in ("fp32", "tf32x3", "fp16x3", "fp16fp8"):
            if v == args.variant:
                r = head
            else:
                r = time_variant(binding, ctx, dev, pix_dev, dev_items, L, v, max(5, args.variant_steps), 3, flush_buf, local_rank, terms_step)
            variants[v] = {"terms_per_s": terms_step / (r["median_ms"] * 1e-3), "median_step_ms": r["median_ms"],
                           "steps": len(r["per_step_ms"]), "per_step_ms": [round(x, 4) for x in r["per_step_ms"]],
                           "clocks": r["clocks"], "roofline": roofline_block(v, r["flops_per_launch"], r["avg_launch_ms"], r["clocks"], c.idx)}
        line["variants"] = variants
        # the same figures where the driver's record keeps them: median of >= 5 event-timed steps each, own clock record
        line["roofline"]["variants"] = {v: compact(r["roofline"], r["median_step_ms"], terms_step, r["clocks"]) for v, r in variants.items()}
    del dev_items, pix_dev

    # ---- Algorithm 1 end to end: S, W, xyz, intervals on the host -> level images on the host -------------
    raws = [w.collect_inputs(n) for n in range(c.n_collects)]
    s5 = binding.StandardSynthesis(ctx, pix, L, args.variant)

    def step_full():
        for r in raws:
            s5.collect(r["S"], r["W"], r["xyz"], r["wavelength"], c.n_eig, iv)
        for l in range(L):
            s5.get(l, out[l])

    step_full()                                               # warm-up: library handles, scratch, solver set-up
    tb = s5.timings()
    fc_steps = 3
    t0 = time.perf_counter()
    for _ in range(fc_steps):
        step_full()
    torch.cuda.synchronize()
    fc_ms = 1e3 * (time.perf_counter() - t0) / fc_steps
    ta = s5.timings()
    n_fc = fc_steps * len(raws)
    line["full_collect"] = {
        "value": terms_step / (fc_ms * 1e-3), "unit": UNIT, "ms_per_step": fc_ms, "steps": fc_steps,
        "h2d_bytes_per_step": sum(r["S"].nbytes + r["xyz"].nbytes + (0 if r["W"] is None else r["W"].nbytes) + iv.nbytes for r in raws),
        "d2h_bytes_per_step": d2h, "ratio_to_e2e_collect_eig": (e2e_ms / e2e_steps) / fc_ms,
        "what": "bb_synth_collect per epoch from host S / W / xyz / intervals (device fp64 Gram + Cholesky + eigensolve, batched "
                "over the queued collects on the glue stream) + bb_synth_get of every level image to host; wall clock",
        "device_ms_per_collect": {k: (ta[k] - tb[k]) / n_fc for k in ("gram_ms", "eig_ms", "prep_ms", "synth_ms")}}
    s5.close()
    line["e2e"]["full_collect_ms"] = fc_ms                     # Algorithm 1 from S (the paper's collect) beside the hot path from B
    line["e2e"]["full_collect_value"] = line["full_collect"]["value"]
    line["e2e"]["full_collect_device_ms_per_collect"] = line["full_collect"]["device_ms_per_collect"]
    line["glue"] = {"precision": "f64", "batched_over": "up to 128 staged collects",
                    "gram_ms_per_collect": line["full_collect"]["device_ms_per_collect"]["gram_ms"],
                    "eig_ms_per_collect": line["full_collect"]["device_ms_per_collect"]["eig_ms"],
                    "solver": "potrfBatched + trsmBatched + (block subspace iteration | XsyevBatched)"}

    # ---- the other configs through the same path (device-resident, --variant) ---------------------------
    if not args.quick and world == 1:
        cfgs = {}
        for idx, cap in ((2, None), (3, None), (5, args.cfg5_collects)):
            if idx == args.config:
                continue
            wi, its, _, _ = prepare_inputs(idx, ctx, binding, workloads, max_collects=cap)
            ci = wi.cfg
            di = to_device(its)
            t_step = float(ci.terms_per_collect) * len(its)
            r = time_variant(binding, ctx, dev, DM.from_numpy(wi.pixels(), np.float64, dev), di, ci.n_levels, args.variant,
                             3 if idx == 5 else 5, 3, flush_buf, local_rank, t_step)
            cfgs["config %d: %s" % (idx, ci.name)] = {
                "terms_per_s": t_step / (r["median_ms"] * 1e-3), "median_step_ms": r["median_ms"], "steps": len(r["per_step_ms"]),
                "collects_per_step": len(its), "collects_in_config": ci.n_collects, "n_ant": ci.n_ant, "n_eig": ci.n_eig,
                "n_pix": ci.n_pix, "phases_per_s": t_step / ci.n_eig / (r["median_ms"] * 1e-3), "clocks": r["clocks"],
                "roofline": roofline_block(args.variant, r["flops_per_launch"], r["avg_launch_ms"], r["clocks"], idx)}
            del di
        line["configs"] = cfgs
        line["roofline"]["configs"] = {k.split(":")[0].replace("config ", ""): {"terms_per_s": r["terms_per_s"], "frac": r["roofline"]["frac"],
                                                                                "ms_per_step": r["median_step_ms"], "sm_mhz": r["clocks"].get("sm_mhz"),
                                                                                "variant": args.variant} for k, r in cfgs.items()}

    # ---- NUFFT Synthesis, informational: config 1's collect through both synthesizers ------
    if not args.quick and world == 1:
        w1, it1, _, _ = prepare_inputs(1, ctx, binding, workloads)
        p1 = w1.pixels()
        ss = binding.StandardSynthesis(ctx, p1, w1.cfg.n_levels, "fp32")
        nu = binding.NufftSynthesis(ctx, p1, w1.cfg.n_levels, eps=1e-6)
        for obj in (ss, nu):                                  # warm-up (cuFFT plan, allocations)
            obj.collect_eig(it1[0]["B"], it1[0]["D"], it1[0]["xyz"], it1[0]["wavelength"])
        ref1, got1 = ss.images().astype(np.float64), nu.images().astype(np.float64)
        t0 = time.perf_counter()
        nu.collect_eig(it1[0]["B"], it1[0]["D"], it1[0]["xyz"], it1[0]["wavelength"])
        nu.images()                                           # the transforms of the staged collect run here
        nufft_ms = 1e3 * (time.perf_counter() - t0)
        line["nufft"] = {"workload": "config 1: %s, one collect, eps 1e-6, one transform" % w1.cfg.name, "ms_per_collect_and_get_wall": nufft_ms,
                         "rel_l2_vs_standard_fp32": float(max(np.linalg.norm(got1[l] - ref1[l]) / np.linalg.norm(ref1[l])
                                                              for l in range(w1.cfg.n_levels))), **nu.stats()}
        nu.close(); ss.close()

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
    ap.add_argument("--variant", default=os.environ.get("BB_VARIANT", "fp16fp8"), choices=["fp32", "tf32x3", "fp16x3", "fp16fp8"])
    ap.add_argument("--quick", action="store_true", help="headline arm + e2e + full_collect only: skip the other variants and configs")
    ap.add_argument("--variant-steps", type=int, default=5, help="timed steps of each non-headline variant (>= 5)")
    ap.add_argument("--cfg5-collects", type=int, default=48, help="collects of config 5 timed per step (of 800)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
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
