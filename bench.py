#!/usr/bin/env python
"""bench.py -- one JSON line per run (contract in the task prompt / DESIGN.md "Measurement").

A "step" is one pass of the whole hot path over one batch of synthetic input: one
modal_simulate call advancing every sample of the workload through all its time steps
(upload & plan construction excluded, as in the paper's protocol: SPEC.md:625).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c4|c0|c1|c2|c3] [--batch B]
  python bench.py --impl reference ...      # the fp64 oracle on the host cores (bounded sample)
  python bench.py --peaks                   # only the machine peaks measured through libmodal.so

value     = sample-steps per second (batch x time steps / s), inputs resident in HBM
e2e       = same metric through modal_simulate_host: host q0 in, host audio out
roofline  = dominant kernel against its bound (algorithmic bytes or flops per launch / CUDA-event time)
secondary = every other BASELINE.json configuration (and C4 batch 1 with a dense uploaded H), device-timed
peaks     = FP32 / FP64 FMA, L2 / HBM / shared-memory / TMEM read bandwidth and exchange-hop latencies measured
            in this run by modal_measure_peaks (csrc/peaks.cuh)
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2505_05940_b200 import workloads as wlmod  # noqa: E402

METRIC = "von_karman_modal_sample_steps_per_s"
UNIT = "sample-steps/s"
# nominal FP32 pipe, used only if modal_measure_peaks is skipped: 148 SMs x 128 FMA lanes x 2 flop x 1.965 GHz
FP32_NOMINAL_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12


def driver_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return d.get("hbm_gbs", 6650.0), "measured (MEASURED_PEAKS.json)", d.get("bf16_tflops_sustained", 1400.0)
    return 6650.0, "fallback (B200_PROFILING.md)", 1400.0


def make_workload(name, batch, n_steps):
    kw = {}
    if batch and name in ("c1", "c3", "c4"):
        kw["batch"] = batch
    if n_steps:
        kw["n_steps"] = n_steps
    return wlmod.by_name(name, **kw)


def algorithmic_work(wl):
    """Per sample-step flops and per-step H bytes."""
    nq, nphi = wl["n_q"], wl["n_phi"]
    if wl["model"] == "vk":
        P = nq * (nq + 1) // 2
        return 2 * nphi * nq * nq + 4 * nphi * nq + 8 * nq, 4 * nphi * P
    return 12 * nq, 0


class ClockSampler(threading.Thread):
    def __init__(self, index=0):
        super().__init__(daemon=True)
        self.rows, self.stop_flag, self.index = [], False, index

    def run(self):
        q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
            "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"
        while not self.stop_flag:
            try:
                o = subprocess.run(["nvidia-smi", "-i", str(self.index), f"--query-gpu={q}", "--format=csv,noheader,nounits"],
                                   capture_output=True, text=True, timeout=5).stdout.strip()
                if o:
                    self.rows.append([s.strip() for s in o.split(",")])
            except Exception:
                pass
            time.sleep(0.1)

    def mark(self):
        return len(self.rows)

    def summary(self, lo=0, hi=None):
        rows = self.rows[lo:hi]
        if not rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unavailable"]}
        sm = sorted(int(r[0]) for r in rows if r[0].isdigit())
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(len(r) > 2 + i and r[2 + i].lower().startswith("active") for r in rows)]
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": int(rows[0][1]) if rows[0][1].isdigit() else None,
                "reasons": reasons, "samples": len(rows)}


def device_time(torch, plan, q0, n_steps, out, steps, warmup, flush=None):
    """Seconds per modal_simulate launch: CUDA events on the launching stream, after warm-up, optional L2 flush between launches."""
    stream = torch.cuda.current_stream().cuda_stream
    for _ in range(max(warmup, 1)):
        plan.simulate(q0, n_steps, out.data_ptr(), first_bad=False, stream=stream)
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for s, e in ev:
        if flush is not None:
            flush.zero_()
        s.record()
        plan.simulate(q0, n_steps, out.data_ptr(), first_bad=False, stream=stream)
        e.record()
    torch.cuda.synchronize()
    return sum(s.elapsed_time(e) for s, e in ev) * 1e-3 / steps


def roofline_for(wl, B, n_steps, per_launch, info, tile_stats, pk, stream=None):
    """Roofline object of one workload: which kernel ran, what bounds it, algorithmic work / time against the measured peak."""
    flops, hbytes = algorithmic_work(wl)
    hbm_peak, peak_src, bf16_peak = driver_peaks()
    fam = int(info[0])
    if fam == 4:
        ach = flops * B * n_steps / per_launch / 1e12
        return {"bound": "tensor", "achieved": ach, "peak": bf16_peak, "unit": "TFLOP/s", "frac": ach / bf16_peak, "traffic": None,
                "peak_source": peak_src + " bf16 sustained", "kernel": "vk_mma_kernel",
                "note": "achieved = F_alg (2 N_phi N_q^2 + ...) x batch x steps / time; the kernel issues 3 bf16 MMAs per MAC (split hi/lo) "
                        "on the K chunks that hold non-zeros only"}
    if fam == 5:
        ach = flops * B * n_steps / per_launch / 1e12
        r = {"bound": "tensor", "achieved": ach, "peak": bf16_peak, "unit": "TFLOP/s", "frac": ach / bf16_peak, "traffic": None,
             "peak_source": peak_src + " bf16 sustained", "kernel": "vk_stream_kernel",
             "note": "H (bf16 hi + lo, K chunks with non-zeros only) is streamed from L2 by TMA every step; rows of H on M, samples on N; "
                     "3 bf16 MMAs per MAC; launches of <= 64 samples"}
        if stream is not None:            # the L2 -> shared memory stream of the step, against the measured L2 read rate
            launches = (B + 63) // 64
            rd = float(stream[11]) * 8192 * n_steps * launches / per_launch / 1e9
            r.update({"h_stream_mib": int(stream[12]), "h_stream_read": rd, "l2_read_peak_64mb": pk.get("l2_read_gbs_64mb") if pk else None,
                      "frac_stream_of_l2": rd / pk["l2_read_gbs_64mb"] if pk else None})
        return r
    if fam == 6:          # dense-team kernel: H of a CTA's modes resident in shared memory, one L2 hop per step: latency-bound at batch 1
        ach = hbytes * n_steps / per_launch / 1e9
        return {"bound": "hbm", "achieved": ach, "peak": hbm_peak, "unit": "GB/s", "frac": ach / hbm_peak, "traffic": None,
                "peak_source": peak_src, "kernel": "vk_dense_kernel", "frac_dense_alg": ach / hbm_peak,
                "note": "algorithmic bytes = the packed H once per step (SURVEY.md 8(d)); the kernel keeps the dense fp32 H in shared memory and "
                        "is bound by the one cross-CTA hop per step, not by bandwidth"}
    if fam == 8:          # replicated-state kernel: H (blocks of the parity structure) resident in shared memory, one L2 hop per step
        ach = hbytes * n_steps / per_launch / 1e9
        tiles, nz = tile_stats
        r = {"bound": "hbm", "achieved": ach, "peak": hbm_peak, "unit": "GB/s", "frac": ach / hbm_peak, "traffic": None,
             "peak_source": peak_src, "kernel": "vk_repl_kernel", "frac_dense_alg": ach / hbm_peak, "tiles": tiles, "tiles_nonzero": nz,
             "achieved_read": 0.0, "frac_read": 0.0}
        if stream is not None:            # Q_REPL_CHECK: what the step really reads is its packed blocks, from shared memory
            rd = float(stream[6]) * 4 * n_steps / per_launch / 1e9
            r.update({"smem_resident_mb": float(stream[6]) * 4 / 1e6, "ctas_with_modes": int(stream[7]), "smem_read": rd,
                      "smem_read_peak": pk.get("smem_read_gbs") if pk else None, "frac_smem": rd / pk["smem_read_gbs"] if pk else None})
        return r
    if fam == 3:
        ach = hbytes * n_steps / per_launch / 1e9
        tiles, nz = tile_stats
        read = nz * 1024 * n_steps / per_launch / 1e9
        return {"bound": "hbm", "achieved": ach, "peak": hbm_peak, "unit": "GB/s", "frac": ach / hbm_peak, "traffic": None,
                "peak_source": peak_src, "kernel": "vk_flow_kernel", "frac_dense_alg": ach / hbm_peak,
                "tiles": tiles, "tiles_nonzero": nz, "achieved_read": read, "frac_read": read / hbm_peak,
                "l2_read_peak_64mb": pk.get("l2_read_gbs_64mb") if pk else None,
                "frac_read_of_l2": read / pk["l2_read_gbs_64mb"] if pk else None}
    if fam == 2:          # small-system kernel: one warp per sample, a dependent chain of a few hundred cycles per step (latency, not a pipe)
        ach = flops * B * n_steps / per_launch / 1e12
        peak = pk["fp32_tflops"] if pk else FP32_NOMINAL_TFLOPS
        return {"bound": "alu", "achieved": ach, "peak": peak, "unit": "TFLOP/s", "frac": ach / peak, "traffic": None,
                "peak_source": "measured in this run (modal_measure_peaks, FP32 FMA)" if pk else "nominal FP32 pipe (peaks skipped)",
                "kernel": "vk_small_kernel", "note": "latency-bound by construction: one warp advances one sample, no barrier, no exchange"}
    # tension / linear kernel: every FMA of the update is fp64 (DFMA), so the bound is the FP64 pipe
    ach = flops * B * n_steps / per_launch / 1e12
    peak = pk["fp64_tflops"] if pk else FP32_NOMINAL_TFLOPS
    return {"bound": "alu", "achieved": ach, "peak": peak, "unit": "TFLOP/s", "frac": ach / peak, "traffic": None,
            "peak_source": "measured in this run (modal_measure_peaks, FP64 FMA)" if pk else "nominal FP32 pipe (peaks skipped)",
            "kernel": "tension_kernel", "frac_of_fp32_pipe": ach / pk["fp32_tflops"] if pk else None}


def run_secondary(mb, torch, sampler, pk, steps=2, warmup=1):
    """Every other configuration of BASELINE.json plus C4 batch 1 with a dense uploaded H, device-timed."""
    res = []
    dev = torch.cuda.current_device()

    def entry(label, wl, plan, q0, B, n_steps, extra=None):
        out = torch.empty((B, n_steps), dtype=torch.float32, device="cuda")
        lo = sampler.mark()
        t = device_time(torch, plan, q0[:B], n_steps, out, steps, warmup)
        info = plan.query(mb.Q_KERNEL_INFO)
        ts = tuple(int(x) for x in plan.query(mb.Q_TILE_STATS)) if wl["model"] == "vk" else (0, 0)
        st, fbad = plan.check(B)
        e = {"workload": label, "batch": B, "time_steps": n_steps, "value": B * n_steps / t, "unit": UNIT,
             "us_per_time_step": 1e6 * t / n_steps, "mode_steps_per_s": B * n_steps * wl["n_q"] / t,
             "realtime_factor_per_sample": (n_steps / wl["sample_rate"]) / t,
             "kernel_family": int(info[0]), "ctas": int(info[1]) * (int(info[2]) if int(info[0]) == 3 else 1),
             "status": int(st), "roofline": roofline_for(wl, B, n_steps, t, info, ts, pk, plan.query(mb.Q_STREAM_LAYOUT) if int(info[0]) == 5 else plan.query(mb.Q_REPL_CHECK) if int(info[0]) == 8 else None),
             "clocks": sampler.summary(lo)}
        nbad = int((fbad >= 0).sum()) if fbad is not None else 0
        if nbad:          # status 3: the explicit scheme itself diverges on these samples (the oracle does too, within a few steps: SPEC.md:298)
            e["unstable_samples"] = nbad
        if extra:
            e.update(extra)
        res.append(e)
        del out

    for name in ("c0", "c1", "c2"):
        wl = wlmod.by_name(name)
        plan, q0 = mb.plan_from_workload(wl, dev)
        entry(wl["name"], wl, plan, q0, wl["batch"], wl["n_steps"])
        plan.close()
    for B in (256, 512, 1024):                              # north_star: tensor-pipe fraction "at batch >= 256"
        wl = wlmod.c3(batch=B)
        plan, q0 = mb.plan_from_workload(wl, dev)
        entry(wl["name"], wl, plan, q0, B, wl["n_steps"])
        plan.close()
    best = max((e for e in res if e["workload"].startswith("c3_")), key=lambda e: e["roofline"]["frac"])
    best["best_c3_batch"] = True
    # reverse pass: C2's mode counts, forward with the trajectory kept on the device, then modal_bptt
    for B in (1, 8):
        wl = wlmod.c2(n_steps=4410) if B == 1 else dict(wlmod.c3(batch=B, n_steps=4410), n_q=100, n_phi=50, name=f"c2_shape_b{B}")
        wl["A"] = np.minimum(wl["A"], 0.5 * wl["h"])
        plan, q0 = mb.plan_from_workload(wl, dev)
        n_steps, nq, nphi = wl["n_steps"], wl["n_q"], wl["n_phi"]
        out = torch.empty((B, n_steps), dtype=torch.float32, device="cuda")
        traj = torch.zeros((B, n_steps, nq), dtype=torch.float64, device="cuda")
        stream = torch.cuda.current_stream().cuda_stream
        qm1 = q0 * (1.0 - 1e-3)                              # any explicit q^-1: the reverse pass differentiates the recurrence it is given
        st, _ = plan.simulate(q0, n_steps, out.data_ptr(), qm1=qm1, stream=stream, traj_dev_ptr=traj.data_ptr())
        gout = torch.randn((B, n_steps), dtype=torch.float32, device="cuda")
        plan.bptt(qm1, n_steps, traj.data_ptr(), gout.data_ptr(), want_H=False, stream=stream)       # warm-up
        ts = []
        for want_H in (False, True):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); plan.bptt(qm1, n_steps, traj.data_ptr(), gout.data_ptr(), want_H=want_H, stream=stream); e1.record()
            torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1) * 1e-3)
        hbm_peak, peak_src, _ = driver_peaks()
        ach = 4.0 * nphi * nq * nq * B * n_steps / ts[0] / 1e9
        res.append({"workload": f"bptt_vk_{nq}x{nphi}_b{B}", "batch": B, "time_steps": n_steps, "value": B * n_steps / ts[0], "unit": UNIT,
                    "us_per_time_step": 1e6 * ts[0] / n_steps, "us_per_time_step_with_grad_H": 1e6 * ts[1] / n_steps, "kernel_family": 7, "status": int(st),
                    "roofline": {"bound": "hbm", "achieved": ach, "peak": hbm_peak, "unit": "GB/s", "frac": ach / hbm_peak, "traffic": None,
                                 "peak_source": peak_src, "kernel": "vk_bptt_kernel",
                                 "frac_of_l2": ach / pk["l2_read_gbs_8mb"] if pk else None,
                                 "note": "reverse step: dense fp32 H (4 N_phi N_q^2 bytes per sample) read once for both contractions, from L2; "
                                         "time includes the gradient copies to the host (modal_bptt is synchronous)"}})
        plan.close()
    wl = wlmod.c4(batch=256)
    plan, q0 = mb.plan_from_workload(wl, dev)
    for B in (16, 64, 256):
        entry(f"c4_vk_400x200_b{B}", wl, plan, q0, B, wl["n_steps"])
    # C4 batch 1 through the FP32 flow kernel (the headline's kernel until the replicated-state kernel; tiles spread over the CTAs, two hops)
    plan.set_option("vk_impl", 1)
    entry("c4_vk_400x200_b1_flow_kernel", wl, plan, q0, 1, wl["n_steps"])
    plan.set_option("vk_impl", 0)
    # C4 batch 1 with a DENSE uploaded tensor (no exact zeros): the paper's H-fitting case -- nothing to skip
    rng = np.random.default_rng(20250505)
    H = rng.normal(size=(wl["n_phi"], wl["n_q"], wl["n_q"]))
    H = H + H.transpose(0, 2, 1)
    plan.coeffs_upload(1, H_full=H)
    del H
    entry("c4_vk_400x200_b1_dense_uploaded_H", wl, plan, q0, 1, wl["n_steps"],
          {"note": "random symmetric H without zeros uploaded through modal_coeffs_upload: every tile is read, frac = dense-schedule fraction"})
    plan.close()
    return res


def run_reference(args):
    """The oracle, as it stands, on the host cores; a bounded sample of the workload per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import oracle as orc
    wl = make_workload(args.workload, args.batch, args.n_steps)
    B, n_full = wl["batch"], wl["n_steps"]
    flops, _ = algorithmic_work(wl)
    # ~1e10 fp64 flop per timed step keeps one step at a few seconds on one core
    cores = orc.num_threads()
    sb = min(B, max(1, cores))
    budget = 6e9 * min(sb, cores)
    n_s = int(max(16, min(n_full, budget / (flops * sb))))
    if n_s == n_full:                      # cheap models (strings): widen the sample over the batch instead
        sb = int(min(B, max(sb, budget / (flops * n_full) // cores * cores)))
    case = orc.assemble(wl, samples=range(sb))
    for _ in range(args.warmup):
        orc.run_case(case, min(n_s, 16))
    t0 = time.perf_counter()
    for _ in range(args.steps):
        orc.run_case(case, n_s)
    dt = time.perf_counter() - t0
    val = sb * n_s * args.steps / dt
    sample = f"{sb} of {B} samples x {n_s} of {n_full} time steps per step (uniform loop, not extrapolated)"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": wl["name"], "n_q": wl["n_q"], "n_phi": wl["n_phi"], "batch": B, "time_steps": n_full},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": min(cores, sb), "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def cpu_baseline(wl, seconds=12.0):
    from oracle import oracle as orc
    B, n_full = wl["batch"], wl["n_steps"]
    flops, _ = algorithmic_work(wl)
    cores = orc.num_threads()
    sb = min(B, max(1, cores))
    n_s = int(max(16, min(n_full, 0.8e9 * seconds * min(sb, cores) / (flops * sb))))
    if n_s == n_full:                      # cheap models (strings): widen the sample over the batch instead
        sb = int(min(B, max(sb, 0.8e9 * seconds * cores / (flops * n_full) // cores * cores)))
    case = orc.assemble(wl, samples=range(sb))
    orc.run_case(case, 4)
    t0 = time.perf_counter()
    orc.run_case(case, n_s)
    dt = time.perf_counter() - t0
    return {"value": sb * n_s / dt, "unit": UNIT, "cores": min(cores, sb), "kind": "oracle (1-core fp64 loop per sample; OpenMP over samples only)",
            "sample": f"{sb} of {B} samples x {n_s} of {n_full} time steps, {dt:.1f} s wall"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c4", choices=["c0", "c1", "c2", "c3", "c4"])
    ap.add_argument("--batch", type=int, default=0)
    ap.add_argument("--n-steps", dest="n_steps", type=int, default=0, help="time steps per simulate call (default: the config's)")
    ap.add_argument("--option", action="append", default=[], help="plan option key=value (modal_plan_set_option), repeatable")
    ap.add_argument("--dense-h", action="store_true", help="upload a dense random symmetric H (no parity zeros) before timing")
    ap.add_argument("--peaks", action="store_true", help="measure and print the machine peaks only")
    ap.add_argument("--no-peaks", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-secondary", action="store_true", help="skip the other configurations reported beside the headline")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist
    from paper_2505_05940_b200 import binding as mb   # raises if libmodal.so is missing: no fallback

    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if args.peaks:
        print(json.dumps({"peaks": mb.measure_peaks(local)}), flush=True)
        return
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    # weak scaling over independent samples: every rank advances its own copy of the workload
    # (rank r draws its excitation from the same recipe; no data-path collective).
    wl = make_workload(args.workload, args.batch, args.n_steps)
    B, n_steps = wl["batch"], wl["n_steps"]
    options = {k: int(v) for k, v in (o.split("=") for o in args.option)}
    plan, q0 = mb.plan_from_workload(wl, local, options=options)
    if args.dense_h:
        rng = np.random.default_rng(20250505)
        H = rng.normal(size=(wl["n_phi"], wl["n_q"], wl["n_q"]))
        plan.coeffs_upload(1, H_full=H + H.transpose(0, 2, 1))
        del H
    out = torch.empty((B, n_steps), dtype=torch.float32, device="cuda")
    out_host = np.empty((B, n_steps), np.float32)
    flush = torch.empty(256 * 1024 * 1024 // 4, dtype=torch.float32, device="cuda")   # 256 MiB > 126 MB L2

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    device_time(torch, plan, q0, n_steps, out, 1, max(args.warmup, 3) - 1)            # warm-up (>= 3 launches with the timed helper's own)
    barrier()
    sampler = ClockSampler(local); sampler.start()
    t_dev = device_time(torch, plan, q0, n_steps, out, args.steps, 1, flush) * args.steps
    barrier()
    head_clocks = sampler.summary()
    st_check, _ = plan.check()                           # one checked completion: a timed-out exchange or an instability is reported, not hidden
    # e2e: host buffers through the C ABI, H2D of the state and D2H of the audio inside the timed region
    plan.simulate_host(q0, n_steps, out=out_host)
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        plan.simulate_host(q0, n_steps, out=out_host)
    torch.cuda.synchronize()
    t_e2e = time.perf_counter() - t0
    tt = torch.tensor([t_dev, t_e2e], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    t_dev, t_e2e = tt.tolist()
    if rank == 0:
        info = plan.query(mb.Q_KERNEL_INFO)
        ts = tuple(int(x) for x in plan.query(mb.Q_TILE_STATS)) if wl["model"] == "vk" else (0, 0)
        pk = None if (args.no_peaks or world > 1) else mb.measure_peaks(local)
        units = world * B * n_steps * args.steps
        value = units / t_dev
        per_launch = t_dev / args.steps
        roof = roofline_for(wl, B, n_steps, per_launch, info, ts, pk,
                            plan.query(mb.Q_STREAM_LAYOUT) if int(info[0]) == 5 else plan.query(mb.Q_REPL_CHECK) if int(info[0]) == 8 else None)
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": 1e3 * per_launch, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f32 force / f64 state" if int(info[0]) != 4 else "bf16 hi+lo operands, f32 accumulate / f64 state", "data": "synthetic",
                "config": {"workload": wl["name"] + ("_dense_uploaded_H" if args.dense_h else ""), "n_q": wl["n_q"], "n_phi": wl["n_phi"],
                           "batch": B, "time_steps": n_steps,
                           "sample_rate": wl["sample_rate"], "l2": "flushed between timed iterations (256 MiB write)",
                           "kernel": {"family": int(info[0]), "ctas_per_team_or_ctas": int(info[1]), "teams_or_groups": int(info[2]),
                                      "threads": int(info[3]), "smem_bytes": int(info[4]), "resident": bool(info[5] & 1),
                                      "grid_team": bool(info[5] & 2)}},
                "mode_steps_per_s": value * wl["n_q"],
                "realtime_factor_per_sample": (n_steps / wl["sample_rate"]) / per_launch,
                "us_per_time_step": 1e6 * per_launch / n_steps, "status_checked": int(st_check),
                "e2e": {"value": units / t_e2e, "unit": UNIT, "h2d_bytes_per_step": int(2 * q0.size * 8),
                        "d2h_bytes_per_step": int(out_host.nbytes + 4 * B)},
                "gpu_launches": args.steps, "clocks": head_clocks, "roofline": roof}
        if pk:
            line["peaks"] = pk
        default_run = world == 1 and args.workload == "c4" and not args.batch and not args.n_steps and not args.dense_h and not options
        if not args.no_secondary and default_run:
            plan.close()
            del out, flush
            line["secondary"] = run_secondary(mb, torch, sampler, pk)
            dense = next(e for e in line["secondary"] if e["workload"].endswith("dense_uploaded_H"))
            roof["dense_schedule"] = {"us_per_time_step": dense["us_per_time_step"], "achieved": dense["roofline"]["achieved"],
                                      "frac": dense["roofline"]["frac"]}
            roof["note"] = ("frac = frac_dense_alg = ALGORITHMIC bytes (SURVEY.md 8(d): the dense packed tensor, 4 n_phi n_q (n_q+1)/2 per time step) "
                            "/ time / measured HBM copy peak.  The sine-basis tensor is 69 % exact zeros by index parity (SURVEY.md 8(f) row 4) and "
                            "symmetric; the replicated-state kernel keeps its non-zero blocks, one per symmetric pair, in shared memory "
                            "(smem_resident_mb over ctas_with_modes CTAs) and reads nothing from HBM inside the loop, so this figure can exceed 1 "
                            "and is NOT a bandwidth achievement: the step is the shared-memory pass over the blocks (smem_read against the measured "
                            "shared-memory rate) plus one cluster hop and one L2 hop (DESIGN.md 7.9).  dense_schedule is the FP32 flow kernel on an "
                            "uploaded H without zeros, which does not fit shared memory: every tile is read each step -- the figure to hold "
                            "against north_star's 60 % for a general H.")
        sampler.stop_flag = True
        if not args.no_cpu_baseline and world == 1:
            line["cpu_baseline"] = cpu_baseline(wl)
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
