#!/usr/bin/env python
"""bench.py -- one JSON line per run (contract in the task prompt / DESIGN.md "Measurement").

A "step" is one pass of the whole hot path over one batch of synthetic input: one
modal_simulate call advancing every sample of the workload through all its time steps
(upload & plan construction excluded, as in the paper's protocol: SPEC.md:625).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c4|c0|c1|c2|c3] [--batch B]
  python bench.py --impl reference ...      # the fp64 oracle on the host cores (bounded sample)

value    = sample-steps per second (batch x time steps / s), inputs resident in HBM
e2e      = same metric through modal_simulate_host: host q0 in, host audio out
roofline = dominant kernel against its bound (algorithmic bytes or flops per launch / CUDA-event time)
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
# nominal FP32 pipe: 148 SMs x 128 FMA lanes x 2 flop x 1.965 GHz (guide: B200_PROFILING.md clocks)
FP32_PEAK_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12
# dram__bytes_read.sum + dram__bytes_write.sum of one C4 batch-1 launch (4410 steps), profiles/r1_c4_b1.md
C4_DRAM_BYTES_PER_LAUNCH = 21.12e6


def peaks():
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


def tensor_roofline(wl, B, n_steps, per_launch, bf16_peak, peak_src):
    """vk_mma_kernel: algorithmic flops (F_alg per sample-step) against the measured bf16 peak.
    The kernel issues three bf16 MMAs per algorithmic MAC (hi*hi + lo*hi + hi*lo) to meet the 1e-4 tolerance."""
    flops, _ = algorithmic_work(wl)
    ach = flops * B * n_steps / per_launch / 1e12
    return {"bound": "tensor", "achieved": ach, "peak": bf16_peak, "unit": "TFLOP/s", "frac": ach / bf16_peak, "traffic": None,
            "peak_source": peak_src + " bf16 sustained", "kernel": "vk_mma_kernel",
            "note": "achieved = F_alg (2 N_phi N_q^2 + ...) x batch x steps / time; the tensor pipe executes 3x that "
                    "(split-bf16), so frac x 3 is the pipe's own utilisation on useful MACs"}


def secondary_c3(mb, torch, steps=2, warmup=1):
    """C3 (batch 256, tensor-core kernel), device-timed only: reported beside the headline workload."""
    wl = wlmod.by_name("c3")
    B, n_steps = wl["batch"], wl["n_steps"]
    plan, q0 = mb.plan_from_workload(wl, torch.cuda.current_device())
    out = torch.empty((B, n_steps), dtype=torch.float32, device="cuda")
    stream = torch.cuda.current_stream().cuda_stream
    for _ in range(warmup):
        plan.simulate(q0, n_steps, out.data_ptr(), first_bad=False, stream=stream)
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for s_, e_ in ev:
        s_.record(); plan.simulate(q0, n_steps, out.data_ptr(), first_bad=False, stream=stream); e_.record()
    torch.cuda.synchronize()
    per_launch = sum(s_.elapsed_time(e_) for s_, e_ in ev) * 1e-3 / steps
    info = plan.query(mb.Q_KERNEL_INFO)
    _, src, bf16_peak = peaks()
    res = {"workload": wl["name"], "value": B * n_steps / per_launch, "unit": UNIT, "us_per_time_step": 1e6 * per_launch / n_steps,
           "mode_steps_per_s": B * n_steps * wl["n_q"] / per_launch, "kernel_family": int(info[0]), "ctas": int(info[1])}
    if int(info[0]) == 4:
        res["roofline"] = tensor_roofline(wl, B, n_steps, per_launch, bf16_peak, src)
    plan.close()
    return res


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

    def summary(self):
        if not self.rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unavailable"]}
        sm = sorted(int(r[0]) for r in self.rows if r[0].isdigit())
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(len(r) > 2 + i and r[2 + i].lower().startswith("active") for r in self.rows)]
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": int(self.rows[0][1]) if self.rows[0][1].isdigit() else None,
                "reasons": reasons, "samples": len(self.rows)}


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
    return {"value": sb * n_s / dt, "unit": UNIT, "cores": min(cores, sb), "kind": "oracle",
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
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-secondary", action="store_true", help="skip the C3 (batch 256, tensor-core) line reported beside the headline")
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
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    # weak scaling over independent samples: every rank advances its own copy of the workload
    # (rank r draws its excitation from the same recipe; no data-path collective).
    wl = make_workload(args.workload, args.batch, args.n_steps)
    B, n_steps = wl["batch"], wl["n_steps"]
    plan, q0 = mb.plan_from_workload(wl, local)
    out = torch.empty((B, n_steps), dtype=torch.float32, device="cuda")
    out_host = np.empty((B, n_steps), np.float32)
    stream = torch.cuda.current_stream().cuda_stream
    flush = torch.empty(256 * 1024 * 1024 // 4, dtype=torch.float32, device="cuda")   # 256 MiB > 126 MB L2

    def step_device():
        plan.simulate(q0, n_steps, out.data_ptr(), first_bad=False, stream=stream)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 1)):
        step_device()
    barrier()
    sampler = ClockSampler(local); sampler.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    for s, e in ev:
        flush.zero_()                         # flush L2 between timed iterations
        s.record()
        step_device()
        e.record()
    barrier()
    sampler.stop_flag = True
    t_dev = sum(s.elapsed_time(e) for s, e in ev) * 1e-3
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
        flops, hbytes = algorithmic_work(wl)
        units = world * B * n_steps * args.steps
        value = units / t_dev
        per_launch = t_dev / args.steps
        hbm_peak, peak_src, bf16_peak = peaks()
        if wl["model"] == "vk" and int(info[0]) == 4:
            roof = tensor_roofline(wl, B, n_steps, per_launch, bf16_peak, peak_src)
        elif wl["model"] == "vk":
            ach = hbytes * n_steps / per_launch / 1e9
            tiles, nz = (int(x) for x in plan.query(mb.Q_TILE_STATS))
            read = nz * 1024 * n_steps / per_launch / 1e9
            roof = {"bound": "hbm", "achieved": ach, "peak": hbm_peak, "unit": "GB/s", "frac": ach / hbm_peak,
                    "traffic": C4_DRAM_BYTES_PER_LAUNCH if (wl["name"], n_steps) == ("c4_vk_400x200_b1", 4410) else None,
                    "peak_source": peak_src, "kernel": "vk_flow_kernel",
                    "tiles": tiles, "tiles_nonzero": nz, "achieved_read": read, "frac_read": read / hbm_peak,
                    "note": "achieved = ALGORITHMIC bytes (SURVEY.md 8(d): the dense packed tensor, 4*n_phi*n_q(n_q+1)/2 per time step, "
                            "once per step for the whole batch) / time.  The kernel keeps the modes grouped by index parity and never "
                            "reads the 16x16 tiles that hold only parity zeros (tiles_nonzero of tiles, SURVEY.md 8(f) row 4), so it can "
                            "exceed the dense-traffic roofline; achieved_read / frac_read count the bytes it does read per step (most "
                            "of them from shared memory, where they stay resident).  traffic = dram read+write bytes of one launch "
                            "(profiles/r1_c4_b1.md): H crosses the HBM pins once per launch"}
        else:
            ach = flops * B * n_steps / per_launch / 1e12
            roof = {"bound": "alu", "achieved": ach, "peak": FP32_PEAK_TFLOPS, "unit": "TFLOP/s", "frac": ach / FP32_PEAK_TFLOPS,
                    "traffic": None, "peak_source": "derived: 148 SM x 128 FP32 lanes x 2 x 1.965 GHz", "kernel": "tension_kernel"}
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": 1e3 * per_launch, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f32 force / f64 state", "data": "synthetic",
                "config": {"workload": wl["name"], "n_q": wl["n_q"], "n_phi": wl["n_phi"], "batch": B, "time_steps": n_steps,
                           "sample_rate": wl["sample_rate"], "l2": "flushed between timed iterations (256 MiB write)",
                           "kernel": {"family": int(info[0]), "cluster_size": int(info[1]), "clusters": int(info[2]),
                                      "threads": int(info[3]), "smem_bytes": int(info[4]), "resident": bool(info[5] & 1),
                                      "grid_team": bool(info[5] & 2)}},
                "mode_steps_per_s": value * wl["n_q"],
                "realtime_factor_per_sample": (n_steps / wl["sample_rate"]) / per_launch,
                "us_per_time_step": 1e6 * per_launch / n_steps,
                "e2e": {"value": units / t_e2e, "unit": UNIT, "h2d_bytes_per_step": int(2 * q0.size * 8),
                        "d2h_bytes_per_step": int(out_host.nbytes + 4 * B)},
                "gpu_launches": args.steps, "clocks": sampler.summary(), "roofline": roof}
        if not args.no_secondary and world == 1 and args.workload == "c4" and not args.batch and not args.n_steps:
            line["secondary"] = secondary_c3(mb, torch)
        if not args.no_cpu_baseline and world == 1:
            line["cpu_baseline"] = cpu_baseline(wl)
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
