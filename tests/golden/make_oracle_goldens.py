"""Writes tests/golden/oracle_*.npz: long fp64 ORACLE runs of the full-size configurations.

The GPU parity tests compare the CUDA path with the oracle over the tolerance window of
BASELINE.json (first 4096 samples; relative L2 over the full run).  At the full sizes the oracle
needs minutes per sample on one host core (C4: 64 MFLOP per step, C3: 8 MFLOP), too long to repeat
inside every ``pytest -m gpu`` run, so its outputs are stored here once.  This script calls ONLY
``oracle/`` (plus the seeded parameter draws of ``workloads.py``, which hold no arithmetic of the
method); nothing in these files ever comes from the CUDA path.  Each file also stores the oracle's
inputs for the chosen samples (q0, omega, nl_scale), which the tests re-derive and compare, so a
stale file fails loudly instead of silently checking against old inputs.

    python tests/golden/make_oracle_goldens.py [c4_b1] [c3] [c4_b16] [c4_b64]     (default: all)

Sample choice (SURVEY.md 8(d) "Oracle timed beside it"): C3 -- 16 samples spanning the amplitude
range, all for 4096 steps and every fourth of them for all 22 050; C4 -- batch 1 for all 4410 steps,
4 samples spanning the amplitude range of the batch-16 and batch-64 draws for all 4410 steps.
"""
from __future__ import annotations

import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from oracle import oracle as orc                                    # noqa: E402
from paper_2505_05940_b200 import workloads as wlmod               # noqa: E402  (parameter draws only)


def spanning(wl, count):
    """`count` sample indices spread evenly over the amplitude range (in plate thicknesses)."""
    order = np.argsort(wl["A"] / wl["h"])
    return sorted(set(order[np.linspace(0, wl["batch"] - 1, count).astype(int)].tolist()))


def run(wl, sub, n_steps):
    case = orc.assemble(wl, samples=sub)
    t0 = time.time()
    ref = orc.run_case(case, n_steps)
    print(f"  {wl['name']}: {len(sub)} samples x {n_steps} steps in {time.time() - t0:.0f} s", flush=True)
    return case, ref


def save(name, **arrays):
    path = os.path.join(HERE, f"oracle_{name}.npz")
    np.savez_compressed(path, **arrays)
    print(f"wrote {path} ({os.path.getsize(path) / 1024:.0f} KiB)", flush=True)


def make_c4(batch):
    wl = wlmod.c4(batch=batch)
    sub = list(range(batch)) if batch <= 4 else spanning(wl, 4)
    case, ref = run(wl, sub, wl["n_steps"])
    save(f"c4_b{batch}", sub=np.array(sub), out=ref["out"], first_bad=ref["first_bad"],
         q0=case.q0, omega=case.omega, nl_scale=case.nl_scale)


def make_c3():
    wl = wlmod.c3()
    sub = spanning(wl, 16)
    full = sub[::4]
    case, ref = run(wl, sub, 4096)
    _, ref_full = run(wl, full, wl["n_steps"])
    save("c3", sub=np.array(sub), out=ref["out"], first_bad=ref["first_bad"],
         sub_full=np.array(full), out_full=ref_full["out"], first_bad_full=ref_full["first_bad"],
         q0=case.q0, omega=case.omega, nl_scale=case.nl_scale)


if __name__ == "__main__":
    which = sys.argv[1:] or ["c4_b1", "c3", "c4_b16", "c4_b64"]
    print(f"oracle threads: {orc.num_threads()}", flush=True)
    for w in which:
        if w == "c3":
            make_c3()
        elif w.startswith("c4_b"):
            make_c4(int(w[4:]))
        else:
            raise SystemExit(f"unknown golden set {w}")
