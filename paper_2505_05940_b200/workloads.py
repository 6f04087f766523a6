"""Seeded synthetic workloads C0..C4 (BASELINE.json ``configs``; recipe in DESIGN.md).

This module only DRAWS PHYSICAL PARAMETERS (geometry, material, loss constants,
excitation bump centre / width / amplitude, pickup position).  It holds none of
the method's arithmetic -- no modes, no coefficients, no projection -- so that
it can serve both the CUDA path and the test oracle, which each derive
everything else themselves.

All randomness: ``numpy.random.Generator(PCG64(20250505 + config_index))``,
one vectorised draw of ``batch`` values per parameter, in the order written
below.  The paper's own benchmark is synthetic too (analytic plate modes, 10 /
50 / 100 modes, 1 s at 44.1 kHz): C0 and C2 are its 10- and
100-mode points, C1 its tension-modulated case scaled to dataset generation,
C3 / C4 the batched and large-tensor extensions BASELINE.json asks for; ``berger`` is the paper's
second benchmark model (tension-modulated plate) on the C0 plate.
"""
from __future__ import annotations

import numpy as np

SEED0 = 20250505
STEEL = dict(E=2.0e11, rho=7860.0, nu=0.3)
SAMPLE_RATE = 44100.0


def _rng(idx: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(SEED0 + idx))


def _plate_common(name, idx, n_q, n_phi, n_steps, batch, ref):
    return dict(name=name, index=idx, model="vk", n_q=n_q, n_phi=n_phi, n_steps=n_steps,
                batch=batch, sample_rate=SAMPLE_RATE, ref=dict(ref), T0=0.0,
                sigma0=0.5, sigma1=1.0e-3, pickup=(0.43, 0.37), **STEEL)


def _fixed_plate(wl, rng, amp_in_h):
    """Same geometry for every sample (C0, C2, C4); bump centre from the seed."""
    B, ref = wl["batch"], wl["ref"]
    wl["Lx"] = np.full(B, ref["Lx"]); wl["Ly"] = np.full(B, ref["Ly"]); wl["h"] = np.full(B, ref["h"])
    wl["W"] = np.full(B, wl["bump_width"])
    wl["A"] = amp_in_h * wl["h"]
    u = rng.random((B, 2))
    wl["x0"] = wl["W"] / 2 + u[:, 0] * (wl["Lx"] - wl["W"])
    wl["y0"] = wl["W"] / 2 + u[:, 1] * (wl["Ly"] - wl["W"])
    return wl


def c0(n_steps=11025):
    """vK plate 0.6 x 0.4 x 0.001 m steel, 10 + 10 modes, batch 1, bump peak 0.5 mm, width 0.1 m."""
    wl = _plate_common("c0_vk_10x10_b1", 0, 10, 10, n_steps, 1, dict(Lx=0.6, Ly=0.4, h=1.0e-3))
    wl["bump_width"] = 0.1
    return _fixed_plate(wl, _rng(0), np.full(1, 0.5))


def c2(n_steps=44100):
    """As C0 with N_q = 100, N_phi = 50 (single-simulation real-time factor)."""
    wl = _plate_common("c2_vk_100x50_b1", 2, 100, 50, n_steps, 1, dict(Lx=0.6, Ly=0.4, h=1.0e-3))
    wl["bump_width"] = 0.1
    return _fixed_plate(wl, _rng(2), np.full(1, 0.5))


def c4(batch=1, n_steps=4410):
    """Plate as C0, N_q = 400, N_phi = 200; batch 1 / 16 / 64; amplitudes a*h, a log-uniform [0.1, 5]."""
    wl = _plate_common(f"c4_vk_400x200_b{batch}", 4, 400, 200, n_steps, batch,
                       dict(Lx=0.6, Ly=0.4, h=1.0e-3))
    wl["bump_width"] = 0.25 * 0.4
    rng = _rng(4)
    a = np.exp(rng.uniform(np.log(0.1), np.log(5.0), batch))
    return _fixed_plate(wl, rng, a)


def c3(batch=256, n_steps=22050):
    """vK plate N_q = 200, N_phi = 100, ``batch`` seeded geometries sharing one coupling tensor."""
    wl = _plate_common(f"c3_vk_200x100_b{batch}", 3, 200, 100, n_steps, batch,
                       dict(Lx=0.6, Ly=0.45, h=1.0e-3))
    rng = _rng(3)
    wl["Lx"] = rng.uniform(0.4, 0.8, batch)
    wl["Ly"] = rng.uniform(0.5, 1.0, batch) * wl["Lx"]
    wl["h"] = rng.uniform(0.5e-3, 2.0e-3, batch)
    a = np.exp(rng.uniform(np.log(0.1), np.log(5.0), batch))
    wl["A"] = a * wl["h"]
    wl["W"] = 0.25 * np.minimum(wl["Lx"], wl["Ly"])
    u = rng.random((batch, 2))
    wl["x0"] = wl["W"] / 2 + u[:, 0] * (wl["Lx"] - wl["W"])
    wl["y0"] = wl["W"] / 2 + u[:, 1] * (wl["Ly"] - wl["W"])
    return wl


def c1(batch=1024, n_steps=44100, n_q=200):
    """Kirchhoff-Carrier stiff strings, 200 modes, ``batch`` parameter sets."""
    rng = _rng(1)
    wl = dict(name=f"c1_kc_string_{n_q}_b{batch}", index=1, model="tension", n_q=n_q, n_phi=0,
              n_steps=n_steps, batch=batch, sample_rate=SAMPLE_RATE, E=STEEL["E"],
              sigma0=0.5, sigma1=1.0e-4, pickup=(0.37,))
    wl["T0s"] = rng.uniform(40.0, 120.0, batch)           # tension, N
    wl["L"] = rng.uniform(0.5, 1.0, batch)                # length, m
    wl["D"] = rng.uniform(1.0e-5, 1.0e-3, batch)          # stiffness E I, N m^2
    wl["rho_lin"] = rng.uniform(1.0e-3, 1.0e-2, batch)    # linear density, kg/m
    wl["A"] = rng.uniform(0.5e-3, 3.0e-3, batch)          # pluck peak, m
    wl["x0"] = rng.uniform(0.1, 0.9, batch) * wl["L"]     # pluck position
    # pluck width: the widest raised cosine that fits, i.e. reaching the nearer end, as a finger
    # pluck does (R13).  A narrow 0.1 L bump strains the string so much (tension more
    # than doubles at 3 mm) that the explicit scheme blows up on a third of the draws.
    wl["W"] = 2.0 * np.minimum(wl["x0"], wl["L"] - wl["x0"])
    wl["area"] = wl["rho_lin"] / STEEL["rho"]             # steel cross-section for tau = E A / 2L
    return wl


def berger(n_q=100, batch=1, n_steps=44100):
    """Berger (tension-modulated) plate of the paper's second benchmark (Fig. 3 bottom; tau of
    PAPER.md:85): the C0 plate with ``n_q`` modes (the paper times 10 / 50 / 100), bump 0.1 m wide, peak
    a*h with a log-uniform in [0.2, 2] drawn from the seed."""
    wl = _plate_common(f"berger_plate_{n_q}_b{batch}", 5, n_q, 0, n_steps, batch, dict(Lx=0.6, Ly=0.4, h=1.0e-3))
    wl["model"] = "berger"
    wl["bump_width"] = 0.1
    rng = _rng(5)
    a = np.exp(rng.uniform(np.log(0.2), np.log(2.0), batch))
    return _fixed_plate(wl, rng, a)


def by_name(name: str, **kw):
    return {"c0": c0, "c1": c1, "c2": c2, "c3": c3, "c4": c4, "berger": berger}[name](**kw)


def shard(wl: dict, rank: int, world: int) -> dict:
    """Batch shard for rank ``rank`` of ``world`` (independent samples, no data-path collective)."""
    B = wl["batch"]
    if not 0 <= rank < world:
        raise ValueError(f"rank {rank} outside [0, {world})")
    if B < world:
        raise ValueError(f"batch {B} < world size {world}: a rank would get no sample (run replicas instead)")
    lo, hi = (B * rank) // world, (B * (rank + 1)) // world
    out = {}
    for k, v in wl.items():
        out[k] = v[lo:hi] if isinstance(v, np.ndarray) and v.shape[:1] == (B,) else v
    out["batch"] = hi - lo
    out["shard"] = (lo, hi)
    return out
