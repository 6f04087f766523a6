"""Multi-GPU host logic on CPU (gloo, world_size 2): the path shards over the batch only
(DESIGN.md section 9): every rank takes a contiguous slice of the samples, derives its own plan
coefficients with the library's host helpers, and no data-path collective is needed; the only
communication is the max-over-ranks of the timing and a barrier (bench.py)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2505_05940_b200 import workloads as wlmod


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close(); return p


def _worker(rank, world, port, batch, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2505_05940_b200 import binding as mb
    wl = wlmod.c3(batch=batch, n_steps=64)
    wl["n_q"], wl["n_phi"] = 24, 6
    part = wlmod.shard(wl, rank, world)
    lo, hi = part["shard"]
    # host-only plan (device -1): per-sample coefficients and excitation of this rank's slice
    plan = mb.Plan(mb.desc_from_workload(part), device=-1)
    om = np.stack([plan.derive_coeffs(Lx=part["Lx"][b], Ly=part["Ly"][b], h=part["h"][b], pickup_x_frac=0.43, pickup_y_frac=0.37)["omega"]
                   for b in range(hi - lo)])
    q0 = np.stack([plan.project_bump(part["Lx"][b], part["Ly"][b], part["x0"][b], part["y0"][b], part["W"][b], part["A"][b])
                   for b in range(hi - lo)])
    # gather what every rank derived (test only: the product path never communicates per step)
    t = torch.zeros(batch, 24 * 2, dtype=torch.float64)
    t[lo:hi] = torch.from_numpy(np.concatenate([om, q0], axis=1))
    dist.all_reduce(t)
    tmax = torch.tensor([float(rank + 1)]); dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
    dist.barrier()
    if rank == 0:
        q.put((t.numpy(), float(tmax)))
    dist.destroy_process_group()


def test_batch_shards_cover_the_batch_once():
    wl = wlmod.c1(batch=10, n_steps=8)
    seen = []
    for r in range(3):
        p = wlmod.shard(wl, r, 3)
        lo, hi = p["shard"]
        assert p["batch"] == hi - lo and np.array_equal(p["L"], wl["L"][lo:hi]) and p["n_q"] == wl["n_q"]
        seen += list(range(lo, hi))
    assert seen == list(range(10))
    with pytest.raises(ValueError):                       # fewer samples than ranks: an empty shard would be refused by the plan
        wlmod.shard(wlmod.c1(batch=2, n_steps=8), 0, 3)


def test_two_ranks_gloo_sharded_derivation_matches_single_rank():
    batch, world = 6, 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, batch, q)) for r in range(world)]
    for p in procs: p.start()
    got, tmax = q.get(timeout=180)
    for p in procs: p.join(60)
    assert all(p.exitcode == 0 for p in procs) and tmax == 2.0
    # single-process reference of the same derivation
    from paper_2505_05940_b200 import binding as mb
    wl = wlmod.c3(batch=batch, n_steps=64); wl["n_q"], wl["n_phi"] = 24, 6
    plan = mb.Plan(mb.desc_from_workload(wl), device=-1)
    for b in range(batch):
        om = plan.derive_coeffs(Lx=wl["Lx"][b], Ly=wl["Ly"][b], h=wl["h"][b], pickup_x_frac=0.43, pickup_y_frac=0.37)["omega"]
        q0 = plan.project_bump(wl["Lx"][b], wl["Ly"][b], wl["x0"][b], wl["y0"][b], wl["W"][b], wl["A"][b])
        assert np.array_equal(got[b, :24], om) and np.array_equal(got[b, 24:], q0)
