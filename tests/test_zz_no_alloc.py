"""modal_vk_simulate_static -- the entry point that allocates nothing (scratch in a static __device__ array) -- against
the existing plan-based path (modal_simulate) on the same inputs, twice in a row: the second call reuses the shared scratch
array with the first call's contents still in it.  Collected last on purpose (pytest -x): a failure here must
not hide any other test.  Runs alone in a fresh process as well as after the other tests."""
import numpy as np
import pytest

from oracle import oracle as orc
from paper_2505_05940_b200 import workloads as wlmod

pytestmark = pytest.mark.gpu

TOL_MAX = 1e-4          # of the signal peak, as tests/test_gpu_parity.py (BASELINE.json's pickup tolerance)


def _case(n_q, n_phi, batch, n_steps):
    wl = wlmod.c3(batch=batch, n_steps=n_steps)
    wl["n_q"], wl["n_phi"] = n_q, n_phi
    wl["A"] = np.minimum(wl["A"], 0.5 * wl["h"])            # weakly non-linear: point-wise comparison over the whole run
    return wl, orc.assemble(wl)


def _existing_path(wl, case, n_steps):
    import torch
    from paper_2505_05940_b200 import binding as mb
    plan = mb.Plan(mb.desc_from_workload(wl), 0)
    B = case.q0.shape[0]
    plan.coeffs_upload(B, omega=case.omega, sigma=case.gamma, nl_scale=case.nl_scale, pickup=case.w, H_full=case.H)
    out = torch.empty((B, n_steps), dtype=torch.float32, device="cuda")
    st, fb = plan.simulate(case.q0, n_steps, out.data_ptr(), qm1=case.qm1, stream=torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert st == 0 and np.all(fb == -1)
    res = out.cpu().numpy().astype(np.float64)
    plan.close()
    return res


@pytest.mark.parametrize("n_q,n_phi,batch,n_steps", [
    (37, 13, 3, 1200),          # teams of 13 CTAs (one in-plane mode each) exchanging through the static scratch
    (100, 50, 20, 300),         # C2's mode counts, teams of 7
])
def test_static_entry_point_matches_existing_path_twice(n_q, n_phi, batch, n_steps):
    import torch
    from paper_2505_05940_b200 import binding as mb
    wl, case = _case(n_q, n_phi, batch, n_steps)
    ref = _existing_path(wl, case, n_steps)
    dev = "cuda"
    cb = case.c1.shape[0]
    assert cb in (1, batch)
    t64 = lambda a: torch.tensor(np.ascontiguousarray(a, np.float64), dtype=torch.float64, device=dev)
    t32 = lambda a: torch.tensor(np.ascontiguousarray(a, np.float64), dtype=torch.float32, device=dev)
    H, c1, c2, c3 = t32(case.H), t64(case.c1), t64(case.c2), t64(case.c3)
    s, w = t32(case.nl_scale), t32(case.w)
    q0, qm1 = t64(case.q0), t64(case.qm1)
    stream = torch.cuda.current_stream().cuda_stream
    peak = np.max(np.abs(ref), axis=1, keepdims=True)
    outs = []
    for call in range(2):                                   # two calls in a row on the same scratch array
        out = torch.full((batch, n_steps), float("nan"), dtype=torch.float32, device=dev)
        fb = torch.full((batch,), 12345, dtype=torch.int32, device=dev)
        mem0 = torch.cuda.memory_allocated()
        mb.vk_simulate_static(n_q, n_phi, batch, n_steps, cb, H.data_ptr(), c1.data_ptr(), c2.data_ptr(), c3.data_ptr(),
                              s.data_ptr(), w.data_ptr(), q0.data_ptr(), qm1.data_ptr(), out.data_ptr(), fb.data_ptr(), stream)
        assert torch.cuda.memory_allocated() == mem0
        torch.cuda.synchronize()
        assert np.all(fb.cpu().numpy() == -1)
        got = out.cpu().numpy().astype(np.float64)
        assert np.all(np.isfinite(got))
        err = np.max(np.abs(got - ref) / peak)
        assert err <= TOL_MAX, (call, err)
        outs.append(got)
    assert np.array_equal(outs[0], outs[1])                 # fixed summation orders, scratch cleared per launch: bit-reproducible


def test_static_entry_point_rejects_sizes_beyond_its_limits():
    from paper_2505_05940_b200 import binding as mb
    with pytest.raises(mb.ModalError) as e:
        mb.vk_simulate_static(mb.STATIC_MAX_NQ + 1, 4, 1, 8, 1, *([16] * 9))
    assert e.value.status == mb.EINCOMPAT and "MODAL_STATIC_MAX_NQ" in e.value.message
    with pytest.raises(mb.ModalError) as e:
        mb.vk_simulate_static(8, 4, 3, 8, 2, *([16] * 9))             # coeff_batch neither 1 nor batch
    assert e.value.status == mb.EINVAL
    with pytest.raises(mb.ModalError) as e:
        mb.vk_simulate_static(8, 4, 1, 8, 1, 0, *([16] * 8))          # NULL H
    assert e.value.status == mb.EINVAL
