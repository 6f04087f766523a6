"""CPU tests of the C-ABI library: it loads, exports every symbol include/modal.h declares,
validates descriptors, and its host-side derivations (mode sets, coefficients, closed-form H,
stability mask, projection) agree with the independent oracle.  No compute call needs a GPU."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from oracle import oracle as orc
from paper_2505_05940_b200 import binding as mb
from paper_2505_05940_b200 import workloads as wlmod

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "modal.h")).read()
    declared = set(re.findall(r"\b(modal_[a-z_]+)\s*\(", hdr))
    assert declared == set(mb.EXPORTS), declared ^ set(mb.EXPORTS)
    for name in declared:
        assert hasattr(mb.lib, name)


def _c0_plan(n_q=10, n_phi=10, **over):
    wl = wlmod.c0()
    wl["n_q"], wl["n_phi"] = n_q, n_phi
    d = mb.desc_from_workload(wl)
    for k, v in over.items():
        setattr(d, k, v)
    return wl, mb.Plan(d, device=-1)


def test_host_only_plan_refuses_to_simulate_no_cpu_fallback():
    wl, plan = _c0_plan()
    out = np.zeros((1, 8), np.float32)
    with pytest.raises(mb.ModalError) as e:
        plan.simulate_host(np.zeros((1, 10)), 8, out=out)
    assert e.value.status == mb.ECUDA and "no CPU fallback" in e.value.message


def test_validation_reports_all_violations():
    wl = wlmod.c0()
    d = mb.desc_from_workload(wl)
    d.rho = -1.0; d.n_q = 0; d.sample_rate = 0.0; d.Lx = 0.0
    with pytest.raises(mb.ModalError) as e:
        mb.Plan(d, device=-1)
    msg = e.value.message
    assert e.value.status == mb.EINVAL
    for frag in ("rho must be positive", "n_q must be at least 1", "sample_rate must be positive", "Lx must be positive"):
        assert frag in msg
    d = mb.desc_from_workload(wlmod.c1(batch=2))
    d.T0 = 0.0; d.D = 0.0
    with pytest.raises(mb.ModalError) as e:
        mb.Plan(d, device=-1)
    assert "degenerate dispersion" in e.value.message


@pytest.mark.parametrize("n_q,n_phi", [(10, 10), (57, 23)])
def test_plate_plan_defaults_match_oracle(n_q, n_phi):
    wl, plan = _c0_plan(n_q, n_phi)
    ref = wl["ref"]
    m, n, lam = orc.rect_modes(ref["Lx"], ref["Ly"], n_q)
    mp, np_, lamp = orc.rect_modes(ref["Lx"], ref["Ly"], n_phi)
    assert np.array_equal(plan.query(mb.Q_MODE_M), m) and np.array_equal(plan.query(mb.Q_MODE_N), n)
    assert np.array_equal(plan.query(mb.Q_PHI_M), mp) and np.array_equal(plan.query(mb.Q_PHI_N), np_)
    assert np.allclose(plan.query(mb.Q_LAMBDA), lam, rtol=1e-14)
    om, ga = orc.omega_gamma(lam, orc.plate_D(wl["E"], ref["h"], wl["nu"]), 0.0, wl["rho"] * ref["h"],
                             wl["sigma0"], wl["sigma1"])
    assert np.allclose(plan.query(mb.Q_OMEGA)[0], om, rtol=1e-13)
    assert np.allclose(plan.query(mb.Q_SIGMA)[0], ga, rtol=1e-13)
    s = wl["E"] / (2 * wl["rho"] * lamp ** 2)
    assert np.allclose(plan.query(mb.Q_NL_SCALE)[0], s, rtol=1e-13)
    w = [orc.rect_mode(m[k], n[k], ref["Lx"], ref["Ly"], 0.43 * ref["Lx"], 0.37 * ref["Ly"]) for k in range(n_q)]
    assert np.allclose(plan.query(mb.Q_PICKUP)[0], w, rtol=1e-12, atol=1e-13)
    H = orc.H_closed(ref["Lx"], ref["Ly"], m, n, mp, np_)
    Hdev = plan.query(mb.Q_H_FULL)
    # two independent closed forms (J-based vs 4-term product-to-sum), compared at fp32 resolution
    assert np.allclose(Hdev, H, rtol=2e-7, atol=1e-7 * np.abs(H).max())
    assert np.array_equal(Hdev == 0, H == 0)                       # parity zeros are exact on both sides
    assert np.array_equal(Hdev, Hdev.transpose(0, 2, 1))
    assert np.all(plan.query(mb.Q_ACTIVE) == 1)


def test_H_upload_roundtrip_and_symmetry_check():
    wl, plan = _c0_plan(21, 7)           # ragged: 21 = 16 + 5
    rng = np.random.default_rng(3)
    H = rng.normal(size=(7, 21, 21)); H = H + H.transpose(0, 2, 1)
    plan.coeffs_upload(1, H_full=H)
    assert np.array_equal(plan.query(mb.Q_H_FULL), orc.f32(H))
    Hbad = H.copy(); Hbad[3, 2, 5] += 1e-3
    with pytest.raises(mb.ModalError) as e:
        plan.coeffs_upload(1, H_full=Hbad)
    assert "not symmetric" in e.value.message


def test_derive_coeffs_other_geometry_matches_oracle_scaling():
    wl = wlmod.c3(batch=4)
    plan = mb.Plan(mb.desc_from_workload(wl), device=-1)
    case = orc.assemble(wl, round_fp32=False)
    for b in range(4):
        r = plan.derive_coeffs(Lx=wl["Lx"][b], Ly=wl["Ly"][b], h=wl["h"][b], pickup_x_frac=0.43, pickup_y_frac=0.37)
        assert np.allclose(r["omega"], case.omega[b], rtol=1e-13)
        assert np.allclose(r["sigma"], case.gamma[b], rtol=1e-13)
        assert np.allclose(r["nl_scale"], case.nl_scale[b], rtol=1e-12)
        wfull = np.array([orc.rect_mode(case.extra["mq"][k], case.extra["nq"][k], wl["Lx"][b], wl["Ly"][b],
                                        0.43 * wl["Lx"][b], 0.37 * wl["Ly"][b]) for k in range(wl["n_q"])])
        assert np.allclose(r["pickup"], wfull, rtol=1e-11, atol=1e-12)
        q0 = plan.project_bump(wl["Lx"][b], wl["Ly"][b], wl["x0"][b], wl["y0"][b], wl["W"][b], wl["A"][b])
        q0o = orc.project_bump_rect(case.extra["mq"], case.extra["nq"], wl["Lx"][b], wl["Ly"][b],
                                    wl["x0"][b], wl["y0"][b], wl["W"][b], wl["A"][b])
        assert np.max(np.abs(q0 - q0o)) < 1e-12 * np.abs(q0o).max()


def test_string_plan_coeffs_mask_and_projection_match_oracle():
    wl = wlmod.c1(batch=8)
    plan, q0 = mb.plan_from_workload(wl, device=-1)
    case = orc.assemble(wl, round_fp32=False)
    assert np.allclose(plan.query(mb.Q_OMEGA), case.omega, rtol=1e-13)
    assert np.allclose(plan.query(mb.Q_SIGMA), case.gamma, rtol=1e-13)
    assert np.allclose(plan.query(mb.Q_NL_SCALE)[:, 0], case.nl_scale, rtol=1e-13)
    assert np.array_equal(plan.query(mb.Q_ACTIVE).astype(bool), case.active)       # reading R11, decided in fp64
    assert 0 < case.active.sum() < case.active.size                                # some strings do lose modes
    assert "masked" in plan.last_error()
    q0o = np.where(case.active, 0, 0) + np.array([orc.project_bump_string(wl["n_q"], wl["L"][b], wl["x0"][b], wl["W"][b], wl["A"][b]) for b in range(8)])
    assert np.max(np.abs(q0 - q0o)) < 1e-13 * np.abs(q0o).max()


def test_workloads_are_seeded_and_shaped_like_baseline_configs():
    a, b = wlmod.c3(batch=16), wlmod.c3(batch=16)
    for k in ("Lx", "Ly", "h", "A", "x0", "y0"):
        assert np.array_equal(a[k], b[k])
    assert np.all((a["Lx"] >= 0.4) & (a["Lx"] <= 0.8)) and np.all((a["Ly"] / a["Lx"] >= 0.5) & (a["Ly"] / a["Lx"] <= 1.0))
    assert np.all((a["A"] / a["h"] >= 0.1) & (a["A"] / a["h"] <= 5.0))
    assert np.all(a["x0"] - a["W"] / 2 >= 0) and np.all(a["x0"] + a["W"] / 2 <= a["Lx"])
    c1 = wlmod.c1()
    assert c1["batch"] == 1024 and c1["n_q"] == 200 and c1["n_steps"] == 44100
    assert np.all((c1["T0s"] >= 40) & (c1["T0s"] <= 120)) and np.all((c1["A"] >= 0.5e-3) & (c1["A"] <= 3e-3))
    assert (wlmod.c0()["n_steps"], wlmod.c2()["n_steps"], wlmod.c4()["n_steps"], wlmod.c3()["n_steps"]) == (11025, 44100, 4410, 22050)
    sh = wlmod.shard(wlmod.c3(batch=10), 1, 4)
    assert sh["batch"] == 3 and sh["shard"] == (2, 5) and len(sh["Lx"]) == 3


def test_berger_plate_plan_defaults_match_oracle():
    """Tension-modulated (Berger) plate, the paper's second benchmark model: the library's
    default coefficients (lambda, omega, gamma, tau/(rho h), pickup) and its bump projection agree with the oracle."""
    wl = wlmod.berger(n_q=50, batch=3, n_steps=64)
    plan = mb.Plan(mb.desc_from_workload(wl), device=-1)
    case = orc.assemble(wl, round_fp32=False)
    assert np.array_equal(plan.query(mb.Q_ACTIVE).astype(bool)[0], case.active[0])
    assert np.allclose(plan.query(mb.Q_LAMBDA), case.lam[0], rtol=1e-13)
    assert np.allclose(plan.query(mb.Q_OMEGA)[0], case.omega[0], rtol=1e-12)
    assert np.allclose(plan.query(mb.Q_SIGMA)[0], case.gamma[0], rtol=1e-12)
    d = plan.derive_coeffs()
    # tau / (rho h) with tau = E h / (2 Lx Ly (1 - nu^2)) written out from PAPER.md:85
    tau_rho = 2.0e11 * 1e-3 / (2 * 0.6 * 0.4 * (1 - 0.09)) / (7860.0 * 1e-3)
    assert abs(d["nl_scale"][0] / tau_rho - 1) < 1e-13 and abs(case.nl_scale[0] / tau_rho - 1) < 1e-13
    assert np.allclose(d["pickup"], case.w[0], rtol=1e-11, atol=1e-12)
    for b in range(3):
        q0 = plan.project_bump(wl["Lx"][b], wl["Ly"][b], wl["x0"][b], wl["y0"][b], wl["W"][b], wl["A"][b])
        assert np.max(np.abs(q0 - case.q0[b])) <= 1e-7 * np.max(np.abs(case.q0[b]))


def test_parity_grouped_modes_leave_whole_tiles_empty_and_queries_stay_in_plan_order():
    """The device order of the transverse modes (grouped by index parity) is internal: H read back through the API is
    in plan order and equals the oracle's closed form; most 16x16 tiles of the packed tensor hold no non-zero entry
    (parity rule m_p+m_q+m_n odd and n_p+n_q+n_n odd), and an uploaded dense H has none."""
    wl = wlmod.c2()
    wl["n_q"], wl["n_phi"] = 100, 20
    plan = mb.Plan(mb.desc_from_workload(wl), device=-1)
    m, n, _ = orc.rect_modes(0.6, 0.4, 100)
    mp, np_, _ = orc.rect_modes(0.6, 0.4, 20)
    H = orc.H_closed(0.6, 0.4, m, n, mp, np_)
    Hq = plan.query(mb.Q_H_FULL)
    assert np.max(np.abs(Hq - H)) <= 1e-6 * np.max(np.abs(H))          # fp32 storage
    total, nz = plan.query(mb.Q_TILE_STATS)
    assert total == 20 * 28 and nz <= 0.55 * total
    # brute-force count of the tiles that can be non-zero when the modes are grouped by parity class
    cls = (np.asarray(m) % 2) * 2 + (np.asarray(n) % 2)
    order = np.argsort(cls, kind="stable")
    Hp = H[:, order][:, :, order]
    cnt = 0
    for k in range(20):
        for I in range(7):
            for J in range(I + 1):
                blk = Hp[k, 16 * I:16 * I + 16, 16 * J:16 * J + 16]
                if I == J:
                    blk = np.tril(blk)
                cnt += bool(np.any(np.float32(blk) != 0))
    assert cnt == nz
    rng = np.random.default_rng(3)
    D = rng.normal(size=(20, 100, 100)); D = D + D.transpose(0, 2, 1)
    plan.coeffs_upload(1, H_full=D)
    assert np.max(np.abs(plan.query(mb.Q_H_FULL) - D)) <= 1e-6 * np.max(np.abs(D))
    total2, nz2 = plan.query(mb.Q_TILE_STATS)
    assert total2 == total and nz2 == total


def test_ftm_plan_refuses_overdamped_mode_naming_it():
    """FTM with omega <= sigma must be an error that names the mode, not NaN
    coefficients; SV proceeds; the oracle applies the same rule (test_ftm_refuses_overdamped_modes)."""
    wl, plan = _c0_plan()
    om = plan.query(mb.Q_OMEGA)[0].copy(); sg = plan.query(mb.Q_SIGMA)[0].copy()
    sg[3] = om[3] * 1.5
    plan.coeffs_upload(1, omega=om, sigma=sg)                      # SV: accepted
    d = mb.desc_from_workload(wl, scheme=mb.FTM)
    pf = mb.Plan(d, device=-1)
    with pytest.raises(mb.ModalError) as e:
        pf.coeffs_upload(1, omega=om, sigma=sg)
    assert e.value.status == mb.EINVAL and "mode 3" in e.value.message and "overdamped" in e.value.message
    sg[3] = om[3]                                                   # critically damped: refused as well
    with pytest.raises(mb.ModalError):
        pf.coeffs_upload(1, omega=om, sigma=sg)


def test_options_api_validates_keys_and_ranges():
    wl, plan = _c0_plan()
    plan.set_option("vk_impl", 2); plan.set_option("flow_g", 4); plan.set_option("timing", 0)
    for key, val in (("vk_impl", 7), ("flow_ns", 99), ("nonsense", 1)):
        with pytest.raises(mb.ModalError) as e:
            plan.set_option(key, val)
        assert e.value.status == mb.EINVAL
    # parity_order re-packs H in the new internal order: the tensor seen through the API does not change
    H1 = plan.query(mb.Q_H_FULL)
    t1 = plan.query(mb.Q_TILE_STATS)
    plan.set_option("parity_order", 0)
    assert np.array_equal(plan.query(mb.Q_H_FULL), H1)
    plan.set_option("parity_order", 1)
    assert np.array_equal(plan.query(mb.Q_H_FULL), H1) and np.array_equal(plan.query(mb.Q_TILE_STATS), t1)


@pytest.mark.parametrize("n_q,n_phi,opts", [(200, 100, {}), (200, 100, dict(mma_split=1)), (37, 13, {}), (16, 1, {}), (1, 1, {}),
                                            (100, 50, dict(parity_order=0))])
def test_batched_kernel_layout_covers_H_exactly_once(n_q, n_phi, opts):
    """Host side of the tcgen05 kernel: the operand slabs of all CTAs together hold every non-zero H^n[k][r] exactly once,
    as bf16 hi + lo within 2^-16 of the fp32 value; class-aligned k blocks give every CTA of the sine-basis plate the same
    number of K chunks."""
    wl = wlmod.c3(batch=4, n_steps=8)
    wl["n_q"], wl["n_phi"] = n_q, n_phi
    plan = mb.Plan(mb.desc_from_workload(wl), device=-1)
    for k, v in opts.items():
        plan.set_option(k, v)
    L = plan.query(mb.Q_MMA_LAYOUT)
    assert L[0] == 1, L
    fits, NKB, NGRP, NG, NC, S, RBT, RBQ, KC, KCL, G, rows_max, kmin, kmax = L[:14]
    assert G == NKB * NGRP <= 148 and NC == NG * RBT <= 256 and 1 <= S <= 3 and S * NC <= 512 and RBT in (32, 64)
    covered, nonzero, err = plan.query(mb.Q_MMA_SLAB_CHECK)
    H = plan.query(mb.Q_H_FULL)
    assert covered == nonzero == np.count_nonzero(H)
    assert err <= 2.0 ** -16
    if n_q == 200 and not opts:
        assert kmin == kmax == 4 and KC == 16            # four parity classes of <= 64 modes: every CTA multiplies one class


@pytest.mark.parametrize("n_q,n_phi", [(400, 200), (130, 40), (60, 80)])
def test_streaming_kernel_layout_covers_H_exactly_once(n_q, n_phi):
    """Host side of the streaming tcgen05 kernel (tensors too large for shared memory, batch 8..64): every non-zero H^n[k][r] sits in
    exactly one K chunk of exactly one (mode, k block) tile, as bf16 hi + lo within 2^-16; the tiles of a CTA fit its 512 TMEM columns
    at 64 samples; every transverse mode has exactly one owner CTA; only K chunks with a non-zero are streamed."""
    wl = wlmod.c4(batch=16, n_steps=8)
    wl["n_q"], wl["n_phi"] = n_q, n_phi
    plan = mb.Plan(mb.desc_from_workload(wl), device=-1)
    L = plan.query(mb.Q_STREAM_LAYOUT)
    assert L[0] == 1, L
    fits, G, NKB, KC, tiles, tmax, tmin, bch, rmax, rmin, nch, chunks, mib, nct = L[:14]
    assert G <= 148 and tmax * 64 <= 512 and tmin >= 1 and rmin >= 1 and bch <= 16 and NKB <= 8
    covered, nonzero, err, rows = plan.query(mb.Q_STREAM_CHECK)
    H = plan.query(mb.Q_H_FULL)
    assert covered == nonzero == np.count_nonzero(H)
    assert err <= 2.0 ** -16 and rows == n_q
    if (n_q, n_phi) == (400, 200):
        # four parity classes of ~100 modes: a tile multiplies only the 7 chunks of its partner class, ~28 % of the dense stream
        assert NKB == 4 and tiles == 800 and nch == 7 and chunks <= 0.3 * 800 * KC
    plan.close()


@pytest.mark.parametrize("n_q,n_phi", [(400, 200), (57, 23), (130, 40)])
def test_replicated_state_kernel_layout_rebuilds_H(n_q, n_phi):
    """Host side of the replicated-state kernel (one sample of a large plate, whole in-plane modes per CTA): the packed blocks --
    one per symmetric pair of parity classes -- and the item descriptors of the threads rebuild every non-zero H^n[k][r] exactly once
    with its fp32 value, mirror images included; at C4 a CTA holds <= 2 modes in <= 160 KiB."""
    wl = wlmod.c4(batch=1, n_steps=8)
    wl["n_q"], wl["n_phi"] = n_q, n_phi
    plan = mb.Plan(mb.desc_from_workload(wl), device=-1)
    found, covered, nonzero, kib, modes, rows, floats, ctas = plan.query(mb.Q_REPL_CHECK)
    H = plan.query(mb.Q_H_FULL)
    assert found == 1 and covered == nonzero == np.count_nonzero(H.astype(np.float32))
    if (n_q, n_phi) == (400, 200):
        assert kib <= 160 and modes == 2 and rows <= 27 and 128 <= ctas <= 132 and floats * 4 < 21e6
    plan.close()


def test_replicated_state_kernel_refuses_a_dense_uploaded_H():
    """An uploaded H without the parity zeros has one block per class pair: it does not fit, and the layout says so."""
    wl = wlmod.c4(batch=1, n_steps=8)
    wl["n_q"], wl["n_phi"] = 96, 24
    plan = mb.Plan(mb.desc_from_workload(wl), device=-1)
    rng = np.random.default_rng(2)
    H = rng.normal(size=(24, 96, 96)); H = H + H.transpose(0, 2, 1)
    plan.coeffs_upload(1, H_full=H)
    assert plan.query(mb.Q_REPL_CHECK)[0] == 0
    plan.close()


def test_batched_kernel_layout_dense_uploaded_H():
    """An uploaded H without the parity zeros (the paper's H-fitting case): every K chunk is listed."""
    wl = wlmod.c3(batch=4, n_steps=8)
    wl["n_q"], wl["n_phi"] = 48, 12
    plan = mb.Plan(mb.desc_from_workload(wl), device=-1)
    rng = np.random.default_rng(1)
    H = rng.normal(size=(12, 48, 48)); H = H + H.transpose(0, 2, 1)
    plan.coeffs_upload(1, H_full=H)
    L = plan.query(mb.Q_MMA_LAYOUT)
    covered, nonzero, err = plan.query(mb.Q_MMA_SLAB_CHECK)
    assert L[0] == 1 and L[12] == L[13] == L[8]          # fewest == most K chunks == all chunks
    assert covered == nonzero == 12 * 48 * 48 and err <= 2.0 ** -16


def test_airy_ritz_basis_library_matches_oracle():
    """SURVEY.md 8(f) row 2 / reading R16: the library's clamped Airy basis (closed-form integrals, symmetry-class Cholesky +
    Jacobi) against the oracle's (Gauss-Legendre quadrature, LAPACK): zeta^4, the coupling tensor the device holds, nl_scale."""
    wl = wlmod.c0()
    wl["n_q"], wl["n_phi"], wl["airy"], wl["n_trial"] = 30, 14, "ritz", 12
    plan = mb.Plan(mb.desc_from_workload(wl), device=-1)
    H_sine = plan.query(mb.Q_H_FULL)
    plan.set_airy_basis(mb.AIRY_CLAMPED_RITZ, 12)
    case = orc.assemble(wl)
    z4, _ = orc.airy_ritz_basis(0.6, 0.4, 14, n_trial=12)
    assert np.allclose(plan.query(mb.Q_AIRY_ZETA4), z4, rtol=1e-10)
    H = plan.query(mb.Q_H_FULL)
    assert np.max(np.abs(H - case.H)) <= 2e-7 * np.abs(case.H).max()           # both rounded to fp32 from values that agree to 1e-10
    assert np.allclose(plan.query(mb.Q_NL_SCALE)[0], wl["E"] / (2 * wl["rho"] * z4), rtol=1e-10)
    assert np.max(np.abs(H - H_sine)) > 0.1 * np.abs(H_sine).max()             # it IS another tensor
    tiles, nz = plan.query(mb.Q_TILE_STATS)
    assert nz < tiles                                                           # reflection symmetry still empties whole tiles
    plan.set_airy_basis(mb.AIRY_SINE)
    assert np.array_equal(plan.query(mb.Q_H_FULL), H_sine)
    with pytest.raises(mb.ModalError):
        plan.set_airy_basis(mb.AIRY_CLAMPED_RITZ, 3)                            # 9 trial functions < 14 modes
