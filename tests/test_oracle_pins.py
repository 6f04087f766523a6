"""Pins of the oracle against things OTHER than itself: values the paper / spec print
(tests/golden/paper_values.txt), closed forms, invariants, textbook special cases and
brute force on tiny inputs.  CPU only.  A pin fails if a plausible mistake is made in the
oracle (dropped term, wrong sign or index, transposed operand)."""
import math
import os

import numpy as np
import pytest
from scipy.special import ellipk

from oracle import oracle as orc

GOLD = {}
with open(os.path.join(os.path.dirname(__file__), "golden", "paper_values.txt")) as fh:
    for line in fh:
        if line.startswith("#") or not line.strip():
            continue
        name, val, tol, _src = [s.strip() for s in line.split("|", 3)]
        GOLD[name] = (float(val), float(tol))


def near_gold(name, x):
    v, tol = GOLD[name]
    assert abs(x - v) <= tol * abs(v) + (0 if tol else 1e-12), (name, x, v)


# ------------------------------------------------------------------ bases ----
def test_string_and_rect_eigenvalues_golden():
    near_gold("lambda1_string_L1", orc.string_lambda(1.0, 1)[0])
    lam = orc.string_lambda(2.0, 3)
    assert np.allclose(lam, [np.pi ** 2 / 4, np.pi ** 2, 9 * np.pi ** 2 / 4], rtol=1e-14)
    m, n, lam = orc.rect_modes(1.0, 1.0, 3)
    near_gold("lambda11_unit_square", lam[0])
    # tie-break: (1,2) before (2,1)
    assert (m[1], n[1]) == (1, 2) and (m[2], n[2]) == (2, 1)
    assert abs(lam[1] - 5 * np.pi ** 2) < 1e-12


def test_rect_modes_vs_bruteforce_lattice():
    # Lx=2, Ly=1, n=10 against exhaustive enumeration of m,n <= 50
    for Lx, Ly, N in [(2.0, 1.0, 10), (0.6, 0.4, 57), (0.6, 0.45, 200)]:
        m, n, lam = orc.rect_modes(Lx, Ly, N)
        mm, nn = np.meshgrid(np.arange(1, 81), np.arange(1, 81), indexing="ij")
        ll = np.sort(((mm * np.pi / Lx) ** 2 + (nn * np.pi / Ly) ** 2).ravel())[:N]
        assert np.allclose(lam, ll, rtol=1e-13)
        assert np.all(np.diff(lam) >= -1e-9)
        assert len({(a, b) for a, b in zip(m, n)}) == N
        assert np.allclose(lam, orc.rect_lambda(m, n, Lx, Ly), rtol=1e-14)


def test_modes_boundary_and_orthonormal():
    Lx, Ly = 0.6, 0.4
    assert abs(orc.rect_mode(3, 2, Lx, Ly, 0.0, 0.1)) < 1e-15
    assert abs(orc.rect_mode(3, 2, Lx, Ly, Lx, 0.1)) < 1e-12
    assert abs(orc.string_mode(1, 1.0, 0.5) - math.sqrt(2.0)) < 1e-14     # SPEC.md:125 (unit norm)
    xg, wg = np.polynomial.legendre.leggauss(40)
    x = 0.5 * Lx * (xg + 1); y = 0.5 * Ly * (xg + 1)
    m, n, _ = orc.rect_modes(Lx, Ly, 6)
    Phi = np.array([[[orc.rect_mode(m[k], n[k], Lx, Ly, xi, yi) for yi in y] for xi in x] for k in range(6)])
    Wt = np.outer(wg, wg) * 0.25 * Lx * Ly
    gram = np.einsum("kab,lab,ab->kl", Phi, Phi, Wt)
    assert np.allclose(gram, np.eye(6), atol=1e-12)


# ----------------------------------------------------------- coefficients ----
def test_omega_gamma_golden_and_textbook_plate():
    om, ga = orc.omega_gamma([np.pi ** 2], 0.0, 1.0, 1.0, 0.0, 0.0)
    assert abs(om[0] - np.pi) < 1e-14 and ga[0] == 0.0
    _, _, lam = orc.rect_modes(1.0, 1.0, 1)
    om, _ = orc.omega_gamma(lam, 5.8328, 0.0, 1.0, 0.0, 0.0)
    near_gold("omega_Dhat5.8328_unit_square_mode11", om[0])
    # textbook simply supported plate: f_mn = (pi/2) sqrt(D/(rho h)) (m^2/Lx^2 + n^2/Ly^2)  (reading R3)
    E, rho, nu, h, Lx, Ly = 2e11, 7860.0, 0.3, 1e-3, 0.6, 0.4
    D = orc.plate_D(E, h, nu)
    m, n, lam = orc.rect_modes(Lx, Ly, 10)
    om, ga = orc.omega_gamma(lam, D, 0.0, rho * h, 0.5, 1e-3)
    f_text = (np.pi / 2) * math.sqrt(E * h ** 3 / (12 * (1 - nu ** 2)) / (rho * h)) * (m ** 2 / Lx ** 2 + n ** 2 / Ly ** 2)
    assert np.allclose(om / (2 * np.pi), f_text, rtol=1e-13)
    assert abs(om[0] / (2 * np.pi) - 21.647) < 2e-3
    assert np.allclose(ga, 0.5 + 1e-3 * lam, rtol=1e-15) and np.all(ga > 0)  # Eq. 14 sign (R9)


def test_tau_golden():
    near_gold("tau_string_unit", orc.tau_string(2.0, 1.0, 1.0))
    near_gold("tau_membrane_unit", orc.tau_membrane(2.0, 1.0, 1.0, 1.0, 0.0))
    near_gold("tau_string_L0.65_A5.0265e-7_E2e11", orc.tau_string(2e11, 5.0265e-7, 0.65))


# ------------------------------------------------------ vK operator and H ----
def test_vk_operator_pins():
    near_gold("vk_operator_centre_unit_square",
              orc.vk_operator(-np.pi ** 2, -np.pi ** 2, 0.0, -np.pi ** 2, -np.pi ** 2, 0.0))
    rng = np.random.default_rng(1)
    a = rng.normal(size=6)
    assert orc.vk_operator(0, 0, 0, *a[:3]) == 0.0                          # linear field
    assert abs(orc.vk_operator(*a) - orc.vk_operator(*a[3:], *a[:3])) < 1e-15
    # the expansion f_xx g_yy + f_yy g_xx - 2 f_xy g_xy
    assert abs(orc.vk_operator(*a) - (a[0] * a[4] + a[1] * a[3] - 2 * a[2] * a[5])) < 1e-14


def test_H_closed_vs_bruteforce_quadrature_and_symmetry():
    Lx, Ly = 0.6, 0.4
    m, n, _ = orc.rect_modes(Lx, Ly, 6)
    H = orc.H_closed(Lx, Ly, m, n, m, n)
    assert np.array_equal(H, H.transpose(0, 2, 1))                         # H^n_pq = H^n_qp exactly
    scale = np.abs(H).max()
    nz = 0
    for k in range(6):
        for i in range(6):
            for j in range(i, 6):
                hq = orc.H_quadrature(Lx, Ly, (m[i], n[i]), (m[j], n[j]), (m[k], n[k]), ng=48)
                assert abs(hq - H[k, i, j]) <= 1e-10 * scale, (k, i, j, hq, H[k, i, j])
                par = (m[i] + m[j] + m[k]) % 2 == 1 and (n[i] + n[j] + n[k]) % 2 == 1
                if not par:
                    assert H[k, i, j] == 0.0                               # parity zeros are exact
                else:
                    nz += 1
    assert nz > 0


def test_H_hand_values_and_geometry_scaling():
    Lx, Ly = 0.6, 0.4
    # by hand: sss(1,1,1) = 4/(3 pi), ccs(1,1,1) = 2/(3 pi)  =>  H^{11}_{11,11} = 64 pi^2 / (3 (Lx Ly)^{5/2})
    h111 = 64 * np.pi ** 2 / (3 * (Lx * Ly) ** 2.5)
    assert abs(orc.H_closed_entry(Lx, Ly, (1, 1), (1, 1), (1, 1)) - h111) < 1e-9 * h111
    # by hand on the unit square, modes (2,1),(2,1) -> (1,1): sss(2,2,1) = 1/2 [J(0,1) - J(4,1)] = 16/(15 pi),
    # ccs(2,2,1) = 1/2 [2/pi - 2/(15 pi)] = 14/(15 pi); y-part as above.
    br = (4 + 4) * (16 / (15 * np.pi)) * (4 / (3 * np.pi)) - 2 * 4 * (14 / (15 * np.pi)) * (2 / (3 * np.pi))
    assert abs(orc.H_closed_entry(1.0, 1.0, (2, 1), (2, 1), (1, 1)) - 8 * np.pi ** 4 * br) < 1e-10
    # same-aspect scaling (reading R14): H ~ (Lx Ly)^(-5/2)
    m, n, _ = orc.rect_modes(Lx, Ly, 8)
    Ha = orc.H_closed(Lx, Ly, m, n, m[:5], n[:5]); Hb = orc.H_closed(1.5 * Lx, 1.5 * Ly, m, n, m[:5], n[:5])
    assert np.allclose(Hb, Ha * (2.25) ** -2.5, rtol=1e-13, atol=0)


def test_H_C_identity_by_independent_quadrature_of_eq11():
    # H^k_{ij} = C^j_{ik};  C^s_{ij} = int Phi_s L(Phi_i, Psi_j)  (Eq. 11)
    Lx, Ly = 0.7, 0.5
    m, n, _ = orc.rect_modes(Lx, Ly, 5)
    for (i, j, k) in [(0, 0, 0), (0, 2, 0), (1, 3, 2), (4, 2, 3), (3, 3, 0), (2, 4, 4)]:
        I, J, K = (m[i], n[i]), (m[j], n[j]), (m[k], n[k])
        Hk = orc.H_quadrature(Lx, Ly, I, J, K, ng=48)
        Cj = orc.C_quadrature(Lx, Ly, J, I, K, ng=48)       # s = j, (i, Psi_k)
        assert abs(Hk - Cj) < 1e-9 * max(1.0, abs(Hk))


# ---------------------------------------------------------------- forces ----
def test_tension_force_pins():
    lam = orc.string_lambda(0.8, 5)
    c = 3.7
    q = np.zeros(5); q[2] = 1.3e-3
    f = orc.tension_force(lam, c, q)
    assert abs(f[2] - c * lam[2] ** 2 * q[2] ** 3) < 1e-18 and np.all(f[[0, 1, 3, 4]] == 0)
    rng = np.random.default_rng(5)
    q = rng.normal(size=5) * 1e-3
    f = orc.tension_force(lam, c, q)
    S = np.sum(lam * q * q)
    assert abs(f @ q - c * S * S) < 1e-15 * abs(c * S * S) + 1e-30 and f @ q > 0
    # Eq. 3 (reading R1): S equals int ||grad w||^2 on the reconstructed displacement
    L = 0.8
    x = np.linspace(0, L, 200001)
    w = sum(q[k] * np.sqrt(2 / L) * np.sin((k + 1) * np.pi * x / L) for k in range(5))
    dw = np.gradient(w, x)
    integ = np.sum(0.5 * (dw[1:] ** 2 + dw[:-1] ** 2) * np.diff(x))
    assert abs(integ - S) < 1e-6 * S
    assert np.allclose(f, c * lam * q * integ, rtol=1e-6)
    # f = grad V, V = (c/4) S^2  (reading R4)
    for k in range(5):
        d = 1e-7
        qp = q.copy(); qp[k] += d; qm = q.copy(); qm[k] -= d
        Vp = orc.potential_nl(orc.TENSION, lam, c, None, qp); Vm = orc.potential_nl(orc.TENSION, lam, c, None, qm)
        assert abs((Vp - Vm) / (2 * d) - f[k]) < 1e-6 * np.abs(f).max()


def test_vk_force_two_stage_equals_naive_and_gradient():
    rng = np.random.default_rng(7)
    Nq, Nphi = 4, 3
    Hq = rng.normal(size=(Nphi, Nq, Nq))                    # not symmetrised: catches transposed operands
    Cc = rng.normal(size=(Nq, Nq, Nphi))
    s = rng.uniform(0.5, 2.0, Nphi); q = rng.normal(size=Nq)
    f_naive = orc.vk_force_naive(Hq, Cc, s, q)
    ref = np.einsum("n,nqr,spn,p,q,r->s", s, Hq, Cc, q, q, q)
    assert np.allclose(f_naive, ref, rtol=1e-12, atol=1e-12)
    # two-stage with C^s_{p,n} = H^n_{p,s}
    Hs = Hq + Hq.transpose(0, 2, 1)
    f2 = orc.vk_force(Hs, s, q)
    Cfrom = np.transpose(Hs, (2, 1, 0))                      # C[s][p][n] = H[n][p][s]
    assert np.allclose(f2, orc.vk_force_naive(Hs, Cfrom, s, q), rtol=1e-12, atol=1e-12)
    # f = grad V, V = 1/4 sum s_n G_n^2 >= 0 ; <f,q> = 4V (readings R4)
    V = orc.potential_nl(orc.VK, None, s, Hs, q)
    assert V > 0 and abs(f2 @ q - 4 * V) < 1e-12 * abs(V)
    for k in range(Nq):
        d = 1e-6
        qp = q.copy(); qp[k] += d; qm = q.copy(); qm[k] -= d
        g = (orc.potential_nl(orc.VK, None, s, Hs, qp) - orc.potential_nl(orc.VK, None, s, Hs, qm)) / (2 * d)
        assert abs(g - f2[k]) < 1e-7 * np.abs(f2).max()
    assert np.all(orc.vk_force(Hs, s, np.zeros(Nq)) == 0)
    assert np.all(orc.vk_force(np.zeros_like(Hs), s, q) == 0)


# --------------------------------------------------------------- schemes ----
def test_scheme_coefficient_limits():
    T = 1 / 44100.0
    om = np.array([2 * np.pi * 100, 2 * np.pi * 5000.0, 0.0]); z = np.zeros(3)
    g, p, r = orc.sv_coeffs(om, z, T)
    assert np.allclose(r, T * T, rtol=1e-15) and np.allclose(g, 2 - om ** 2 * T * T, rtol=1e-14) and np.all(p == -1.0)
    ga = np.array([5.0, 40.0, 1.0])
    g, p, r = orc.sv_coeffs(om, ga, T)                     # Eq. 21-23 simplified: r = T^2/(1+gT), p = -(1-gT)/(1+gT)
    assert np.allclose(r, T * T / (1 + ga * T), rtol=1e-15)
    assert np.allclose(p, -(1 - ga * T) / (1 + ga * T), rtol=1e-14)
    a1, a2, b1 = orc.ftm_coeffs(om[:2], z[:2], T)
    assert np.all(a2 == 1.0)
    a1, _, _ = orc.ftm_coeffs(np.array([np.pi / 2 / T]), np.zeros(1), T)
    assert abs(a1[0]) < 1e-12
    # b1 / r -> 1 as T -> 0 (reading R7: both schemes apply the same per-unit-mass force)
    for Ts, tol in [(1e-4, 1e-2), (1e-6, 1e-4)]:
        _, _, r = orc.sv_coeffs(om[:1], ga[:1], Ts); _, _, b1 = orc.ftm_coeffs(om[:1], ga[:1], Ts)
        assert abs(b1[0] / r[0] - 1) < tol


def _run_linear(scheme, om, ga, T, q0, qm1, n):
    c1, c2, c3 = orc.scheme_coeffs(scheme, om, ga, T)
    return orc.simulate(orc.LINEAR, c1, c2, c3, np.ones_like(om), q0, qm1, n)["out"][0]


def test_sv_linear_closed_form_damped_sinusoid():
    # q^n = rho^n (A cos n theta + B sin n theta), rho = sqrt(-p), theta = arccos(g / (2 sqrt(-p)))
    T = 1 / 44100.0
    om = np.array([2 * np.pi * 440.0]); ga = np.array([3.0])
    g, p, r = orc.sv_coeffs(om, ga, T)
    rho = math.sqrt(-p[0]); th = math.acos(g[0] / (2 * rho))
    q0, qm1 = 1e-3, 0.9995e-3
    A = q0
    B = (A * math.cos(th) - qm1 * rho) / math.sin(th)      # from q^{-1} = rho^{-1}(A cos th - B sin th)
    n = np.arange(20000)
    exact = rho ** n * (A * np.cos(n * th) + B * np.sin(n * th))
    out = _run_linear(orc.SV, om, ga, T, [[q0]], [[qm1]], 20000)
    assert np.max(np.abs(out - exact)) < 1e-12 * 1e-3 * 50
    assert abs(rho - math.exp(-ga[0] * T)) < 1e-12          # decay per step matches e^{-gamma T} to O(T^3)
    assert abs(th / T - om[0]) / om[0] < (om[0] * T) ** 2   # frequency warp is O((omega T)^2)


def test_ftm_reproduces_continuous_damped_sinusoid_exactly():
    T = 1 / 44100.0
    om = np.array([2 * np.pi * 440.0]); ga = np.array([3.0])
    wt = math.sqrt(om[0] ** 2 - ga[0] ** 2)
    def q(t):
        return 1e-3 * math.exp(-ga[0] * t) * (math.cos(wt * t) + ga[0] / wt * math.sin(wt * t))
    n = 44100
    out = _run_linear(orc.FTM, om, ga, T, [[q(0.0)]], [[q(-T)]], n)
    exact = np.array([q(k * T) for k in range(n)])
    assert np.max(np.abs(out - exact)) < 1e-10 * 1e-3


def test_ftm_impulse_response_closed_form():
    # unit impulse at n = 0, single lossless mode: q^{n+1} = b1 sin(w(n+1)T)/sin(wT)
    T = 1 / 44100.0
    om = np.array([2 * np.pi * 1000.0]); ga = np.zeros(1)
    c1, c2, c3 = orc.scheme_coeffs(orc.FTM, om, ga, T)
    n = 1000
    fext = np.zeros((1, n)); fext[0, 0] = 1.0
    out = orc.simulate(orc.LINEAR, c1, c2, c3, np.ones(1), [[0.0]], [[0.0]], n,
                       fext=fext, fext_gain=np.ones((1, 1)))["out"][0]
    k = np.arange(n)
    exact = c3[0] * np.sin(om[0] * k * T) / math.sin(om[0] * T)
    assert np.max(np.abs(out - exact)) < 1e-9 * c3[0] * 100


def test_simulate_conventions_zero_determinism_instability():
    T = 1 / 44100.0
    om = np.array([1000.0, 3000.0]); ga = np.array([1.0, 2.0])
    c1, c2, c3 = orc.scheme_coeffs(orc.SV, om, ga, T)
    w = np.array([0.3, -0.7])
    z = orc.simulate(orc.LINEAR, c1, c2, c3, w, np.zeros((1, 2)), np.zeros((1, 2)), 100)
    assert np.all(z["out"] == 0) and z["first_bad"][0] == -1
    q0 = np.array([[1e-3, 2e-3]])
    a = orc.simulate(orc.LINEAR, c1, c2, c3, w, q0, q0, 50, want_traj=True, want_final=True)
    b = orc.simulate(orc.LINEAR, c1, c2, c3, w, q0, q0, 50)
    assert np.array_equal(a["out"], b["out"])                                # determinism
    assert abs(a["out"][0, 0] - w @ q0[0]) < 1e-18                           # out[0] = w . q^0 (R10)
    assert np.array_equal(a["traj"][0, 0], q0[0])
    assert abs(a["out"][0, 1] - w @ ((c1 + c2) * q0[0])) < 1e-18             # first update
    assert np.array_equal(a["q_final"][0, 0], a["traj"][0, 49])
    # unstable mode (omega T > 2) blows up; the first non-finite step index is reported
    om_bad = np.array([2.5 / T]); c1, c2, c3 = orc.scheme_coeffs(orc.SV, om_bad, np.zeros(1), T)
    r = orc.simulate(orc.LINEAR, c1, c2, c3, np.ones(1), [[1.0]], [[1.0]], 5000, want_traj=True)
    fb = r["first_bad"][0]
    assert fb > 0 and np.all(np.isfinite(r["traj"][0, :fb])) and not np.isfinite(r["traj"][0, fb, 0])


# --------------------------------------------- Duffing closed form (R2, R4) ----
def _measured_frequency(x, T):
    """Mean frequency from interpolated downward zero crossings."""
    s = np.where((x[:-1] > 0) & (x[1:] <= 0))[0]
    t = (s + x[s] / (x[s] - x[s + 1])) * T
    return (len(t) - 1) / (t[-1] - t[0])


def _duffing_exact_freq(w0, kappa, a):
    mpar = kappa * a * a / (2 * (w0 ** 2 + kappa * a * a))
    return math.sqrt(w0 ** 2 + kappa * a * a) / (4 * ellipk(mpar))


@pytest.mark.parametrize("kind", ["tension", "vk"])
def test_single_mode_is_duffing_with_elliptic_period(kind):
    """One active mode: q'' + w0^2 q + kappa q^3 = 0, exact period 4K(m)/sqrt(w0^2 + kappa a^2),
    m = kappa a^2 / (2 (w0^2 + kappa a^2)).  The SV frequency converges to it at 2nd order."""
    w0 = 2 * np.pi * 100.0
    a = 1e-3
    if kind == "tension":
        lam = np.array([50.0]); c = 0.25 * w0 ** 2 / (lam[0] ** 2 * a * a)      # kappa a^2 = w0^2/4
        kappa = c * lam[0] ** 2
        kw = dict(lam=lam[None], nl_scale=c); model = orc.TENSION
    else:
        H = np.array([[[7461.5725]]]); s = np.array([0.25 * w0 ** 2 / (H[0, 0, 0] ** 2 * a * a)])
        kappa = s[0] * H[0, 0, 0] ** 2                                            # f = s H^2 q^3
        kw = dict(nl_scale=s[None], H=H); model = orc.VK
    f_exact = _duffing_exact_freq(w0, kappa, a)
    assert 1.08 < f_exact / 100.0 < 1.10                                          # hardening: pitch rises
    errs = []
    for over in (1, 2, 4):
        T = 1 / (44100.0 * over)
        om = np.array([w0]); ga = np.zeros(1)
        c1, c2, c3 = orc.scheme_coeffs(orc.SV, om, ga, T)
        q0 = np.array([[a]])
        if model == orc.VK:
            qm1 = orc.start_state(model, q0[0], om, T, nl_scale=kw["nl_scale"][0], H=kw["H"])[None]
        else:
            qm1 = orc.start_state(model, q0[0], om, T, lam=kw["lam"][0], nl_scale=kw["nl_scale"])[None]
        out = orc.simulate(model, c1, c2, c3, np.ones(1), q0, qm1, int(44100 * over * 0.5), **kw)["out"][0]
        errs.append(_measured_frequency(out, T) - f_exact)
    assert abs(errs[0]) < 5e-3                                                    # ~1e-5 relative at 44.1 kHz
    assert 3.3 < errs[0] / errs[1] < 4.7 and 3.0 < errs[1] / errs[2] < 5.0        # 2nd order


# ------------------------------------------------------- energy and order ----
def _small_vk_case(amp, lossless=True, Nq=6, Nphi=6):
    Lx, Ly, h, E, rho, nu = 0.6, 0.4, 1e-3, 2e11, 7860.0, 0.3
    m, n, lam = orc.rect_modes(Lx, Ly, Nq)
    H = orc.H_closed(Lx, Ly, m, n, m[:Nphi], n[:Nphi])
    om, ga = orc.omega_gamma(lam, orc.plate_D(E, h, nu), 0.0, rho * h, 0.0 if lossless else 0.5, 0.0 if lossless else 1e-3)
    s = E / (2 * rho * lam[:Nphi] ** 2)
    q0 = orc.project_bump_rect(m, n, Lx, Ly, 0.27, 0.17, 0.3, amp * h)
    return dict(H=H, om=om, ga=ga, s=s, q0=q0, m=m, n=n, Lx=Lx, Ly=Ly, h=h)


def test_linear_lossless_energy_is_conserved_exactly():
    c = _small_vk_case(0.5)
    T = 1 / 44100.0
    c1, c2, c3 = orc.scheme_coeffs(orc.SV, c["om"], c["ga"], T)
    qm1 = orc.start_state(orc.LINEAR, c["q0"], c["om"], T)
    r = orc.simulate(orc.LINEAR, c1, c2, c3, np.ones(6), c["q0"][None], qm1[None], 11025, want_traj=True)
    e = orc.energy(orc.LINEAR, T, c["om"], r["traj"][0])
    assert (e.max() - e.min()) / e.mean() < 1e-11
    # the energy is the textbook one at rest: 1/2 sum omega^2 q0^2 up to O(T^2)
    assert abs(e[0] / (0.5 * np.sum(c["om"] ** 2 * c["q0"] ** 2)) - 1) < 1e-3


@pytest.mark.parametrize("amp,osc_bound", [(0.5, 5e-6), (2.0, 1e-4)])
def test_nonlinear_lossless_energy_bounded_no_drift(amp, osc_bound):
    c = _small_vk_case(amp)
    T = 1 / 44100.0
    c1, c2, c3 = orc.scheme_coeffs(orc.SV, c["om"], c["ga"], T)
    qm1 = orc.start_state(orc.VK, c["q0"], c["om"], T, nl_scale=c["s"], H=c["H"])
    r = orc.simulate(orc.VK, c1, c2, c3, np.ones(6), c["q0"][None], qm1[None], 11025,
                     nl_scale=c["s"][None], H=c["H"], want_traj=True)
    e = orc.energy(orc.VK, T, c["om"], r["traj"][0], nl_scale=c["s"], H=c["H"])
    k = len(e) // 10
    assert (e.max() - e.min()) / e.mean() < osc_bound
    assert abs(e[-k:].mean() - e[:k].mean()) / e.mean() < osc_bound / 5
    # non-linear share of the energy is what the amplitude implies (hardening, V_nl > 0)
    V = orc.potential_nl(orc.VK, None, c["s"], c["H"], c["q0"])
    assert V > 0 and abs(e[0] - (0.5 * np.sum(c["om"] ** 2 * c["q0"] ** 2) + V)) < 2e-3 * e[0]


def test_damped_energy_decreases():
    c = _small_vk_case(1.0, lossless=False)
    T = 1 / 44100.0
    c1, c2, c3 = orc.scheme_coeffs(orc.SV, c["om"], c["ga"], T)
    qm1 = orc.start_state(orc.VK, c["q0"], c["om"], T, nl_scale=c["s"], H=c["H"])
    r = orc.simulate(orc.VK, c1, c2, c3, np.ones(6), c["q0"][None], qm1[None], 8000,
                     nl_scale=c["s"][None], H=c["H"], want_traj=True)
    e = orc.energy(orc.VK, T, c["om"], r["traj"][0], nl_scale=c["s"], H=c["H"])
    sm = np.convolve(e, np.ones(400) / 400, mode="valid")
    assert np.all(np.diff(sm[::400]) < 0)


def test_second_order_convergence_with_symmetric_start():
    """Whole-run error vs a 16x oversampled run drops ~4x when T halves (needs the 2nd-order start, R8)."""
    c = _small_vk_case(1.0, lossless=False)
    def run(over):
        T = 1 / (44100.0 * over)
        c1, c2, c3 = orc.scheme_coeffs(orc.SV, c["om"], c["ga"], T)
        qm1 = orc.start_state(orc.VK, c["q0"], c["om"], T, nl_scale=c["s"], H=c["H"])
        o = orc.simulate(orc.VK, c1, c2, c3, np.ones(6), c["q0"][None], qm1[None], 2048 * over,
                         nl_scale=c["s"][None], H=c["H"])["out"][0]
        return o[::over]
    ref = run(16)
    e1 = np.max(np.abs(run(1) - ref)); e2 = np.max(np.abs(run(2) - ref)); e4 = np.max(np.abs(run(4) - ref))
    assert 3.5 < e1 / e2 < 4.6 and 3.5 < e2 / e4 < 4.8


# ------------------------------------------------------------ projection ----
def test_string_pluck_projection_closed_form():
    L, x0, W, A, N = 0.8, 0.31, 0.08, 2e-3, 40
    q = orc.project_bump_string(N, L, x0, W, A)
    k = np.arange(1, N + 1) * np.pi / L
    beta = 2 * np.pi / W
    part1 = 2 * np.sin(k * W / 2) / k
    part2 = np.sin((beta - k) * W / 2) / (beta - k) + np.sin((beta + k) * W / 2) / (beta + k)
    exact = 0.5 * A * np.sqrt(2 / L) * np.sin(k * x0) * (part1 + part2)
    assert np.allclose(q, exact, rtol=0, atol=1e-14)


def test_plate_bump_projection_reconstructs_peak_and_is_quadrature_independent():
    Lx, Ly, x0, y0, W, A = 0.6, 0.4, 0.23, 0.19, 0.2, 5e-4
    m, n, _ = orc.rect_modes(Lx, Ly, 300)
    q = orc.project_bump_rect(m, n, Lx, Ly, x0, y0, W, A)
    q2 = orc.project_bump_rect(m, n, Lx, Ly, x0, y0, W, A, nr=160, nth=512)
    assert np.max(np.abs(q - q2)) < 1e-15
    peak = sum(q[k] * orc.rect_mode(m[k], n[k], Lx, Ly, x0, y0) for k in range(300))
    assert abs(peak - A) < 0.02 * A
    # cartesian brute force on the bounding square for the first modes
    xg, wg = np.polynomial.legendre.leggauss(400)
    X = x0 + 0.5 * W * xg[:, None]; Y = y0 + 0.5 * W * xg[None, :]
    R = np.hypot(X - x0, Y - y0)
    w0 = np.where(R < W / 2, 0.5 * A * (1 + np.cos(2 * np.pi * R / W)), 0.0)
    for k in range(5):
        phi = 2 / np.sqrt(Lx * Ly) * np.sin(m[k] * np.pi * X / Lx) * np.sin(n[k] * np.pi * Y / Ly)
        brute = np.sum(np.outer(wg, wg) * w0 * phi) * 0.25 * W * W
        assert abs(brute - q[k]) < 1e-6 * abs(q[0])


# ---------------------------------------------- glue of assemble(): mask rule and geometry fold ----
def test_geometry_fold_of_assemble_equals_own_geometry_tensor():
    """Reading R14 / SURVEY.md C18: assemble() keeps ONE tensor H_ref and folds (c_b / c_ref)^2 into s_n[b].
    Pin: the force from (H_ref, folded s) equals the force from the sample's OWN tensor, H_closed on its own
    (Lx, Ly) at a DIFFERENT aspect ratio with the same index sets, and the plain scale E / (2 rho zeta_b^4)."""
    wl = dict(name="fold", model="vk", n_q=14, n_phi=9, n_steps=8, batch=3, sample_rate=44100.0,
              ref=dict(Lx=0.6, Ly=0.45, h=1e-3), T0=0.0, sigma0=0.5, sigma1=1e-3, pickup=(0.43, 0.37),
              E=2.0e11, rho=7860.0, nu=0.3,
              Lx=np.array([0.47, 0.8, 0.6]), Ly=np.array([0.47 * 0.52, 0.8 * 0.97, 0.45]), h=np.array([0.7e-3, 1.9e-3, 1e-3]),
              A=np.array([1e-3, 1e-3, 1e-3]), W=np.array([0.1, 0.15, 0.1]), x0=np.array([0.2, 0.3, 0.3]), y0=np.array([0.12, 0.4, 0.2]))
    case = orc.assemble(wl, round_fp32=False)
    mq, nq, mphi, nphi = (case.extra[k] for k in ("mq", "nq", "mphi", "nphi"))
    rng = np.random.default_rng(3)
    for b in range(3):
        Lx, Ly = wl["Lx"][b], wl["Ly"][b]
        H_own = orc.H_closed(Lx, Ly, mq, nq, mphi, nphi)
        s_own = wl["E"] / (2.0 * wl["rho"] * orc.rect_lambda(mphi, nphi, Lx, Ly) ** 2)
        q = rng.normal(size=14) * 1e-3
        f_fold = orc.vk_force(case.H, case.nl_scale[b], q)
        f_own = orc.vk_force(H_own, s_own, q)
        assert np.allclose(f_fold, f_own, rtol=1e-11, atol=1e-14 * np.abs(f_own).max()), b
    # the two off-reference samples really have another aspect ratio (the pin would be vacuous otherwise)
    assert abs(wl["Ly"][0] / wl["Lx"][0] - 0.75) > 0.2 and abs(wl["Ly"][1] / wl["Lx"][1] - 0.75) > 0.2


def test_mask_rule_sv_keeps_what_the_scheme_carries():
    """Reading R11 / SURVEY.md C12: SV needs omega T < 2.  A lossless linear mode at omega T = 1.89 stays bounded
    over 1e5 steps, at omega T = 2.01 it diverges; active_mask keeps the first and drops the second."""
    T = 1.0 / 44100.0
    for wT, bounded in [(1.89, True), (2.01, False)]:
        om = np.array([wT / T]); ga = np.zeros(1)
        g, p, r = orc.sv_coeffs(om, ga, T)
        q0 = np.array([[1.0]]); qm1 = np.array([[1.0]])
        res = orc.simulate(orc.LINEAR, g, p, r, np.ones(1), q0, qm1, 100000)
        peak = np.nanmax(np.abs(res["out"]))
        assert (np.isfinite(peak) and peak < 20.0) == bounded, (wT, peak)
        assert bool(orc.active_mask(orc.SV, om, ga, T)[0]) == bounded
    assert orc.active_mask(orc.SV, np.array([1.8999 / T, 1.9 / T]), np.zeros(2), T).tolist() == [True, False]


def test_mask_rule_ftm_stops_short_of_the_aliasing_limit():
    """FTM is exact at the samples for any damped frequency, so its limit is aliasing, not stability: the sampled
    response of a mode at w~ T = 1.06 pi is indistinguishable from that of 0.94 pi.  active_mask keeps w~ < 0.95 pi / T."""
    T = 1.0 / 44100.0
    ga = np.array([3.0])
    def response(wt_T):
        wt = wt_T * np.pi / T
        om = np.sqrt(wt ** 2 + ga ** 2)
        a1, a2, b1 = orc.ftm_coeffs(om, ga, T)
        q0 = np.array([[1.0]])
        qm1 = np.array([[np.exp(ga[0] * T) * (np.cos(wt * T) - ga[0] / wt * np.sin(wt * T))]])      # exact q(-T)
        return om, orc.simulate(orc.LINEAR, -a1, -a2, b1, np.ones(1), q0, qm1, 4000)["out"][0]
    om_lo, lo = response(0.94)
    om_hi, hi = response(1.06)
    n = np.arange(4000)
    exact = np.exp(-ga[0] * n * T) * (np.cos(0.94 * np.pi * n) + ga[0] / (0.94 * np.pi / T) * np.sin(0.94 * np.pi * n))
    assert np.max(np.abs(lo - exact)) < 1e-9                       # the kept mode is reproduced exactly
    assert np.max(np.abs(hi - lo)) < 2e-3                          # the aliased one cannot be told apart from it
    assert orc.active_mask(orc.FTM, om_lo, ga, T)[0] and not orc.active_mask(orc.FTM, om_hi, ga, T)[0]
    w = lambda x: np.sqrt((x * np.pi / T) ** 2 + ga ** 2)
    assert orc.active_mask(orc.FTM, w(0.9499), ga, T)[0] and not orc.active_mask(orc.FTM, w(0.9501), ga, T)[0]


def test_ftm_refuses_overdamped_modes():
    """the FTM coefficients need underdamped modes; an active overdamped mode is an error naming it."""
    T = 1.0 / 44100.0
    om = np.array([2000.0, 50.0, 3000.0]); ga = np.array([1.0, 60.0, 2.0])
    with pytest.raises(ValueError, match="mode 1"):
        orc.scheme_coeffs(orc.FTM, om, ga, T, np.ones(3, bool))
    orc.scheme_coeffs(orc.FTM, om, ga, T, np.array([True, False, True]))     # a masked mode is not asked for coefficients
    orc.scheme_coeffs(orc.SV, om, ga, T)                                      # SV proceeds


# ---------------------------------- in-plane basis of reading R16: clamped (Airy) modes by Rayleigh-Ritz ----
def _ritz_fields(c_n, Lx, Ly, x, y):
    """Psi, Psi_xx, Psi_yy, Psi_xy of one mode on the tensor grid x (x) y, from the trial functions' own derivatives."""
    nt = c_n.shape[0]
    Tx, dTx, ddTx = orc._ritz_trial(nt, x / Lx)
    Ty, dTy, ddTy = orc._ritz_trial(nt, y / Ly)
    f = lambda a, b: np.einsum("ij,ig,jh->gh", c_n, a, b)
    return f(Tx, Ty), f(ddTx, Ty) / Lx ** 2, f(Tx, ddTy) / Ly ** 2, f(dTx, dTy) / (Lx * Ly)


def test_airy_ritz_square_plate_textbook_value_and_upper_bounds():
    """Clamped square plate: the fundamental frequency parameter zeta_1^2 L^2 is 35.99 in the textbooks (35.985 to five
    figures); Rayleigh-Ritz values are upper bounds that can only fall when the trial space grows."""
    prev = None
    for nt in (4, 8, 12, 16):
        z4, _ = orc.airy_ritz_basis(1.0, 1.0, 4, n_trial=nt)
        lam = np.sqrt(z4)
        assert lam[0] >= 35.985
        if prev is not None:
            assert np.all(lam <= prev * (1 + 1e-12))
        prev = lam
    assert prev[0] < 35.995 and abs(prev[1] - prev[2]) < 1e-6 * prev[1]          # 35.99; modes (2,1) / (1,2) degenerate on the square
    assert abs(prev[1] - 73.40) < 0.05 and abs(prev[3] - 108.22) < 0.15            # 73.39, 108.2 in the same tables
    # scaling: zeta^4 ~ L^-4 at fixed aspect
    za, _ = orc.airy_ritz_basis(0.6, 0.4, 5, n_trial=10)
    zb, _ = orc.airy_ritz_basis(1.2, 0.8, 5, n_trial=10)
    assert np.allclose(za, 16.0 * zb, rtol=1e-10)


def test_airy_ritz_modes_orthonormal_clamped_and_weakly_biharmonic():
    """By 2-D Gauss-Legendre quadrature of the evaluated functions (not the Kronecker assembly): the modes are orthonormal,
    vanish with their normal slope on the edges, and satisfy the weak eigen-equation  int Lap Psi Lap v = zeta^4 int Psi v
    against every trial function v; the Rayleigh quotient with int (Lap Psi)^2 gives zeta^4 back."""
    Lx, Ly, nt = 0.6, 0.4, 10
    z4, c = orc.airy_ritz_basis(Lx, Ly, 6, n_trial=nt)
    xg, wg = np.polynomial.legendre.leggauss(96)
    x, wx = 0.5 * Lx * (xg + 1), 0.5 * Lx * wg
    y, wy = 0.5 * Ly * (xg + 1), 0.5 * Ly * wg
    W = wx[:, None] * wy[None, :]
    F = [_ritz_fields(c[n], Lx, Ly, x, y) for n in range(6)]
    gram = np.array([[np.sum(W * F[a][0] * F[b][0]) for b in range(6)] for a in range(6)])
    assert np.allclose(gram, np.eye(6), atol=1e-9)
    for n in range(6):
        lap = F[n][1] + F[n][2]
        assert abs(np.sum(W * lap * lap) / z4[n] - 1.0) < 1e-8
        for (i, j) in ((1, 1), (2, 3), (5, 2)):                                   # a few trial functions as test functions
            e = np.zeros((nt, nt)); e[i - 1, j - 1] = 1.0
            v, vxx, vyy, _ = _ritz_fields(e, Lx, Ly, x, y)
            lhs, rhs = np.sum(W * lap * (vxx + vyy)), z4[n] * np.sum(W * F[n][0] * v)
            assert abs(lhs - rhs) <= 1e-7 * (abs(lhs) + abs(rhs)) + 1e-6 * np.sqrt(z4[n])
    # boundary: value and normal derivative (finite difference of the evaluated function)
    h = 1e-6
    for n in range(6):
        for yy in (0.07, 0.21, 0.33):
            assert abs(orc.airy_ritz_eval(c, Lx, Ly, 0.0, yy)[n]) < 1e-10 and abs(orc.airy_ritz_eval(c, Lx, Ly, Lx, yy)[n]) < 1e-9
            assert abs(orc.airy_ritz_eval(c, Lx, Ly, h, yy)[n]) / h < 1e-3 * np.abs(F[n][0]).max()
        assert abs(orc.airy_ritz_eval(c, Lx, Ly, 0.3, h)[n]) / h < 1e-3 * np.abs(F[n][0]).max()


def test_H_airy_ritz_vs_bruteforce_quadrature_symmetry_and_HC_identity():
    """Eq. 10 by brute-force 2-D quadrature of Psi_n L(Phi_p, Phi_q) (operator of Eq. 7 through orc.vk_operator) against the
    separable evaluation; symmetry in (p, q); and Eq. 11: C^s_{p,n} = int Phi_s L(Phi_p, Psi_n) equals H^n_{p,s},
    which holds because Psi and its normal slope vanish on the edges."""
    Lx, Ly, nt = 0.6, 0.4, 8
    z4, c = orc.airy_ritz_basis(Lx, Ly, 5, n_trial=nt)
    mq, nq, _ = orc.rect_modes(Lx, Ly, 6)
    H = orc.H_airy_ritz(Lx, Ly, mq, nq, c)
    assert np.max(np.abs(H - H.transpose(0, 2, 1))) <= 1e-9 * np.abs(H).max()
    xg, wg = np.polynomial.legendre.leggauss(72)
    x, wx = 0.5 * Lx * (xg + 1), 0.5 * Lx * wg
    y, wy = 0.5 * Ly * (xg + 1), 0.5 * Ly * wg
    W = wx[:, None] * wy[None, :]
    amp = 2.0 / np.sqrt(Lx * Ly)

    def phi(k):     # value, xx, yy, xy of transverse sine mode k on the grid
        ax, ay = mq[k] * np.pi / Lx, nq[k] * np.pi / Ly
        sx, cx, sy, cy = np.sin(ax * x)[:, None], np.cos(ax * x)[:, None], np.sin(ay * y)[None, :], np.cos(ay * y)[None, :]
        return amp * sx * sy, -amp * ax ** 2 * sx * sy, -amp * ay ** 2 * sx * sy, amp * ax * ay * cx * cy

    vkop = np.vectorize(orc.vk_operator)
    for (n, p, q) in ((0, 0, 0), (0, 1, 1), (1, 0, 1), (2, 3, 0), (4, 5, 2), (3, 2, 2)):
        psi, pxx, pyy, pxy = _ritz_fields(c[n], Lx, Ly, x, y)
        fp, fq = phi(p), phi(q)
        brute = np.sum(W * psi * vkop(fp[1], fp[2], fp[3], fq[1], fq[2], fq[3]))
        assert abs(brute - H[n, p, q]) <= 1e-7 * np.abs(H).max(), (n, p, q, brute, H[n, p, q])
        c_spn = np.sum(W * fq[0] * vkop(fp[1], fp[2], fp[3], pxx, pyy, pxy))        # s = q: C^q_{p,n}
        assert abs(c_spn - H[n, p, q]) <= 1e-6 * np.abs(H).max(), (n, p, q, c_spn, H[n, p, q])
    # reflection symmetry of the rectangle: ~3/4 of the entries vanish, as for the sine basis
    assert 0.2 < np.mean(np.abs(H) > 1e-9 * np.abs(H).max()) < 0.3


# ------------------------------------------------ reverse pass ----
def _bptt_problem(seed=0, Nq=7, Nphi=5, N=48):
    rng = np.random.default_rng(seed)
    H = rng.normal(size=(Nphi, Nq, Nq)); H = H + H.transpose(0, 2, 1)
    T = 1 / 44100
    om = rng.uniform(500, 9000, Nq); ga = rng.uniform(0.5, 30, Nq)
    c1, c2, c3 = orc.scheme_coeffs(orc.SV, om, ga, T)
    w = rng.normal(size=Nq); s = rng.uniform(1e7, 1e8, Nphi)
    q0 = rng.normal(size=Nq) * 1e-2; qm1 = q0 + rng.normal(size=Nq) * 1e-4
    gout = rng.normal(size=N)
    return dict(c1=c1, c2=c2, c3=c3, w=w, s=s, H=H, q0=q0, qm1=qm1), gout, N


def test_bptt_adjoint_matches_finite_differences_of_the_forward_oracle():
    """PAPER.md:281-285.  The adjoint recurrence (numpy) against central differences of the INDEPENDENT forward code
    (modal_oracle.c through `simulate`) for a linear functional L = sum_n gout_n out_n: every gradient array, including H
    (perturbed as a symmetric pair: dL/d(pair) = g[k][r] + g[r][k]).  A wrong sign, a dropped Jacobian term, a transposed
    index or an off-by-one in the step index fails here."""
    P, gout, N = _bptt_problem()

    def L(**over):
        a = {**P, **over}
        r = orc.simulate(orc.VK, a["c1"][None], a["c2"][None], a["c3"][None], a["w"][None], a["q0"][None], a["qm1"][None], N,
                         nl_scale=a["s"][None], H=a["H"])
        return float(gout @ r["out"][0])

    g = orc.bptt_vk(P["c1"], P["c2"], P["c3"], P["w"], P["s"], P["H"], P["q0"], P["qm1"], gout)
    # the non-linear part must matter in this problem, or the Jacobian terms would go unchecked
    g_lin = orc.bptt_vk(P["c1"], P["c2"], P["c3"], P["w"], 0 * P["s"], P["H"], P["q0"], P["qm1"], gout)
    assert np.linalg.norm(g["q0"] - g_lin["q0"]) > 1e-3 * np.linalg.norm(g["q0"])
    for name, eps in (("q0", 1e-7), ("qm1", 1e-7), ("c1", 1e-7), ("c2", 1e-7), ("c3", 1e-12), ("w", 1e-6), ("s", 1e3)):
        for idx in range(P[name].shape[0]):
            hi = P[name].copy(); hi[idx] += eps
            lo = P[name].copy(); lo[idx] -= eps
            fd = (L(**{name: hi}) - L(**{name: lo})) / (2 * eps)
            assert abs(fd - g[name][idx]) <= 2e-5 * np.max(np.abs(g[name])) + 1e-7 * abs(fd), (name, idx, fd, g[name][idx])
    rng = np.random.default_rng(1)
    for _ in range(12):
        m, k, r = rng.integers(0, 5), rng.integers(0, 7), rng.integers(0, 7)
        eps = 1e-5
        hi = P["H"].copy(); lo = P["H"].copy()
        for (a, b) in {(k, r), (r, k)}:
            hi[m, a, b] += eps; lo[m, a, b] -= eps
        fd = (L(H=hi) - L(H=lo)) / (2 * eps)
        want = g["H"][m, k, r] + (g["H"][m, r, k] if k != r else 0.0)
        assert abs(fd - want) <= 2e-5 * np.max(np.abs(g["H"])) + 1e-6 * abs(fd), (m, k, r, fd, want)


def test_bptt_linear_case_is_the_transposed_impulse_response():
    """With s = 0 the recurrence is linear and time-invariant: dL/dq0_k = sum_n gout_n w_k h_k[n], h_k the response of
    mode k to q^0 = 1, q^-1 = 0 ... which for the homogeneous recurrence is the textbook two-term solution."""
    P, gout, N = _bptt_problem(seed=3)
    g = orc.bptt_vk(P["c1"], P["c2"], P["c3"], P["w"], 0 * P["s"], P["H"], P["q0"], P["qm1"], gout)
    h0 = np.zeros((N, 7)); h1 = np.zeros((N, 7))       # responses to (q0, qm1) = (1, 0) and (0, 1)
    a, b = np.ones(7), np.zeros(7)
    c, d = np.zeros(7), np.ones(7)
    for n in range(N):
        h0[n], h1[n] = a, c
        a, b = P["c1"] * a + P["c2"] * b, a
        c, d = P["c1"] * c + P["c2"] * d, c
    assert np.allclose(g["q0"], P["w"] * (gout @ h0), rtol=1e-12, atol=1e-14)
    assert np.allclose(g["qm1"], P["w"] * (gout @ h1), rtol=1e-12, atol=1e-14)
    assert np.all(g["s"] == 0) or np.allclose(g["H"], 0)


@pytest.mark.parametrize("scheme", [orc.SV, orc.FTM])
def test_scheme_coefficient_derivatives_by_finite_differences(scheme):
    T = 1 / 44100
    om = np.array([300.0, 2500.0, 20000.0, 60000.0]); ga = np.array([0.5, 3.0, 40.0, 200.0])
    d = orc.dcoeffs_domega_dgamma(scheme, om, ga, T)
    for var, eps in (("w", 1e-3), ("g", 1e-4)):
        hi = orc.scheme_coeffs(scheme, om + (eps if var == "w" else 0), ga + (eps if var == "g" else 0), T)
        lo = orc.scheme_coeffs(scheme, om - (eps if var == "w" else 0), ga - (eps if var == "g" else 0), T)
        for i, c in enumerate(("c1", "c2", "c3")):
            fd = (hi[i] - lo[i]) / (2 * eps)
            assert np.allclose(d[f"{c}_{var}"], fd, rtol=2e-6, atol=1e-9 * np.max(np.abs(fd)) + 1e-18), (c, var, d[f"{c}_{var}"], fd)


def test_bptt_tension_adjoint_matches_finite_differences_of_the_forward_oracle():
    """The adjoint of the tension-modulated recurrence (strings / Berger plates) against central differences of the forward C oracle."""
    rng = np.random.default_rng(5)
    Nq, N = 9, 60
    T = 1 / 44100
    om = rng.uniform(500, 9000, Nq); ga = rng.uniform(0.5, 30, Nq)
    c1, c2, c3 = orc.scheme_coeffs(orc.SV, om, ga, T)
    lam = np.sort(rng.uniform(10, 900, Nq)); w = rng.normal(size=Nq); cval = 4.0e6
    q0 = rng.normal(size=Nq) * 2e-3; qm1 = q0 + rng.normal(size=Nq) * 1e-5
    gout = rng.normal(size=N)
    P = dict(c1=c1, c2=c2, c3=c3, w=w, q0=q0, qm1=qm1)

    def L(cv=cval, **over):
        a = {**P, **over}
        r = orc.simulate(orc.TENSION, a["c1"][None], a["c2"][None], a["c3"][None], a["w"][None], a["q0"][None], a["qm1"][None], N,
                         lam=lam[None], nl_scale=np.array([cv]))
        return float(gout @ r["out"][0])

    g = orc.bptt_tension(c1, c2, c3, w, lam, cval, q0, qm1, gout)
    g_lin = orc.bptt_tension(c1, c2, c3, w, lam, 0.0, q0, qm1, gout)
    assert np.linalg.norm(g["q0"] - g_lin["q0"]) > 1e-3 * np.linalg.norm(g["q0"])          # the non-linear terms matter here
    for name, eps in (("q0", 1e-8), ("qm1", 1e-8), ("c1", 1e-7), ("c2", 1e-7), ("c3", 1e-13), ("w", 1e-6)):
        for idx in range(Nq):
            hi = P[name].copy(); hi[idx] += eps
            lo = P[name].copy(); lo[idx] -= eps
            fd = (L(**{name: hi}) - L(**{name: lo})) / (2 * eps)
            assert abs(fd - g[name][idx]) <= 5e-5 * np.max(np.abs(g[name])) + 1e-7 * abs(fd), (name, idx, fd, g[name][idx])
    fd = (L(cv=cval * (1 + 1e-5)) - L(cv=cval * (1 - 1e-5))) / (2e-5 * cval)
    assert abs(fd - g["c"]) <= 1e-5 * abs(g["c"]), (fd, g["c"])
