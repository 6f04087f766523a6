"""ORACLE (test infrastructure, NOT the product) -- Python side.

ctypes loader for ``modal_oracle.c`` plus the O(N) glue of the method written
with numpy in fp64, in the paper's order: modes -> omega/gamma -> mask ->
scheme coefficients -> coupling tensor -> initial projection -> two-step start
-> stepping.  Citations are PAPER.md line numbers; readings R1..R14 are the
ones listed in DESIGN.md.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline /
``--impl reference`` legs may import this module.  It imports nothing from
``paper_2505_05940_b200``: workloads are passed in as plain dicts by the caller.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "modal_oracle.c")
_LIB = os.path.join(_HERE, "libmodal_oracle.so")

LINEAR, TENSION, VK = 0, 1, 2

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int)


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, OpenMP over batch samples only)."""
    if force or (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(
            ["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class _SimArgs(C.Structure):
    _fields_ = [
        ("model", C.c_int), ("Nq", C.c_int), ("Nphi", C.c_int),
        ("batch", C.c_int), ("n_steps", C.c_int), ("coeff_batch", C.c_int),
        ("c1", _dp), ("c2", _dp), ("c3", _dp), ("w", _dp), ("lambda_", _dp),
        ("nl_scale", _dp), ("H", _dp), ("q0", _dp), ("qm1", _dp),
        ("fext", _dp), ("fext_gain", _dp), ("out", _dp), ("first_bad", _ip),
        ("traj", _dp), ("q_final", _dp),
    ]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        L = _lib
        L.orc_string_mode.restype = C.c_double
        L.orc_string_mode.argtypes = [C.c_int, C.c_double, C.c_double]
        L.orc_rect_mode.restype = C.c_double
        L.orc_rect_mode.argtypes = [C.c_int, C.c_int] + [C.c_double] * 4
        L.orc_tau_string.restype = C.c_double
        L.orc_tau_string.argtypes = [C.c_double] * 3
        L.orc_tau_membrane.restype = C.c_double
        L.orc_tau_membrane.argtypes = [C.c_double] * 5
        L.orc_vk_operator.restype = C.c_double
        L.orc_vk_operator.argtypes = [C.c_double] * 6
        L.orc_H_quadrature.restype = C.c_double
        L.orc_H_quadrature.argtypes = [C.c_double, C.c_double] + [C.c_int] * 7 + [_dp, _dp]
        L.orc_C_quadrature.restype = C.c_double
        L.orc_C_quadrature.argtypes = [C.c_double, C.c_double] + [C.c_int] * 7 + [_dp, _dp]
        L.orc_H_closed_entry.restype = C.c_double
        L.orc_H_closed_entry.argtypes = [C.c_double, C.c_double] + [C.c_int] * 6
        L.orc_tension_S.restype = C.c_double
        L.orc_potential_nl.restype = C.c_double
        L.orc_potential_nl.argtypes = [C.c_int, C.c_int, C.c_int, _dp, _dp, _dp, _dp]
        L.orc_simulate.argtypes = [C.POINTER(_SimArgs)]
        L.orc_simulate.restype = C.c_int
        L.orc_energy.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, C.c_double,
                                 _dp, _dp, _dp, _dp, _dp, _dp]
        L.orc_energy.restype = None
    return _lib


def _d(a):
    """contiguous fp64 view + ctypes pointer (None -> NULL)."""
    if a is None:
        return None, None
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(_dp)


def _i(a):
    a = np.ascontiguousarray(a, dtype=np.int32)
    return a, a.ctypes.data_as(_ip)


def num_threads() -> int:
    return int(lib().orc_num_threads())


# ---------------------------------------------------------------- bases ----
def string_lambda(L: float, N: int) -> np.ndarray:
    out = np.empty(N)
    lib().orc_string_lambda(C.c_double(L), C.c_int(N), out.ctypes.data_as(_dp))
    return out


def string_mode(m: int, L: float, x: float) -> float:
    return lib().orc_string_mode(m, L, x)


def rect_modes(Lx: float, Ly: float, N: int):
    m = np.empty(N, np.int32); n = np.empty(N, np.int32); lam = np.empty(N)
    rc = lib().orc_rect_modes(C.c_double(Lx), C.c_double(Ly), C.c_int(N),
                              m.ctypes.data_as(_ip), n.ctypes.data_as(_ip), lam.ctypes.data_as(_dp))
    assert rc == 0
    return m, n, lam


def rect_mode(m: int, n: int, Lx: float, Ly: float, x: float, y: float) -> float:
    return lib().orc_rect_mode(int(m), int(n), Lx, Ly, x, y)


def rect_lambda(m, n, Lx, Ly) -> np.ndarray:
    """lambda for a GIVEN index set on another geometry (reading R14: index sets fixed)."""
    m = np.asarray(m, np.float64); n = np.asarray(n, np.float64)
    return (m * np.pi / Lx) ** 2 + (n * np.pi / Ly) ** 2


def omega_gamma(lam, D, T0, rho_m, sigma0, sigma1):
    lam, lp = _d(lam)
    om = np.empty_like(lam); ga = np.empty_like(lam)
    lib().orc_omega_gamma(C.c_int(lam.size), lp, C.c_double(D), C.c_double(T0), C.c_double(rho_m),
                          C.c_double(sigma0), C.c_double(sigma1),
                          om.ctypes.data_as(_dp), ga.ctypes.data_as(_dp))
    return om, ga


def tau_string(E, A, L):
    return lib().orc_tau_string(E, A, L)


def tau_membrane(E, h, Lx, Ly, nu):
    return lib().orc_tau_membrane(E, h, Lx, Ly, nu)


def plate_D(E, h, nu):
    """Bending stiffness of a thin plate, D = E h^3 / (12 (1 - nu^2))."""
    return E * h ** 3 / (12.0 * (1.0 - nu * nu))


# ------------------------------------------------------------ couplings ----
def vk_operator(fxx, fyy, fxy, gxx, gyy, gxy):
    return lib().orc_vk_operator(fxx, fyy, fxy, gxx, gyy, gxy)


def H_closed(Lx, Ly, mq, nq, mphi, nphi) -> np.ndarray:
    mq, mqp = _i(mq); nq, nqp = _i(nq); mphi, mpp = _i(mphi); nphi, npp = _i(nphi)
    Nq, Nphi = mq.size, mphi.size
    H = np.empty((Nphi, Nq, Nq))
    lib().orc_H_closed(C.c_double(Lx), C.c_double(Ly), C.c_int(Nq), mqp, nqp,
                       C.c_int(Nphi), mpp, npp, H.ctypes.data_as(_dp))
    return H


def H_closed_entry(Lx, Ly, p, q, n):
    return lib().orc_H_closed_entry(Lx, Ly, int(p[0]), int(p[1]), int(q[0]), int(q[1]), int(n[0]), int(n[1]))


def H_quadrature(Lx, Ly, i, j, k, ng=64):
    xg, wg = np.polynomial.legendre.leggauss(ng)
    xg, xp = _d(xg); wg, wp = _d(wg)
    return lib().orc_H_quadrature(Lx, Ly, int(i[0]), int(i[1]), int(j[0]), int(j[1]),
                                  int(k[0]), int(k[1]), ng, xp, wp)


def C_quadrature(Lx, Ly, s, i, j, ng=64):
    xg, wg = np.polynomial.legendre.leggauss(ng)
    xg, xp = _d(xg); wg, wp = _d(wg)
    return lib().orc_C_quadrature(Lx, Ly, int(s[0]), int(s[1]), int(i[0]), int(i[1]),
                                  int(j[0]), int(j[1]), ng, xp, wp)


# --------------------------------------------------------------- forces ----
def tension_force(lam, c, q):
    lam, lp = _d(lam); q, qp = _d(q)
    f = np.empty_like(q)
    lib().orc_tension_force(C.c_int(q.size), lp, C.c_double(c), qp, f.ctypes.data_as(_dp))
    return f


def vk_G(H, q):
    H, Hp = _d(H); q, qp = _d(q)
    Nphi, Nq = H.shape[0], H.shape[1]
    G = np.empty(Nphi)
    lib().orc_vk_G(C.c_int(Nq), C.c_int(Nphi), Hp, qp, G.ctypes.data_as(_dp))
    return G


def vk_force(H, s, q):
    H, Hp = _d(H); s, sp = _d(s); q, qp = _d(q)
    Nphi, Nq = H.shape[0], H.shape[1]
    f = np.empty(Nq); work = np.empty(Nphi)
    lib().orc_vk_force(C.c_int(Nq), C.c_int(Nphi), Hp, sp, qp,
                       f.ctypes.data_as(_dp), work.ctypes.data_as(_dp))
    return f


def vk_force_naive(Hq, Cc, scale, q):
    Hq, Hp = _d(Hq); Cc, Cp = _d(Cc); scale, sp = _d(scale); q, qp = _d(q)
    Nphi, Nq = Hq.shape[0], Hq.shape[1]
    f = np.empty(Nq)
    lib().orc_vk_force_naive(C.c_int(Nq), C.c_int(Nphi), Hp, Cp, sp, qp, f.ctypes.data_as(_dp))
    return f


def potential_nl(model, lam, nl_scale, H, q):
    q, qp = _d(q)
    lam, lp = _d(lam); nl_scale, sp = _d(np.atleast_1d(nl_scale)); H, Hp = _d(H)
    Nphi = 0 if H is None else H.shape[0]
    return lib().orc_potential_nl(model, q.size, Nphi, lp, sp, Hp, qp)


# -------------------------------------------------------------- schemes ----
def sv_coeffs(omega, gamma, T):
    omega, op = _d(omega); gamma, gp = _d(gamma)
    g = np.empty_like(omega); p = np.empty_like(omega); r = np.empty_like(omega)
    lib().orc_sv_coeffs(C.c_int(omega.size), op, gp, C.c_double(T),
                        g.ctypes.data_as(_dp), p.ctypes.data_as(_dp), r.ctypes.data_as(_dp))
    return g, p, r


def ftm_coeffs(omega, gamma, T):
    omega, op = _d(omega); gamma, gp = _d(gamma)
    a1 = np.empty_like(omega); a2 = np.empty_like(omega); b1 = np.empty_like(omega)
    lib().orc_ftm_coeffs(C.c_int(omega.size), op, gp, C.c_double(T),
                         a1.ctypes.data_as(_dp), a2.ctypes.data_as(_dp), b1.ctypes.data_as(_dp))
    return a1, a2, b1


def simulate(model, c1, c2, c3, w, q0, qm1, n_steps, *, lam=None, nl_scale=None, H=None,
             fext=None, fext_gain=None, want_traj=False, want_final=False):
    """Run the two-step recurrence for every sample.

    c1,c2,c3,w (and lam / nl_scale) are [coeff_batch][Nq] with coeff_batch 1 or batch.
    Returns dict(out[batch][n_steps], first_bad[batch], traj?, q_final?).
    """
    q0 = np.atleast_2d(np.asarray(q0, np.float64))
    batch, Nq = q0.shape
    c1 = np.atleast_2d(np.asarray(c1, np.float64))
    cb = c1.shape[0]
    assert cb in (1, batch)
    a = _SimArgs()
    keep = []

    def put(name, arr, shape=None):
        if arr is None:
            setattr(a, name, None)
            return None
        arr = np.ascontiguousarray(arr, np.float64)
        if shape is not None:
            assert arr.size == int(np.prod(shape)), (name, arr.shape, shape)
        keep.append(arr)
        setattr(a, name, arr.ctypes.data_as(_dp))
        return arr

    Nphi = 0 if H is None else int(np.asarray(H).shape[0])
    a.model, a.Nq, a.Nphi, a.batch, a.n_steps, a.coeff_batch = model, Nq, Nphi, batch, n_steps, cb
    put("c1", c1, (cb, Nq)); put("c2", c2, (cb, Nq)); put("c3", c3, (cb, Nq)); put("w", w, (cb, Nq))
    put("lambda_", lam, (cb, Nq) if lam is not None else None)
    if model == VK:
        put("nl_scale", nl_scale, (cb, Nphi))
    elif model == TENSION:
        put("nl_scale", np.atleast_1d(nl_scale), (cb,))
    else:
        a.nl_scale = None
    put("H", H)
    put("q0", q0, (batch, Nq)); put("qm1", qm1, (batch, Nq))
    put("fext", fext, (batch, n_steps) if fext is not None else None)
    put("fext_gain", fext_gain, (batch, Nq) if fext_gain is not None else None)
    out = np.empty((batch, n_steps)); keep.append(out); a.out = out.ctypes.data_as(_dp)
    fb = np.empty(batch, np.int32); a.first_bad = fb.ctypes.data_as(_ip)
    traj = qf = None
    if want_traj:
        traj = np.empty((batch, n_steps, Nq)); a.traj = traj.ctypes.data_as(_dp)
    if want_final:
        qf = np.empty((batch, 2, Nq)); a.q_final = qf.ctypes.data_as(_dp)
    lib().orc_simulate(C.byref(a))
    return {"out": out, "first_bad": fb, "traj": traj, "q_final": qf}


def energy(model, T, omega, traj, *, lam=None, nl_scale=None, H=None):
    """Discrete energy h^{n+1/2} of ONE sample's trajectory [n_steps][Nq] (reading R12)."""
    traj, tp = _d(traj); omega, op = _d(omega)
    n_steps, Nq = traj.shape
    lam, lp = _d(lam); H, Hp = _d(H)
    nl_scale, sp = _d(None if nl_scale is None else np.atleast_1d(nl_scale))
    Nphi = 0 if H is None else H.shape[0]
    e = np.empty(n_steps - 1)
    lib().orc_energy(model, Nq, Nphi, n_steps, C.c_double(T), op, lp, sp, Hp, tp, e.ctypes.data_as(_dp))
    return e


# ------------------------------------------------- excitation projection ----
def project_bump_rect(m, n, Lx, Ly, x0, y0, W, A, nr=96, nth=256):
    """q_k^0 = int_S w0 Phi_k dS for the raised-cosine bump (reading R13)
    w0 = (A/2)(1 + cos(2 pi r / W)) for r < W/2, r = |(x,y) - (x0,y0)|, else 0.
    Polar quadrature on the disc: Gauss-Legendre in r, trapezoid in theta."""
    xr, wr = np.polynomial.legendre.leggauss(nr)
    r = 0.25 * W * (xr + 1.0); wr = 0.25 * W * wr
    th = 2.0 * np.pi * np.arange(nth) / nth
    X = x0 + r[:, None] * np.cos(th)[None, :]
    Y = y0 + r[:, None] * np.sin(th)[None, :]
    w0 = 0.5 * A * (1.0 + np.cos(2.0 * np.pi * r / W))
    wt = (wr * r * w0)[:, None] * (2.0 * np.pi / nth)
    q = np.empty(len(m))
    c = 2.0 / np.sqrt(Lx * Ly)
    for k in range(len(m)):
        phi = c * np.sin(m[k] * np.pi * X / Lx) * np.sin(n[k] * np.pi * Y / Ly)
        q[k] = np.sum(wt * phi)
    return q


def project_bump_string(N, L, x0, W, A, ng=256):
    """1-D raised-cosine pluck w0 = (A/2)(1 + cos(2 pi (x-x0)/W)), |x-x0| < W/2."""
    xg, wg = np.polynomial.legendre.leggauss(ng)
    x = x0 + 0.5 * W * xg; wq = 0.5 * W * wg
    w0 = 0.5 * A * (1.0 + np.cos(2.0 * np.pi * (x - x0) / W))
    mm = np.arange(1, N + 1)
    phi = np.sqrt(2.0 / L) * np.sin(mm[:, None] * np.pi * x[None, :] / L)
    return phi @ (wq * w0)


# ------------------------------------------------------ case assembly ------
SV, FTM = 0, 1


@dataclass
class Case:
    """Everything orc_simulate needs for a set of samples, plus by-products."""
    model: int
    scheme: int
    T: float
    Nq: int
    Nphi: int
    omega: np.ndarray          # [B][Nq]
    gamma: np.ndarray          # [B][Nq]
    active: np.ndarray         # [B][Nq] bool (reading R11)
    c1: np.ndarray; c2: np.ndarray; c3: np.ndarray      # [B][Nq]
    w: np.ndarray              # [B][Nq] pickup weights (0 on masked modes)
    lam: np.ndarray            # [B][Nq]
    nl_scale: np.ndarray       # VK [B][Nphi]; TENSION [B]
    H: np.ndarray | None       # [Nphi][Nq][Nq] shared
    q0: np.ndarray             # [B][Nq]
    qm1: np.ndarray            # [B][Nq]
    extra: dict = field(default_factory=dict)


def f32(x):
    """Round to fp32 and widen back: the values the GPU stores (harness rule)."""
    return np.asarray(x, np.float64).astype(np.float32).astype(np.float64)


def scheme_coeffs(scheme, omega, gamma, T, active=None):
    """(c1, c2, c3) of q+ = c1 q + c2 q- + c3 (fext - f): SV (g, p, r) or FTM (-a1, -a2, b1) (reading R7).
    The FTM coefficients exist for underdamped modes only ("overdamped mode -> error naming
    the mode"): an active mode with omega <= gamma is refused."""
    if scheme == SV:
        return sv_coeffs(omega, gamma, T)
    bad = np.asarray(omega) <= np.asarray(gamma)
    if active is not None:
        bad = bad & np.asarray(active, bool)
    if np.any(bad):
        raise ValueError(f"FTM scheme: mode {int(np.argmax(bad))} is critically damped or overdamped (omega <= gamma)")
    a1, a2, b1 = ftm_coeffs(omega, gamma, T)
    return -a1, -a2, b1


def active_mask(scheme, omega, gamma, T):
    """Reading R11: SV modes with omega T >= 1.9 and FTM modes with w~ >= 0.95 pi / T are inactive."""
    if scheme == SV:
        return omega * T < 1.9
    wt = np.sqrt(np.maximum(omega ** 2 - gamma ** 2, 0.0))
    return wt < 0.95 * np.pi / T


def start_state(model, q0, omega, T, *, lam=None, nl_scale=None, H=None):
    """Reading R8: zero initial velocity, q^{-1} = q^0 + (T^2/2)(-omega^2 q^0 - f_nl(q^0))."""
    if model == VK:
        f = vk_force(H, nl_scale, q0)
    elif model == TENSION:
        f = tension_force(lam, float(nl_scale), q0)
    else:
        f = np.zeros_like(q0)
    return q0 + 0.5 * T * T * (-(omega ** 2) * q0 - f)


def assemble(wl: dict, samples=None, *, scheme=SV, lossless=False, round_fp32=True) -> Case:
    """Build the oracle's inputs for workload dict ``wl`` (see workloads.py) for the given
    sample indices.  ``round_fp32``: arrays the GPU keeps in fp32 (H, s_n, w, lambda,
    tau/rho) are rounded to fp32 first so both sides see identical values."""
    B = wl["batch"]
    samples = list(range(B)) if samples is None else list(samples)
    T = 1.0 / wl["sample_rate"]
    Nq = wl["n_q"]
    rnd = f32 if round_fp32 else (lambda x: np.asarray(x, np.float64))
    s0 = 0.0 if lossless else wl["sigma0"]
    s1 = 0.0 if lossless else wl["sigma1"]
    rows = {k: [] for k in ("omega", "gamma", "active", "c1", "c2", "c3", "w", "lam", "nl", "q0", "qm1")}
    H = None
    if wl["model"] == "vk":
        model, Nphi = VK, wl["n_phi"]
        ref = wl["ref"]
        mq, nq, _ = rect_modes(ref["Lx"], ref["Ly"], Nq)            # index sets: reference geometry
        mphi, nphi, _ = rect_modes(ref["Lx"], ref["Ly"], Nphi)      # reading R5
        ritz = wl.get("airy", "sine") == "ritz"                      # reading R16 instead of R5 (workload key, default sine)
        if ritz:
            z4_ref, c_airy = airy_ritz_basis(ref["Lx"], ref["Ly"], Nphi, n_trial=wl["n_trial"])
            H = rnd(H_airy_ritz(ref["Lx"], ref["Ly"], mq, nq, c_airy))
        else:
            H = rnd(H_closed(ref["Lx"], ref["Ly"], mq, nq, mphi, nphi))
        c_ref = (ref["Lx"] * ref["Ly"]) ** -2.5
        for b in samples:
            Lx, Ly, h = wl["Lx"][b], wl["Ly"][b], wl["h"][b]
            lam = rect_lambda(mq, nq, Lx, Ly)
            om, ga = omega_gamma(lam, plate_D(wl["E"], h, wl["nu"]), wl["T0"], wl["rho"] * h, s0, s1)
            act = active_mask(scheme, om, ga, T)
            if ritz:
                # the Ritz modes keep their shape only at the reference aspect ratio, where zeta^4 ~ L^-4
                assert abs(Ly / Lx - ref["Ly"] / ref["Lx"]) < 1e-12, "reading R16: per-sample geometry at the reference aspect ratio only"
                zeta4 = z4_ref * (ref["Lx"] / Lx) ** 4
            else:
                zeta4 = rect_lambda(mphi, nphi, Lx, Ly) ** 2            # zeta_n^4 = lambda_n^2 (R5)
            c_b = (Lx * Ly) ** -2.5
            s = rnd(wl["E"] / (2.0 * wl["rho"] * zeta4) * (c_b / c_ref) ** 2)   # reading R14
            xp, yp = wl["pickup"][0] * Lx, wl["pickup"][1] * Ly
            w = np.array([rect_mode(mq[k], nq[k], Lx, Ly, xp, yp) for k in range(Nq)])
            w = rnd(np.where(act, w, 0.0))
            q0 = project_bump_rect(mq, nq, Lx, Ly, wl["x0"][b], wl["y0"][b], wl["W"][b], wl["A"][b])
            q0 = np.where(act, q0, 0.0)
            c1, c2, c3 = scheme_coeffs(scheme, om, ga, T, act)
            c3 = np.where(act, c3, 0.0)
            qm1 = np.where(act, start_state(VK, q0, om, T, nl_scale=s, H=H), 0.0)
            for k, v in zip(rows, (om, ga, act, c1, c2, c3, w, lam, s, q0, qm1)):
                rows[k].append(v)
        extra = {"mq": mq, "nq": nq, "mphi": mphi, "nphi": nphi}
    elif wl["model"] == "berger":
        # Berger plate: tension modulation (Eq. 8) on the rectangular sine basis with
        # tau_membrane of PAPER.md:85 (Eq. 4), per unit mass rho h (reading R3)
        model, Nphi = TENSION, 0
        ref = wl["ref"]
        mq, nq, _ = rect_modes(ref["Lx"], ref["Ly"], Nq)
        for b in samples:
            Lx, Ly, h = wl["Lx"][b], wl["Ly"][b], wl["h"][b]
            lam = rect_lambda(mq, nq, Lx, Ly)
            om, ga = omega_gamma(lam, plate_D(wl["E"], h, wl["nu"]), wl["T0"], wl["rho"] * h, s0, s1)
            act = active_mask(scheme, om, ga, T)
            c = float(rnd(tau_membrane(wl["E"], h, Lx, Ly, wl["nu"]) / (wl["rho"] * h)))
            lam_r = rnd(lam)
            xp, yp = wl["pickup"][0] * Lx, wl["pickup"][1] * Ly
            w = np.array([rect_mode(mq[k], nq[k], Lx, Ly, xp, yp) for k in range(Nq)])
            w = rnd(np.where(act, w, 0.0))
            q0 = project_bump_rect(mq, nq, Lx, Ly, wl["x0"][b], wl["y0"][b], wl["W"][b], wl["A"][b])
            q0 = np.where(act, q0, 0.0)
            c1, c2, c3 = scheme_coeffs(scheme, om, ga, T, act)
            c3 = np.where(act, c3, 0.0)
            qm1 = np.where(act, start_state(TENSION, q0, om, T, lam=lam_r, nl_scale=c), 0.0)
            for k, v in zip(rows, (om, ga, act, c1, c2, c3, w, lam_r, c, q0, qm1)):
                rows[k].append(v)
        extra = {"mq": mq, "nq": nq}
    else:
        model = TENSION if wl["model"] == "tension" else LINEAR
        Nphi = 0
        for b in samples:
            L = wl["L"][b]
            lam = string_lambda(L, Nq)
            om, ga = omega_gamma(lam, wl["D"][b], wl["T0s"][b], wl["rho_lin"][b], s0, s1)
            act = active_mask(scheme, om, ga, T)
            tau = tau_string(wl["E"], wl["area"][b], L)
            c = float(rnd(tau / wl["rho_lin"][b])) if model == TENSION else 0.0
            lam_r = rnd(lam)
            xp = wl["pickup"][0] * L
            w = np.array([string_mode(m, L, xp) for m in range(1, Nq + 1)])
            w = rnd(np.where(act, w, 0.0))
            q0 = np.where(act, project_bump_string(Nq, L, wl["x0"][b], wl["W"][b], wl["A"][b]), 0.0)
            c1, c2, c3 = scheme_coeffs(scheme, om, ga, T, act)
            c3 = np.where(act, c3, 0.0)
            qm1 = np.where(act, start_state(model, q0, om, T, lam=lam_r, nl_scale=c), 0.0)
            for k, v in zip(rows, (om, ga, act, c1, c2, c3, w, lam_r, c, q0, qm1)):
                rows[k].append(v)
        extra = {}
    A = {k: np.array(v) for k, v in rows.items()}
    return Case(model=model, scheme=scheme, T=T, Nq=Nq, Nphi=Nphi, omega=A["omega"], gamma=A["gamma"],
                active=A["active"], c1=A["c1"], c2=A["c2"], c3=A["c3"], w=A["w"], lam=A["lam"],
                nl_scale=A["nl"], H=H, q0=A["q0"], qm1=A["qm1"], extra=extra)


def run_case(case: Case, n_steps: int, **kw):
    return simulate(case.model, case.c1, case.c2, case.c3, case.w, case.q0, case.qm1, n_steps,
                    lam=case.lam if case.model == TENSION else None,
                    nl_scale=case.nl_scale if case.model != LINEAR else None,
                    H=case.H, **kw)


# ------------------------------------------------------- in-plane basis, reading B ----
# PAPER.md:53, 123 say the in-plane (Airy) eigenfunctions Psi_n and eigenvalues zeta_n^4 come from "a separate
# eigendecomposition of the Airy stress function" by "a Galerkin type approach" and give no formula.  For a plate whose edges
# are free to move in the plane the Airy function obeys Psi = dPsi/dn = 0 on the boundary, i.e. the CLAMPED-plate problem
#     Lap Lap Psi = zeta^4 Psi,   Psi = dPsi/dn = 0 on the edges                       (reading R16)
# which has no closed form.  Rayleigh-Ritz on the trial space  T_i(x / Lx) T_j(y / Ly),  T_i(s) = sin(pi s) sin(i pi s),
# i, j = 1 .. n_trial  (every T_i and its slope vanish at s = 0 and 1):
#     K c = zeta^4 M c,   K = int (Lap u)(Lap v) dS,   M = int u v dS.
# This oracle does every integral by Gauss-Legendre QUADRATURE and the eigenproblem with scipy.linalg.eigh; the library uses
# closed-form integrals and its own eigensolver (csrc/host_math.hpp), so comparing the two is a real cross-check.
def _ritz_trial(n_trial, s):
    """T_i(s), T_i'(s), T_i''(s) for i = 1..n_trial at the points s (unit interval)."""
    i = np.arange(1, n_trial + 1)[:, None]
    a, b = np.sin(np.pi * s)[None, :], np.sin(i * np.pi * s)
    da, db = np.pi * np.cos(np.pi * s)[None, :], i * np.pi * np.cos(i * np.pi * s)
    dda, ddb = -np.pi ** 2 * a, -(i * np.pi) ** 2 * b
    return a * b, da * b + a * db, dda * b + 2 * da * db + a * ddb


def airy_ritz_basis(Lx, Ly, n_phi, n_trial=12, ng=160):
    """The n_phi lowest clamped-plate (Airy) modes on [0, Lx] x [0, Ly]: zeta4 [n_phi] ascending and coefficients
    c [n_phi][n_trial][n_trial] with Psi_n(x, y) = sum_ij c[n, i, j] T_i(x / Lx) T_j(y / Ly), unit L2 norm, sign fixed by
    making the largest coefficient positive.  All integrals by ng-point Gauss-Legendre quadrature."""
    from scipy.linalg import eigh
    xg, wg = np.polynomial.legendre.leggauss(ng)
    s, w = 0.5 * (xg + 1.0), 0.5 * wg
    T, dT, ddT = _ritz_trial(n_trial, s)
    A0, A1, A2 = (T * w) @ T.T, (dT * w) @ dT.T, (ddT * w) @ ddT.T       # int T_i T_j, T_i' T_j', T_i'' T_j'' on the unit interval
    # int (u_xx + u_yy)(v_xx + v_yy) with int u_xx v_yy = int u_xy v_xy for clamped trial functions (two integrations by parts)
    M = Lx * Ly * np.kron(A0, A0)
    K = Lx * Ly * (np.kron(A2, A0) / Lx ** 4 + 2.0 * np.kron(A1, A1) / (Lx * Ly) ** 2 + np.kron(A0, A2) / Ly ** 4)
    lam, vec = eigh(K, M)
    zeta4 = lam[:n_phi]
    c = vec[:, :n_phi].T.reshape(n_phi, n_trial, n_trial).copy()
    for n in range(n_phi):
        k = np.argmax(np.abs(c[n]))
        if c[n].flat[k] < 0:
            c[n] = -c[n]
    return zeta4, c


def airy_ritz_eval(c, Lx, Ly, x, y):
    """Psi_n(x, y) for every n (c from airy_ritz_basis)."""
    nt = c.shape[1]
    Tx = _ritz_trial(nt, np.atleast_1d(x / Lx))[0][:, 0]
    Ty = _ritz_trial(nt, np.atleast_1d(y / Ly))[0][:, 0]
    return np.einsum("nij,i,j->n", c, Tx, Ty)


def H_airy_ritz(Lx, Ly, mq, nq, c, ng=200):
    """H^n_pq = int Psi_n L(Phi_p, Phi_q) dS (Eq. 10, operator of Eq. 7) for the sine transverse modes
    (mq, nq) and the Ritz in-plane modes c, by separable Gauss-Legendre quadrature:
        L(Phi_p, Phi_q) = Phi_p,xx Phi_q,yy + Phi_p,yy Phi_q,xx - 2 Phi_p,xy Phi_q,xy."""
    mq = np.asarray(mq, float); nq = np.asarray(nq, float)
    xg, wg = np.polynomial.legendre.leggauss(ng)
    s, w = 0.5 * (xg + 1.0), 0.5 * wg
    nt = c.shape[1]
    T = _ritz_trial(nt, s)[0]                                               # [nt][ng]
    sx, cx = np.sin(np.pi * mq[:, None] * s), np.cos(np.pi * mq[:, None] * s)   # transverse factors on the unit interval
    sy, cy = np.sin(np.pi * nq[:, None] * s), np.cos(np.pi * nq[:, None] * s)
    # 1-D integrals  int T_i sin sin  and  int T_i cos cos   -> [nt][Nq][Nq]
    SSx = np.einsum("ig,pg,qg,g->ipq", T, sx, sx, w); CCx = np.einsum("ig,pg,qg,g->ipq", T, cx, cx, w)
    SSy = np.einsum("jg,pg,qg,g->jpq", T, sy, sy, w); CCy = np.einsum("jg,pg,qg,g->jpq", T, cy, cy, w)
    ax, ay = np.pi * mq / Lx, np.pi * nq / Ly                               # wavenumbers
    # Phi = (2 / sqrt(Lx Ly)) sin sin; dS = Lx Ly ds dt
    pref = 4.0 / (Lx * Ly) * Lx * Ly
    A = (ax[:, None] ** 2) * (ay[None, :] ** 2)                              # Phi_p,xx Phi_q,yy -> a_xp^2 a_yq^2 (signs cancel)
    Bc = (ax * ay)[:, None] * (ax * ay)[None, :]
    H = np.empty((c.shape[0], len(mq), len(mq)))
    for n in range(c.shape[0]):
        Sx = np.einsum("ij,ipq->jpq", c[n], SSx); Cx = np.einsum("ij,ipq->jpq", c[n], CCx)
        t1 = np.einsum("jpq,jpq->pq", Sx, SSy)                              # sum_ij c_ij SSx_i SSy_j
        t2 = np.einsum("jpq,jpq->pq", Cx, CCy)
        H[n] = pref * ((A + A.T) * t1 - 2.0 * Bc * t2)
    return H


# ------------------------------------------- reverse pass ----
def bptt_vk(c1, c2, c3, w, nl_scale, H, q0, qm1, gout):
    """Backpropagation through time of ONE von Karman sample ("gradients ... by backpropagation through
    the time integrator"; the paper uses autodiff, this is the same adjoint written out).

    Forward, as `simulate` (Eq. 19/20, no external force), n = 0 .. N-1, N = len(gout):
        out_n = w . q^n,     q^{n+1} = c1 q^n + c2 q^{n-1} - c3 f(q^n),
        f_k(q) = sum_m s_m G_m t_mk,  t_m = H^m q,  G_m = q . t_m                       (Eq. 9)
    Loss: any L(out) with gout[n] = dL/d out_n.  Adjoint a^n = dL/dq^n (total), a^N = a^{N+1} = 0:
        a^n = w gout_n + c1 a^{n+1} + c2 a^{n+2} - J(q^n)^T (c3 a^{n+1}),
        J_kj = df_k/dq_j = sum_m s_m [ (H^m q + H^mT q)_j t_mk + G_m H^m_kj ]
    Returns dL/d{q0, qm1, c1, c2, c3, w, s (nl_scale), H}; H entries are treated as independent (no symmetry constraint).
    Plain numpy fp64, one einsum per stage and step; small sizes only.
    """
    c1, c2, c3, w, s = (np.asarray(x, np.float64) for x in (c1, c2, c3, w, nl_scale))
    H = np.asarray(H, np.float64); q0 = np.asarray(q0, np.float64); qm1 = np.asarray(qm1, np.float64)
    gout = np.asarray(gout, np.float64)
    N, Nq = gout.shape[0], q0.shape[0]
    # forward, stored
    q = np.empty((N + 1, Nq)); q[0] = q0
    prev = qm1
    for n in range(N):
        t = np.einsum("mkr,r->mk", H, q[n])
        G = t @ q[n]
        f = (s * G) @ t
        q[n + 1] = c1 * q[n] + c2 * prev - c3 * f
        prev = q[n]
    g = {k: np.zeros(Nq) for k in ("c1", "c2", "c3", "w")}
    g["s"] = np.zeros_like(s); g["H"] = np.zeros_like(H)
    a1 = np.zeros(Nq); a2 = np.zeros(Nq)            # a^{n+1}, a^{n+2}
    for n in range(N - 1, -1, -1):
        qn = q[n]; qp = q[n - 1] if n > 0 else qm1
        t = np.einsum("mkr,r->mk", H, qn)           # t_m = H^m q
        tt = np.einsum("mkr,k->mr", H, qn)          # H^mT q
        G = t @ qn
        f = (s * G) @ t
        mu = c3 * a1
        d = t @ mu                                  # t_m . mu
        # J^T mu = sum_m s_m [ (t_m + tt_m) d_m + G_m H^mT mu ]
        JTmu = (s * d) @ (t + tt) + np.einsum("m,mkj,k->j", s * G, H, mu)
        g["c1"] += a1 * qn; g["c2"] += a1 * qp; g["c3"] -= a1 * f
        g["w"] += gout[n] * qn
        g["s"] -= d * G
        g["H"] -= (s * d)[:, None, None] * np.multiply.outer(qn, qn)[None] + (s * G)[:, None, None] * np.multiply.outer(mu, qn)[None]
        a0 = w * gout[n] + c1 * a1 + c2 * a2 - JTmu
        a2, a1 = a1, a0
    g["q0"] = a1                                     # a^0
    g["qm1"] = c2 * a2                               # q^{-1} enters q^1 only: c2 a^1
    return g


def dcoeffs_domega_dgamma(scheme, omega, gamma, T):
    """Partial derivatives of (c1, c2, c3) wrt omega and gamma, for the chain rule to the physical parameters:
    SV (Eq. 21-23): c1 = (2 - w^2 T^2)/(1 + gT), c2 = -(1 - gT)/(1 + gT), c3 = T^2/(1 + gT);
    FTM (reading R7): c1 = 2 e^{-gT} cos(wt T), c2 = -e^{-2gT}, c3 = T e^{-gT} sin(wt T)/wt, wt = sqrt(w^2 - g^2).
    Returns dict d{c1,c2,c3}_d{w,g}."""
    w_, g_ = np.asarray(omega, np.float64), np.asarray(gamma, np.float64)
    if scheme == SV:
        den = 1.0 + g_ * T
        return dict(c1_w=-2 * w_ * T * T / den, c1_g=-(2 - w_ ** 2 * T * T) * T / den ** 2,
                    c2_w=np.zeros_like(w_), c2_g=2 * T / den ** 2,
                    c3_w=np.zeros_like(w_), c3_g=-T ** 3 / den ** 2)
    wt = np.sqrt(w_ ** 2 - g_ ** 2)
    e = np.exp(-g_ * T); sn, cs = np.sin(wt * T), np.cos(wt * T)
    wt_w, wt_g = w_ / wt, -g_ / wt
    dc3_dwt = T * e * (T * cs * wt - sn) / wt ** 2
    return dict(c1_w=-2 * e * sn * T * wt_w, c1_g=-2 * T * e * cs - 2 * e * sn * T * wt_g,
                c2_w=np.zeros_like(w_), c2_g=2 * T * np.exp(-2 * g_ * T),
                c3_w=dc3_dwt * wt_w, c3_g=-T * T * e * sn / wt + dc3_dwt * wt_g)


def bptt_tension(c1, c2, c3, w, lam, c, q0, qm1, gout):
    """Backpropagation through time of ONE tension-modulated sample (Kirchhoff-Carrier string / Berger plate; the paper's
    non-linear string fits): as `bptt_vk` with f_mu = c lam_mu q_mu S, S = sum_nu lam_nu q_nu^2
    (Eq. 8, reading R2).  J_mu,j = c [lam_mu S delta_mu,j + 2 lam_mu q_mu lam_j q_j] (symmetric), so
    J^T mu = c [S lam mu + 2 (sum lam q mu) lam q].  Returns dL/d{q0, qm1, c1, c2, c3, w, c}; numpy fp64."""
    c1, c2, c3, w, lam = (np.asarray(x, np.float64) for x in (c1, c2, c3, w, lam))
    q0 = np.asarray(q0, np.float64); qm1 = np.asarray(qm1, np.float64); gout = np.asarray(gout, np.float64)
    c = float(c)
    N, Nq = gout.shape[0], q0.shape[0]
    q = np.empty((N + 1, Nq)); q[0] = q0
    prev = qm1
    for n in range(N):
        S = float(lam @ (q[n] ** 2))
        q[n + 1] = c1 * q[n] + c2 * prev - c3 * (c * lam * q[n] * S)
        prev = q[n]
    g = {k: np.zeros(Nq) for k in ("c1", "c2", "c3", "w")}
    g["c"] = 0.0
    a1 = np.zeros(Nq); a2 = np.zeros(Nq)
    for n in range(N - 1, -1, -1):
        qn = q[n]; qp = q[n - 1] if n > 0 else qm1
        S = float(lam @ (qn ** 2))
        f = c * lam * qn * S
        mu = c3 * a1
        D = float((lam * qn) @ mu)
        JTmu = c * (S * lam * mu + 2.0 * D * lam * qn)
        g["c1"] += a1 * qn; g["c2"] += a1 * qp; g["c3"] -= a1 * f
        g["w"] += gout[n] * qn
        g["c"] -= D * S
        a0 = w * gout[n] + c1 * a1 + c2 * a2 - JTmu
        a2, a1 = a1, a0
    g["q0"] = a1
    g["qm1"] = c2 * a2
    return g
