"""Thin ctypes binding over libmodal.so (include/modal.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels of the library; this module never
computes.  Importing it loads the library and raises if it is missing -- there is no CPU
fallback.  torch is used only by callers for device buffers and streams.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmodal.so")

OK, EINVAL, EINCOMPAT, EUNSTABLE, ECUDA, ENOMEM = range(6)
LINEAR, TENSION, VK = 0, 1, 2
SV, FTM = 0, 1
STRING, RECT = 0, 1
(Q_MODE_M, Q_MODE_N, Q_PHI_M, Q_PHI_N, Q_LAMBDA, Q_OMEGA, Q_SIGMA, Q_NL_SCALE, Q_PICKUP, Q_ACTIVE,
 Q_H_FULL, Q_COEFF_BATCH, Q_KERNEL_INFO, Q_TILE_STATS, Q_MMA_LAYOUT, Q_MMA_SLAB_CHECK, Q_AIRY_ZETA4, Q_STREAM_LAYOUT, Q_STREAM_CHECK, Q_REPL_CHECK) = range(20)
AIRY_SINE, AIRY_CLAMPED_RITZ = 0, 1

_dp = C.POINTER(C.c_double)
_fp = C.POINTER(C.c_float)
_ip = C.POINTER(C.c_int)


class PlanDesc(C.Structure):
    _fields_ = [("model", C.c_int), ("scheme", C.c_int), ("geom", C.c_int), ("bc", C.c_int),
                ("Lx", C.c_double), ("Ly", C.c_double), ("h", C.c_double),
                ("E", C.c_double), ("rho", C.c_double), ("nu", C.c_double),
                ("T0", C.c_double), ("D", C.c_double), ("area", C.c_double),
                ("sigma0", C.c_double), ("sigma1", C.c_double),
                ("pickup_x", C.c_double), ("pickup_y", C.c_double),
                ("n_q", C.c_int), ("n_phi", C.c_int), ("sample_rate", C.c_double),
                ("max_batch", C.c_int), ("max_steps", C.c_int)]


class Coeffs(C.Structure):
    _fields_ = [("coeff_batch", C.c_int), ("omega", _dp), ("sigma", _dp), ("nl_scale", _dp),
                ("lambda_", _dp), ("pickup", _dp), ("H_full", _dp)]


class Init(C.Structure):
    _fields_ = [("q0", _dp), ("qm1", _dp), ("fext_signal", C.c_void_p), ("fext_gain", _dp),
                ("traj_dev", C.c_void_p)]


class BpttArgs(C.Structure):
    _fields_ = [("qm1", _dp), ("traj_dev", C.c_void_p), ("gout_dev", C.c_void_p)] + [(n, _dp) for n in (
        "grad_q0", "grad_qm1", "grad_omega", "grad_sigma", "grad_c1", "grad_c2", "grad_c3", "grad_pickup", "grad_nl_scale", "grad_H")]


class SampleGeom(C.Structure):
    _fields_ = [("Lx", C.c_double), ("Ly", C.c_double), ("h", C.c_double), ("T0", C.c_double),
                ("D", C.c_double), ("rho", C.c_double), ("area", C.c_double),
                ("pickup_x_frac", C.c_double), ("pickup_y_frac", C.c_double)]


EXPORTS = ["modal_plan_create", "modal_coeffs_upload", "modal_simulate", "modal_simulate_host",
           "modal_plan_check", "modal_plan_set_option", "modal_plan_set_airy_basis", "modal_plan_destroy", "modal_last_error",
           "modal_plan_query", "modal_derive_coeffs", "modal_project_bump", "modal_measure_peaks", "modal_vk_simulate_static", "modal_bptt"]

if not os.path.exists(LIB_PATH):
    raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2505_05940_b200.build` "
                      "(there is no CPU fallback)")
lib = C.CDLL(LIB_PATH)
lib.modal_plan_create.argtypes = [C.POINTER(PlanDesc), C.c_int, C.POINTER(C.c_void_p)]
lib.modal_coeffs_upload.argtypes = [C.c_void_p, C.POINTER(Coeffs)]
lib.modal_simulate.argtypes = [C.c_void_p, C.c_int, C.c_int, C.POINTER(Init), C.c_void_p, _ip, C.c_void_p]
lib.modal_simulate_host.argtypes = [C.c_void_p, C.c_int, C.c_int, C.POINTER(Init), _fp, _ip]
lib.modal_plan_check.argtypes = [C.c_void_p, _ip]
lib.modal_bptt.argtypes = [C.c_void_p, C.c_int, C.c_int, C.POINTER(BpttArgs), C.c_void_p]
lib.modal_plan_set_option.argtypes = [C.c_void_p, C.c_char_p, C.c_int]
lib.modal_plan_set_airy_basis.argtypes = [C.c_void_p, C.c_int, C.c_int]
lib.modal_plan_destroy.argtypes = [C.c_void_p]
lib.modal_plan_destroy.restype = None
lib.modal_last_error.argtypes = [C.c_void_p]
lib.modal_last_error.restype = C.c_char_p
lib.modal_plan_query.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_ulonglong]
lib.modal_derive_coeffs.argtypes = [C.c_void_p, C.POINTER(SampleGeom), _dp, _dp, _dp, _dp, _dp]
lib.modal_project_bump.argtypes = [C.c_void_p] + [C.c_double] * 6 + [_dp]


class Peaks(C.Structure):
    _fields_ = [(n, C.c_double) for n in (
        "sm_clock_mhz", "fp32_tflops", "fp64_tflops", "l2_read_gbs_8mb", "l2_read_gbs_64mb", "hbm_read_gbs", "smem_read_gbs",
        "smem_bytes_per_clk_sm", "tmem_read_bytes_per_clk_sm", "hop_cycles_idle", "hop_cycles_loaded",
        "relacq_hop_cycles_idle", "relacq_hop_cycles_loaded")]


lib.modal_measure_peaks.argtypes = [C.c_int, C.POINTER(Peaks)]
lib.modal_vk_simulate_static.argtypes = [C.c_int] * 5 + [C.c_void_p] * 11 + [C.c_char_p, C.c_int]
STATIC_MAX_NQ, STATIC_SCRATCH_BYTES = 256, 1 << 20


def vk_simulate_static(n_q, n_phi, batch, n_steps, coeff_batch, H, c1, c2, c3, s, w, q0, qm1, out, first_bad=0, stream=0):
    """modal_vk_simulate_static: every array argument is a DEVICE address (int); nothing is allocated, nothing synchronised."""
    err = C.create_string_buffer(512)
    st = lib.modal_vk_simulate_static(n_q, n_phi, batch, n_steps, coeff_batch, H, c1, c2, c3, s, w, q0, qm1, out,
                                      first_bad or None, stream or None, err, 512)
    if st != OK:
        raise ModalError(st, err.value.decode())
    return st


def measure_peaks(device: int = 0) -> dict:
    """modal_measure_peaks: FP32 / FP64 FMA, L2 / HBM / shared-memory / TMEM read bandwidth, exchange-hop latencies."""
    pk = Peaks()
    st = lib.modal_measure_peaks(device, C.byref(pk))
    if st != OK:
        raise RuntimeError(f"modal_measure_peaks: status {st}")
    return {n: getattr(pk, n) for n, _ in Peaks._fields_}


class ModalError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"modal status {status}: {msg}")
        self.status = status
        self.message = msg


def _arr(a, dtype=np.float64):
    return None if a is None else np.ascontiguousarray(a, dtype=dtype)


def _ptr(a, t=_dp):
    return None if a is None else a.ctypes.data_as(t)


class Plan:
    """modal_plan_create / modal_coeffs_upload / modal_simulate / modal_plan_destroy."""

    def __init__(self, desc: PlanDesc, device: int = 0):
        self.desc = desc
        self._h = C.c_void_p()
        st = lib.modal_plan_create(C.byref(desc), device, C.byref(self._h))
        if st != OK:
            raise ModalError(st, lib.modal_last_error(None).decode())
        self.n_q, self.n_phi = desc.n_q, desc.n_phi

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            lib.modal_plan_destroy(self._h)
            self._h = C.c_void_p()

    __del__ = close

    def last_error(self) -> str:
        return lib.modal_last_error(self._h).decode()

    def _check(self, st, allow=()):
        if st != OK and st not in allow:
            raise ModalError(st, self.last_error())
        return st

    def coeffs_upload(self, coeff_batch=1, omega=None, sigma=None, nl_scale=None, lam=None,
                      pickup=None, H_full=None):
        keep = [_arr(x) for x in (omega, sigma, nl_scale, lam, pickup, H_full)]
        c = Coeffs(coeff_batch, *[_ptr(k) for k in keep])
        return self._check(lib.modal_coeffs_upload(self._h, C.byref(c)))

    def simulate(self, q0, n_steps, out_dev_ptr: int, qm1=None, first_bad=True, stream: int = 0,
                 fext_dev_ptr: int = 0, fext_gain=None, traj_dev_ptr: int = 0):
        """out_dev_ptr: device address of a [batch][n_steps] fp32 buffer (e.g. tensor.data_ptr()).
        Returns (status, first_bad or None)."""
        q0 = _arr(np.atleast_2d(q0)); qm1 = None if qm1 is None else _arr(np.atleast_2d(qm1))
        g = _arr(fext_gain)
        batch = q0.shape[0]
        init = Init(_ptr(q0), _ptr(qm1), fext_dev_ptr or None, _ptr(g), traj_dev_ptr or None)
        fb = np.empty(batch, np.int32) if first_bad else None
        st = lib.modal_simulate(self._h, batch, n_steps, C.byref(init), C.c_void_p(out_dev_ptr),
                                _ptr(fb, _ip), C.c_void_p(stream))
        self._check(st, allow=(EUNSTABLE,))
        return st, fb

    def check(self, batch=None):
        """modal_plan_check: completes the last (asynchronous) simulate.  Returns (status, first_bad or None)."""
        fb = None if batch is None else np.empty(batch, np.int32)
        st = lib.modal_plan_check(self._h, _ptr(fb, _ip))
        self._check(st, allow=(EUNSTABLE,))
        return st, fb

    def bptt(self, qm1, n_steps, traj_dev_ptr, gout_dev_ptr, want_H=False, stream=0):
        """modal_bptt: gradients of a loss on the audio (gout = dL/d out, device) through the stored trajectory (device)."""
        qm1 = _arr(np.atleast_2d(qm1))
        B = qm1.shape[0]
        g = {n: np.zeros((B, self.n_q)) for n in ("q0", "qm1", "omega", "sigma", "c1", "c2", "c3", "pickup")}
        g["nl_scale"] = np.zeros((B, max(self.n_phi, 1)))            # tension / linear plans: one scale per sample
        if want_H and self.n_phi > 0:
            g["H"] = np.zeros((self.n_phi, self.n_q, self.n_q))
        a = BpttArgs(_ptr(qm1, _dp), traj_dev_ptr, gout_dev_ptr, *[_ptr(g[n], _dp) for n in ("q0", "qm1", "omega", "sigma", "c1", "c2", "c3", "pickup", "nl_scale")],
                     _ptr(g.get("H"), _dp))
        self._check(lib.modal_bptt(self._h, B, int(n_steps), C.byref(a), stream or None))
        return g

    def set_airy_basis(self, basis: int, n_trial: int = 0):
        return self._check(lib.modal_plan_set_airy_basis(self._h, int(basis), int(n_trial)))

    def set_option(self, key: str, value: int):
        return self._check(lib.modal_plan_set_option(self._h, key.encode(), int(value)))

    def simulate_host(self, q0, n_steps, qm1=None, out=None):
        q0 = _arr(np.atleast_2d(q0)); qm1 = None if qm1 is None else _arr(np.atleast_2d(qm1))
        batch = q0.shape[0]
        if out is None:
            out = np.empty((batch, n_steps), np.float32)
        init = Init(_ptr(q0), _ptr(qm1), None, None, None)
        fb = np.empty(batch, np.int32)
        st = lib.modal_simulate_host(self._h, batch, n_steps, C.byref(init), _ptr(out, _fp), _ptr(fb, _ip))
        self._check(st, allow=(EUNSTABLE,))
        return out, fb, st

    def query(self, what):
        nq, nphi = self.n_q, self.n_phi
        cb = np.zeros(1, np.int32)
        lib.modal_plan_query(self._h, Q_COEFF_BATCH, cb.ctypes.data_as(C.c_void_p), 4)
        cb = int(cb[0])
        nnl = nphi if self.desc.model == VK else 1
        shape, dt = {
            Q_MODE_M: ((nq,), np.int32), Q_MODE_N: ((nq,), np.int32),
            Q_PHI_M: ((nphi,), np.int32), Q_PHI_N: ((nphi,), np.int32),
            Q_LAMBDA: ((nq,), np.float64), Q_OMEGA: ((cb, nq), np.float64), Q_SIGMA: ((cb, nq), np.float64),
            Q_NL_SCALE: ((cb, nnl), np.float64), Q_PICKUP: ((cb, nq), np.float64),
            Q_ACTIVE: ((cb, nq), np.int32), Q_H_FULL: ((nphi, nq, nq), np.float64),
            Q_COEFF_BATCH: ((1,), np.int32), Q_KERNEL_INFO: ((8,), np.int32), Q_TILE_STATS: ((2,), np.int32),
            Q_MMA_LAYOUT: ((16,), np.int32), Q_MMA_SLAB_CHECK: ((3,), np.float64),
            Q_AIRY_ZETA4: ((nphi,), np.float64), Q_STREAM_LAYOUT: ((16,), np.int32), Q_STREAM_CHECK: ((4,), np.float64),
            Q_REPL_CHECK: ((8,), np.float64)}[what]
        a = np.zeros(shape, dt)
        self._check(lib.modal_plan_query(self._h, what, a.ctypes.data_as(C.c_void_p), a.nbytes))
        return a

    def derive_coeffs(self, **geom):
        g = SampleGeom(**geom)
        nq = self.n_q
        nnl = self.n_phi if self.desc.model == VK else 1
        om, sg, lam, pk = (np.empty(nq) for _ in range(4))
        nl = np.empty(nnl)
        self._check(lib.modal_derive_coeffs(self._h, C.byref(g), _ptr(om), _ptr(sg), _ptr(nl), _ptr(lam), _ptr(pk)))
        return dict(omega=om, sigma=sg, nl_scale=nl, lam=lam, pickup=pk)

    def project_bump(self, Lx, Ly, x0, y0, W, A):
        q0 = np.empty(self.n_q)
        self._check(lib.modal_project_bump(self._h, Lx, Ly, x0, y0, W, A, _ptr(q0)))
        return q0


# ---------------------------------------------------------------------------------------
# Workload -> plan + inputs, using only the library's own host helpers (no oracle).
# ---------------------------------------------------------------------------------------
def desc_from_workload(wl: dict, scheme=SV, lossless=False, max_batch=None, max_steps=None) -> PlanDesc:
    s0 = 0.0 if lossless else wl["sigma0"]
    s1 = 0.0 if lossless else wl["sigma1"]
    if wl["model"] in ("vk", "berger"):
        ref = wl["ref"]
        return PlanDesc(model=VK if wl["model"] == "vk" else TENSION, scheme=scheme, geom=RECT, bc=0, Lx=ref["Lx"], Ly=ref["Ly"], h=ref["h"],
                        E=wl["E"], rho=wl["rho"], nu=wl["nu"], T0=wl["T0"], D=0.0, area=0.0,
                        sigma0=s0, sigma1=s1, pickup_x=wl["pickup"][0] * ref["Lx"], pickup_y=wl["pickup"][1] * ref["Ly"],
                        n_q=wl["n_q"], n_phi=wl["n_phi"], sample_rate=wl["sample_rate"],
                        max_batch=max_batch or wl["batch"], max_steps=max_steps or wl["n_steps"])
    model = TENSION if wl["model"] == "tension" else LINEAR
    return PlanDesc(model=model, scheme=scheme, geom=STRING, bc=0, Lx=float(wl["L"][0]), Ly=0.0, h=0.0,
                    E=wl["E"], rho=float(wl["rho_lin"][0]), nu=0.0, T0=float(wl["T0s"][0]), D=float(wl["D"][0]),
                    area=float(wl["area"][0]), sigma0=s0, sigma1=s1, pickup_x=wl["pickup"][0] * float(wl["L"][0]),
                    pickup_y=0.0, n_q=wl["n_q"], n_phi=0, sample_rate=wl["sample_rate"],
                    max_batch=max_batch or wl["batch"], max_steps=max_steps or wl["n_steps"])


def plan_from_workload(wl: dict, device=0, scheme=SV, lossless=False, options=None):
    """Create a plan for a workload dict (workloads.py), upload per-sample coefficients where the
    samples differ in geometry, and project the excitation.  Returns (plan, q0[batch][n_q])."""
    plan = Plan(desc_from_workload(wl, scheme, lossless), device)
    for k, v in (options or {}).items():
        plan.set_option(k, v)
    B = wl["batch"]
    q0 = np.empty((B, wl["n_q"]))
    if wl["model"] in ("vk", "berger"):
        same = all(np.all(wl[k] == wl[k][0]) for k in ("Lx", "Ly", "h")) and \
            wl["Lx"][0] == wl["ref"]["Lx"] and wl["Ly"][0] == wl["ref"]["Ly"] and wl["h"][0] == wl["ref"]["h"]
        if not same:
            rows = [plan.derive_coeffs(Lx=wl["Lx"][b], Ly=wl["Ly"][b], h=wl["h"][b],
                                       pickup_x_frac=wl["pickup"][0], pickup_y_frac=wl["pickup"][1]) for b in range(B)]
            lam = dict(lam=[r["lam"] for r in rows]) if wl["model"] == "berger" else {}
            plan.coeffs_upload(B, omega=[r["omega"] for r in rows], sigma=[r["sigma"] for r in rows],
                               nl_scale=[r["nl_scale"] for r in rows], pickup=[r["pickup"] for r in rows], **lam)
        for b in range(B):
            q0[b] = plan.project_bump(wl["Lx"][b], wl["Ly"][b], wl["x0"][b], wl["y0"][b], wl["W"][b], wl["A"][b])
    else:
        rows = [plan.derive_coeffs(Lx=wl["L"][b], T0=wl["T0s"][b], D=wl["D"][b], rho=wl["rho_lin"][b],
                                   area=wl["area"][b], pickup_x_frac=wl["pickup"][0]) for b in range(B)]
        plan.coeffs_upload(B, omega=[r["omega"] for r in rows], sigma=[r["sigma"] for r in rows],
                           nl_scale=[r["nl_scale"] for r in rows], lam=[r["lam"] for r in rows],
                           pickup=[r["pickup"] for r in rows])
        for b in range(B):
            q0[b] = plan.project_bump(wl["L"][b], 0.0, wl["x0"][b], 0.0, wl["W"][b], wl["A"][b])
    return plan, q0
