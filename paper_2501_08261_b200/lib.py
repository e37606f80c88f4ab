"""ctypes binding of liblisa_td.so -- argument marshalling only.

Every function has the name and argument order of its C entry point in include/lisa_td.h
(minus the ``lisa_td_`` prefix).  Array arguments are torch CUDA float64 tensors (device
pointers are passed through, the current torch stream is the stream argument); ``*_host``
arguments are CPU tensors / numpy arrays.  Nothing is computed here, and there is no CPU
fallback: a missing library or a failing call raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "liblisa_td.so")

EXPORTS = [
    "lisa_td_last_error", "lisa_td_version", "lisa_td_orbit_table_create", "lisa_td_orbit_table_destroy", "lisa_td_modes_to_pol", "lisa_td_link_response",
    "lisa_td_link_response_up2",
    "lisa_td_laser_links", "lisa_td_tdi2", "lisa_td_tdi2_static", "lisa_td_response_tdi_workspace_bytes",
    "lisa_td_response_tdi", "lisa_td_plan_create", "lisa_td_plan_destroy", "lisa_td_loglike",
    "lisa_td_loglike_channels",
    "lisa_td_spectrum", "lisa_td_fisher", "lisa_td_psd_weights", "lisa_td_pipeline_create",
    "lisa_td_pipeline_destroy", "lisa_td_pipeline_host", "lisa_td_pipeline_host_up2", "lisa_td_check",
    "lisa_td_loglike_from_modes_workspace_bytes", "lisa_td_loglike_from_modes",
]
PROBE_LIB_PATH = os.path.join(_HERE, "liblisa_td_probe.so")  # bench-only, csrc/lisa_td_probe.h


class LisaTdError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"liblisa_td error {code}: {msg}")
        self.code = code


class Orbit(C.Structure):
    """lisa_td_orbit"""
    _fields_ = [("kind", C.c_int), ("L_m", C.c_double), ("a_m", C.c_double),
                ("year_s", C.c_double), ("phase0", C.c_double), ("t_ref", C.c_double),
                ("r_static", (C.c_double * 3) * 3), ("L_static", C.c_double * 6),
                ("table", C.c_void_p), ("tt_order", C.c_int), ("tdi_nested", C.c_int)]


class OrbitTable:
    """lisa_td_orbit_table: device copy of tabulated spacecraft positions [n_tab][3][3] (metres)."""

    def __init__(self, r_tab, t_tab0, dt_tab, order=7):
        r = np.ascontiguousarray(r_tab, dtype=np.float64)
        if r.ndim != 3 or r.shape[1:] != (3, 3):
            raise ValueError("r_tab must be [n_tab][3][3]")
        self._h = C.c_void_p()
        _check(load().lisa_td_orbit_table_create(C.byref(self._h), r.shape[0], float(t_tab0), float(dt_tab),
                                                 int(order), r.ctypes.data_as(C.c_void_p)))

    def close(self):
        if self._h:
            load().lisa_td_orbit_table_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def make_orbit(d: dict) -> Orbit:
    o = Orbit()
    if d["kind"] == "static":
        o.kind = 0
        for i in range(3):
            for j in range(3):
                o.r_static[i][j] = float(d["r_static"][i][j])
        for k in range(6):
            o.L_static[k] = float(d["L_static"][k])
    elif d["kind"] == "kepler1":
        o.kind = 1
        o.L_m, o.a_m, o.year_s = float(d["L_m"]), float(d["a_m"]), float(d["year_s"])
        o.phase0, o.t_ref = float(d.get("phase0", 0.0)), float(d.get("t_ref", 0.0))
    elif d["kind"] == "table":
        # the handle (device copy) is created once and cached in the description
        if "_lisa_table" not in d:
            d["_lisa_table"] = OrbitTable(d["r_tab"], d["t_tab0"], d["dt_tab"], d.get("tab_order", 7))
        o.kind = 2
        o.table = d["_lisa_table"]._h
    else:
        raise ValueError(d["kind"])
    o.tt_order = int(d.get("tt_order", 0))  # delay model, reading A22
    o.tdi_nested = int(d.get("nested", 0))
    return o


_lib = None


def load() -> C.CDLL:
    """Load the CUDA library (raises if it has not been built: there is no fallback)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} not built; run `python -m paper_2501_08261_b200.build`")
    L = C.CDLL(LIB_PATH)
    vp, dbl, i32, i64 = C.c_void_p, C.c_double, C.c_int, C.c_longlong
    L.lisa_td_last_error.restype = C.c_char_p
    L.lisa_td_version.restype = i32
    L.lisa_td_orbit_table_create.argtypes = [C.POINTER(vp), i32, dbl, dbl, i32, vp]
    L.lisa_td_orbit_table_destroy.argtypes = [vp]
    L.lisa_td_modes_to_pol.argtypes = [i32, i64, i32, C.POINTER(i32), C.POINTER(i32)] + [vp] * 11 + [vp]
    L.lisa_td_link_response.argtypes = [i32, i64, dbl, dbl, i32, i64, vp, vp, vp, vp,
                                        C.POINTER(Orbit), vp, vp]
    L.lisa_td_link_response_up2.argtypes = L.lisa_td_link_response.argtypes
    L.lisa_td_laser_links.argtypes = [i64, dbl, dbl, i32, i64, vp, C.POINTER(Orbit), vp, vp]
    L.lisa_td_tdi2.argtypes = [i32, i64, dbl, dbl, i32, i32, i32, i64, i64, vp, C.POINTER(Orbit),
                               vp, vp]
    L.lisa_td_tdi2_static.argtypes = [i32, i64, dbl, dbl, i32, i32, i32, i64, i64, vp, C.POINTER(Orbit),
                                      vp, i32, vp]
    L.lisa_td_response_tdi_workspace_bytes.restype = i64
    L.lisa_td_response_tdi_workspace_bytes.argtypes = [i32, i64]
    L.lisa_td_response_tdi.argtypes = [i32, i64, dbl, dbl, i32, i64, i32, i32, i64, i64, vp, vp, vp,
                                       vp, C.POINTER(Orbit), vp, vp, i64, vp]
    L.lisa_td_plan_create.argtypes = [C.POINTER(vp), i32, i64]
    L.lisa_td_plan_destroy.argtypes = [vp]
    L.lisa_td_loglike.argtypes = [vp, i32, i64, vp, vp, vp, i64, i64, vp, vp, vp, vp]
    L.lisa_td_loglike_channels.argtypes = [vp, i32, i64, i32, vp, vp, vp, i64, i64, vp, vp, vp, vp]
    L.lisa_td_spectrum.argtypes = [vp, i32, i64, vp, vp, vp]
    L.lisa_td_fisher.argtypes = [vp, i32, i64, vp, vp, vp, i64, i64, vp, vp]
    L.lisa_td_psd_weights.argtypes = [i64, dbl, dbl, dbl, dbl, i32, vp]
    L.lisa_td_pipeline_create.argtypes = [C.POINTER(vp), i32, i64, i32, i32]
    L.lisa_td_pipeline_destroy.argtypes = [vp]
    L.lisa_td_pipeline_host.argtypes = ([vp, i32, i64, i32, C.POINTER(i32), C.POINTER(i32)] + [vp] * 10
                                        + [dbl, dbl, i32, i64, i32, i64, i64, C.POINTER(Orbit), vp, vp,
                                           i64, i64, vp, vp, vp])
    L.lisa_td_pipeline_host_up2.argtypes = L.lisa_td_pipeline_host.argtypes
    L.lisa_td_check.argtypes = [vp]
    L.lisa_td_loglike_from_modes_workspace_bytes.restype = i64
    L.lisa_td_loglike_from_modes_workspace_bytes.argtypes = [i32, i64]
    L.lisa_td_loglike_from_modes.argtypes = ([vp, i32, i64, i32, C.POINTER(i32), C.POINTER(i32)] + [vp] * 10
                                             + [dbl, dbl, i32, i64, i32, i64, i64, C.POINTER(Orbit), vp, vp, i64, i64,
                                                vp, vp, vp, vp, i64, vp])
    _lib = L
    return L


def _check(rc):
    if rc != 0:
        raise LisaTdError(rc, load().lisa_td_last_error().decode())


def _dev(t, name="tensor"):
    """device pointer of a CUDA float64 contiguous tensor (None -> NULL)"""
    if t is None:
        return None
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
        raise TypeError(f"{name}: expected a contiguous CUDA float64 tensor")
    return C.c_void_p(t.data_ptr())


def _host(a):
    """pointer of a CPU float64 contiguous tensor / numpy array (None -> NULL)"""
    if a is None:
        return None
    if isinstance(a, torch.Tensor):
        if a.is_cuda or a.dtype != torch.float64 or not a.is_contiguous():
            raise TypeError("expected a contiguous CPU float64 tensor")
        return C.c_void_p(a.data_ptr())
    if not (isinstance(a, np.ndarray) and a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]):
        raise TypeError("expected a C-contiguous float64 numpy array")
    return C.c_void_p(a.ctypes.data)


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _ints(v):
    a = (C.c_int * len(v))(*[int(x) for x in v])
    return a


def last_error() -> str:
    return load().lisa_td_last_error().decode()


def version() -> int:
    return load().lisa_td_version()


def check():
    """lisa_td_check on the current torch stream: synchronises, raises if a kernel flagged a delay
    outside the host-side orbit bounds."""
    _check(load().lisa_td_check(_stream()))


def debug_force_generic(mode):
    """TEST-ONLY dispatch switch (not an ABI call): sets the environment variable LISA_TD_DISPATCH,
    which the library reads at every call.  1 = generic kernels, 2 = five-mode S1 without TMA,
    0 / False = normal."""
    os.environ["LISA_TD_DISPATCH"] = str(int(mode))


def modes_to_pol(B, N, l, m, amp, phase, alpha, beta, gamma, iota, phi, psi, euler0, hplus, hcross):
    _check(load().lisa_td_modes_to_pol(B, N, len(l), _ints(l), _ints(m), _dev(amp), _dev(phase),
                                       _dev(alpha), _dev(beta), _dev(gamma), _dev(iota), _dev(phi),
                                       _dev(psi), _dev(euler0), _dev(hplus), _dev(hcross), _stream()))


def link_response(B, N, t0, dt, order, margin_y, hplus, hcross, lam, beta_sky, orbit, y):
    o = make_orbit(orbit)
    _check(load().lisa_td_link_response(B, N, t0, dt, order, margin_y, _dev(hplus), _dev(hcross),
                                        _dev(lam), _dev(beta_sky), C.byref(o), _dev(y), _stream()))


def link_response_up2(B, N, t0, dt, order, margin_y, hplus_c, hcross_c, lam, beta_sky, orbit, y):
    o = make_orbit(orbit)
    _check(load().lisa_td_link_response_up2(B, N, t0, dt, order, margin_y, _dev(hplus_c), _dev(hcross_c),
                                            _dev(lam), _dev(beta_sky), C.byref(o), _dev(y), _stream()))


def laser_links(N, t0, dt, order, margin, p, orbit, y):
    o = make_orbit(orbit)
    _check(load().lisa_td_laser_links(N, t0, dt, order, margin, _dev(p), C.byref(o), _dev(y), _stream()))


def tdi2(B, N, t0, dt, order, generation, out_kind, margin_lo, margin_hi, y, orbit, tdi):
    o = make_orbit(orbit)
    _check(load().lisa_td_tdi2(B, N, t0, dt, order, generation, out_kind, margin_lo, margin_hi,
                               _dev(y), C.byref(o), _dev(tdi), _stream()))


TDI2_STATIC_MAX_N = 65536  # LISA_TD_TDI2_STATIC_MAX_N of include/lisa_td.h


def tdi2_static(B, N, t0, dt, order, generation, out_kind, margin_lo, margin_hi, y, orbit, tdi, check=True):
    """lisa_td_tdi2 with its scratch in the library's static device array: allocates nothing, N <= TDI2_STATIC_MAX_N"""
    o = make_orbit(orbit)
    _check(load().lisa_td_tdi2_static(B, N, t0, dt, order, generation, out_kind, margin_lo, margin_hi,
                                      _dev(y), C.byref(o), _dev(tdi), 1 if check else 0, _stream()))


def response_tdi_workspace_bytes(B, N) -> int:
    return load().lisa_td_response_tdi_workspace_bytes(B, N)


def response_tdi(B, N, t0, dt, order, margin_y, generation, out_kind, margin_lo, margin_hi, hplus,
                 hcross, lam, beta_sky, orbit, tdi, workspace):
    o = make_orbit(orbit)
    _check(load().lisa_td_response_tdi(B, N, t0, dt, order, margin_y, generation, out_kind, margin_lo,
                                       margin_hi, _dev(hplus), _dev(hcross), _dev(lam), _dev(beta_sky),
                                       C.byref(o), _dev(tdi), _dev(workspace),
                                       workspace.numel() * workspace.element_size(), _stream()))


class Plan:
    """lisa_td_plan (cuFFT plan + spectrum scratch)."""

    def __init__(self, B, N):
        self._h = C.c_void_p()
        _check(load().lisa_td_plan_create(C.byref(self._h), B, N))
        self.B, self.N = B, N

    def close(self):
        if self._h:
            load().lisa_td_plan_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def loglike(plan: Plan, B, N, tdi, data_spec, weight, kmin, kmax, loglike_out, dh=None, hh=None):
    _check(load().lisa_td_loglike(plan._h, B, N, _dev(tdi), _dev(data_spec), _dev(weight), kmin, kmax,
                                  _dev(loglike_out), _dev(dh), _dev(hh), _stream()))


def loglike_channels(plan: Plan, B, N, n_channels, tdi, data_spec, weight, kmin, kmax, loglike_out, dh=None, hh=None):
    _check(load().lisa_td_loglike_channels(plan._h, B, N, int(n_channels), _dev(tdi), _dev(data_spec), _dev(weight),
                                           kmin, kmax, _dev(loglike_out), _dev(dh), _dev(hh), _stream()))


def loglike_from_modes_workspace_bytes(B, N) -> int:
    return load().lisa_td_loglike_from_modes_workspace_bytes(B, N)


def loglike_from_modes(plan: Plan, B, N, l, m, amp, phase, alpha, beta, gamma, iota, phi, psi, lam, beta_sky, t0, dt,
                       order, margin_y, generation, margin_lo, margin_hi, orbit, data_spec, weight, kmin, kmax,
                       loglike_out, dh, hh, workspace):
    o = make_orbit(orbit)
    _check(load().lisa_td_loglike_from_modes(
        plan._h, B, N, len(l), _ints(l), _ints(m), _dev(amp), _dev(phase), _dev(alpha), _dev(beta), _dev(gamma),
        _dev(iota), _dev(phi), _dev(psi), _dev(lam), _dev(beta_sky), t0, dt, order, margin_y, generation, margin_lo,
        margin_hi, C.byref(o), _dev(data_spec), _dev(weight), kmin, kmax, _dev(loglike_out), _dev(dh), _dev(hh),
        _dev(workspace), workspace.numel() * workspace.element_size(), _stream()))


def spectrum(plan: Plan, B, N, tdi, spec):
    _check(load().lisa_td_spectrum(plan._h, B, N, _dev(tdi), _dev(spec), _stream()))


def fisher(plan: Plan, D, N, tdi, delta, weight, kmin, kmax, fisher_out):
    delta = np.ascontiguousarray(delta, dtype=np.float64)
    assert delta.size == D
    _check(load().lisa_td_fisher(plan._h, D, N, _dev(tdi), _host(delta), _dev(weight), kmin, kmax,
                                 _dev(fisher_out), _stream()))


def psd_weights(N, dt, acc_noise, oms_noise, arm_s, generation) -> np.ndarray:
    w = np.zeros((3, N // 2 + 1))
    _check(load().lisa_td_psd_weights(N, dt, acc_noise, oms_noise, arm_s, generation, _host(w)))
    return w


class Pipeline:
    """lisa_td_pipeline: S1..S5 from host buffers."""

    def __init__(self, chunk_B, N, n_modes, twisted):
        self._h = C.c_void_p()
        _check(load().lisa_td_pipeline_create(C.byref(self._h), chunk_B, N, n_modes, int(twisted)))

    def close(self):
        if self._h:
            load().lisa_td_pipeline_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def pipeline_host(pipe: Pipeline, B, N, l, m, amp, phase, alpha, beta, gamma, iota, phi, psi, lam,
                  beta_sky, t0, dt, order, margin_y, generation, margin_lo, margin_hi, orbit,
                  data_spec, weight, kmin, kmax, loglike_out, dh=None, hh=None):
    o = make_orbit(orbit)
    _check(load().lisa_td_pipeline_host(
        pipe._h, B, N, len(l), _ints(l), _ints(m), _host(amp), _host(phase), _host(alpha), _host(beta),
        _host(gamma), _host(iota), _host(phi), _host(psi), _host(lam), _host(beta_sky), t0, dt, order,
        margin_y, generation, margin_lo, margin_hi, C.byref(o), _host(data_spec), _host(weight), kmin,
        kmax, _host(loglike_out), _host(dh), _host(hh)))


def pipeline_host_up2(pipe: Pipeline, B, N, l, m, amp_c, phase_c, alpha_c, beta_c, gamma_c, iota, phi, psi, lam,
                      beta_sky, t0, dt, order, margin_y, generation, margin_lo, margin_hi, orbit,
                      data_spec, weight, kmin, kmax, loglike_out, dh=None, hh=None):
    """mode / angle arrays on the 2 dt grid: [B][M][N/2+1], [B][N/2+1]"""
    o = make_orbit(orbit)
    _check(load().lisa_td_pipeline_host_up2(
        pipe._h, B, N, len(l), _ints(l), _ints(m), _host(amp_c), _host(phase_c), _host(alpha_c), _host(beta_c),
        _host(gamma_c), _host(iota), _host(phi), _host(psi), _host(lam), _host(beta_sky), t0, dt, order,
        margin_y, generation, margin_lo, margin_hi, C.byref(o), _host(data_spec), _host(weight), kmin,
        kmax, _host(loglike_out), _host(dh), _host(hh)))


_probe = None


def _probe_lib() -> C.CDLL:
    """liblisa_td_probe.so: fp64 throughput probes for bench.py (csrc/lisa_td_probe.h), not product ABI"""
    global _probe
    if _probe is None:
        if not os.path.exists(PROBE_LIB_PATH):
            raise ImportError(f"{PROBE_LIB_PATH} not built; run `python -m paper_2501_08261_b200.build`")
        P = C.CDLL(PROBE_LIB_PATH)
        vp, i32, i64 = C.c_void_p, C.c_int, C.c_longlong
        P.lisa_td_probe_dfma.argtypes = [i64, i32, i32, vp, C.POINTER(C.c_float), vp]
        P.lisa_td_probe_fp64_pipes.argtypes = [i64, i32, i32, i32, vp, C.POINTER(C.c_float), vp]
        P.lisa_td_probe_fp64_operands.argtypes = [i32, i64, i32, vp, C.POINTER(C.c_float), vp]
        _probe = P
    return _probe


def probe_dfma(iters, blocks, threads, sink) -> float:
    ms = C.c_float()
    if _probe_lib().lisa_td_probe_dfma(iters, blocks, threads, _dev(sink), C.byref(ms), _stream()) != 0:
        raise RuntimeError("lisa_td_probe_dfma failed")
    return ms.value


def probe_fp64_operands(pattern, iters, blocks, sink) -> float:
    ms = C.c_float(0.0)
    if _probe_lib().lisa_td_probe_fp64_operands(pattern, iters, blocks, _dev(sink), C.byref(ms), _stream()) != 0:
        raise RuntimeError("lisa_td_probe_fp64_operands failed")
    return ms.value


def probe_fp64_pipes(iters, blocks, dfma_warps, dmma_warps, sink) -> float:
    ms = C.c_float()
    if _probe_lib().lisa_td_probe_fp64_pipes(iters, blocks, dfma_warps, dmma_warps, _dev(sink), C.byref(ms), _stream()) != 0:
        raise RuntimeError("lisa_td_probe_fp64_pipes failed")
    return ms.value
