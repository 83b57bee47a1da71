"""Thin Python binding of the C ABI in include/gpw.h (argument marshalling only).

Every step of the path runs in the CUDA kernels of libgpw.so; PyTorch is used for device memory and
streams.  There is no CPU fallback: if the library is missing it is built with nvcc, and if that fails
or no CUDA device is present the eval calls raise.

    plan = gpw_build_pairs(cell, natm, xyz, nshl, shl_atom, shl_l, shl_nprim, shl_prim_off,
                           prim_exp, prim_coef, nlevel, mesh, tau, rel_cutoff, hermi)
    gpw_eval_rho(plan, D, deriv, rho_levels)      # torch CUDA float64 tensors, rho overwritten
    gpw_eval_mat(plan, v_levels, deriv, F)        # F overwritten
    gpw_eval_grad(plan, v_levels, deriv, D, grad) # grad [natm, 3] overwritten
"""
from __future__ import annotations

import ctypes
import os
from typing import List, Optional, Sequence

import numpy as np

from . import build as _build

GPW_MAX_LEVEL = 8
GPW_OK, GPW_EINVAL, GPW_ENOMEM, GPW_ECUDA, GPW_EUNSUPPORTED = 0, -1, -2, -3, -4


class GpwError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"gpw error {code}: {msg}")
        self.code = code


class gpw_info(ctypes.Structure):
    _fields_ = [("nao", ctypes.c_int), ("nshl", ctypes.c_int), ("nlevel", ctypes.c_int),
                ("hermi", ctypes.c_int), ("on_device", ctypes.c_int),
                ("ntask", ctypes.c_long),
                ("ntask_level", ctypes.c_long * GPW_MAX_LEVEL),
                ("nvisit_level", ctypes.c_long * GPW_MAX_LEVEL),
                ("nvisit_class", ctypes.c_long * (GPW_MAX_LEVEL * 16)),
                ("nitem", ctypes.c_long), ("ncoef_total", ctypes.c_long),
                ("build_seconds", ctypes.c_double), ("device_bytes", ctypes.c_long)]


class gpw_task(ctypes.Structure):
    _fields_ = [("shl_a", ctypes.c_int), ("prim_a", ctypes.c_int), ("shl_b", ctypes.c_int),
                ("prim_b", ctypes.c_int), ("T", ctypes.c_int * 3), ("level", ctypes.c_int),
                ("R", ctypes.c_double)]


class gpw_visit(ctypes.Structure):
    _fields_ = [("task", ctypes.c_int), ("block", ctypes.c_int * 3)]


NCOMP = {0: 1, 1: 4, 2: 5}   # components of a level array per deriv (include/gpw.h)
_dp = ctypes.POINTER(ctypes.c_double)
_ip = ctypes.POINTER(ctypes.c_int)
_lib = None

EXPORTS = ["gpw_build_pairs", "gpw_eval_rho", "gpw_eval_mat", "gpw_eval_grad", "gpw_interp_up", "gpw_restrict_down",
           "gpw_hartree", "gpw_gspace_gradient", "gpw_gspace_divergence",
           "gpw_eval_mat_static", "gpw_eval_rho_host", "gpw_eval_mat_host", "gpw_plan_wait", "gpw_plan_set_partition", "gpw_plan_partition_bounds",
           "gpw_plan_info", "gpw_plan_export_tasks", "gpw_plan_export_visits", "gpw_free_plan", "gpw_last_error", "gpw_dfma_peak", "gpw_dmma_peak",
           "gpw_plan_set_timing", "gpw_plan_get_timing"]


__all__ = [n for n in EXPORTS if n != "gpw_last_error"] + ["GpwError", "Plan", "load_library", "model_flops", "EXPORTS", "GPW_STATIC_MOM_DOUBLES"]


def load_library():
    """dlopen libgpw.so (building it first if it is missing or stale)."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.build()
    L = ctypes.CDLL(path)
    L.gpw_last_error.restype = ctypes.c_char_p
    L.gpw_build_pairs.restype = ctypes.c_int
    L.gpw_build_pairs.argtypes = [_dp, ctypes.c_int, _dp, ctypes.c_int, _ip, _ip, _ip, _ip, _dp, _dp,
                                  ctypes.c_int, _ip, ctypes.c_double, ctypes.c_double, ctypes.c_int,
                                  ctypes.POINTER(ctypes.c_void_p)]
    L.gpw_eval_rho.restype = ctypes.c_int
    L.gpw_eval_rho.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int,
                               ctypes.POINTER(ctypes.c_void_p), ctypes.c_void_p]
    L.gpw_eval_mat.restype = ctypes.c_int
    L.gpw_eval_mat.argtypes = [ctypes.c_void_p, ctypes.POINTER(ctypes.c_void_p), ctypes.c_int,
                               ctypes.c_void_p, ctypes.c_void_p]
    L.gpw_eval_mat_static.restype = ctypes.c_int
    L.gpw_eval_mat_static.argtypes = [ctypes.c_void_p, ctypes.POINTER(ctypes.c_void_p), ctypes.c_int,
                                      ctypes.c_void_p, ctypes.c_void_p]
    L.gpw_eval_grad.restype = ctypes.c_int
    L.gpw_eval_grad.argtypes = [ctypes.c_void_p, ctypes.POINTER(ctypes.c_void_p), ctypes.c_int,
                                ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
    L.gpw_interp_up.restype = ctypes.c_int
    L.gpw_interp_up.argtypes = [ctypes.c_void_p, ctypes.POINTER(ctypes.c_void_p), ctypes.c_int,
                                ctypes.c_void_p, ctypes.c_void_p]
    L.gpw_restrict_down.restype = ctypes.c_int
    L.gpw_restrict_down.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int,
                                    ctypes.POINTER(ctypes.c_void_p), ctypes.c_void_p]
    L.gpw_eval_rho_host.restype = ctypes.c_int
    L.gpw_eval_rho_host.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int, ctypes.POINTER(ctypes.c_void_p), ctypes.c_void_p]
    L.gpw_eval_mat_host.restype = ctypes.c_int
    L.gpw_eval_mat_host.argtypes = [ctypes.c_void_p, ctypes.POINTER(ctypes.c_void_p), ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p]
    L.gpw_plan_wait.restype = ctypes.c_int
    L.gpw_plan_wait.argtypes = [ctypes.c_void_p, ctypes.c_void_p]
    L.gpw_plan_set_partition.restype = ctypes.c_int
    L.gpw_plan_set_partition.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int]
    L.gpw_plan_partition_bounds.restype = ctypes.c_int
    L.gpw_plan_partition_bounds.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_int, _ip, _ip]
    for name in ("gpw_hartree", "gpw_gspace_gradient", "gpw_gspace_divergence"):
        getattr(L, name).restype = ctypes.c_int
        getattr(L, name).argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
    L.gpw_plan_info.restype = ctypes.c_int
    L.gpw_plan_info.argtypes = [ctypes.c_void_p, ctypes.POINTER(gpw_info)]
    L.gpw_plan_export_tasks.restype = ctypes.c_int
    L.gpw_plan_export_tasks.argtypes = [ctypes.c_void_p, ctypes.POINTER(gpw_task), ctypes.c_long,
                                        ctypes.POINTER(ctypes.c_long)]
    L.gpw_plan_export_visits.restype = ctypes.c_int
    L.gpw_plan_export_visits.argtypes = [ctypes.c_void_p, ctypes.POINTER(gpw_visit), ctypes.c_long,
                                         ctypes.POINTER(ctypes.c_long)]
    L.gpw_plan_set_timing.restype = ctypes.c_int
    L.gpw_plan_set_timing.argtypes = [ctypes.c_void_p, ctypes.c_int]
    L.gpw_plan_get_timing.restype = ctypes.c_int
    L.gpw_plan_get_timing.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.POINTER(ctypes.c_float)]
    L.gpw_dfma_peak.restype = ctypes.c_int
    L.gpw_dfma_peak.argtypes = [ctypes.c_double, _dp, _ip]
    L.gpw_dmma_peak.restype = ctypes.c_int
    L.gpw_dmma_peak.argtypes = [ctypes.c_double, _dp, _dp]
    L.gpw_free_plan.restype = None
    L.gpw_free_plan.argtypes = [ctypes.c_void_p]
    _lib = L
    return L


def _check(rc: int):
    if rc != GPW_OK:
        raise GpwError(rc, load_library().gpw_last_error().decode())


class Plan:
    """Owner of an opaque gpw_plan*."""

    def __init__(self, handle: int, mesh: np.ndarray):
        self._h = ctypes.c_void_p(handle)
        self.mesh = mesh
        self.info = gpw_plan_info(self)
        self.nao = self.info["nao"]
        self.nlevel = self.info["nlevel"]

    def __del__(self):
        gpw_free_plan(self)


def gpw_build_pairs(cell, natm, xyz, nshl, shl_atom, shl_l, shl_nprim, shl_prim_off, prim_exp,
                    prim_coef, nlevel, mesh, tau, rel_cutoff, hermi) -> Plan:
    L = load_library()
    cell = np.ascontiguousarray(cell, np.float64).reshape(9)
    xyz = np.ascontiguousarray(xyz, np.float64).reshape(-1)
    ia = [np.ascontiguousarray(a, np.int32) for a in (shl_atom, shl_l, shl_nprim, shl_prim_off)]
    pe = np.ascontiguousarray(prim_exp, np.float64)
    pc = np.ascontiguousarray(prim_coef, np.float64)
    mesh = np.ascontiguousarray(mesh, np.int32).reshape(-1, 3)
    out = ctypes.c_void_p()
    rc = L.gpw_build_pairs(cell.ctypes.data_as(_dp), int(natm), xyz.ctypes.data_as(_dp), int(nshl),
                           *[a.ctypes.data_as(_ip) for a in ia], pe.ctypes.data_as(_dp),
                           pc.ctypes.data_as(_dp), int(nlevel), mesh.ctypes.data_as(_ip), float(tau),
                           float(rel_cutoff), int(hermi), ctypes.byref(out))
    _check(rc)
    return Plan(out.value, mesh.copy())


def gpw_free_plan(plan: Plan):
    h = getattr(plan, "_h", None)
    if h is not None and h.value:
        load_library().gpw_free_plan(h)
        plan._h = ctypes.c_void_p()


def gpw_plan_info(plan: Plan) -> dict:
    info = gpw_info()
    _check(load_library().gpw_plan_info(plan._h, ctypes.byref(info)))
    nl = info.nlevel
    return {
        "nao": info.nao, "nshl": info.nshl, "nlevel": nl, "hermi": info.hermi,
        "on_device": bool(info.on_device), "ntask": info.ntask,
        "ntask_level": [info.ntask_level[i] for i in range(nl)],
        "nvisit_level": [info.nvisit_level[i] for i in range(nl)],
        "nvisit_class": np.array(list(info.nvisit_class), dtype=np.int64).reshape(GPW_MAX_LEVEL, 4, 4)[:nl],
        "nitem": info.nitem, "ncoef_total": info.ncoef_total, "build_seconds": info.build_seconds,
        "device_bytes": info.device_bytes,
    }


def gpw_plan_export_tasks(plan: Plan):
    """(ints[ntask, 8] = shl_a, prim_a, shl_b, prim_b, T0, T1, T2, level ; R[ntask])"""
    L = load_library()
    n = ctypes.c_long()
    _check(L.gpw_plan_export_tasks(plan._h, None, 0, ctypes.byref(n)))
    buf = (gpw_task * max(1, n.value))()
    _check(L.gpw_plan_export_tasks(plan._h, buf, n.value, ctypes.byref(n)))
    ints = np.zeros((n.value, 8), np.int32)
    R = np.zeros(n.value)
    for i in range(n.value):
        t = buf[i]
        ints[i] = (t.shl_a, t.prim_a, t.shl_b, t.prim_b, t.T[0], t.T[1], t.T[2], t.level)
        R[i] = t.R
    return ints, R


def gpw_plan_export_visits(plan: Plan) -> np.ndarray:
    """ints[nvisit, 4] = task (row of gpw_plan_export_tasks), unwrapped block coordinates b1, b2, b3."""
    L = load_library()
    n = ctypes.c_long()
    _check(L.gpw_plan_export_visits(plan._h, None, 0, ctypes.byref(n)))
    buf = np.zeros((max(1, n.value), 4), np.int32)
    _check(L.gpw_plan_export_visits(plan._h, buf.ctypes.data_as(ctypes.POINTER(gpw_visit)), n.value, ctypes.byref(n)))
    return buf[:n.value]


def _stream_ptr(stream) -> ctypes.c_void_p:
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return ctypes.c_void_p(s.cuda_stream)


def _check_grid(t, shape, what):
    import torch
    if not (t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and tuple(t.shape) == shape):
        raise ValueError(f"{what}: need a contiguous CUDA float64 tensor of shape {shape}, got {tuple(t.shape)} {t.dtype} {t.device}")


def gpw_eval_rho(plan: Plan, D, deriv: int, rho: Sequence, stream=None):
    """rho[level] (CUDA float64 [ncomp, N1, N2, N3]) is overwritten with the collocated density."""
    nc = NCOMP[int(deriv)]
    _check_grid(D, (plan.nao, plan.nao), "D")
    for lev in range(plan.nlevel):
        _check_grid(rho[lev], (nc,) + tuple(int(x) for x in plan.mesh[lev]), f"rho[{lev}]")
    ptrs = (ctypes.c_void_p * plan.nlevel)(*[r.data_ptr() for r in rho])
    _check(load_library().gpw_eval_rho(plan._h, ctypes.c_void_p(D.data_ptr()), int(deriv), ptrs, _stream_ptr(stream)))


def gpw_eval_mat(plan: Plan, v: Sequence, deriv: int, F, stream=None):
    """F (CUDA float64 [nao, nao]) is overwritten with the integrated matrix (includes dV)."""
    nc = NCOMP[int(deriv)]
    _check_grid(F, (plan.nao, plan.nao), "F")
    for lev in range(plan.nlevel):
        _check_grid(v[lev], (nc,) + tuple(int(x) for x in plan.mesh[lev]), f"v[{lev}]")
    ptrs = (ctypes.c_void_p * plan.nlevel)(*[x.data_ptr() for x in v])
    _check(load_library().gpw_eval_mat(plan._h, ptrs, int(deriv), ctypes.c_void_p(F.data_ptr()), _stream_ptr(stream)))


GPW_STATIC_MOM_DOUBLES = 1 << 21


def gpw_eval_mat_static(plan: Plan, v: Sequence, deriv: int, F, stream=None):
    """gpw_eval_mat with the moment workspace in the library's static device array: no allocation inside the call;
    plans whose workspace exceeds GPW_STATIC_MOM_DOUBLES are rejected (GpwError, GPW_EUNSUPPORTED)."""
    nc = NCOMP[int(deriv)]
    _check_grid(F, (plan.nao, plan.nao), "F")
    for lev in range(plan.nlevel):
        _check_grid(v[lev], (nc,) + tuple(int(x) for x in plan.mesh[lev]), f"v[{lev}]")
    ptrs = (ctypes.c_void_p * plan.nlevel)(*[x.data_ptr() for x in v])
    _check(load_library().gpw_eval_mat_static(plan._h, ptrs, int(deriv), ctypes.c_void_p(F.data_ptr()), _stream_ptr(stream)))


def _check_host(t, shape, what):
    import torch
    if not (not t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and tuple(t.shape) == shape):
        raise ValueError(f"{what}: need a contiguous host float64 tensor of shape {shape}, got {tuple(t.shape)} {t.dtype} {t.device}")


def gpw_eval_rho_host(plan: Plan, D, deriv: int, rho: Sequence, stream=None):
    """Host-buffer variant: D and rho[level] are HOST tensors (pinned for overlap); complete after gpw_plan_wait."""
    nc = NCOMP[int(deriv)]
    _check_host(D, (plan.nao, plan.nao), "D")
    for lev in range(plan.nlevel):
        _check_host(rho[lev], (nc,) + tuple(int(x) for x in plan.mesh[lev]), f"rho[{lev}]")
    ptrs = (ctypes.c_void_p * plan.nlevel)(*[r.data_ptr() for r in rho])
    _check(load_library().gpw_eval_rho_host(plan._h, ctypes.c_void_p(D.data_ptr()), int(deriv), ptrs, _stream_ptr(stream)))


def gpw_eval_mat_host(plan: Plan, v: Sequence, deriv: int, F, stream=None):
    """Host-buffer variant: v[level] and F are HOST tensors (pinned for overlap); complete after gpw_plan_wait."""
    nc = NCOMP[int(deriv)]
    _check_host(F, (plan.nao, plan.nao), "F")
    for lev in range(plan.nlevel):
        _check_host(v[lev], (nc,) + tuple(int(x) for x in plan.mesh[lev]), f"v[{lev}]")
    ptrs = (ctypes.c_void_p * plan.nlevel)(*[x.data_ptr() for x in v])
    _check(load_library().gpw_eval_mat_host(plan._h, ptrs, int(deriv), ctypes.c_void_p(F.data_ptr()), _stream_ptr(stream)))


def gpw_plan_wait(plan: Plan, stream=None):
    """Make the stream wait for every host-buffer call issued so far on the plan."""
    _check(load_library().gpw_plan_wait(plan._h, _stream_ptr(stream)))


def gpw_plan_set_partition(plan: Plan, rank: int, nranks: int):
    """Shard the eval calls: this process evaluates the n1 slab `rank` of `nranks` on every level (include/gpw.h)."""
    _check(load_library().gpw_plan_set_partition(plan._h, int(rank), int(nranks)))


def gpw_plan_partition_bounds(plan: Plan, level: int, rank: int, nranks: int):
    """(n1_lo, n1_hi): the grid-index range along n1 that `rank` of `nranks` owns on `level`."""
    lo, hi = ctypes.c_int(), ctypes.c_int()
    _check(load_library().gpw_plan_partition_bounds(plan._h, int(level), int(rank), int(nranks), ctypes.byref(lo), ctypes.byref(hi)))
    return lo.value, hi.value


def gpw_eval_grad(plan: Plan, v: Sequence, deriv: int, D, grad, stream=None):
    """grad (CUDA float64 [natm, 3]) is overwritten with dE/dR of E = sum dV [v0 rho + w . grad rho] at fixed v, w."""
    nc = NCOMP[int(deriv)]
    _check_grid(D, (plan.nao, plan.nao), "D")
    if not (grad.is_cuda and grad.is_contiguous() and grad.dim() == 2 and grad.shape[1] == 3 and str(grad.dtype) == "torch.float64"):
        raise ValueError("grad: need a contiguous CUDA float64 tensor of shape [natm, 3]")
    for lev in range(plan.nlevel):
        _check_grid(v[lev], (nc,) + tuple(int(x) for x in plan.mesh[lev]), f"v[{lev}]")
    ptrs = (ctypes.c_void_p * plan.nlevel)(*[x.data_ptr() for x in v])
    _check(load_library().gpw_eval_grad(plan._h, ptrs, int(deriv), ctypes.c_void_p(D.data_ptr()),
                                        ctypes.c_void_p(grad.data_ptr()), _stream_ptr(stream)))


def gpw_interp_up(plan: Plan, rho: Sequence, ncomp: int, rho_fine, stream=None):
    for lev in range(plan.nlevel):
        _check_grid(rho[lev], (int(ncomp),) + tuple(int(x) for x in plan.mesh[lev]), f"rho[{lev}]")
    _check_grid(rho_fine, (int(ncomp),) + tuple(int(x) for x in plan.mesh[0]), "rho_fine")
    ptrs = (ctypes.c_void_p * plan.nlevel)(*[r.data_ptr() for r in rho])
    _check(load_library().gpw_interp_up(plan._h, ptrs, int(ncomp), ctypes.c_void_p(rho_fine.data_ptr()), _stream_ptr(stream)))


def gpw_restrict_down(plan: Plan, v_fine, ncomp: int, v: Sequence, stream=None):
    for lev in range(plan.nlevel):
        _check_grid(v[lev], (int(ncomp),) + tuple(int(x) for x in plan.mesh[lev]), f"v[{lev}]")
    _check_grid(v_fine, (int(ncomp),) + tuple(int(x) for x in plan.mesh[0]), "v_fine")
    ptrs = (ctypes.c_void_p * plan.nlevel)(*[x.data_ptr() for x in v])
    _check(load_library().gpw_restrict_down(plan._h, ctypes.c_void_p(v_fine.data_ptr()), int(ncomp), ptrs, _stream_ptr(stream)))


def _gspace(name, plan, x, xshape, y, yshape, stream):
    m = tuple(int(v) for v in plan.mesh[0])
    _check_grid(x, xshape + m, "input")
    _check_grid(y, yshape + m, "output")
    _check(getattr(load_library(), name)(plan._h, ctypes.c_void_p(x.data_ptr()), ctypes.c_void_p(y.data_ptr()), _stream_ptr(stream)))


def gpw_hartree(plan: Plan, rho_fine, vh_fine, stream=None):
    """vh_fine [N1, N2, N3] is overwritten with the Hartree potential of rho_fine (Eq. 5-6), both on the finest mesh."""
    _gspace("gpw_hartree", plan, rho_fine, (), vh_fine, (), stream)


def gpw_gspace_gradient(plan: Plan, rho_fine, grad_fine, stream=None):
    """grad_fine [3, N1, N2, N3] is overwritten with the Fourier gradient of rho_fine (Eq. 10)."""
    _gspace("gpw_gspace_gradient", plan, rho_fine, (), grad_fine, (3,), stream)


def gpw_gspace_divergence(plan: Plan, w_fine, div_fine, stream=None):
    """div_fine [N1, N2, N3] is overwritten with the Fourier divergence of w_fine [3, N1, N2, N3] (Eq. 14)."""
    _gspace("gpw_gspace_divergence", plan, w_fine, (3,), div_fine, (), stream)


def gpw_plan_set_timing(plan: Plan, enable: bool):
    _check(load_library().gpw_plan_set_timing(plan._h, int(bool(enable))))


def gpw_plan_get_timing(plan: Plan, which: int):
    """Kernel durations (ms) of the last eval_rho (which=0: pre-pass, collocation) or eval_mat
    (which=1: integration, post-pass); waits for that call to finish."""
    ms = (ctypes.c_float * 2)()
    _check(load_library().gpw_plan_get_timing(plan._h, int(which), ms))
    return float(ms[0]), float(ms[1])


def gpw_dfma_peak(min_seconds: float = 0.5):
    """(TFLOP/s of a register-only FP64 FMA loop on the current device, SM count)."""
    t, n = ctypes.c_double(), ctypes.c_int()
    _check(load_library().gpw_dfma_peak(float(min_seconds), ctypes.byref(t), ctypes.byref(n)))
    return t.value, n.value


def gpw_dmma_peak(min_seconds: float = 0.3):
    """(TFLOP/s of mma.sync.m8n8k4.f64 alone, TFLOP/s of DMMA + DFMA issued together) on the current device."""
    a, b = ctypes.c_double(), ctypes.c_double()
    _check(load_library().gpw_dmma_peak(float(min_seconds), ctypes.byref(a), ctypes.byref(b)))
    return a.value, b.value


# ---- flop model of SURVEY.md 8(d): what the direct evaluation of Alg. 1/2 must compute per visited point
def model_flops(info: dict, deriv: int) -> float:
    """Model FP64 flops of ONE eval_rho (or one eval_mat) call: sum over (level, la, lb) of
    64 * visits * W, W0 = 2 nca ncb + 2 (nca + ncb) + 4, W1 = 4 nca ncb + 10 (nca + ncb) + 8."""
    nc = [1, 3, 6, 10]
    total = 0.0
    cls = info["nvisit_class"]
    for la in range(4):
        for lb in range(4):
            n = float(cls[:, la, lb].sum())
            w0 = 2 * nc[la] * nc[lb] + 2 * (nc[la] + nc[lb]) + 4
            w1 = 4 * nc[la] * nc[lb] + 10 * (nc[la] + nc[lb]) + 8
            total += 64.0 * n * (w0, w1, w1 + w0)[int(deriv)]   # deriv = 2: the tau contraction counted as one more W0
    return total
