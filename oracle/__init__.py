"""CPU oracle for the multigrid GPW collocation / integration hot path.

TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only ``tests/``,
``__graft_entry__.smoke()`` and the ``cpu_baseline`` / ``--impl reference``
legs of ``bench.py`` may import this package.  It shares no code with the CUDA
path (``paper_2603_24881_b200``) and never imports it; the only common module
is the seeded input generator ``paper_2603_24881_b200.inputs`` (no arithmetic
of the method).

Parts:
  gpw_oracle.c   truncated definition T1..T8 (what the GPU path must reproduce
                 to 1e-11), plain C + OpenMP, called through ctypes here
  dense.py       plain definition C.1: Eq. (3)/(4) of the paper with brute-force
                 sums over all lattice images, numpy (tiny cells only)
  overlap.py     analytic periodic overlap matrix (closed form), numpy

Parity status: every function is pinned by ``tests/test_oracle_*.py`` (see
DESIGN.md "Pins"); nothing here is "parity unpinned".
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import List, Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gpw_oracle.c")
_LIB = os.path.join(_HERE, "libgpw_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile gpw_oracle.c with gcc -O2 -fopenmp (building the checker is not using it)."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
        return _LIB
    cmd = ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c99", "-D_GNU_SOURCE",
           "-o", _LIB, _SRC, "-lm"]
    subprocess.check_call(cmd)
    return _LIB


_dp = ctypes.POINTER(ctypes.c_double)
_ip = ctypes.POINTER(ctypes.c_int)
_ucp = ctypes.POINTER(ctypes.c_ubyte)


def _load():
    global _lib
    if _lib is not None:
        return _lib
    build()
    L = ctypes.CDLL(_LIB)
    L.orc_create.restype = ctypes.c_void_p
    L.orc_create.argtypes = [_dp, ctypes.c_int, _dp, ctypes.c_int, _ip, _ip, _ip, _ip, _dp, _dp,
                             ctypes.c_int, _ip, ctypes.c_double, ctypes.c_double]
    L.orc_free.argtypes = [ctypes.c_void_p]
    L.orc_ntask.restype = ctypes.c_long
    L.orc_ntask.argtypes = [ctypes.c_void_p]
    L.orc_nao.restype = ctypes.c_int
    L.orc_nao.argtypes = [ctypes.c_void_p]
    L.orc_get_tasks.argtypes = [ctypes.c_void_p, _ip, _dp]
    L.orc_visit_counts.argtypes = [ctypes.c_void_p, ctypes.POINTER(ctypes.c_long)]
    L.orc_last_visit_counts.argtypes = [ctypes.c_void_p, ctypes.POINTER(ctypes.c_long)]
    L.orc_export_visits.restype = ctypes.c_long
    L.orc_export_visits.argtypes = [ctypes.c_void_p, ctypes.c_long, _ip]
    L.orc_eval_rho.restype = ctypes.c_int
    L.orc_eval_rho.argtypes = [ctypes.c_void_p, _dp, ctypes.c_int, ctypes.POINTER(_dp),
                               ctypes.POINTER(_ucp)]
    L.orc_eval_mat.restype = ctypes.c_int
    L.orc_eval_mat.argtypes = [ctypes.c_void_p, ctypes.POINTER(_dp), ctypes.c_int, _dp, _ucp]
    L.orc_eval_grad.restype = ctypes.c_int
    L.orc_eval_grad.argtypes = [ctypes.c_void_p, ctypes.POINTER(_dp), ctypes.c_int, _dp, _dp]
    L.orc_prim_radius.restype = ctypes.c_double
    L.orc_prim_radius.argtypes = [ctypes.c_int, ctypes.c_double, ctypes.c_double, ctypes.c_double]
    L.orc_pair_radius.restype = ctypes.c_double
    L.orc_pair_radius.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_double,
                                  ctypes.c_double, ctypes.c_double, ctypes.c_double]
    L.orc_num_threads.restype = ctypes.c_int
    _lib = L
    return L


def _d(a):
    return a.ctypes.data_as(_dp)


def _i(a):
    return a.ctypes.data_as(_ip)


def num_threads() -> int:
    return int(_load().orc_num_threads())


def prim_radius(l: int, a: float, coef: float, tau: float) -> float:
    return float(_load().orc_prim_radius(l, a, coef, tau))


def pair_radius(la, lb, ap, kappa, dA, dB, tau) -> float:
    return float(_load().orc_pair_radius(la, lb, ap, kappa, dA, dB, tau))


_NCOMP = {0: 1, 1: 4, 2: 5}   # value | + gradient (T8) | + kinetic-energy density (T10)


class Oracle:
    """Truncated-definition evaluator (T1..T8) for one set of inputs.

    Takes the same flat arrays as ``gpw_build_pairs`` (include/gpw.h); always
    enumerates ORDERED pairs (no use of D's symmetry, reading A14)."""

    def __init__(self, cell, natm, xyz, nshl, shl_atom, shl_l, shl_nprim, shl_prim_off,
                 prim_exp, prim_coef, nlevel, mesh, tau, rel_cutoff, hermi=None):
        L = _load()
        self._L = L
        self.cell = np.ascontiguousarray(cell, np.float64).reshape(3, 3)
        self.xyz = np.ascontiguousarray(xyz, np.float64).reshape(-1, 3)
        self.shl_atom = np.ascontiguousarray(shl_atom, np.int32)
        self.shl_l = np.ascontiguousarray(shl_l, np.int32)
        self.shl_nprim = np.ascontiguousarray(shl_nprim, np.int32)
        self.shl_prim_off = np.ascontiguousarray(shl_prim_off, np.int32)
        self.prim_exp = np.ascontiguousarray(prim_exp, np.float64)
        self.prim_coef = np.ascontiguousarray(prim_coef, np.float64)
        self.mesh = np.ascontiguousarray(mesh, np.int32).reshape(-1, 3)
        self.nlevel = int(nlevel)
        self.nshl = int(nshl)
        self._h = L.orc_create(_d(self.cell), int(natm), _d(self.xyz), int(nshl), _i(self.shl_atom),
                               _i(self.shl_l), _i(self.shl_nprim), _i(self.shl_prim_off),
                               _d(self.prim_exp), _d(self.prim_coef), int(nlevel), _i(self.mesh),
                               float(tau), float(rel_cutoff))
        if not self._h:
            raise ValueError("orc_create failed (singular cell?)")
        self.nao = int(L.orc_nao(self._h))
        self.ntask = int(L.orc_ntask(self._h))

    @classmethod
    def from_inputs(cls, inp) -> "Oracle":
        return cls(*inp.abi_args())

    def __del__(self):
        h = getattr(self, "_h", None)
        if h:
            self._L.orc_free(h)
            self._h = None

    def tasks(self):
        """(ints[ntask,8] = shl_a, prim_a, shl_b, prim_b, T0, T1, T2, level ; R[ntask])"""
        ints = np.zeros((self.ntask, 8), np.int32)
        R = np.zeros(self.ntask, np.float64)
        if self.ntask:
            self._L.orc_get_tasks(self._h, _i(ints), _d(R))
        return ints, R

    def visit_counts(self) -> np.ndarray:
        """[nlevel,4,4] number of (ordered task, 4x4x4 tile) visits per (la, lb)."""
        out = np.zeros((self.nlevel, 4, 4), dtype=np.int64)
        self._L.orc_visit_counts(self._h, out.ctypes.data_as(ctypes.POINTER(ctypes.c_long)))
        return out

    def visits(self) -> np.ndarray:
        """ints[nvisit, 4] = task (row of tasks()), unwrapped tile coordinates beta_1, beta_2, beta_3 (T6)."""
        n = int(self._L.orc_export_visits(self._h, 0, None))
        buf = np.zeros((max(1, n), 4), np.int32)
        self._L.orc_export_visits(self._h, n, _i(buf))
        return buf[:n]

    def last_visit_counts(self) -> np.ndarray:
        """[nlevel,4,4] visits evaluated by the last eval_rho / eval_mat call (bookkeeping for timing)."""
        out = np.zeros((self.nlevel, 4, 4), dtype=np.int64)
        self._L.orc_last_visit_counts(self._h, out.ctypes.data_as(ctypes.POINTER(ctypes.c_long)))
        return out

    def eval_rho(self, D: np.ndarray, deriv: int = 0,
                 tile_masks: Optional[Sequence[Optional[np.ndarray]]] = None) -> List[np.ndarray]:
        D = np.ascontiguousarray(D, np.float64)
        assert D.shape == (self.nao, self.nao)
        nc = _NCOMP[int(deriv)]
        rho = [np.zeros((nc,) + tuple(int(x) for x in m)) for m in self.mesh]
        ptrs = (_dp * self.nlevel)(*[_d(r) for r in rho])
        mptr = None
        keep = []
        if tile_masks is not None:
            arr = []
            for lev, m in enumerate(tile_masks):
                if m is None:
                    arr.append(ctypes.cast(None, _ucp))
                else:
                    mm = np.ascontiguousarray(m, np.uint8).reshape(-1)
                    assert mm.size == int(np.prod(self.mesh[lev] // 4))
                    keep.append(mm)
                    arr.append(mm.ctypes.data_as(_ucp))
            mptr = (_ucp * self.nlevel)(*arr)
        rc = self._L.orc_eval_rho(self._h, _d(D), int(deriv), ptrs, mptr)
        assert rc == 0
        return rho

    def eval_mat(self, v: Sequence[np.ndarray], deriv: int = 0,
                 pair_mask: Optional[np.ndarray] = None) -> np.ndarray:
        nc = _NCOMP[int(deriv)]
        vv = []
        for lev in range(self.nlevel):
            a = np.ascontiguousarray(v[lev], np.float64)
            assert a.shape == (nc,) + tuple(int(x) for x in self.mesh[lev]), a.shape
            vv.append(a)
        ptrs = (_dp * self.nlevel)(*[_d(a) for a in vv])
        F = np.zeros((self.nao, self.nao))
        pm = None
        if pair_mask is not None:
            pmask = np.ascontiguousarray(pair_mask, np.uint8).reshape(self.nshl, self.nshl)
            pm = pmask.ctypes.data_as(_ucp)
        rc = self._L.orc_eval_mat(self._h, ptrs, int(deriv), _d(F), pm)
        assert rc == 0
        return F

    def eval_grad(self, v: Sequence[np.ndarray], deriv: int, D: np.ndarray) -> np.ndarray:
        """[natm, 3] nuclear gradient of sum_alpha dV sum_r [v0 rho + w . grad rho] at fixed v, w (T11)."""
        assert deriv in (0, 1)
        nc = _NCOMP[int(deriv)]
        vv = []
        for lev in range(self.nlevel):
            a = np.ascontiguousarray(v[lev], np.float64)
            assert a.shape == (nc,) + tuple(int(x) for x in self.mesh[lev]), a.shape
            vv.append(a)
        ptrs = (_dp * self.nlevel)(*[_d(a) for a in vv])
        D = np.ascontiguousarray(D, np.float64)
        assert D.shape == (self.nao, self.nao)
        g = np.zeros((self.xyz.shape[0], 3))
        rc = self._L.orc_eval_grad(self._h, ptrs, int(deriv), _d(D), _d(g))
        assert rc == 0
        return g
