"""Analytic periodic overlap matrix S^per = sum_T <phi_mu | phi_nu^T>.

TEST INFRASTRUCTURE (see oracle/__init__.py).  Textbook closed form, used as the
pin "v = 1  =>  F = S" and "sum_n rho(r_n) dV = Tr(D S)" (DESIGN.md pins G4/G5):
Eq. (4) of the paper with v_Hxc = 1 is the overlap integral, and the uniform-grid
quadrature of Eq. (29) is spectrally accurate for well-resolved Gaussians.

1-D integrals by the Obara-Saika recurrence over the whole real line:
  S_00        = sqrt(pi/p) exp(-mu X_AB^2),  p = a + b, mu = a b / p
  S_{i+1,j}   = X_PA S_ij + (i S_{i-1,j} + j S_{i,j-1}) / (2p)
  S_{i,j+1}   = X_PB S_ij + (i S_{i-1,j} + j S_{i,j-1}) / (2p)
"""
from __future__ import annotations

import math

import numpy as np


def _cart_powers(l):
    return [(lx, ly, l - lx - ly) for lx in range(l, -1, -1) for ly in range(l - lx, -1, -1)]


def overlap_1d(la: int, lb: int, a: float, b: float, A: float, B: float) -> np.ndarray:
    """S[i, j] = int (x-A)^i (x-B)^j exp(-a (x-A)^2 - b (x-B)^2) dx, i <= la, j <= lb."""
    p = a + b
    mu = a * b / p
    P = (a * A + b * B) / p
    PA, PB = P - A, P - B
    S = np.zeros((la + 2, lb + 2))
    S[0, 0] = math.sqrt(math.pi / p) * math.exp(-mu * (A - B) ** 2)
    for i in range(la + 1):
        for j in range(lb + 1):
            lowi = S[i - 1, j] if i > 0 else 0.0
            lowj = S[i, j - 1] if j > 0 else 0.0
            rec = (i * lowi + j * lowj) / (2 * p)
            if i + 1 <= la:
                S[i + 1, j] = PA * S[i, j] + rec
            if j + 1 <= lb:
                S[i, j + 1] = PB * S[i, j] + rec
    return S[: la + 1, : lb + 1]


def periodic_overlap(inp, eps: float = 1e-24, kinetic: bool = False) -> np.ndarray:
    """S^per[nao, nao] for the contracted Cartesian basis of ``inp``; with kinetic=True the periodic
    kinetic-energy matrix T^per = sum_T 1/2 <grad phi_mu | grad phi_nu^T> instead (textbook: per axis
    D_ij = int (d/dx g_i)(d/dx g_j) = i j S_{i-1,j-1} - 2b i S_{i-1,j+1} - 2a j S_{i+1,j-1} + 4ab S_{i+1,j+1},
    T = 1/2 (D_x S_y S_z + S_x D_y S_z + S_x S_y D_z)) -- the pin of Eq. (15)-(16) with v_tau = 1."""
    cell = np.asarray(inp.cell, float)
    binv = np.linalg.inv(cell)
    bnorm = np.linalg.norm(binv, axis=0)
    ao_loc = inp.ao_loc
    S = np.zeros((inp.nao, inp.nao))
    for sa in range(inp.nshl):
        la = int(inp.shl_l[sa])
        A = np.asarray(inp.xyz[int(inp.shl_atom[sa])], float)
        pa_ = _cart_powers(la)
        for sb in range(inp.nshl):
            lb = int(inp.shl_l[sb])
            B = np.asarray(inp.xyz[int(inp.shl_atom[sb])], float)
            pb_ = _cart_powers(lb)
            blk = np.zeros((len(pa_), len(pb_)))
            pax, pbx = np.array(pa_), np.array(pb_)
            for ka in range(int(inp.shl_nprim[sa])):
                ia = int(inp.shl_prim_off[sa]) + ka
                a, ca = float(inp.prim_exp[ia]), float(inp.prim_coef[ia])
                for kb in range(int(inp.shl_nprim[sb])):
                    ib = int(inp.shl_prim_off[sb]) + kb
                    b, cb = float(inp.prim_exp[ib]), float(inp.prim_coef[ib])
                    mu = a * b / (a + b)
                    # exp(-mu d^2) * polynomial growth < eps  ->  reach in |A - B - T|
                    reach = math.sqrt((math.log(abs(ca * cb) / eps) + 8.0 * (la + lb + 1)) / mu)
                    f = (A - B) @ binv
                    lo = np.ceil(f - reach * bnorm).astype(int)
                    hi = np.floor(f + reach * bnorm).astype(int)
                    for t1 in range(lo[0], hi[0] + 1):
                        for t2 in range(lo[1], hi[1] + 1):
                            for t3 in range(lo[2], hi[2] + 1):
                                Bt = B + t1 * cell[0] + t2 * cell[1] + t3 * cell[2]
                                s1 = [overlap_1d(la + 1, lb + 1, a, b, A[x], Bt[x]) for x in range(3)]
                                sx, sy, sz = (t[: la + 1, : lb + 1] for t in s1)
                                if not kinetic:
                                    blk += ca * cb * (sx[np.ix_(pax[:, 0], pbx[:, 0])] *
                                                      sy[np.ix_(pax[:, 1], pbx[:, 1])] *
                                                      sz[np.ix_(pax[:, 2], pbx[:, 2])])
                                    continue
                                d1 = []
                                for x in range(3):
                                    S1 = np.pad(s1[x], ((1, 0), (1, 0)))       # S1[i + 1, j + 1] = S_ij, S_{-1,.} = 0
                                    i = np.arange(la + 1)[:, None]
                                    j = np.arange(lb + 1)[None, :]
                                    d1.append(i * j * S1[i, j] - 2 * b * i * S1[i, j + 2] - 2 * a * j * S1[i + 2, j]
                                              + 4 * a * b * S1[i + 2, j + 2])
                                pick = lambda t, x: t[np.ix_(pax[:, x], pbx[:, x])]
                                blk += 0.5 * ca * cb * (pick(d1[0], 0) * pick(sy, 1) * pick(sz, 2) +
                                                        pick(sx, 0) * pick(d1[1], 1) * pick(sz, 2) +
                                                        pick(sx, 0) * pick(sy, 1) * pick(d1[2], 2))
            S[ao_loc[sa]:ao_loc[sa + 1], ao_loc[sb]:ao_loc[sb + 1]] = blk
    return S
