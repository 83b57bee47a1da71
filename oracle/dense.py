"""Plain definition (C.1 of DESIGN.md) of collocation and integration: numpy only.

TEST INFRASTRUCTURE (see oracle/__init__.py).  Tiny cells only.

Follows the paper literally, with NO truncation radius, NO tiles and NO
screening of pairs:

  Phi_mu(r)  = sum_S phi_mu(r - S)            Eq. (1)-(2) at k = 0
  rho(r_n)   = sum_{mu,nu} D_mu,nu Phi_mu(r_n) Phi_nu(r_n)          Eq. (3)
  F_mu,nu    = dV sum_n v(r_n) Phi_mu(r_n) Phi_nu(r_n)              Eq. (4) with the
               quadrature weight dV = Omega / N_grid of Eq. (29)
  deriv = 1  : rho_c = d_c rho ; F += dV sum_n w_c d_c(Phi_mu Phi_nu)   Eq. (11)

i.e. rho = diag(Phi D Phi^T) and F = dV Phi^T diag(v) Phi.  The image sum runs
over every lattice vector S whose primitive can exceed 1e-22 anywhere in the cell.

Multigrid: every primitive pair belongs to exactly one level
(rule T5, by a_p = a_mu + a_nu); rho_alpha uses only that level's pairs and
F = sum_alpha F_alpha.  This is expressed with a 0/1 mask on the
primitive-resolved density matrix.
"""
from __future__ import annotations

import math
from typing import List, Sequence

import numpy as np


def _cart_powers(l):
    return [(lx, ly, l - lx - ly) for lx in range(l, -1, -1) for ly in range(l - lx, -1, -1)]


def grid_points(cell: np.ndarray, mesh) -> np.ndarray:
    """r_n = (n1/N1) a1 + (n2/N2) a2 + (n3/N3) a3, C order with n3 fastest (u0 = 0)."""
    n1, n2, n3 = (int(x) for x in mesh)
    u = np.stack(np.meshgrid(np.arange(n1) / n1, np.arange(n2) / n2, np.arange(n3) / n3,
                             indexing="ij"), axis=-1).reshape(-1, 3)
    return u @ np.asarray(cell, float)


def _prim_reach(l, a, coef, eps=1e-22):
    r = 1.0
    for _ in range(60):
        val = (math.log(abs(coef) / eps) + l * math.log(max(r, 1.0))) / a
        r = math.sqrt(max(val, 1.0))
    return r + 1.0


def prim_ao_matrix(inp, level: int, deriv: int):
    """Primitive-resolved periodised AO values on one level.

    Returns (Phi[ncomp, Ngrid, nprimao], prim_ao_exp[nprimao], expand[nprimao] -> contracted AO index).
    Column order: shells in input order; inside a shell the primitives in order,
    each with its Cartesian components (decreasing lx, then ly)."""
    cell = np.asarray(inp.cell, float)
    binv = np.linalg.inv(cell)          # u = r @ binv ; b_i = binv[:, i]
    bnorm = np.linalg.norm(binv, axis=0)
    r = grid_points(cell, inp.mesh[level])
    ncomp = 4 if deriv else 1      # deriv = 2 (tau) needs the same first derivatives as deriv = 1
    cols, exps, expand = [], [], []
    ao_loc = inp.ao_loc
    for s in range(inp.nshl):
        l = int(inp.shl_l[s])
        A = np.asarray(inp.xyz[int(inp.shl_atom[s])], float)
        fA = A @ binv
        pw = _cart_powers(l)
        for k in range(int(inp.shl_nprim[s])):
            p = int(inp.shl_prim_off[s]) + k
            a, coef = float(inp.prim_exp[p]), float(inp.prim_coef[p])
            reach = _prim_reach(l, a, coef)
            lo = np.floor(-fA - reach * bnorm).astype(int)
            hi = np.ceil(1.0 - fA + reach * bnorm).astype(int)
            vals = np.zeros((ncomp, r.shape[0], len(pw)))
            for s1 in range(lo[0], hi[0] + 1):
                for s2 in range(lo[1], hi[1] + 1):
                    for s3 in range(lo[2], hi[2] + 1):
                        S = s1 * cell[0] + s2 * cell[1] + s3 * cell[2]
                        d = r - (A + S)
                        e = coef * np.exp(-a * np.einsum("ij,ij->i", d, d))
                        for ic, (lx, ly, lz) in enumerate(pw):
                            px, py, pz = d[:, 0] ** lx, d[:, 1] ** ly, d[:, 2] ** lz
                            vals[0, :, ic] += px * py * pz * e
                            if deriv:
                                dpx = -2 * a * d[:, 0] ** (lx + 1) + (lx * d[:, 0] ** (lx - 1) if lx else 0.0)
                                dpy = -2 * a * d[:, 1] ** (ly + 1) + (ly * d[:, 1] ** (ly - 1) if ly else 0.0)
                                dpz = -2 * a * d[:, 2] ** (lz + 1) + (lz * d[:, 2] ** (lz - 1) if lz else 0.0)
                                vals[1, :, ic] += dpx * py * pz * e
                                vals[2, :, ic] += px * dpy * pz * e
                                vals[3, :, ic] += px * py * dpz * e
            cols.append(vals)
            exps.extend([a] * len(pw))
            expand.extend(range(int(ao_loc[s]), int(ao_loc[s + 1])))
    return np.concatenate(cols, axis=2), np.array(exps), np.array(expand, dtype=np.int64)


def level_cutoffs(inp) -> np.ndarray:
    """E_alpha = 0.5 min_i (pi N_alpha,i |b_i|)^2  (rule T5)."""
    binv = np.linalg.inv(np.asarray(inp.cell, float))
    bnorm = np.linalg.norm(binv, axis=0)
    return np.array([0.5 * np.min((math.pi * np.asarray(m, float) * bnorm) ** 2) for m in inp.mesh])


def pair_levels(inp, prim_ao_exp: np.ndarray) -> np.ndarray:
    """level[p, q] of every primitive-AO pair: the coarsest alpha with
    E_alpha >= rel_cutoff (a_p + a_q), else level 0 (rule T5)."""
    ecut = level_cutoffs(inp)
    ap = prim_ao_exp[:, None] + prim_ao_exp[None, :]
    lev = np.zeros(ap.shape, dtype=np.int64)
    done = np.zeros(ap.shape, dtype=bool)
    for a in range(inp.nlevel - 1, -1, -1):
        ok = (~done) & (ecut[a] >= inp.rel_cutoff * ap)
        lev[ok] = a
        done |= ok
    return lev


def dense_rho(inp, D: np.ndarray, deriv: int = 0) -> List[np.ndarray]:
    """rho_alpha on every level from the plain definition."""
    out = []
    for level in range(inp.nlevel):
        Phi, pexp, expand = prim_ao_matrix(inp, level, deriv)
        lev = pair_levels(inp, pexp)
        Dp = D[np.ix_(expand, expand)] * (lev == level)
        n1, n2, n3 = (int(x) for x in inp.mesh[level])
        t = Phi[0] @ Dp
        comps = [np.einsum("ij,ij->i", t, Phi[0])]
        if deriv:
            for c in (1, 2, 3):
                comps.append(np.einsum("ij,ij->i", Phi[c] @ Dp, Phi[0]) + np.einsum("ij,ij->i", t, Phi[c]))
        if deriv == 2:      # Eq. (15): tau = 1/2 sum_c diag(Phi_c D Phi_c^T)
            comps.append(0.5 * sum(np.einsum("ij,ij->i", Phi[c] @ Dp, Phi[c]) for c in (1, 2, 3)))
        out.append(np.stack(comps).reshape(len(comps), n1, n2, n3))
    return out


def dense_mat(inp, v: Sequence[np.ndarray], deriv: int = 0) -> np.ndarray:
    """F = sum_alpha F_alpha from the plain definition (includes dV)."""
    omega = abs(np.linalg.det(np.asarray(inp.cell, float)))
    F = np.zeros((inp.nao, inp.nao))
    for level in range(inp.nlevel):
        Phi, pexp, expand = prim_ao_matrix(inp, level, deriv)
        lev = pair_levels(inp, pexp)
        ng = Phi.shape[1]
        dV = omega / ng
        vl = np.asarray(v[level], float).reshape(-1, ng)
        Fp = Phi[0].T @ (vl[0][:, None] * Phi[0])
        if deriv:
            for c in (1, 2, 3):
                X = Phi[c].T @ (vl[c][:, None] * Phi[0])
                Fp += X + X.T
        if deriv == 2:      # Eq. (16) with the 1/2 of PAPER.md:265-268: 1/2 dV sum_c Phi_c^T diag(v_tau) Phi_c
            for c in (1, 2, 3):
                Fp += 0.5 * Phi[c].T @ (vl[4][:, None] * Phi[c])
        Fp = dV * Fp * (lev == level)
        np.add.at(F, (expand[:, None], expand[None, :]), Fp)
    return F
