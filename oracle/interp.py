"""Oracle for the inter-level Fourier combination, Eq. (7)-(8) of the paper.

TEST INFRASTRUCTURE, NOT THE PRODUCT (see oracle/__init__.py).  Plain numpy, FP64.

Definition followed (reading A17).  Level alpha has mesh N_alpha = (N1, N2, N3) and grid points
r_n = sum_i (n_i / N_i) a_i.  Its plane waves are G_m = 2 pi sum_i m_i b_i with b_i the i-th COLUMN of
inverse(cell) (so that G_m . r_n = 2 pi sum_i m_i n_i / N_i) and integer m_i in [-N_i/2, N_i/2).  The
Fourier coefficients of a grid function f are

    F(f)(G_m) = (1 / N_grid) sum_n f(r_n) exp(-i G_m . r_n)            (so that f(r_n) = sum_m F(f)(G_m) exp(+i G_m . r_n))

Eq. (8):  rho~_alpha(G) = F(rho_alpha)(G) if |G| < G_alpha, else 0, with the cutoff
G_alpha = min_i pi N_alpha,i |b_i| (the sphere inscribed in the level's FFT box) and, in addition, every
Nyquist plane |m_i| = N_alpha,i / 2 dropped (for a cubic cell the sphere already excludes them).  A plane
wave that sits ON the sphere up to rounding (|G|^2 within 1e-12 relative of G_alpha^2; e.g. m = (12,16,0)
on a cubic 40^3 level) counts as |G| >= G_alpha, so that the decision does not depend on the order of the
floating-point operations (TIE below).
Eq. (7):  rho~(G) = sum_alpha rho~_alpha(G), evaluated on the finest mesh:
    interp_up:      rho_fine(r_n) = sum_G rho~(G) exp(+i G . r_n)
The paper transforms v back "for each of the multiple grids":
    restrict_down:  v_alpha(r_n) = sum_{|G| < G_alpha} F(v_fine)(G) exp(+i G . r_n)
which is the adjoint of interp_up in the sense dV_fine <I rho_alpha, v_fine> = dV_alpha <rho_alpha, R v_fine>.

Two codings: the FFT one below (numpy.fft as the library step) and ``*_bruteforce`` which writes the two
sums above out term by term (tiny meshes only); tests/test_oracle_interp.py pins one against the other and
both against closed forms (plane waves, conservation of the integral, adjointness).
"""
from __future__ import annotations

from typing import List, Sequence

import numpy as np


TIE = 1e-12   # relative width, in |G|^2, of "on the cutoff sphere"


def _bvec(cell) -> np.ndarray:
    """Columns b_i of inverse(cell): u_i = r . b_i."""
    return np.linalg.inv(np.asarray(cell, np.float64).reshape(3, 3))


def g_cut(cell, mesh) -> float:
    """G_alpha = min_i pi N_i |b_i|."""
    binv = _bvec(cell)
    return float(min(np.pi * int(mesh[i]) * np.linalg.norm(binv[:, i]) for i in range(3)))


def _freqs(n: int) -> np.ndarray:
    """signed integer frequencies in FFT order: 0, 1, ..., n/2-1, -n/2, ..., -1"""
    m = np.arange(n)
    return np.where(m < n - n // 2, m, m - n)


def keep_mask(cell, mesh) -> np.ndarray:
    """Boolean [N1,N2,N3] in FFT order: plane wave m is kept on this level (Eq. 8)."""
    binv = _bvec(cell)
    N = [int(x) for x in mesh]
    m1, m2, m3 = np.meshgrid(_freqs(N[0]), _freqs(N[1]), _freqs(N[2]), indexing="ij")
    G = 2.0 * np.pi * (m1[..., None] * binv[:, 0] + m2[..., None] * binv[:, 1] + m3[..., None] * binv[:, 2])
    g2 = (G * G).sum(-1)
    gc = g_cut(cell, mesh)
    ok = g2 < gc * gc * (1.0 - TIE)
    for mi, n in ((m1, N[0]), (m2, N[1]), (m3, N[2])):
        ok &= (2 * np.abs(mi) < n)
    return ok


def _embed_index(n_from: int, n_to: int) -> np.ndarray:
    """position on an n_to-point FFT axis of every signed frequency of an n_from-point axis (n_from <= n_to)"""
    return np.mod(_freqs(n_from), n_to)


def interp_up(cell, meshes, rho: Sequence[np.ndarray]) -> np.ndarray:
    """rho[alpha]: [N1,N2,N3] real on level alpha (finest first).  Returns the total on the finest mesh."""
    Nf = [int(x) for x in meshes[0]]
    spec = np.zeros(Nf, np.complex128)
    for mesh, r in zip(meshes, rho):
        N = [int(x) for x in mesh]
        r = np.asarray(r, np.float64)
        assert list(r.shape) == N
        c = np.fft.fftn(r) / float(np.prod(N))
        c = np.where(keep_mask(cell, mesh), c, 0.0)
        ix = np.ix_(_embed_index(N[0], Nf[0]), _embed_index(N[1], Nf[1]), _embed_index(N[2], Nf[2]))
        spec[ix] += c
    out = np.fft.ifftn(spec) * float(np.prod(Nf))
    return np.ascontiguousarray(out.real)


def restrict_down(cell, meshes, v_fine: np.ndarray) -> List[np.ndarray]:
    """v_fine: [N1,N2,N3] real on the finest mesh.  Returns v_alpha on every level (finest first)."""
    Nf = [int(x) for x in meshes[0]]
    v_fine = np.asarray(v_fine, np.float64)
    assert list(v_fine.shape) == Nf
    c = np.fft.fftn(v_fine) / float(np.prod(Nf))
    out = []
    for mesh in meshes:
        N = [int(x) for x in mesh]
        ix = np.ix_(_embed_index(N[0], Nf[0]), _embed_index(N[1], Nf[1]), _embed_index(N[2], Nf[2]))
        ca = np.where(keep_mask(cell, mesh), c[ix], 0.0)
        out.append(np.ascontiguousarray((np.fft.ifftn(ca) * float(np.prod(N))).real))
    return out


# ------------------------------------------------------------------------------------------------
# the same two sums written out term by term (O(N_grid^2); tiny meshes only) -- no FFT, no index tricks


def _kept_waves(cell, mesh):
    """list of (m, G) kept on this level, by looping over all signed integer triples"""
    binv = _bvec(cell)
    N = [int(x) for x in mesh]
    gc = g_cut(cell, mesh)
    out = []
    for m1 in range(-(N[0] // 2), N[0] - N[0] // 2):
        for m2 in range(-(N[1] // 2), N[1] - N[1] // 2):
            for m3 in range(-(N[2] // 2), N[2] - N[2] // 2):
                if 2 * abs(m1) >= N[0] or 2 * abs(m2) >= N[1] or 2 * abs(m3) >= N[2]:
                    continue
                G = 2.0 * np.pi * (m1 * binv[:, 0] + m2 * binv[:, 1] + m3 * binv[:, 2])
                if float(G @ G) < gc * gc * (1.0 - TIE):
                    out.append(((m1, m2, m3), G))
    return out


def _points(cell, mesh) -> np.ndarray:
    cell = np.asarray(cell, np.float64).reshape(3, 3)
    N = [int(x) for x in mesh]
    n1, n2, n3 = np.meshgrid(np.arange(N[0]), np.arange(N[1]), np.arange(N[2]), indexing="ij")
    frac = np.stack([n1 / N[0], n2 / N[1], n3 / N[2]], -1).reshape(-1, 3)
    return frac @ cell   # r_n = sum_i (n_i/N_i) a_i, rows of cell are a_i


def interp_up_bruteforce(cell, meshes, rho: Sequence[np.ndarray]) -> np.ndarray:
    rf = _points(cell, meshes[0])
    out = np.zeros(rf.shape[0], np.complex128)
    for mesh, r in zip(meshes, rho):
        ra = _points(cell, mesh)
        f = np.asarray(r, np.float64).reshape(-1)
        for _, G in _kept_waves(cell, mesh):
            coef = (f * np.exp(-1j * (ra @ G))).sum() / f.size
            out += coef * np.exp(1j * (rf @ G))
    return out.real.reshape([int(x) for x in meshes[0]])


def restrict_down_bruteforce(cell, meshes, v_fine: np.ndarray) -> List[np.ndarray]:
    rf = _points(cell, meshes[0])
    f = np.asarray(v_fine, np.float64).reshape(-1)
    res = []
    for mesh in meshes:
        ra = _points(cell, mesh)
        out = np.zeros(ra.shape[0], np.complex128)
        for _, G in _kept_waves(cell, mesh):
            coef = (f * np.exp(-1j * (rf @ G))).sum() / f.size
            out += coef * np.exp(1j * (ra @ G))
        res.append(out.real.reshape([int(x) for x in mesh]))
    return res
