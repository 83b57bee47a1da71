"""Oracle for the G-space steps of the Fock build: Hartree potential and Fourier derivatives.

TEST INFRASTRUCTURE, NOT THE PRODUCT (see oracle/__init__.py).  Plain numpy, FP64.

Conventions as in oracle/interp.py: mesh N = (N1, N2, N3), grid points r_n = sum_i (n_i / N_i) a_i, plane waves
G_m = 2 pi sum_i m_i b_i (b_i = i-th column of inverse(cell)), integer m_i in [-N_i/2, N_i/2), Fourier coefficients
F(f)(G_m) = (1 / N_grid) sum_n f(r_n) exp(-i G_m . r_n), so that f(r_n) = sum_m F(f)(G_m) exp(+i G_m . r_n).

    hartree      Eq. (5)-(6), first term of Eq. (6):
                 v_H(r) = sum_{G != 0} (4 pi / |G|^2) F(rho)(G) exp(i G . r)
                 (Eq. 5 writes (1/Omega) sum_G v~(G) e^{iGr} with the continuous transform rho~ = Omega F(rho): the same.)
    gradient     Eq. (10):   grad rho (r) = sum_G i G F(rho)(G) exp(i G . r)
    divergence   Eq. (14):   div w (r)    = sum_G i G . F(w)(G) exp(i G . r)

Reading A26: plane waves on a Nyquist plane (|m_i| = N_i / 2, even N_i) are dropped in all three --
there exp(i G . r_n) with +N_i/2 and -N_i/2 coincide on the grid while G (and, in a non-orthogonal cell, |G|^2)
does not, so the result would depend on an arbitrary choice; a resolved density has no weight there.

Two codings of hartree: the FFT one (numpy.fft as the library step) and hartree_direct, the sum over G written
out term by term from closed-form coefficients; tests/test_oracle_gspace.py pins them against each other on a
periodic Gaussian charge, whose F(rho)(G) = exp(-|G|^2 / 4 alpha) / Omega is known in closed form.
"""
from __future__ import annotations

import numpy as np


def _bvec(cell) -> np.ndarray:
    return np.linalg.inv(np.asarray(cell, np.float64).reshape(3, 3))


def _freqs(n: int) -> np.ndarray:
    m = np.arange(n)
    return np.where(m < n - n // 2, m, m - n)


def gvectors(cell, mesh):
    """(G[N1,N2,N3,3] in FFT order, nyquist[N1,N2,N3] boolean)."""
    binv = _bvec(cell)
    N = [int(x) for x in mesh]
    m = np.stack(np.meshgrid(_freqs(N[0]), _freqs(N[1]), _freqs(N[2]), indexing="ij"), -1)
    G = 2.0 * np.pi * m @ binv.T           # G_c = 2 pi sum_i m_i binv[c, i]
    nyq = np.zeros(N, bool)
    for ax in range(3):
        if N[ax] % 2 == 0:
            nyq |= np.abs(m[..., ax]) == N[ax] // 2
    return G, nyq


def hartree(cell, rho: np.ndarray) -> np.ndarray:
    """v_H on the mesh of rho (Eq. 5-6): 4 pi / |G|^2 on every coefficient, G = 0 and Nyquist planes dropped."""
    G, nyq = gvectors(cell, rho.shape)
    G2 = np.einsum("...c,...c->...", G, G)
    rk = np.fft.fftn(rho) / rho.size
    ker = np.zeros_like(G2)
    ok = (G2 > 0) & ~nyq
    ker[ok] = 4.0 * np.pi / G2[ok]
    return np.fft.ifftn(rk * ker).real * rho.size


def gradient(cell, rho: np.ndarray) -> np.ndarray:
    """[3, N1, N2, N3]: Eq. (10)."""
    G, nyq = gvectors(cell, rho.shape)
    rk = np.fft.fftn(rho) / rho.size
    rk[nyq] = 0.0
    return np.stack([np.fft.ifftn(1j * G[..., c] * rk).real * rho.size for c in range(3)])


def divergence(cell, w: np.ndarray) -> np.ndarray:
    """[N1, N2, N3] from w[3, N1, N2, N3]: Eq. (14)."""
    G, nyq = gvectors(cell, w.shape[1:])
    acc = np.zeros(w.shape[1:], complex)
    for c in range(3):
        wk = np.fft.fftn(w[c]) / w[c].size
        wk[nyq] = 0.0
        acc += 1j * G[..., c] * wk
    return np.fft.ifftn(acc).real * w[0].size


def hartree_direct(cell, mesh, coef, mmax: int) -> np.ndarray:
    """v_H(r_n) = sum_{0 < |m_i| <= mmax} (4 pi / |G_m|^2) coef(G_m) exp(i G_m . r_n), the sum of Eq. (5) written out
    (no FFT) for Fourier coefficients given in closed form by coef(G[..., 3]) -> complex."""
    binv = _bvec(cell)
    N = [int(x) for x in mesh]
    u = np.stack(np.meshgrid(*[np.arange(n) / n for n in N], indexing="ij"), -1)      # fractional coordinates
    out = np.zeros(N)
    rng = np.arange(-mmax, mmax + 1)
    for m1 in rng:
        for m2 in rng:
            for m3 in rng:
                if m1 == 0 and m2 == 0 and m3 == 0:
                    continue
                m = np.array([m1, m2, m3], float)
                G = 2.0 * np.pi * binv @ m
                c = coef(G)
                out += (4.0 * np.pi / (G @ G) * c * np.exp(2j * np.pi * (u @ m))).real
    return out
