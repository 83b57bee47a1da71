"""Pins of oracle/gspace.py (-m "not gpu"): Hartree potential (Eq. 5-6) and Fourier derivatives (Eq. 10, 14)."""
import numpy as np

from oracle import gspace


CELL = np.array([[7.0, 0.3, 0.0], [0.4, 6.5, 0.5], [-0.3, 0.2, 6.0]])


def _points(cell, mesh):
    u = np.stack(np.meshgrid(*[np.arange(n) / n for n in mesh], indexing="ij"), -1)
    return u @ cell


def _periodic_gaussian(cell, mesh, alpha, centre):
    """rho(r) = sum_T (alpha/pi)^{3/2} exp(-alpha |r - c - T|^2): unit charge per cell."""
    r = _points(cell, mesh)
    out = np.zeros(mesh)
    for t1 in range(-3, 4):
        for t2 in range(-3, 4):
            for t3 in range(-3, 4):
                d = r - centre - (t1 * cell[0] + t2 * cell[1] + t3 * cell[2])
                out += (alpha / np.pi) ** 1.5 * np.exp(-alpha * np.einsum("...c,...c->...", d, d))
    return out


def test_hartree_of_a_periodic_gaussian_charge_closed_form():
    """A unit Gaussian charge has F(rho)(G) = exp(-|G|^2 / 4 alpha) exp(-i G . c) / Omega; summing
    4 pi / |G|^2 times that over G term by term (no FFT) must reproduce the FFT route from the sampled rho."""
    mesh, alpha, c = (24, 24, 20), 0.7, np.array([2.0, 3.1, 2.7])
    omega = abs(np.linalg.det(CELL))
    rho = _periodic_gaussian(CELL, mesh, alpha, c)
    assert abs(rho.sum() * omega / rho.size - 1.0) < 1e-12
    v = gspace.hartree(CELL, rho)
    coef = lambda G: np.exp(-(G @ G) / (4 * alpha)) * np.exp(-1j * (G @ c)) / omega
    want = gspace.hartree_direct(CELL, mesh, coef, mmax=9)      # exp(-G^2/4 alpha) < 1e-17 beyond |m| = 9
    assert np.abs(v - want).max() < 1e-12 * np.abs(want).max()
    assert abs(v.mean()) < 1e-14          # the G = 0 term is dropped


def test_hartree_of_a_plane_wave_and_poisson_equation():
    mesh = (16, 12, 20)
    binv = np.linalg.inv(CELL)
    m = np.array([2, -1, 3])
    G = 2 * np.pi * binv @ m
    r = _points(CELL, mesh)
    rho = np.cos(r @ G + 0.3)
    v = gspace.hartree(CELL, rho)
    assert np.abs(v - 4 * np.pi / (G @ G) * rho).max() < 1e-13 * np.abs(v).max()
    # -laplace v_H = 4 pi (rho - mean): div grad through the Fourier derivatives
    rho2 = _periodic_gaussian(CELL, (24, 24, 20), 0.9, np.array([3.0, 3.0, 3.0]))
    v2 = gspace.hartree(CELL, rho2)
    lap = gspace.divergence(CELL, gspace.gradient(CELL, v2))
    assert np.abs(-lap - 4 * np.pi * (rho2 - rho2.mean())).max() < 1e-10 * np.abs(rho2).max() * 4 * np.pi


def test_gradient_and_divergence_of_plane_waves_and_nyquist_dropped():
    mesh = (12, 16, 8)
    binv = np.linalg.inv(CELL)
    r = _points(CELL, mesh)
    G = 2 * np.pi * binv @ np.array([1, 2, -3])
    f = np.sin(r @ G)
    g = gspace.gradient(CELL, f)
    for c in range(3):
        assert np.abs(g[c] - G[c] * np.cos(r @ G)).max() < 1e-13 * np.abs(G).max()
    w = np.stack([np.sin(r @ G) * k for k in (0.5, -1.0, 2.0)])
    d = gspace.divergence(CELL, w)
    assert np.abs(d - (G @ np.array([0.5, -1.0, 2.0])) * np.cos(r @ G)).max() < 1e-12
    # a pure Nyquist wave (m_3 = N_3 / 2) is dropped by all three operators
    n = np.arange(mesh[2])
    ny = np.broadcast_to(np.cos(np.pi * n), mesh).copy()
    assert np.abs(gspace.gradient(CELL, ny)).max() < 1e-14
    assert np.abs(gspace.hartree(CELL, ny)).max() < 1e-14
    assert np.abs(gspace.divergence(CELL, np.stack([ny, ny, ny]))).max() < 1e-14
