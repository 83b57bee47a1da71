"""Pins of the interpolation oracle (oracle/interp.py; Eq. 7-8).

The paper prints no worked example for Eq. (7)-(8); the oracle is pinned to what the mathematics fixes:
the two sums written out term by term (no FFT), plane waves (transferred exactly below the cutoff,
annihilated above it), the integral of the density, a resolved periodic Gaussian, and adjointness.
"""
import numpy as np
import pytest

from oracle import interp

CUBIC = np.diag([7.0, 7.0, 7.0])
TRICLINIC = np.array([[6.0, 0.4, 0.3], [0.5, 7.0, -0.2], [0.1, 0.6, 6.5]])
MESHES = np.array([[12, 8, 8], [8, 4, 8], [4, 4, 4]])


def points(cell, mesh):
    N = [int(x) for x in mesh]
    n = np.stack(np.meshgrid(*[np.arange(k) for k in N], indexing="ij"), -1).astype(float)
    return (n / np.array(N, float)) @ cell


@pytest.mark.parametrize("cell", [CUBIC, TRICLINIC])
def test_fft_coding_equals_term_by_term_sums(cell):
    rng = np.random.default_rng(7)
    rho = [rng.standard_normal(tuple(m)) for m in MESHES]
    a = interp.interp_up(cell, MESHES, rho)
    b = interp.interp_up_bruteforce(cell, MESHES, rho)
    assert np.abs(a - b).max() <= 1e-13 * np.abs(b).max()
    vf = rng.standard_normal(tuple(MESHES[0]))
    ra = interp.restrict_down(cell, MESHES, vf)
    rb = interp.restrict_down_bruteforce(cell, MESHES, vf)
    for x, y in zip(ra, rb):
        assert np.abs(x - y).max() <= 1e-13 * max(np.abs(y).max(), 1e-300)


def test_cutoff_is_the_inscribed_sphere():
    # cubic cell edge a, mesh N: G_alpha = pi N / a
    assert interp.g_cut(CUBIC, [12, 12, 12]) == pytest.approx(np.pi * 12 / 7.0, rel=1e-15)
    # anisotropic mesh: the smallest axis decides
    assert interp.g_cut(CUBIC, [12, 8, 16]) == pytest.approx(np.pi * 8 / 7.0, rel=1e-15)
    # kept waves of a 4^3 cubic level: |m| < 2 -> the 3x3x3 cube of m in {-1,0,1} with |m|^2 < 4 (all 27)
    assert int(interp.keep_mask(CUBIC, [4, 4, 4]).sum()) == 27
    # 8^3: |m|^2 < 16 and |m_i| < 4
    m = np.arange(-3, 4)
    want = sum(1 for a in m for b in m for c in m if a * a + b * b + c * c < 16)
    assert int(interp.keep_mask(CUBIC, [8, 8, 8]).sum()) == want


@pytest.mark.parametrize("cell", [CUBIC, TRICLINIC])
def test_plane_wave_below_cutoff_is_transferred_exactly(cell):
    meshes = np.array([[16, 16, 12], [8, 8, 8]])
    binv = np.linalg.inv(cell)
    m = np.array([1, -2, 1])
    G = 2 * np.pi * (binv @ m)
    assert np.linalg.norm(G) < interp.g_cut(cell, meshes[1])
    coarse = np.cos(points(cell, meshes[1]) @ G + 0.3)
    zero = np.zeros(tuple(meshes[0]))
    up = interp.interp_up(cell, meshes, [zero, coarse])
    want = np.cos(points(cell, meshes[0]) @ G + 0.3)
    assert np.abs(up - want).max() <= 1e-13
    # and down: the same wave on the fine mesh arrives unchanged on every level
    down = interp.restrict_down(cell, meshes, want)
    assert np.abs(down[0] - want).max() <= 1e-13
    assert np.abs(down[1] - coarse).max() <= 1e-13


def test_plane_wave_above_cutoff_is_dropped():
    meshes = np.array([[16, 16, 16], [8, 8, 8]])
    binv = np.linalg.inv(CUBIC)
    m = np.array([3, 3, 0])            # representable on 8^3 (|m_i| < 4) but |m| = 4.24 >= 4
    G = 2 * np.pi * (binv @ m)
    coarse = np.cos(points(CUBIC, meshes[1]) @ G)
    up = interp.interp_up(CUBIC, meshes, [np.zeros((16, 16, 16)), coarse])
    assert np.abs(up).max() <= 1e-14
    fine = np.cos(points(CUBIC, meshes[0]) @ G)
    down = interp.restrict_down(CUBIC, meshes, fine)
    assert np.abs(down[1]).max() <= 1e-14
    assert np.abs(down[0] - fine).max() <= 1e-13   # |m| = 4.24 < 8 on the fine level


def test_nyquist_plane_is_dropped():
    meshes = np.array([[8, 8, 8]])
    n = np.arange(8)
    f = np.zeros((8, 8, 8)) + ((-1.0) ** n)[:, None, None]   # m = (4,0,0)
    assert np.abs(interp.interp_up(CUBIC, meshes, [f])).max() <= 1e-15


@pytest.mark.parametrize("cell", [CUBIC, TRICLINIC])
def test_integral_is_conserved(cell):
    rng = np.random.default_rng(3)
    rho = [rng.standard_normal(tuple(m)) for m in MESHES]
    vol = abs(np.linalg.det(cell))
    want = sum(r.sum() * vol / r.size for r in rho)
    up = interp.interp_up(cell, MESHES, rho)
    got = up.sum() * vol / up.size
    assert got == pytest.approx(want, rel=1e-13)


@pytest.mark.parametrize("cell", [CUBIC, TRICLINIC])
def test_adjointness(cell):
    rng = np.random.default_rng(5)
    rho = [rng.standard_normal(tuple(m)) for m in MESHES]
    vf = rng.standard_normal(tuple(MESHES[0]))
    vol = abs(np.linalg.det(cell))
    lhs = (interp.interp_up(cell, MESHES, rho) * vf).sum() * vol / vf.size
    down = interp.restrict_down(cell, MESHES, vf)
    rhs = sum((r * d).sum() * vol / r.size for r, d in zip(rho, down))
    assert lhs == pytest.approx(rhs, rel=1e-12)


def test_resolved_periodic_gaussian_is_interpolated_to_its_closed_form():
    # f(r) = sum_S exp(-a |r - c - S|^2) with a h_coarse^2 = 0.19: its spectrum beyond the coarse cutoff
    # is exp(-G_c^2/(4a)) = exp(-pi^2/(4 a h^2)) ~ 2e-6 relative; interpolation error is of that order
    a, L = 0.25, 7.0
    cell = np.diag([L, L, L])
    meshes = np.array([[16, 16, 16], [8, 8, 8]])
    c = np.array([3.1, 3.6, 2.9])

    def f(mesh):
        r = points(cell, mesh)
        out = np.zeros(r.shape[:-1])
        for s1 in range(-4, 5):
            for s2 in range(-4, 5):
                for s3 in range(-4, 5):
                    d = r - c - L * np.array([s1, s2, s3])
                    out += np.exp(-a * (d * d).sum(-1))
        return out

    up = interp.interp_up(cell, meshes, [np.zeros((16, 16, 16)), f(meshes[1])])
    want = f(meshes[0])
    err = np.abs(up - want).max() / np.abs(want).max()
    assert err < 2e-4
    # ... and a softer Gaussian converges: error falls by orders of magnitude with a
    a = 0.12
    up2 = interp.interp_up(cell, meshes, [np.zeros((16, 16, 16)), f(meshes[1])])
    err2 = np.abs(up2 - f(meshes[0])).max() / np.abs(f(meshes[0])).max()
    assert err2 < 1e-8 and err2 < 1e-3 * err


def test_band_limited_fine_field_is_its_own_image():
    # a field made only of kept waves of level 0 passes through up (as level 0) and down unchanged
    rng = np.random.default_rng(11)
    meshes = np.array([[12, 12, 8]])
    keep = interp.keep_mask(TRICLINIC, meshes[0])
    spec = np.where(keep, np.fft.fftn(rng.standard_normal((12, 12, 8))), 0.0)
    f = np.fft.ifftn(spec).real
    assert np.abs(interp.interp_up(TRICLINIC, meshes, [f]) - f).max() <= 1e-14
    assert np.abs(interp.restrict_down(TRICLINIC, meshes, f)[0] - f).max() <= 1e-14


def test_wave_on_the_cutoff_sphere_is_dropped_whatever_the_rounding():
    # cubic 40^3 level: m = (12,16,0) has |m|^2 = 400 = (N/2)^2 exactly -> |G| = G_alpha -> dropped; for
    # several edge lengths (different roundings of 2 pi m / L) the decision must be the same
    for L in (7.0, 7.3, 9.123456789, 37.2):
        keep = interp.keep_mask(np.diag([L, L, L]), [40, 40, 40])
        assert not keep[12, 16, 0] and not keep[16, 12, 0] and not keep[0, -12, 16]
        assert keep[12, 15, 0] and keep[11, 16, 3]
        m = np.arange(-19, 20)
        want = sum(1 for a in m for b in m for c in m if a * a + b * b + c * c < 400)
        assert int(keep.sum()) == want
