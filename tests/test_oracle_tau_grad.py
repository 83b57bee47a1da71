"""Pins of the oracle's meta-GGA (deriv = 2, Eq. 15-16) and nuclear-gradient (Alg. 3) evaluators (-m "not gpu").

Nothing here touches the CUDA path.  Each test checks oracle/gpw_oracle.c against something other than itself:
the plain definition (oracle/dense.py), the analytic kinetic-energy matrix (oracle/overlap.py), closed forms,
finite differences of the energy.
"""
import dataclasses
import math

import numpy as np
import pytest

import oracle
from oracle import dense, overlap
from paper_2603_24881_b200 import inputs


def relmax(a, b):
    return float(np.abs(np.asarray(a) - np.asarray(b)).max() / max(np.abs(np.asarray(b)).max(), 1e-300))


def volume(inp):
    return abs(np.linalg.det(inp.cell))


# ---------------------------------------------------------------- tau: plain definition, closed forms
@pytest.mark.parametrize("kind", ["cubic", "wrap"])
def test_tau_truncated_matches_plain_definition(kind):
    """Untruncated brute force over all lattice images (numpy) against the truncated evaluator.  The radius R_t of
    T4 bounds phi_a phi_b, not its derivatives: every derivative costs a factor <= 2 a R_t + l / R_t at the
    truncation surface, so the truncation error of tau (two derivatives) is ~(2 a_p R_t)^2 times that of rho --
    2e-7 at tau = 1e-10 on these cells -- and vanishes with tau like the others (second half)."""
    inp = inputs.make_small(kind, deriv=2)
    o = oracle.Oracle.from_inputs(inp)
    D = inp.D()
    v = [inp.v(l) for l in range(inp.nlevel)]
    assert v[0].shape[0] == 5
    rho_d, F_d = dense.dense_rho(inp, D, 2), dense.dense_mat(inp, v, 2)
    for tau, tol4 in ((1e-10, 2e-7), (1e-18, 1e-12)):
        o = oracle.Oracle.from_inputs(dataclasses.replace(inp, tau=tau))
        rho = o.eval_rho(D, 2)
        for a, b in zip(rho, rho_d):
            assert a.shape[0] == 5
            for c in range(4):
                assert relmax(a[c], b[c]) < min(1e-8, tol4)
            assert relmax(a[4], b[4]) < tol4
        assert relmax(o.eval_mat(v, 2), F_d) < tol4


def test_tau_components_0_to_3_do_not_depend_on_deriv():
    inp = inputs.make_small("contracted", deriv=2)
    o = oracle.Oracle.from_inputs(inp)
    D = inp.D()
    r2, r1 = o.eval_rho(D, 2), o.eval_rho(D, 1)
    for a, b in zip(r2, r1):
        assert np.array_equal(a[:4], b)
    v = [inp.v(l) for l in range(inp.nlevel)]
    vz = [np.concatenate([x[:4], 0 * x[4:]]) for x in v]
    assert relmax(o.eval_mat(vz, 2), o.eval_mat([x[:4] for x in v], 1)) < 1e-14


def test_tau_single_s_primitive_closed_form():
    """phi = c exp(-a |r - A|^2):  grad phi = -2a (r - A) phi, so tau = 1/2 D 4 a^2 |r - A|^2 phi^2 (cell so large
    that images do not matter; tau = 1e-16 so that truncation does not either)."""
    a, coef, d = 0.45, 0.9, 1.7
    cell = np.eye(3) * 14.0
    A = np.array([6.2, 7.2, 7.1])
    inp = inputs.make_custom(cell, [A], [[(0, [a], [coef])]], [[40, 40, 40]], C=np.ones((1, 1)), tau=1e-16, deriv=2)
    o = oracle.Oracle.from_inputs(inp)
    tau = o.eval_rho(d * np.ones((1, 1)), 2)[0][4]
    r = dense.grid_points(cell, inp.mesh[0]) - A
    r2 = np.einsum("ij,ij->i", r, r)
    want = 0.5 * d * 4 * a * a * r2 * (coef * np.exp(-a * r2)) ** 2
    assert relmax(tau.reshape(-1), want) < 1e-12


def test_v_tau_equal_one_gives_analytic_kinetic_matrix_and_kinetic_energy():
    """Eq. (16) with v_tau = 1 and v_Hxc = 0 is the kinetic-energy matrix 1/2 <grad phi_mu | grad phi_nu>;
    sum_r tau dV = Tr(D T).  Well-resolved grid, tau = 1e-13: the quadrature is exact to rounding."""
    inp = dataclasses.replace(inputs.make_small("resolved", deriv=2), tau=1e-13)
    T = overlap.periodic_overlap(inp, kinetic=True)
    assert np.abs(T - T.T).max() < 1e-14 and np.all(np.linalg.eigvalsh(T) > 0)
    o = oracle.Oracle.from_inputs(inp)
    v = []
    for lev in range(inp.nlevel):
        x = np.zeros((5,) + tuple(int(n) for n in inp.mesh[lev]))
        x[4] = 1.0
        v.append(x)
    F = o.eval_mat(v, 2)
    assert relmax(F, T) < 5e-11
    D = inp.D()
    rho = o.eval_rho(D, 2)
    ekin = sum(r[4].sum() * volume(inp) / r[4].size for r in rho)
    assert abs(ekin - np.sum(D * T)) < 5e-11 * abs(np.sum(D * T))
    # free-space closed form: the kinetic energy of a normalised s Gaussian is 3a/2
    big = inputs.make_custom(np.eye(3) * 60.0, [[30.0, 30.0, 30.0]], [[(0, [0.37], [inputs.gto_norm(0, 0.37)])]], [[4, 4, 4]])
    assert abs(overlap.periodic_overlap(big, kinetic=True)[0, 0] - 1.5 * 0.37) < 1e-13


@pytest.mark.parametrize("kind", ["triclinic", "wrap"])
def test_tau_adjointness(kind):
    inp = inputs.make_small(kind, deriv=2)
    o = oracle.Oracle.from_inputs(inp)
    D = np.random.default_rng(11).standard_normal((inp.nao, inp.nao))          # not symmetric on purpose
    v = [inp.v(l) for l in range(inp.nlevel)]
    rho, F = o.eval_rho(D, 2), o.eval_mat(v, 2)
    lhs = sum(np.sum(r * vv) * volume(inp) / r[0].size for r, vv in zip(rho, v))
    rhs = np.sum(D * F)
    assert abs(lhs - rhs) < 1e-12 * max(abs(lhs), np.abs(D).max() * np.abs(F).max())


# ---------------------------------------------------------------- nuclear gradient
def _energy(inp, D, v, deriv):
    """E = sum_alpha dV sum_r [v0 rho + w . grad rho] from the collocation evaluator."""
    rho = oracle.Oracle.from_inputs(inp).eval_rho(D, deriv)
    return sum(np.sum(r * vv) * volume(inp) / r[0].size for r, vv in zip(rho, v))


def _mini(kind, deriv):
    """Two-atom cells on coarse meshes, sized for 13 evaluations at tau = 1e-18."""
    if kind == "cubic":
        return dataclasses.replace(inputs.make_small("cubic", deriv=deriv, tau=1e-18), mesh=np.array([[16, 16, 16]], np.int32))
    # sheared cell, s p d f | p d (one shell with three primitives), two levels
    cell = np.array([[5.5, 0.4, 0.3], [0.6, 5.0, -0.4], [-0.5, 0.7, 4.8]])
    xyz = np.array([[1.0, 1.4, 1.9], [3.1, 2.9, 2.4]])
    n = inputs.gto_norm
    shells = [[(0, [0.55], [n(0, 0.55)]), (1, [0.7], [n(1, 0.7)]), (2, [0.9], [n(2, 0.9)]), (3, [0.8], [n(3, 0.8)])],
              [(1, [1.3, 0.6, 0.45], [0.3 * n(1, 1.3), 0.5 * n(1, 0.6), 0.4 * n(1, 0.45)]), (2, [0.5], [n(2, 0.5)])]]
    return inputs.make_custom(cell, xyz, shells, [[16, 12, 12], [8, 8, 8]], tau=1e-18, rel_cutoff=6.0, deriv=deriv, seed=8)


@pytest.mark.parametrize("kind,deriv", [("cubic", 0), ("sheared", 0), ("sheared", 1)])
def test_nuclear_gradient_against_finite_differences_of_the_energy(kind, deriv):
    """dE/dR_A by central differences of E(R) with v, w fixed; tau tiny so that the visit set does not matter.
    A smooth v (a few plane waves) keeps the finite-difference error at delta^2."""
    base = _mini(kind, deriv)
    if kind == "sheared":
        assert len(set(oracle.Oracle.from_inputs(base).tasks()[0][:, 7])) == 2      # both levels populated
    rng = np.random.default_rng(4)
    D = rng.standard_normal((base.nao, base.nao))          # not symmetric on purpose
    binv = np.linalg.inv(base.cell)
    v = []
    for lev in range(base.nlevel):
        r = dense.grid_points(base.cell, base.mesh[lev])
        comps = []
        for c in range(base.ncomp):
            m = rng.integers(-1, 2, 3)
            comps.append(np.cos(2 * np.pi * (r @ binv) @ m + rng.uniform(0, 6)) * rng.uniform(0.5, 1.5))
        v.append(np.stack(comps).reshape((base.ncomp,) + tuple(int(x) for x in base.mesh[lev])))
    g = oracle.Oracle.from_inputs(base).eval_grad(v, deriv, D)
    assert g.shape == (base.natm, 3)
    delta = 1e-4
    for A in range(base.natm):
        for c in range(3):
            e = np.zeros_like(base.xyz); e[A, c] = delta
            fd = (_energy(dataclasses.replace(base, xyz=base.xyz + e), D, v, deriv) -
                  _energy(dataclasses.replace(base, xyz=base.xyz - e), D, v, deriv)) / (2 * delta)
            assert abs(g[A, c] - fd) < 2e-7 * np.abs(g).max(), (A, c, g[A, c], fd)


def test_nuclear_gradient_translational_sum_rule():
    """A rigid shift of all atoms shifts rho: sum_A dE/dR_A = -dV sum_r v0 grad rho (deriv = 0, any truncation,
    because every pair moves rigidly with its two centres)."""
    inp = inputs.make_small("wrap", deriv=0)
    o = oracle.Oracle.from_inputs(inp)
    D = inp.D()
    v = [inp.v(l) for l in range(inp.nlevel)]
    g = o.eval_grad(v, 0, D)
    rho1 = o.eval_rho(D, 1)
    want = np.array([-sum(np.sum(r[1 + c] * vv[0]) * volume(inp) / vv[0].size for r, vv in zip(rho1, v)) for c in range(3)])
    assert np.abs(g.sum(axis=0) - want).max() < 1e-12 * np.abs(g).max()
