"""Pins of the CPU oracle (-m "not gpu").  Nothing here touches the CUDA path.

Each test checks oracle/gpw_oracle.c (the truncated definition the GPU must
match) against something other than itself: the plain definition with
brute-force lattice sums (oracle/dense.py, numpy), closed forms, invariants.
Pin numbers G1..G12 refer to DESIGN.md "Pins".
"""
import dataclasses
import math
import os

import numpy as np
import pytest

import oracle
from oracle import dense, overlap
from paper_2603_24881_b200 import inputs

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def relmax(a, b):
    return float(np.abs(np.asarray(a) - np.asarray(b)).max() / max(np.abs(np.asarray(b)).max(), 1e-300))


def volume(inp):
    return abs(np.linalg.det(inp.cell))


# ---------------------------------------------------------------- radii (T1, T4; Eq. 20)
@pytest.mark.parametrize("l", [0, 1, 2, 3])
@pytest.mark.parametrize("a", [0.08, 0.7, 12.0])
def test_prim_radius_is_largest_root_of_eq20(l, a):
    tau = 1e-10
    coef = inputs.gto_norm(l, a)
    r = oracle.prim_radius(l, a, coef, tau)
    f = lambda x: x * x * coef * x ** l * math.exp(-a * x * x)
    assert abs(f(r) / tau - 1.0) < 1e-9
    # largest root: monotonically below tau beyond r
    xs = r * (1.0 + np.linspace(1e-6, 3.0, 400))
    assert all(f(x) < tau for x in xs)


@pytest.mark.parametrize("la,lb", [(0, 0), (1, 2), (3, 3), (2, 0)])
def test_pair_radius_is_largest_root(la, lb):
    tau, ap, kappa, dA, dB = 1e-10, 0.9, 0.37, 0.8, 0.45
    R = oracle.pair_radius(la, lb, ap, kappa, dA, dB, tau)
    f = lambda x: x * x * kappa * (x + dA) ** la * (x + dB) ** lb * math.exp(-ap * x * x)
    assert abs(f(R) / tau - 1.0) < 1e-9
    xs = R * (1.0 + np.linspace(1e-6, 3.0, 400))
    assert all(f(x) < tau for x in xs)


def test_envelope_bounds_every_component():
    """T4's envelope kappa (r+dA)^la (r+dB)^lb exp(-a_p r^2) bounds |phi_a,i phi_b,j| at distance r from P."""
    rng = np.random.default_rng(3)
    la, lb, aa, ab = 3, 2, 0.6, 1.1
    A, B = np.array([0.3, -0.2, 0.5]), np.array([1.1, 0.9, -0.4])
    ap = aa + ab
    P = (aa * A + ab * B) / ap
    ca, cb = inputs.gto_norm(la, aa), inputs.gto_norm(lb, ab)
    kappa = ca * cb * math.exp(-aa * ab / ap * np.sum((A - B) ** 2))
    dA, dB = np.linalg.norm(P - A), np.linalg.norm(P - B)
    for _ in range(200):
        d = rng.standard_normal(3)
        r = rng.uniform(0.0, 6.0)
        x = P + r * d / np.linalg.norm(d)
        env = kappa * (r + dA) ** la * (r + dB) ** lb * math.exp(-ap * r * r)
        for (ax, ay, az) in inputs.cart_powers(la):
            for (bx, by, bz) in inputs.cart_powers(lb):
                va = ca * np.prod((x - A) ** [ax, ay, az]) * math.exp(-aa * np.sum((x - A) ** 2))
                vb = cb * np.prod((x - B) ** [bx, by, bz]) * math.exp(-ab * np.sum((x - B) ** 2))
                assert abs(va * vb) <= env * (1 + 1e-12)


# ---------------------------------------------------------------- task set, levels, tiles (T2, T5, T6)
def test_task_set_levels_and_tiles_by_brute_force():
    inp = inputs.make_small("triclinic")
    o = oracle.Oracle.from_inputs(inp)
    ints, R = o.tasks()
    cell = inp.cell
    binv = np.linalg.inv(cell)
    # radii by bisection on Eq. (20), independent of the oracle's fixed-point iteration
    def rad(l, a, c):
        f = lambda x: math.log(c) + (l + 2) * math.log(x) - a * x * x - math.log(inp.tau)
        lo, hi = math.sqrt((l + 2) / (2 * a)), 100.0
        for _ in range(200):
            mid = 0.5 * (lo + hi)
            lo, hi = (mid, hi) if f(mid) > 0 else (lo, mid)
        return lo
    prad = [rad(int(inp.shl_l[s]), float(inp.prim_exp[s]), float(inp.prim_coef[s])) for s in range(inp.nshl)]
    got = {tuple(int(x) for x in row[[0, 2, 4, 5, 6]]) for row in ints}
    rr = np.linspace(1e-3, 40.0, 40000)
    n_in = n_out = 0
    for sa in range(inp.nshl):
        for sb in range(inp.nshl):
            A, B = inp.xyz[inp.shl_atom[sa]], inp.xyz[inp.shl_atom[sb]]
            aa, ab = float(inp.prim_exp[sa]), float(inp.prim_exp[sb])
            la, lb = int(inp.shl_l[sa]), int(inp.shl_l[sb])
            for t1 in range(-4, 5):
                for t2 in range(-4, 5):
                    for t3 in range(-4, 5):
                        Bt = B + t1 * cell[0] + t2 * cell[1] + t3 * cell[2]
                        key = (sa, sb, t1, t2, t3)
                        if not np.linalg.norm(A - Bt) < prad[sa] + prad[sb]:
                            assert key not in got          # T2: radii must overlap
                            continue
                        # T4: the pair survives iff its envelope r^2 E(r) reaches tau somewhere
                        ap = aa + ab
                        P = (aa * A + ab * Bt) / ap
                        dA, dB = np.linalg.norm(P - A), np.linalg.norm(P - Bt)
                        kap = inp.prim_coef[sa] * inp.prim_coef[sb] * math.exp(-aa * ab / ap * np.sum((A - Bt) ** 2))
                        peak = np.max(rr ** 2 * kap * (rr + dA) ** la * (rr + dB) ** lb * np.exp(-ap * rr ** 2))
                        if peak > inp.tau * 1.01:
                            assert key in got
                            n_in += 1
                        elif peak < inp.tau * 0.99:
                            assert key not in got
                            n_out += 1
    assert n_in > 100 and n_out > 100 and n_in <= len(got)
    # levels by the numpy rule in oracle/dense.py (independent coding of T5)
    ecut = dense.level_cutoffs(inp)
    for row in ints:
        ap = inp.prim_exp[row[1]] + inp.prim_exp[row[3]]
        ok = [a for a in range(inp.nlevel) if ecut[a] >= inp.rel_cutoff * ap]
        assert row[7] == (max(ok) if ok else 0)
    # tiles (T6) by brute force over a generous index box, for a sample of tasks
    counts = o.visit_counts()
    rng = np.random.default_rng(0)
    total = np.zeros_like(counts)
    for t in range(len(ints)):
        sa, pa, sb, pb, t1, t2, t3, lev = (int(x) for x in ints[t])
        aa, ab = inp.prim_exp[pa], inp.prim_exp[pb]
        A = inp.xyz[inp.shl_atom[sa]]
        Bt = inp.xyz[inp.shl_atom[sb]] + t1 * cell[0] + t2 * cell[1] + t3 * cell[2]
        P = (aa * A + ab * Bt) / (aa + ab)
        N = inp.mesh[lev].astype(int)
        u = P @ binv
        w = R[t] * np.linalg.norm(binv, axis=0) * N
        lo = np.floor(u * N - w).astype(int) - 1
        hi = np.ceil(u * N + w).astype(int) + 1
        g = np.stack(np.meshgrid(*[np.arange(lo[i], hi[i] + 1) for i in range(3)], indexing="ij"), -1).reshape(-1, 3)
        r = (g / N) @ cell
        inside = np.einsum("ij,ij->i", r - P, r - P) <= R[t] ** 2
        tiles = {tuple(x) for x in np.floor_divide(g[inside], 4)}
        total[lev, inp.shl_l[sa], inp.shl_l[sb]] += len(tiles)
    assert np.array_equal(total, counts)


# ---------------------------------------------------------------- G1/G2: against the plain definition
@pytest.mark.parametrize("kind,deriv", [("cubic", 1), ("triclinic", 0), ("ortho", 0), ("wrap", 1), ("contracted", 0)])
def test_truncated_matches_plain_definition(kind, deriv):
    """north_star: untruncated brute force over all lattice images on tiny cells, rel 1e-8 at tau = 1e-10."""
    inp = inputs.make_small(kind, deriv=deriv)
    o = oracle.Oracle.from_inputs(inp)
    D = inp.D()
    v = [inp.v(l) for l in range(inp.nlevel)]
    rho, rho_d = o.eval_rho(D, deriv), dense.dense_rho(inp, D, deriv)
    for a, b in zip(rho, rho_d):
        for c in range(a.shape[0]):
            assert relmax(a[c], b[c]) < 1e-8
    F, F_d = o.eval_mat(v, deriv), dense.dense_mat(inp, v, deriv)
    assert relmax(F, F_d) < 1e-8


def test_truncation_error_scales_with_tau_and_vanishes():
    base = inputs.make_small("cubic", deriv=1)
    D = base.D()
    v = [base.v(l) for l in range(base.nlevel)]
    rho_d, F_d = dense.dense_rho(base, D, 1), dense.dense_mat(base, v, 1)
    errs = []
    for tau in (1e-6, 1e-9, 1e-12, 1e-20):
        inp = dataclasses.replace(base, tau=tau)
        o = oracle.Oracle.from_inputs(inp)
        e1 = max(relmax(a, b) for a, b in zip(o.eval_rho(D, 1), rho_d))
        e2 = relmax(o.eval_mat(v, 1), F_d)
        errs.append(max(e1, e2))
    assert errs[0] > errs[1] > errs[2]
    assert errs[0] < 1e-3 and errs[1] < 1e-6 and errs[2] < 1e-9
    assert errs[3] < 1e-13      # G1: two independent codings of Eq. (3)/(4) agree to rounding


# ---------------------------------------------------------------- G4/G5: analytic overlap, electron count
def test_v_equal_one_gives_analytic_overlap_and_electron_count():
    """Eq. (4) with v = 1 is the overlap; sum_n rho dV = Tr(D S).  Well-resolved grid
    (a_p h^2 <= 0.04 on the finest level), tau = 1e-13: quadrature is exact to rounding."""
    inp = dataclasses.replace(inputs.make_small("resolved"), tau=1e-13, v_const=1.0)
    S = overlap.periodic_overlap(inp)
    o = oracle.Oracle.from_inputs(inp)
    ints, _ = o.tasks()
    assert len(set(ints[:, 7])) == 2          # both levels populated
    F = o.eval_mat([inp.v(l) for l in range(inp.nlevel)], 0)
    assert relmax(F, S) < 2e-11
    D = inp.D()
    rho = o.eval_rho(D, 0)
    nel = sum(r.sum() * volume(inp) / r.size for r in rho)
    assert abs(nel - np.sum(D * S)) < 2e-11 * abs(np.sum(D * S))
    # closed-form diagonal (tests/golden/closed_forms.txt): same basis in a cell large enough that image
    # terms vanish, so the periodic overlap's diagonal is the free-space self overlap
    gold = np.loadtxt(os.path.join(GOLDEN, "closed_forms.txt"))
    free = {tuple(int(x) for x in row[:3]): row[3] for row in gold}
    big = dataclasses.replace(inp, cell=inp.cell * 6.0)
    Sb = overlap.periodic_overlap(big)
    loc = big.ao_loc
    for s in range(big.nshl):
        for i, pw in enumerate(inputs.cart_powers(int(big.shl_l[s]))):
            key = tuple(sorted(pw, reverse=True))
            assert abs(Sb[loc[s] + i, loc[s] + i] - free[key]) < 1e-12


def test_overlap_closed_form_free_space():
    """oracle/overlap.py against the textbook self-overlaps in tests/golden/closed_forms.txt."""
    gold = np.loadtxt(os.path.join(GOLDEN, "closed_forms.txt"))
    for lx, ly, lz, val in gold:
        l = int(lx + ly + lz)
        a = 0.83
        n = inputs.gto_norm(l, a)
        s = 1.0
        for k in (int(lx), int(ly), int(lz)):
            s *= overlap.overlap_1d(k, k, a, a, 0.3, 0.3)[k, k]
        assert abs(n * n * s - val) < 1e-14


# ---------------------------------------------------------------- G6: adjointness
@pytest.mark.parametrize("kind,deriv", [("triclinic", 1), ("contracted", 0), ("wrap", 1)])
def test_adjointness(kind, deriv):
    """sum_alpha dV_alpha <rho_alpha[D], v_alpha> = Tr(D F[v]) exactly (same visit set both ways)."""
    inp = inputs.make_small(kind, deriv=deriv)
    o = oracle.Oracle.from_inputs(inp)
    rng = np.random.default_rng(11)
    D = rng.standard_normal((inp.nao, inp.nao))          # not symmetric on purpose
    v = [inp.v(l) for l in range(inp.nlevel)]
    rho = o.eval_rho(D, deriv)
    F = o.eval_mat(v, deriv)
    lhs = sum(np.sum(r * vv) * volume(inp) / r[0].size for r, vv in zip(rho, v))
    rhs = np.sum(D * F)
    assert abs(lhs - rhs) < 1e-12 * max(abs(lhs), np.abs(D).max() * np.abs(F).max())


# ---------------------------------------------------------------- G7: one s primitive, closed form
def test_single_s_primitive_closed_form():
    a, coef = 0.45, 0.9
    cell = np.array([[6.0, 0, 0], [0.8, 5.5, 0], [0.3, -0.6, 5.0]])
    A = np.array([1.2, 2.2, 3.1])
    inp = inputs.make_custom(cell, [A], [[(0, [a], [coef])]], [[24, 24, 20]], C=np.ones((1, 1)), tau=1e-16)
    o = oracle.Oracle.from_inputs(inp)
    rho = o.eval_rho(np.ones((1, 1)), 0)[0][0]
    r = dense.grid_points(cell, inp.mesh[0])
    # rho = (sum_S coef exp(-a|r-A-S|^2))^2 = coef^2 sum_{S,S'} ...
    phi = np.zeros(r.shape[0])
    for s1 in range(-6, 7):
        for s2 in range(-6, 7):
            for s3 in range(-6, 7):
                d = r - A - (s1 * cell[0] + s2 * cell[1] + s3 * cell[2])
                phi += coef * np.exp(-a * np.einsum("ij,ij->i", d, d))
    assert relmax(rho.reshape(-1), phi ** 2) < 1e-13


# ---------------------------------------------------------------- G8: translation covariance
def test_translation_by_grid_step_and_lattice_vector():
    inp = inputs.make_small("triclinic", deriv=0)
    D = inp.D()
    v = [inp.v(l) for l in range(inp.nlevel)]
    o = oracle.Oracle.from_inputs(inp)
    rho0, F0 = o.eval_rho(D, 0), o.eval_mat(v, 0)
    # shift by one grid step of the coarse level along a2 (= 2... steps of nothing on level 0: use common step)
    # common step: a2/4 is 8 steps on level 0 (N2=32) and 4 steps on level 1 (N2=16)
    shift = inp.cell[1] / 4.0
    inp2 = dataclasses.replace(inp, xyz=inp.xyz + shift)
    o2 = oracle.Oracle.from_inputs(inp2)
    rho2 = o2.eval_rho(D, 0)
    for lev, (r0, r2) in enumerate(zip(rho0, rho2)):
        k = int(inp.mesh[lev][1]) // 4
        assert relmax(r2[0], np.roll(r0[0], k, axis=1)) < 1e-12
    v2 = [np.roll(vv, int(inp.mesh[lev][1]) // 4, axis=2) for lev, vv in enumerate(v)]
    assert relmax(o2.eval_mat(v2, 0), F0) < 1e-12
    # shift by a lattice vector: nothing changes
    inp3 = dataclasses.replace(inp, xyz=inp.xyz + inp.cell[0] - inp.cell[2])
    o3 = oracle.Oracle.from_inputs(inp3)
    for r0, r3 in zip(rho0, o3.eval_rho(D, 0)):
        assert relmax(r3, r0) < 1e-12
    assert relmax(o3.eval_mat(v, 0), F0) < 1e-12


# ---------------------------------------------------------------- G9: symmetry, deriv consistency
def test_symmetry_and_deriv_consistency():
    inp = inputs.make_small("contracted", deriv=1)
    o = oracle.Oracle.from_inputs(inp)
    D = inp.D()
    v = [inp.v(l) for l in range(inp.nlevel)]
    F1 = o.eval_mat(v, 1)
    assert np.abs(F1 - F1.T).max() < 1e-13 * np.abs(F1).max()
    rho1, rho0 = o.eval_rho(D, 1), o.eval_rho(D, 0)
    for a, b in zip(rho1, rho0):
        assert relmax(a[0], b[0]) < 1e-14
    F0 = o.eval_mat([vv[:1] for vv in v], 0)
    Fz = o.eval_mat([np.concatenate([vv[:1], 0 * vv[1:]]) for vv in v], 1)
    assert relmax(Fz, F0) < 1e-14


# ---------------------------------------------------------------- G10: gradient
def test_gradient_against_finite_difference_of_rigid_shift():
    """d_c rho = -d/dR_c rho under a rigid shift of all atoms; tau tiny so the visit set does not matter."""
    base = inputs.make_small("cubic", deriv=1, tau=1e-18)
    D = base.D()
    g = oracle.Oracle.from_inputs(base).eval_rho(D, 1)[0]
    delta = 1e-4
    for c in range(3):
        e = np.zeros(3); e[c] = delta
        rp = oracle.Oracle.from_inputs(dataclasses.replace(base, xyz=base.xyz + e)).eval_rho(D, 0)[0][0]
        rm = oracle.Oracle.from_inputs(dataclasses.replace(base, xyz=base.xyz - e)).eval_rho(D, 0)[0][0]
        fd = -(rp - rm) / (2 * delta)
        assert relmax(g[1 + c], fd) < 2e-7


def test_gradient_against_fourier_derivative_and_integral_of_gradient():
    """Eq. (10): grad rho = F^-1(iG rho~) on a well-resolved grid; constant w, v0 = 0 gives F ~ 0."""
    inp = dataclasses.replace(inputs.make_small("resolved", deriv=1), tau=1e-13,
                              mesh=inputs.make_small("resolved").mesh[:1], rel_cutoff=1e-9)
    o = oracle.Oracle.from_inputs(inp)
    D = inp.D()
    rho = o.eval_rho(D, 1)[0]
    N = inp.mesh[0].astype(int)
    binv = np.linalg.inv(inp.cell)                      # columns b_i
    m = [np.fft.fftfreq(int(n), 1.0 / int(n)) for n in N]
    M = np.stack(np.meshgrid(*m, indexing="ij"), -1)    # integer frequencies
    G = 2 * np.pi * M @ binv.T                           # G = 2 pi sum_i m_i b_i
    rk = np.fft.fftn(rho[0])
    for c in range(3):
        gk = 1j * G[..., c] * rk
        # drop the Nyquist planes (even meshes) where the derivative is ambiguous
        for ax, n in enumerate(N):
            if n % 2 == 0:
                sl = [slice(None)] * 3; sl[ax] = int(n) // 2
                gk[tuple(sl)] = 0
        gr = np.fft.ifftn(gk).real
        assert relmax(rho[1 + c], gr) < 1e-9
    v = np.zeros((4,) + tuple(int(x) for x in N))
    v[1], v[2], v[3] = 0.7, -1.3, 0.4
    F = o.eval_mat([v], 1)
    S = overlap.periodic_overlap(inp)
    assert np.abs(F).max() < 1e-10 * np.abs(S).max()


# ---------------------------------------------------------------- masked (sampled) evaluation
# The full-size GPU parity tests (cfg 2-4) compare against eval_rho(tile_masks=...) / eval_mat(pair_mask=...):
# the mask branch of task_tiles and the tile_mask / pair_mask branches of build_visits.  They are pinned here
# against the unmasked evaluators (themselves pinned above), not against the CUDA path.
@pytest.mark.parametrize("kind,deriv", [("triclinic", 1), ("wrap", 0), ("contracted", 1)])
def test_masked_rho_equals_unmasked_on_marked_blocks_and_zero_elsewhere(kind, deriv):
    inp = inputs.make_small(kind, deriv=deriv)
    o = oracle.Oracle.from_inputs(inp)
    D = inp.D()
    full = o.eval_rho(D, deriv)
    full_counts = o.last_visit_counts()
    rng = np.random.default_rng(21)
    masks = []
    for lev in range(inp.nlevel):
        T = (inp.mesh[lev] // 4).astype(int)
        m = (rng.random(tuple(T)) < 0.3).astype(np.uint8)
        # blocks on the cell faces are reached only through wrapped (folded) visits of pairs near the far face
        m[0, :, -1] = 1
        m[-1, 0, :] = 1
        masks.append(m)
    if inp.nlevel > 1:
        masks[-1] = None          # a level that is not sampled at all
    got = o.eval_rho(D, deriv, tile_masks=masks)
    sub_counts = o.last_visit_counts()
    assert 0 < sub_counts.sum() < full_counts.sum()
    for lev in range(inp.nlevel):
        if masks[lev] is None:
            assert not np.any(got[lev])
            assert sub_counts[lev].sum() == 0
            continue
        pm = np.repeat(np.repeat(np.repeat(masks[lev].astype(bool), 4, 0), 4, 1), 4, 2)
        for c in range(full[lev].shape[0]):
            assert np.array_equal(got[lev][c][pm], full[lev][c][pm])      # same visits, same order: bit for bit
            assert not np.any(got[lev][c][~pm])
        assert np.any(full[lev][0][~pm])                                    # the complement was not empty


@pytest.mark.parametrize("kind,deriv", [("triclinic", 1), ("wrap", 0), ("contracted", 1)])
def test_masked_mat_equals_unmasked_on_marked_shell_blocks(kind, deriv):
    inp = inputs.make_small(kind, deriv=deriv)
    o = oracle.Oracle.from_inputs(inp)
    v = [inp.v(l) for l in range(inp.nlevel)]
    full = o.eval_mat(v, deriv)
    full_counts = o.last_visit_counts()
    rng = np.random.default_rng(22)
    pmask = (rng.random((inp.nshl, inp.nshl)) < 0.35).astype(np.uint8)
    pmask[0, inp.nshl - 1] = 1
    pmask[inp.nshl - 1, 0] = 0            # not symmetric on purpose: (a,b) and (b,a) are separate blocks
    got = o.eval_mat(v, deriv, pair_mask=pmask)
    sub_counts = o.last_visit_counts()
    assert 0 < sub_counts.sum() < full_counts.sum()
    loc = inp.ao_loc
    for sa in range(inp.nshl):
        for sb in range(inp.nshl):
            blk = (slice(loc[sa], loc[sa + 1]), slice(loc[sb], loc[sb + 1]))
            if pmask[sa, sb]:
                assert np.array_equal(got[blk], full[blk])
            else:
                assert not np.any(got[blk])
    assert np.any(full[loc[-2]:, :loc[1]])   # the unmarked block (last shell, first shell) is not empty in the full F


def test_masked_visit_counts_add_up_over_a_partition_of_the_blocks():
    """The masked evaluator visits every (task, block) exactly once over a partition of the stored blocks
    (no visit lost or doubled by the wrapped block id of the mask lookup)."""
    inp = inputs.make_small("wrap", deriv=0)
    o = oracle.Oracle.from_inputs(inp)
    D = inp.D()
    total = o.visit_counts()
    T = (inp.mesh[0] // 4).astype(int)
    part = np.random.default_rng(5).integers(0, 3, tuple(T))
    acc = np.zeros_like(total)
    rho = np.zeros((1,) + tuple(int(x) for x in inp.mesh[0]))
    for k in range(3):
        r = o.eval_rho(D, 0, tile_masks=[(part == k).astype(np.uint8)])
        acc += o.last_visit_counts()
        rho += r[0]
    assert np.array_equal(acc, total)
    assert np.array_equal(rho, o.eval_rho(D, 0)[0])
