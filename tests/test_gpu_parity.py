"""Parity of the CUDA path (through the C ABI) with the CPU oracle, element by element (-m gpu).

Tolerance: 1e-11 relative to the max-norm, per level and component for rho, over all entries for F
(north_star; T9).  Levels the oracle leaves exactly zero must be exactly zero."""
import dataclasses

import numpy as np
import pytest

import oracle
import paper_2603_24881_b200 as gpw
from paper_2603_24881_b200 import inputs

from gpu_util import TOL, check_rho, gpu_grad, gpu_mat, gpu_rho, relmax, tile_mask_to_points

pytestmark = pytest.mark.gpu


def _plan(inp, hermi=None):
    a = list(inp.abi_args())
    if hermi is not None:
        a[14] = hermi
    p = gpw.gpw_build_pairs(*a)
    assert p.info["on_device"], "no device copy of the plan: the CUDA path did not run"
    return p


@pytest.mark.parametrize("kind", ["cubic", "triclinic", "ortho", "wrap", "contracted", "resolved"])
@pytest.mark.parametrize("deriv", [0, 1, 2])
@pytest.mark.parametrize("hermi", [1, 0])
def test_small_cells_full_parity(kind, deriv, hermi):
    """deriv = 2: the fifth component is tau (Eq. 15) / the v_tau term of F (Eq. 16), SURVEY 8(f) item 2."""
    inp = inputs.make_small(kind, deriv=deriv, hermi=hermi)
    o = oracle.Oracle.from_inputs(inp)
    plan = _plan(inp)
    D = inp.D()
    if not hermi:   # ordered pairs must work for a non-symmetric D
        D = D + 0.2 * np.random.default_rng(3).standard_normal(D.shape)
    check_rho(gpu_rho(plan, D, deriv), o.eval_rho(D, deriv))
    v = [inp.v(l) for l in range(inp.nlevel)]
    F, Fo = gpu_mat(plan, v, deriv), o.eval_mat(v, deriv)
    assert np.isfinite(F).all()
    assert relmax(F, Fo) <= TOL


@pytest.mark.parametrize("kind", ["cubic", "triclinic", "ortho", "wrap", "contracted", "resolved"])
@pytest.mark.parametrize("deriv", [0, 1])
@pytest.mark.parametrize("hermi", [1, 0])
def test_small_cells_nuclear_gradient(kind, deriv, hermi):
    """gpw_eval_grad (Alg. 3) against the oracle's orc_eval_grad: relative to the largest component."""
    inp = inputs.make_small(kind, deriv=deriv, hermi=hermi)
    o = oracle.Oracle.from_inputs(inp)
    plan = _plan(inp)
    D = inp.D()
    if not hermi:
        D = D + 0.2 * np.random.default_rng(3).standard_normal(D.shape)
    v = [inp.v(l) for l in range(inp.nlevel)]
    g = gpu_grad(plan, v, deriv, D, inp.natm)
    go = o.eval_grad(v, deriv, D)
    assert np.isfinite(g).all()
    assert relmax(g, go) <= TOL
    # the calls of the other kinds on the same plan are not disturbed by the gradient's workspace
    assert relmax(gpu_mat(plan, v, deriv), o.eval_mat(v, deriv)) <= TOL


def test_config1_meta_gga_and_gradient_sampled():
    """cfg 1 (32 waters) with deriv = 2 on a sample of blocks / shell pairs, and the nuclear gradient in full."""
    inp = dataclasses.replace(inputs.make_config(1), deriv=2)
    o = oracle.Oracle.from_inputs(inp)
    plan = _plan(inp)
    D = inp.D()
    rng = np.random.default_rng(11)
    masks = [(rng.random(int(np.prod(m // 4))) < 0.05).astype(np.uint8) for m in inp.mesh]
    ro = o.eval_rho(D, 2, tile_masks=masks)
    rg = gpu_rho(plan, D, 2)
    for lev in range(inp.nlevel):
        pm = tile_mask_to_points(masks[lev], inp.mesh[lev])
        for c in range(5):
            den = np.abs(rg[lev][c]).max()
            if den > 0:
                assert np.abs(rg[lev][c][pm] - ro[lev][c][pm]).max() / den <= TOL
    v = [inp.v(l) for l in range(inp.nlevel)]
    pmask = (rng.random((inp.nshl, inp.nshl)) < 0.05).astype(np.uint8)
    Fo = o.eval_mat(v, 2, pair_mask=pmask)
    F = gpu_mat(plan, v, 2)
    ao = np.concatenate([[0], np.cumsum([(l + 1) * (l + 2) // 2 for l in inp.shl_l])])
    sel = np.zeros((inp.nao, inp.nao), bool)
    for a, b in zip(*np.nonzero(pmask)):
        sel[ao[a]:ao[a + 1], ao[b]:ao[b + 1]] = True
    assert np.abs(F[sel] - Fo[sel]).max() / np.abs(F).max() <= TOL
    v1 = [x[:4] for x in v]
    assert relmax(gpu_grad(plan, v1, 1, D, inp.natm), o.eval_grad(v1, 1, D)) <= TOL


def test_hermi_uses_both_triangles_of_D():
    """hermi = 1 processes unordered pairs with D_ab + D_ba: equals the ordered sum for any D."""
    inp = inputs.make_small("contracted", deriv=1, hermi=1)
    D = np.random.default_rng(5).standard_normal((inp.nao, inp.nao))
    o = oracle.Oracle.from_inputs(inp)
    check_rho(gpu_rho(_plan(inp), D, 1), o.eval_rho(D, 1))


def test_config0_full():
    inp = inputs.make_config(0)
    o = oracle.Oracle.from_inputs(inp)
    plan = _plan(inp)
    D = inp.D()
    for deriv in (0, 1):
        check_rho(gpu_rho(plan, D, deriv), o.eval_rho(D, deriv))
        v = [inp.v(l, 4 if deriv else 1) for l in range(inp.nlevel)]
        assert relmax(gpu_mat(plan, v, deriv), o.eval_mat(v, deriv)) <= TOL


def test_config1_full_32_water():
    inp = inputs.make_config(1)
    o = oracle.Oracle.from_inputs(inp)
    plan = _plan(inp)
    D = inp.D()
    rho = gpu_rho(plan, D, 0)
    check_rho(rho, o.eval_rho(D, 0))
    v = [inp.v(l) for l in range(inp.nlevel)]
    F = gpu_mat(plan, v, 0)
    assert relmax(F, o.eval_mat(v, 0)) <= TOL
    # adjointness on the GPU outputs alone (pin G6)
    vol = abs(np.linalg.det(inp.cell))
    lhs = sum(np.sum(r * x) * vol / r[0].size for r, x in zip(rho, v))
    assert abs(lhs - np.sum(D * F)) <= 1e-11 * max(abs(lhs), 1.0)


def _full_size_parity(inp, tile_frac, pair_frac, seed=0):
    """Full-size launch (the configuration bench.py times) against the oracle -- on everything (frac = 1) or on a
    seeded sample: all visits of the sampled blocks (rho) and of the sampled shell pairs (F).  The masked
    evaluation of the oracle is pinned on the CPU (tests/test_oracle_pins.py).  Errors are relative to the
    ORACLE's max-norm (T9) over what it evaluated; on a sample that is at most the full max-norm, so the
    test is at least as strict as T9."""
    rng = np.random.default_rng(seed)
    o = oracle.Oracle.from_inputs(inp)
    plan = _plan(inp)
    D = inp.D()
    got = gpu_rho(plan, D, inp.deriv)
    if tile_frac >= 1.0:
        check_rho(got, o.eval_rho(D, inp.deriv))
    else:
        masks = []
        for lev in range(inp.nlevel):
            nt = int(np.prod(inp.mesh[lev] // 4))
            m = rng.random(nt) < max(tile_frac, min(1.0, 64.0 / nt))
            masks.append(m.astype(np.uint8))
        want = o.eval_rho(D, inp.deriv, tile_masks=masks)
        for lev in range(inp.nlevel):
            pm = tile_mask_to_points(masks[lev], inp.mesh[lev])
            for c in range(want[lev].shape[0]):
                assert np.isfinite(got[lev][c]).all()
                ref = np.abs(want[lev][c][pm]).max()
                if ref == 0.0:
                    assert not np.any(got[lev][c][pm])
                    continue
                e = np.abs(got[lev][c][pm] - want[lev][c][pm]).max() / ref
                assert e <= TOL, f"rho level {lev} comp {c}: rel err {e:.3e}"
    v = [inp.v(l) for l in range(inp.nlevel)]
    F = gpu_mat(plan, v, inp.deriv)
    assert np.isfinite(F).all()
    if pair_frac >= 1.0:
        assert relmax(F, o.eval_mat(v, inp.deriv)) <= TOL
    else:
        pmask = (rng.random((inp.nshl, inp.nshl)) < pair_frac).astype(np.uint8)
        Fo = o.eval_mat(v, inp.deriv, pair_mask=pmask)
        loc = inp.ao_loc
        sel = np.zeros((inp.nao, inp.nao), bool)
        for sa, sb in zip(*np.nonzero(pmask)):
            sel[loc[sa]:loc[sa + 1], loc[sb]:loc[sb + 1]] = True
        e = np.abs(F[sel] - Fo[sel]).max() / np.abs(Fo[sel]).max()
        assert e <= TOL, f"F rel err {e:.3e}"
    assert np.abs(F - F.T).max() <= 1e-12 * np.abs(F).max()
    # adjointness on the full GPU outputs (pin G6): exact for any truncation
    vol = abs(np.linalg.det(inp.cell))
    lhs = sum(np.sum(r * x) * vol / r[0].size for r, x in zip(got, v))
    assert abs(lhs - np.sum(D * F)) <= 1e-11 * max(abs(lhs), 1.0)


def test_config3_f_shells_triclinic_full():
    """cfg 3 (f shells, triclinic) in full: every grid point of every level and every entry of F."""
    _full_size_parity(inputs.make_config(3), tile_frac=1.0, pair_frac=1.0)


def test_config2_256_water_gga_40_percent():
    """cfg 2, the launch configuration bench.py times: 40 % of the blocks of every level, 40 % of the shell pairs."""
    _full_size_parity(inputs.make_config(2), tile_frac=0.4, pair_frac=0.4)


def test_config4_512_water_gga_f_3_percent():
    """The largest instance (20480 AOs, five levels, 2.1e8 block visits) in the launch configuration bench.py
    times: 3 % of the blocks and of the shell pairs (SURVEY 8(c) contingency for cfg 4: at least 2 %)."""
    _full_size_parity(inputs.make_config(4), tile_frac=0.03, pair_frac=0.03)


@pytest.mark.parametrize("kind", ["cubic", "triclinic", "ortho", "wrap", "contracted", "resolved"])
def test_device_built_lists_equal_oracle_visit_set(kind):
    """Pin G12 as a set, on the lists built on the device: every (pair, lattice image, unwrapped block) triple
    is one of the oracle's T6 visits and vice versa."""
    from test_abi_host import visit_set
    inp = inputs.make_small(kind)
    o = oracle.Oracle.from_inputs(inp)
    plan = _plan(inp, hermi=0)
    got = visit_set(gpw.gpw_plan_export_tasks(plan)[0], gpw.gpw_plan_export_visits(plan))
    assert np.array_equal(got, visit_set(o.tasks()[0], o.visits()))


@pytest.mark.parametrize("kind", ["cubic", "triclinic", "ortho", "wrap", "contracted", "resolved"])
def test_device_built_lists_match_oracle_visit_counts(kind):
    """Pin G12 on the device-built lists: per (level, la, lb) the number of (pair, image, block) visits equals the
    oracle's own enumeration (ordered pairs)."""
    inp = inputs.make_small(kind)
    o = oracle.Oracle.from_inputs(inp)
    plan = _plan(inp, hermi=0)
    ocnt = o.visit_counts()
    assert np.array_equal(plan.info["nvisit_class"], ocnt)
    assert sum(plan.info["nvisit_level"]) == int(ocnt.sum())


def test_device_built_lists_config1_visit_counts():
    inp = inputs.make_config(1)
    o = oracle.Oracle.from_inputs(inp)
    ocnt = o.visit_counts()
    assert np.array_equal(_plan(inp, hermi=0).info["nvisit_class"], ocnt)
    # unordered pairs: every canonical pair but the self pairs stands for two ordered ones
    c1 = _plan(inp, hermi=1).info["nvisit_class"]
    self_visits = 2 * (c1 + np.transpose(c1, (0, 2, 1))) - (ocnt + np.transpose(ocnt, (0, 2, 1)))
    assert (self_visits >= 0).all() and int(self_visits.sum()) % 2 == 0


# ------------------------------------------------------------------------------------------ edge cases
def test_empty_plan_and_empty_levels():
    base = inputs.make_small("cubic", deriv=1)
    # (i) threshold so loose that every primitive is dropped: outputs are exactly zero
    inp = dataclasses.replace(base, tau=1e6)
    plan = _plan(inp)
    assert plan.info["ntask"] == 0
    rho = gpu_rho(plan, inp.D(), 1)
    assert all(not np.any(r) for r in rho)
    assert not np.any(gpu_mat(plan, [inp.v(l) for l in range(inp.nlevel)], 1))
    # (ii) a coarse level no pair is assigned to stays exactly zero
    inp = dataclasses.replace(base, mesh=np.array([[28, 28, 28], [8, 8, 8]], np.int32))
    o = oracle.Oracle.from_inputs(inp)
    plan = _plan(inp)
    assert plan.info["ntask_level"][1] == 0
    rho = gpu_rho(plan, inp.D(), 1)
    assert not np.any(rho[1])
    check_rho(rho, o.eval_rho(inp.D(), 1))


def test_single_s_primitive_and_minimal_mesh():
    """One s function on the smallest legal mesh (one 4x4x4 block per axis pair, many wraps)."""
    cell = np.eye(3) * 3.0
    inp = inputs.make_custom(cell, [[0.4, 1.1, 2.0]], [[(0, [0.9], [1.3])]], [[4, 8, 4]], C=np.ones((1, 1)),
                             tau=1e-10, deriv=1)
    o = oracle.Oracle.from_inputs(inp)
    plan = _plan(inp)
    D = np.ones((1, 1))
    check_rho(gpu_rho(plan, D, 1), o.eval_rho(D, 1))
    v = [inp.v(0)]
    assert relmax(gpu_mat(plan, v, 1), o.eval_mat(v, 1)) <= TOL


def test_long_visit_lists_split_into_items():
    """Diffuse f shells on a coarse mesh: every block is visited by every pair many times over, so the
    lists are cut into several work items that accumulate atomically."""
    cell = np.array([[6.0, 0.3, 0.0], [0.0, 6.2, 0.4], [0.5, 0.0, 5.8]])
    rng = np.random.default_rng(9)
    xyz = rng.uniform(0, 6, (6, 3))
    shells = [[(0, [0.21], [1.0]), (1, [0.17], [0.8]), (2, [0.25], [0.6]), (3, [0.19], [0.5])] for _ in range(6)]
    inp = inputs.make_custom(cell, xyz, shells, [[12, 12, 12]], tau=1e-10, deriv=1, seed=2)
    o = oracle.Oracle.from_inputs(inp)
    plan = _plan(inp)
    assert plan.info["nitem"] > 27          # more items than blocks
    D = inp.D()
    check_rho(gpu_rho(plan, D, 1), o.eval_rho(D, 1))
    v = [inp.v(0)]
    assert relmax(gpu_mat(plan, v, 1), o.eval_mat(v, 1)) <= TOL


def test_repeat_calls_overwrite_outputs():
    inp = inputs.make_small("cubic", deriv=0)
    plan = _plan(inp)
    D = inp.D()
    r1 = gpu_rho(plan, D, 0)
    r2 = gpu_rho(plan, 2.0 * D, 0)
    assert relmax(r2[0], 2.0 * r1[0]) <= 1e-13
    v = [inp.v(0)]
    assert relmax(gpu_mat(plan, v, 0), gpu_mat(plan, v, 0)) <= 1e-13


def test_eval_on_a_side_stream_and_two_plans_interleaved():
    """The eval calls are asynchronous on the caller's stream and keep no state between plans: two plans
    used alternately on a non-default stream give the same results as each alone on the default stream."""
    import torch
    a = inputs.make_small("cubic", deriv=1)
    b = inputs.make_small("triclinic", deriv=1)
    pa, pb = _plan(a), _plan(b)
    ref = {}
    for name, inp, plan in (("a", a, pa), ("b", b, pb)):
        v = [inp.v(l) for l in range(inp.nlevel)]
        ref[name] = (gpu_rho(plan, inp.D(), 1), gpu_mat(plan, v, 1))
    side = torch.cuda.Stream()
    out = {}
    with torch.cuda.stream(side):
        for rep in range(2):
            for name, inp, plan in (("a", a, pa), ("b", b, pb)):
                D = torch.as_tensor(inp.D(), device="cuda")
                rho = [torch.full((4,) + tuple(int(x) for x in m), float("nan"), dtype=torch.float64, device="cuda") for m in plan.mesh]
                vd = [torch.as_tensor(inp.v(l), device="cuda") for l in range(inp.nlevel)]
                F = torch.full((plan.nao, plan.nao), float("nan"), dtype=torch.float64, device="cuda")
                gpw.gpw_eval_rho(plan, D, 1, rho)
                gpw.gpw_eval_mat(plan, vd, 1, F)
                out[name] = (rho, F)
    side.synchronize()
    for name in ("a", "b"):
        rho, F = out[name]
        for got, want in zip(rho, ref[name][0]):
            assert relmax(got.cpu().numpy(), want) <= 1e-13
        assert relmax(F.cpu().numpy(), ref[name][1]) <= 1e-13


def test_host_buffer_entry_points_match_the_resident_path():
    """gpw_eval_rho_host / gpw_eval_mat_host (pinned host arrays in, host arrays out, copies on the library's own
    streams): the same results as the device-pointer calls, also when several calls are queued before the wait."""
    import torch
    inp = inputs.make_small("triclinic", deriv=1)
    plan = _plan(inp)
    D = inp.D()
    v = [inp.v(l) for l in range(inp.nlevel)]
    rho_ref = gpu_rho(plan, D, 1)
    F_ref = gpu_mat(plan, v, 1)
    Dh = torch.as_tensor(np.ascontiguousarray(D)).pin_memory()
    vh = [torch.as_tensor(np.ascontiguousarray(x)).pin_memory() for x in v]
    rho_h = [torch.full(x.shape, float("nan"), dtype=torch.float64).pin_memory() for x in v]
    Fh = torch.full((inp.nao, inp.nao), float("nan"), dtype=torch.float64).pin_memory()
    for _ in range(3):   # queued back to back: the staging buffers are reused without a race
        gpw.gpw_eval_rho_host(plan, Dh, 1, rho_h)
        gpw.gpw_eval_mat_host(plan, vh, 1, Fh)
    gpw.gpw_plan_wait(plan)
    torch.cuda.synchronize()
    for a, b in zip(rho_h, rho_ref):
        assert relmax(a.numpy(), b) <= 1e-13
    assert relmax(Fh.numpy(), F_ref) <= 1e-13
    # pageable memory works too (no overlap), and a different deriv reallocates the staging grids
    rho0 = [torch.empty((1,) + tuple(x.shape[1:]), dtype=torch.float64) for x in v]
    gpw.gpw_eval_rho_host(plan, torch.as_tensor(np.ascontiguousarray(D)), 0, rho0)
    gpw.gpw_plan_wait(plan)
    torch.cuda.synchronize()
    for a, b in zip(rho0, rho_ref):
        assert relmax(a.numpy()[0], b[0]) <= 1e-13


@pytest.mark.parametrize("kind", ["cubic", "triclinic", "wrap", "contracted"])
@pytest.mark.parametrize("hermi", [0, 1])
def test_device_screened_pairs_equal_oracle_task_set(kind, hermi):
    """Pair screening on the device (pairs_device.cu; T2-T5) against the oracle's enumeration: the same set of
    (shell a, prim a, shell b, prim b, T, level) with the same radii; hermi = 1: the canonical half (A14)."""
    inp = inputs.make_small(kind, hermi=hermi)
    o = oracle.Oracle.from_inputs(inp)
    oi, oR = o.tasks()
    gi, gR = gpw.gpw_plan_export_tasks(_plan(inp))
    want = {tuple(int(x) for x in r): float(R) for r, R in zip(oi, oR)}
    if hermi:
        want = {k: R for k, R in want.items()
                if k[1] > k[3] or (k[1] == k[3] and (k[4], k[5], k[6]) >= (0, 0, 0))}
    got = {tuple(int(x) for x in r): float(R) for r, R in zip(gi, gR)}
    assert set(got) == set(want)
    assert max(abs(got[k] - want[k]) / want[k] for k in got) <= 1e-13


@pytest.mark.parametrize("nranks", [2, 3])
def test_sharded_plan_slabs_sum_to_the_whole(nranks):
    """gpw_plan_set_partition: every rank evaluates its n1 slab of every level.  Run here one rank after the other on
    one GPU (no kernel waits for another): the rho slabs are disjoint, tile the grid and equal the unsharded rho to
    rounding, the partial F and gradients sum to the unsharded result."""
    inp = inputs.make_small("triclinic", deriv=1)
    plan = _plan(inp)
    D = inp.D()
    v = [inp.v(l) for l in range(inp.nlevel)]
    rho_full, F_full = gpu_rho(plan, D, 1), gpu_mat(plan, v, 1)
    g_full = gpu_grad(plan, v, 1, D, inp.natm)
    rho_sum = [np.zeros_like(r) for r in rho_full]
    F_sum, g_sum = np.zeros_like(F_full), np.zeros_like(g_full)
    for rank in range(nranks):
        gpw.gpw_plan_set_partition(plan, rank, nranks)
        rho = gpu_rho(plan, D, 1)
        for lev, r in enumerate(rho):
            lo, hi = gpw.gpw_plan_partition_bounds(plan, lev, rank, nranks)
            assert not np.any(r[:, :lo]) and not np.any(r[:, hi:])            # nothing outside the owned slab
            if hi > lo:                                                       # the slab itself: the same work items
                assert relmax(r[:, lo:hi], rho_full[lev][:, lo:hi]) <= 1e-13  # (atomics on split blocks: not bit for bit)
            rho_sum[lev] += r
        # v outside the owned slab is never read: poison it
        vp = []
        for lev, x in enumerate(v):
            lo, hi = gpw.gpw_plan_partition_bounds(plan, lev, rank, nranks)
            y = np.full_like(x, np.nan)
            y[:, lo:hi] = x[:, lo:hi]
            vp.append(y)
        F_sum += gpu_mat(plan, vp, 1)
        g_sum += gpu_grad(plan, vp, 1, D, inp.natm)
    gpw.gpw_plan_set_partition(plan, 0, 1)
    for a, b in zip(rho_sum, rho_full):
        assert relmax(a, b) <= 1e-13
    assert relmax(F_sum, F_full) <= 1e-13 and relmax(g_sum, g_full) <= 1e-13
    assert relmax(gpu_rho(plan, D, 1)[0], rho_full[0]) <= 1e-13              # back to the whole
