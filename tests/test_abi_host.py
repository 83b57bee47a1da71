"""C-ABI library: loads, exports every symbol of include/gpw.h, argument validation, and the host plan
builder (gpw_build_pairs) against the oracle's own enumeration (pin G12).  No GPU, no compute calls."""
import ctypes
import os
import re

import numpy as np
import pytest

import oracle
import paper_2603_24881_b200 as gpw
from paper_2603_24881_b200 import binding, inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "gpw.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(gpw_[a-z_]+)\s*\(", hdr))
    assert {"gpw_build_pairs", "gpw_eval_rho", "gpw_eval_mat"} <= declared
    lib = gpw.load_library()
    for name in declared:
        assert hasattr(lib, name), name
    assert declared == set(binding.EXPORTS)


def _build(inp, hermi=None, **kw):
    args = list(inp.abi_args())
    if hermi is not None:
        args[14] = hermi
    return gpw.gpw_build_pairs(*args)


def test_argument_validation():
    inp = inputs.make_small("cubic")
    a = list(inp.abi_args())

    def expect(code, idx, val):
        b = list(a)
        b[idx] = val
        with pytest.raises(gpw.GpwError) as e:
            gpw.gpw_build_pairs(*b)
        assert e.value.code == code

    expect(binding.GPW_EINVAL, 11, np.array([[30, 28, 28]]))            # mesh not a multiple of 4
    expect(binding.GPW_EINVAL, 12, 0.0)                                   # tau
    expect(binding.GPW_EINVAL, 0, np.zeros((3, 3)))                       # singular cell
    expect(binding.GPW_EUNSUPPORTED, 5, np.array([4] * inp.nshl, np.int32))   # g shells
    expect(binding.GPW_EINVAL, 8, -inp.prim_exp)                          # exponent <= 0
    expect(binding.GPW_EINVAL, 14, 2)                                     # hermi
    # a coarse level finer than level 0 on one axis (the spectrum embedding of gpw_interp_up would not fit)
    b = list(inputs.make_small("triclinic").abi_args())
    b[11] = np.array([[36, 32, 28], [20, 36, 16]])
    with pytest.raises(gpw.GpwError) as e:
        gpw.gpw_build_pairs(*b)
    assert e.value.code == binding.GPW_EINVAL


def test_pair_too_sharp_for_the_mesh_is_refused():
    """A primitive so sharp that exp(-a_p d^2) underflows at the corner of its own 4x4x4 blocks would come out as
    zeros from the corner-anchored Gaussian recursion (Eq. 24-25): gpw_build_pairs refuses it instead."""
    cell = np.eye(3) * 8.0
    ok = inputs.make_custom(cell, [[1.0, 2.0, 3.0]], [[(0, [40.0], [1.0])]], [[32, 32, 32]], C=np.ones((1, 1)))
    gpw.gpw_build_pairs(*ok.abi_args())                       # a_p h^2 = 5: crude quadrature, still representable
    sharp = inputs.make_custom(cell, [[1.0, 2.0, 3.0]], [[(0, [400.0], [1.0])]], [[32, 32, 32]], C=np.ones((1, 1)))
    with pytest.raises(gpw.GpwError) as e:
        gpw.gpw_build_pairs(*sharp.abi_args())
    assert e.value.code == binding.GPW_EUNSUPPORTED and "sharp" in str(e.value)


@pytest.mark.parametrize("kind", ["triclinic", "ortho", "wrap", "contracted"])
def test_plan_matches_oracle_enumeration(kind):
    inp = inputs.make_small(kind)
    o = oracle.Oracle.from_inputs(inp)
    oi, oR = o.tasks()
    ocnt = o.visit_counts()
    # ordered pairs: identical set, radii and per-class visit counts
    p0 = _build(inp, hermi=0)
    ints, R = gpw.gpw_plan_export_tasks(p0)
    assert len(ints) == len(oi)
    key = lambda rows, rr: sorted((tuple(int(x) for x in r), float(x)) for r, x in zip(rows, rr))
    got, want = key(ints, R), key(oi, oR)
    assert [g[0] for g in got] == [w[0] for w in want]
    assert max(abs(g[1] - w[1]) for g, w in zip(got, want)) < 1e-12
    assert np.array_equal(p0.info["nvisit_class"], ocnt)
    assert sum(p0.info["nvisit_level"]) == int(ocnt.sum())
    # unordered pairs (hermi): the canonical half; mirrored pairs (b, a, -T) complete the ordered set
    p1 = _build(inp, hermi=1)
    ints1, R1 = gpw.gpw_plan_export_tasks(p1)
    full = set()
    for r in ints1:
        sa, pa, sb, pb, t0, t1, t2, lev = (int(x) for x in r)
        full.add((sa, pa, sb, pb, t0, t1, t2, lev))
        full.add((sb, pb, sa, pa, -t0, -t1, -t2, lev))
        assert pa > pb or (pa == pb and (t0, t1, t2) >= (0, 0, 0))
    assert full == {w[0] for w in want}
    # visits: every canonical pair but the self pairs (a == b, T == 0) stands for two ordered pairs
    c1 = p1.info["nvisit_class"]
    sym = c1 + np.transpose(c1, (0, 2, 1))
    osym = ocnt + np.transpose(ocnt, (0, 2, 1))
    self_visits = 2 * sym - osym
    assert (self_visits >= 0).all() and int(self_visits.sum()) > 0 and int(self_visits.sum()) % 2 == 0


def visit_set(tasks_ints, visits):
    """Sorted unique rows (shl_a, prim_a, shl_b, prim_b, T0, T1, T2, level, b1, b2, b3) of a task table and its
    visit rows; a (pair, block) visit listed twice fails."""
    rows = np.concatenate([np.asarray(tasks_ints)[visits[:, 0]], visits[:, 1:]], axis=1).astype(np.int64)
    uniq = np.unique(rows, axis=0)
    assert len(uniq) == len(rows), "a (pair, block) visit is listed twice"
    return uniq


@pytest.mark.parametrize("kind", ["triclinic", "wrap", "contracted"])
def test_visit_lists_equal_oracle_visit_set(kind):
    """Pin G12 as a SET: every (pair, lattice image, unwrapped block) triple of the plan's collocation lists is one
    of the oracle's T6 visits and vice versa (ordered pairs).  Without a GPU this checks the host list builder;
    tests/test_gpu_parity.py repeats it on the device-built lists."""
    inp = inputs.make_small(kind)
    o = oracle.Oracle.from_inputs(inp)
    want = visit_set(o.tasks()[0], o.visits())
    plan = _build(inp, hermi=0)
    got = visit_set(gpw.gpw_plan_export_tasks(plan)[0], gpw.gpw_plan_export_visits(plan))
    assert np.array_equal(got, want)
    assert len(got) == int(o.visit_counts().sum())


def test_eval_without_device_fails_loudly():
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA device present")
    inp = inputs.make_small("cubic")
    plan = _build(inp)
    assert not plan.info["on_device"]
    lib = gpw.load_library()
    dummy = (ctypes.c_void_p * plan.nlevel)(*[8] * plan.nlevel)
    rc = lib.gpw_eval_rho(plan._h, ctypes.c_void_p(8), 0, dummy, None)
    assert rc == binding.GPW_ECUDA
    assert b"no CPU path" in lib.gpw_last_error()
    rc = lib.gpw_eval_mat(plan._h, dummy, 0, ctypes.c_void_p(8), None)
    assert rc == binding.GPW_ECUDA
    rc = lib.gpw_interp_up(plan._h, dummy, 1, ctypes.c_void_p(8), None)
    assert rc == binding.GPW_ECUDA and b"no CPU path" in lib.gpw_last_error()
    rc = lib.gpw_restrict_down(plan._h, ctypes.c_void_p(8), 1, dummy, None)
    assert rc == binding.GPW_ECUDA and b"no CPU path" in lib.gpw_last_error()


def test_model_flops_convention():
    inp = inputs.make_small("cubic")
    plan = _build(inp, hermi=0)
    cls = plan.info["nvisit_class"]
    nc = [1, 3, 6, 10]
    want0 = sum(64 * int(cls[:, a, b].sum()) * (2 * nc[a] * nc[b] + 2 * (nc[a] + nc[b]) + 4) for a in range(4) for b in range(4))
    want1 = sum(64 * int(cls[:, a, b].sum()) * (4 * nc[a] * nc[b] + 10 * (nc[a] + nc[b]) + 8) for a in range(4) for b in range(4))
    assert gpw.model_flops(plan.info, 0) == want0 and gpw.model_flops(plan.info, 1) == want1
