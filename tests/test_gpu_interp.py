"""Parity of gpw_interp_up / gpw_restrict_down (cuFFT path, through the C ABI) with oracle/interp.py (-m gpu).

Eq. (7)-(8).  Tolerance 1e-11 relative to the max-norm (the FFTs are orthogonal transforms:
rounding is O(log N) ulp)."""
import numpy as np
import pytest

import paper_2603_24881_b200 as gpw
from oracle import interp
from paper_2603_24881_b200 import inputs

from gpu_util import TOL, relmax

pytestmark = pytest.mark.gpu


def _run(inp, ncomp, seed):
    import torch
    plan = gpw.gpw_build_pairs(*inp.abi_args())
    assert plan.info["on_device"]
    rng = np.random.default_rng(seed)
    meshes = [tuple(int(x) for x in m) for m in inp.mesh]
    rho = [rng.standard_normal((ncomp,) + m) for m in meshes]
    rho_d = [torch.as_tensor(r, device="cuda") for r in rho]
    fine = torch.full((ncomp,) + meshes[0], float("nan"), dtype=torch.float64, device="cuda")
    gpw.gpw_interp_up(plan, rho_d, ncomp, fine)
    torch.cuda.synchronize()
    got = fine.cpu().numpy()
    for k in range(ncomp):
        want = interp.interp_up(inp.cell, inp.mesh, [r[k] for r in rho])
        assert relmax(got[k], want) <= TOL
    for r, rd in zip(rho, rho_d):   # inputs untouched
        assert np.array_equal(r, rd.cpu().numpy())
    vf = rng.standard_normal((ncomp,) + meshes[0])
    vf_d = torch.as_tensor(vf, device="cuda")
    v_d = [torch.full((ncomp,) + m, float("nan"), dtype=torch.float64, device="cuda") for m in meshes]
    gpw.gpw_restrict_down(plan, vf_d, ncomp, v_d)
    torch.cuda.synchronize()
    assert np.array_equal(vf, vf_d.cpu().numpy())
    for k in range(ncomp):
        want = interp.restrict_down(inp.cell, inp.mesh, vf[k])
        for lev in range(len(meshes)):
            assert relmax(v_d[lev][k].cpu().numpy(), want[lev]) <= TOL
    # adjointness on the GPU outputs alone: dV_f <I rho, v_f> = sum_alpha dV_alpha <rho_alpha, R v_f>
    vol = abs(float(np.linalg.det(inp.cell)))
    lhs = float((fine * vf_d).sum()) * vol / np.prod(meshes[0])
    rhs = sum(float((a * b).sum()) * vol / np.prod(m) for a, b, m in zip(rho_d, v_d, meshes))
    assert abs(lhs - rhs) <= 1e-12 * max(abs(lhs), abs(rhs), 1e-300) * 1e2


@pytest.mark.parametrize("kind", ["cubic", "triclinic"])
def test_small_cells(kind):
    inp = inputs.make_small(kind)
    _run(inp, 1, 1)
    _run(inp, 4, 2)


def test_config1_meshes_with_sphere_ties():
    # cubic 100/60/36/20: integer triples with |m|^2 = (N/2)^2 exist (e.g. (6,8,0) on 20^3): the tie rule decides
    _run(inputs.make_config(1), 1, 3)


def test_config3_triclinic_meshes():
    _run(inputs.make_config(3), 2, 4)


def test_plane_wave_is_transferred_exactly():
    import torch
    inp = inputs.make_config(3)
    plan = gpw.gpw_build_pairs(*inp.abi_args())
    meshes = [tuple(int(x) for x in m) for m in inp.mesh]
    binv = np.linalg.inv(inp.cell)
    G = 2 * np.pi * (binv @ np.array([2.0, -3.0, 1.0]))

    def wave(mesh):
        n = np.stack(np.meshgrid(*[np.arange(k) for k in mesh], indexing="ij"), -1).astype(float)
        return np.cos(((n / np.array(mesh, float)) @ inp.cell) @ G + 0.7)

    rho = [np.zeros((1,) + m) for m in meshes]
    rho[-1][0] = wave(meshes[-1])      # lives on the coarsest level only
    fine = torch.empty((1,) + meshes[0], dtype=torch.float64, device="cuda")
    gpw.gpw_interp_up(plan, [torch.as_tensor(r, device="cuda") for r in rho], 1, fine)
    assert np.abs(fine[0].cpu().numpy() - wave(meshes[0])).max() <= 1e-12


@pytest.mark.parametrize("kind", ["triclinic", "ortho", "cubic"])
def test_gspace_operators_match_oracle(kind):
    """gpw_hartree (Eq. 5-6), gpw_gspace_gradient (Eq. 10), gpw_gspace_divergence (Eq. 14) on the finest mesh
    against oracle/gspace.py (numpy FFT); random fields, so every plane wave is exercised."""
    import torch
    from oracle import gspace
    inp = inputs.make_small(kind)
    plan = gpw.gpw_build_pairs(*inp.abi_args())
    m = tuple(int(x) for x in inp.mesh[0])
    rng = np.random.default_rng(21)
    rho = rng.standard_normal(m)
    w = rng.standard_normal((3,) + m)
    rho_d, w_d = torch.as_tensor(rho, device="cuda"), torch.as_tensor(w, device="cuda")
    vh = torch.full(m, float("nan"), dtype=torch.float64, device="cuda")
    gr = torch.full((3,) + m, float("nan"), dtype=torch.float64, device="cuda")
    dv = torch.full(m, float("nan"), dtype=torch.float64, device="cuda")
    gpw.gpw_hartree(plan, rho_d, vh)
    gpw.gpw_gspace_gradient(plan, rho_d, gr)
    gpw.gpw_gspace_divergence(plan, w_d, dv)
    torch.cuda.synchronize()
    assert np.array_equal(rho, rho_d.cpu().numpy()) and np.array_equal(w, w_d.cpu().numpy())   # inputs untouched
    assert relmax(vh.cpu().numpy(), gspace.hartree(inp.cell, rho)) <= TOL
    want = gspace.gradient(inp.cell, rho)
    for c in range(3):
        assert relmax(gr[c].cpu().numpy(), want[c]) <= TOL
    assert relmax(dv.cpu().numpy(), gspace.divergence(inp.cell, w)) <= TOL
    # Eq. (13): <w, grad rho> = -<div w, rho> on the GPU outputs alone
    lhs, rhs = float((w_d * gr).sum()), -float((dv * rho_d).sum())
    assert abs(lhs - rhs) <= 1e-11 * max(abs(lhs), abs(rhs))
