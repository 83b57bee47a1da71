"""gpw_eval_mat_static: the integration with its moment workspace in the library's static device array (include/gpw.h),
for callers that cannot call cudaMalloc.  Checked against the existing path (gpw_eval_mat) on the same inputs, to the
tolerance of the parity tests, on calls in a row that leave each other's moments behind in the shared array.

Collected last on purpose (the suite runs with pytest -x); passes alone in a fresh process and after the others."""
import numpy as np
import pytest

import paper_2603_24881_b200 as gpw
from paper_2603_24881_b200 import inputs

from gpu_util import TOL, gpu_mat, relmax

pytestmark = pytest.mark.gpu


def _plan(inp):
    p = gpw.gpw_build_pairs(*inp.abi_args())
    assert p.info["on_device"], "no device copy of the plan: the CUDA path did not run"
    return p


def _static_mat(plan, vd, deriv):
    import torch
    F = torch.full((plan.nao, plan.nao), float("nan"), dtype=torch.float64, device="cuda")
    gpw.gpw_eval_mat_static(plan, vd, deriv, F)
    torch.cuda.synchronize()
    return F.cpu().numpy()


@pytest.mark.parametrize("deriv", [0, 1, 2])
def test_static_workspace_matches_eval_mat_on_calls_in_a_row(deriv):
    """Two plans of different pair layouts used alternately, then one of them twice with different potentials: every
    call finds the previous call's moments in the array and must clear what it accumulates into."""
    import torch
    a = inputs.make_small("triclinic", deriv=deriv)     # f shells: both class ranges, register and group post-pass
    b = inputs.make_small("contracted", deriv=deriv)
    pa, pb = _plan(a), _plan(b)
    va = [a.v(l) for l in range(a.nlevel)]
    vb = [b.v(l) for l in range(b.nlevel)]
    va2 = [1.0 - 0.5 * x[..., ::-1, :].copy() for x in va]   # a second, different potential on plan a
    want = {"a": gpu_mat(pa, va, deriv), "b": gpu_mat(pb, vb, deriv), "a2": gpu_mat(pa, va2, deriv)}
    assert relmax(want["a2"], want["a"]) > 1e-3, "the second potential must change the result"
    dev = {k: [torch.as_tensor(np.ascontiguousarray(x), device="cuda") for x in v] for k, v in (("a", va), ("b", vb), ("a2", va2))}
    _static_mat(pa, dev["a"], deriv)   # first use: looks up the array's address, loads the kernels
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for key, plan in (("a", pa), ("b", pb), ("a", pa), ("a2", pa), ("a2", pa), ("b", pb)):
        F = _static_mat(plan, dev[key], deriv)
        assert np.isfinite(F).all()
        assert relmax(F, want[key]) <= TOL, f"call on {key}: rel err {relmax(F, want[key]):.3e}"
    # nothing was allocated on the device by those calls (the outputs come from torch's cache of the first call)
    assert torch.cuda.mem_get_info()[0] >= free0


def test_static_workspace_config1_fits_and_matches():
    """config 1 (32 H2O, 58 684 pairs): 0.65 M doubles of moments, inside the 2 M limit; two calls in a row."""
    import torch
    inp = inputs.make_config(1)
    plan = _plan(inp)
    assert plan.info["ncoef_total"] <= gpw.GPW_STATIC_MOM_DOUBLES
    deriv = 1
    v = [inp.v(l, ncomp=4) for l in range(inp.nlevel)]
    want = gpu_mat(plan, v, deriv)
    vd = [torch.as_tensor(np.ascontiguousarray(x), device="cuda") for x in v]
    for _ in range(2):
        assert relmax(_static_mat(plan, vd, deriv), want) <= TOL


def test_static_workspace_rejects_a_plan_beyond_the_limit():
    """config 2 (256 H2O) with deriv = 2 needs its moments of degree L and, behind them, those of degree L + 2: more
    than the static array holds.  A clear error, nothing launched, F untouched."""
    import torch
    inp = inputs.make_config(2)
    plan = _plan(inp)
    assert 2 * plan.info["ncoef_total"] > gpw.GPW_STATIC_MOM_DOUBLES   # the degree-(L+2) block is the larger of the two
    vd = [torch.zeros((5,) + tuple(int(x) for x in m), dtype=torch.float64, device="cuda") for m in plan.mesh]
    F = torch.full((plan.nao, plan.nao), 7.0, dtype=torch.float64, device="cuda")
    with pytest.raises(gpw.GpwError) as e:
        gpw.gpw_eval_mat_static(plan, vd, 2, F)
    assert e.value.code == gpw.binding.GPW_EUNSUPPORTED
    assert "GPW_STATIC_MOM_DOUBLES" in str(e.value)
    torch.cuda.synchronize()
    assert bool((F == 7.0).all())
