"""Helpers of the -m gpu parity tests: run the CUDA path through the binding, compare with the oracle."""
import numpy as np

import paper_2603_24881_b200 as gpw

TOL = 1e-11   # north_star: relative, max-norm, on rho (per level and component) and F


def gpu_rho(plan, D, deriv):
    import torch
    nc = {0: 1, 1: 4, 2: 5}[int(deriv)]
    Dd = torch.as_tensor(np.ascontiguousarray(D), device="cuda")
    rho = [torch.full((nc,) + tuple(int(x) for x in m), float("nan"), dtype=torch.float64, device="cuda")
           for m in plan.mesh]
    gpw.gpw_eval_rho(plan, Dd, deriv, rho)
    torch.cuda.synchronize()
    return [r.cpu().numpy() for r in rho]


def gpu_mat(plan, v, deriv):
    import torch
    vd = [torch.as_tensor(np.ascontiguousarray(x), device="cuda") for x in v]
    F = torch.full((plan.nao, plan.nao), float("nan"), dtype=torch.float64, device="cuda")
    gpw.gpw_eval_mat(plan, vd, deriv, F)
    torch.cuda.synchronize()
    return F.cpu().numpy()


def gpu_grad(plan, v, deriv, D, natm):
    import torch
    vd = [torch.as_tensor(np.ascontiguousarray(x), device="cuda") for x in v]
    Dd = torch.as_tensor(np.ascontiguousarray(D), device="cuda")
    g = torch.full((natm, 3), float("nan"), dtype=torch.float64, device="cuda")
    gpw.gpw_eval_grad(plan, vd, deriv, Dd, g)
    torch.cuda.synchronize()
    return g.cpu().numpy()


def relmax(a, b):
    a, b = np.asarray(a), np.asarray(b)
    den = np.abs(b).max() if b.size else 0.0
    if den == 0.0:
        return 0.0 if not np.any(a) else float("inf")
    return float(np.abs(a - b).max() / den)


def check_rho(got, want, tol=TOL):
    worst = 0.0
    for lev, (g, w) in enumerate(zip(got, want)):
        assert g.shape == w.shape
        assert np.isfinite(g).all(), f"level {lev}: non-finite output"
        for c in range(w.shape[0]):
            e = relmax(g[c], w[c])
            assert e <= tol, f"rho level {lev} comp {c}: rel err {e:.3e}"
            worst = max(worst, e)
    return worst


def tile_mask_to_points(mask, mesh):
    """[T1,T2,T3] block mask -> [N1,N2,N3] boolean point mask."""
    m = np.asarray(mask, bool).reshape([int(x) // 4 for x in mesh])
    return np.repeat(np.repeat(np.repeat(m, 4, 0), 4, 1), 4, 2)
