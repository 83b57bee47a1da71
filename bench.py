#!/usr/bin/env python
"""bench.py -- one JSON line for the multigrid GPW collocation + integration hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2] [--deriv d] [--tau t] [--rel-cutoff c] [--impl reference]

A step is one pass of the hot path on one synthetic workload: gpw_eval_rho on every level followed by
gpw_eval_mat (the plan of gpw_build_pairs is built once beforehand; setup time is reported, not timed
into the metric).  The metric is BASELINE.json's: FP64 GFLOP/s of eval_rho + eval_mat, counted with the
fixed flop model of SURVEY.md 8(d) (what the direct evaluation of Alg. 1/2 must compute per visited
grid point), the same convention for every kernel design.  The roofline object is for the dominant
kernel against the FP64 FMA peak; cpu_baseline is the oracle (oracle/, test infrastructure) timed on a
bounded sample of the same workload on this box's host cores.  --impl reference times that oracle alone.
With N > 1 (torchrun) every rank runs its own independent workload of the same shape (weak scaling, no
data-path collective): the path is specified for one GPU.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "fp64_model_gflops_eval_rho_plus_eval_mat"
UNIT = "GFLOP/s"
NOMINAL_FP64_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12   # SMs x FP64 lanes x 2 x max SM clock


class ClockSampler(threading.Thread):
    """nvidia-smi clocks and throttle reasons during the timed region (B200_PROFILING.md recipe)."""

    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index = index
        self.rows = []
        self.proc = None

    def run(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.FIELDS}", "--format=csv,noheader,nounits", "-lms", "100",
                 "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            for line in self.proc.stdout:
                self.rows.append((time.time(), [x.strip() for x in line.split(",")]))
        except Exception:
            pass

    def stop(self):
        if self.proc is not None:
            self.proc.terminate()

    def summary(self, t0: float, t1: float) -> dict:
        rows = [r for (t, r) in self.rows if t0 <= t <= t1 and len(r) >= 7] or [r for (_, r) in self.rows if len(r) >= 7]
        if not rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        sm = [float(r[0]) for r in rows]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(r[3 + i].lower().startswith("active") for r in rows)]
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(rows[0][1]), "reasons": reasons,
                "power_w_max": max(float(r[2]) for r in rows), "samples": len(rows)}


def csrc_sha() -> str:
    """Hash of the kernel sources: ties the committed ncu figures (profiles/traffic.json) to the build they were taken on."""
    import hashlib
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2603_24881_b200", "csrc")
    for f in sorted(os.listdir(d)):
        if f.endswith((".cu", ".cuh", ".h", ".cpp")):
            h.update(f.encode())
            h.update(open(os.path.join(d, f), "rb").read())
    return h.hexdigest()[:16]


def model_flops_from_counts(counts, deriv: int) -> float:
    nc = [1, 3, 6, 10]
    tot = 0.0
    for la in range(4):
        for lb in range(4):
            w0 = 2 * nc[la] * nc[lb] + 2 * (nc[la] + nc[lb]) + 4
            w1 = 4 * nc[la] * nc[lb] + 10 * (nc[la] + nc[lb]) + 8
            w = (w0, w1, w1 + w0)[int(deriv)]   # deriv = 2: the tau contraction counted as one more value-like contraction
            tot += 64.0 * float(counts[:, la, lb].sum()) * w
    return tot


def rank_seed(config: int, rank: int):
    """Seed of rank's workload: rank 0 takes the config's own seed, every other rank an independent workload
    of the same shape (weak scaling, no data-path collective)."""
    from paper_2603_24881_b200 import inputs
    return None if rank == 0 else inputs.BASE_SEED + config + 1000 * rank


def reduce_over_ranks(ms_step: float, flops_step: float, dist, device):
    """Whole-job figures: the slowest rank's time per step and the flops of all ranks."""
    if dist is None:
        return ms_step, flops_step
    import torch
    t = torch.tensor([ms_step], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    f = torch.tensor([flops_step], dtype=torch.float64, device=device)
    dist.all_reduce(f, op=dist.ReduceOp.SUM)
    return float(t.item()), float(f.item())


def time_oracle_sample(inp, budget_s: float = 20.0):
    """The oracle as it stands on a bounded, seeded sample of the workload: all visits of a random set
    of 4x4x4 blocks (eval_rho) and of a random set of shell pairs (eval_mat).  Returns (GFLOP/s in the
    bench's unit, cores, description).  The oracle sums ORDERED pairs; its visits count half, so that
    the figure is in the same unit as the GPU's (unordered pairs, hermi = 1)."""
    import oracle
    o = oracle.Oracle.from_inputs(inp)
    rng = np.random.default_rng(12345)
    D = inp.D() if inp.nao <= 8192 else None
    if D is None:   # very large nao: a random symmetric matrix has the same cost
        D = rng.standard_normal((inp.nao, inp.nao))
    tot_vis = float(o.visit_counts().sum())
    # size the sample from a rough rate (visits per second) measured on a tiny first bite
    frac_t, frac_p = 2e-4, 2e-4
    best = None
    for _ in range(3):
        masks = [(rng.random(int(np.prod(m // 4))) < frac_t).astype(np.uint8) for m in inp.mesh]
        pmask = (rng.random((inp.nshl, inp.nshl)) < frac_p).astype(np.uint8)
        v = [inp.v(l) for l in range(inp.nlevel)]
        t0 = time.time()
        o.eval_rho(D, inp.deriv, tile_masks=masks)
        t1 = time.time()
        c_rho = o.last_visit_counts()
        o.eval_mat(v, inp.deriv, pair_mask=pmask)
        t2 = time.time()
        c_mat = o.last_visit_counts()
        fl = 0.5 * (model_flops_from_counts(c_rho, inp.deriv) + model_flops_from_counts(c_mat, inp.deriv))
        el = t2 - t0
        best = (fl / el / 1e9, f"{int(c_rho.sum())} block visits of {int(sum(m.sum() for m in masks))} random 4x4x4 blocks "
                f"(eval_rho, {t1 - t0:.1f} s) + {int(c_mat.sum())} block visits of {int(pmask.sum())} random shell pairs "
                f"(eval_mat, {t2 - t1:.1f} s) of {inp.name}; ordered-pair visits counted half")
        best = best + (el,)
        if el > 0.5 * budget_s:
            break
        scale = min(50.0, 0.8 * budget_s / max(el, 1e-3))
        frac_t, frac_p = min(1.0, frac_t * scale), min(1.0, frac_p * scale)
    return best[0], oracle.num_threads(), best[1], best[2]


def run_reference(args, inp):
    vals, secs = [], []
    desc, cores = "", 0
    for i in range(args.warmup + args.steps):
        g, cores, desc, el = time_oracle_sample(inp, budget_s=max(4.0, 60.0 / max(1, args.warmup + args.steps)))
        if i >= args.warmup:
            vals.append(g)
            secs.append(el)
    val = float(np.mean(vals))
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * float(np.mean(secs)),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": inp.name},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config index (default 2: 256 waters, GGA)")
    ap.add_argument("--deriv", type=int, default=None, choices=[0, 1, 2],
                    help="override the config's derivative level (2 = meta-GGA: a fifth component, tau / v_tau)")
    ap.add_argument("--tau", type=float, default=None, help="override the screening threshold of Eq. 20 (configs: 1e-10; the paper used 1e-6)")
    ap.add_argument("--rel-cutoff", type=float, default=None, help="override the level-assignment constant (configs: 20; reading A6)")
    ap.add_argument("--shard", action="store_true",
                    help="N > 1: ONE workload sharded over the ranks (gpw_plan_set_partition: an n1 slab of every level per "
                         "rank, partial F summed by an NCCL all-reduce inside the step; strong scaling) instead of one "
                         "independent workload per rank")
    ap.add_argument("--impl", default="gpw", choices=["gpw", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    import dataclasses
    from paper_2603_24881_b200 import inputs

    def workload(seed=None):
        inp = inputs.make_config(args.config, seed=seed)
        over = {k: v for k, v in (("deriv", args.deriv), ("tau", args.tau), ("rel_cutoff", args.rel_cutoff)) if v is not None}
        if over:
            inp = dataclasses.replace(inp, name=inp.name + "".join(f"+{k}={v:g}" for k, v in over.items()), **over)
        return inp

    if args.impl == "reference":
        if rank == 0:
            run_reference(args, workload())
        return

    import torch
    import paper_2603_24881_b200 as gpw
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU path)"
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    W = max(3, args.warmup)

    # every rank its own independent workload of the same shape (weak scaling); --shard: the same workload on every
    # rank, each evaluating its slab
    shard = args.shard and world > 1
    inp = workload(None if shard else rank_seed(args.config, rank))
    deriv, nc = inp.deriv, inp.ncomp
    t0 = time.time()
    plan = gpw.gpw_build_pairs(*inp.abi_args())
    build_s = time.time() - t0
    info = plan.info
    assert info["on_device"]
    flops_step = 2.0 * gpw.model_flops(info, deriv)       # eval_rho + eval_mat
    flops_call = gpw.model_flops(info, deriv)
    if shard:
        gpw.gpw_plan_set_partition(plan, rank, world)
        flops_step /= world      # summed over the ranks again below: the job's flops are those of the one workload

    # resident inputs / outputs
    C = torch.as_tensor(inp.C, device="cuda")
    D = (C @ C.T).contiguous()
    gen = torch.Generator(device="cuda").manual_seed(inp.seed)
    shapes = [(nc,) + tuple(int(x) for x in m) for m in inp.mesh]
    v = [torch.randn(s, dtype=torch.float64, device="cuda", generator=gen) for s in shapes]
    rho = [torch.empty(s, dtype=torch.float64, device="cuda") for s in shapes]
    F = torch.empty((inp.nao, inp.nao), dtype=torch.float64, device="cuda")
    grid_bytes = sum(int(np.prod(s)) * 8 for s in shapes)
    resident_bytes = 2 * grid_bytes + 2 * inp.nao * inp.nao * 8

    peak_meas, nsm = gpw.gpw_dfma_peak(0.5)
    peak_dmma, peak_mixed = gpw.gpw_dmma_peak(0.3)

    def step():
        gpw.gpw_eval_rho(plan, D, deriv, rho)
        gpw.gpw_eval_mat(plan, v, deriv, F)
        if shard:
            dist.all_reduce(F)       # the path's one exchange: the partial Fock matrices (NCCL over NVLink)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(W):
        step()
    sampler = ClockSampler(local_rank)
    sampler.start()
    time.sleep(0.3)
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    marks = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    tw0 = time.time()
    e0.record()
    marks[0].record()
    for i in range(args.steps):   # nothing but the K steps (and one event record each) between the two brackets
        step()
        marks[i + 1].record()
    e1.record()
    barrier()
    tw1 = time.time()
    ms_total = e0.elapsed_time(e1)
    clocks = sampler.summary(tw0, tw1)
    sampler.stop()
    per_step = np.array([marks[i].elapsed_time(marks[i + 1]) for i in range(args.steps)])
    ms_step = ms_total / args.steps
    # kernel durations from the library's own events on the launching stream, outside the timed region
    gpw.gpw_plan_set_timing(plan, True)
    kts = []
    for _ in range(max(3, min(args.steps, 10))):
        step()
        a = gpw.gpw_plan_get_timing(plan, 0)
        b = gpw.gpw_plan_get_timing(plan, 1)
        kts.append([a[0], a[1], b[0], b[1]])
    gpw.gpw_plan_set_timing(plan, False)
    kt = np.median(np.array(kts), axis=0)
    kt_min = np.min(np.array(kts), axis=0)
    ms_step, flops_all = reduce_over_ranks(ms_step, flops_step, dist, "cuda")
    value = flops_all / (ms_step * 1e-3) / 1e9

    # parity-side sanity on the very buffers that were timed: adjointness <rho[D], v> dV = Tr(D F[v])
    vol = abs(float(np.linalg.det(inp.cell)))
    lhs = sum(float((r * x).sum()) * vol / r[0].numel() for r, x in zip(rho, v))
    rhs = float((D * F).sum())
    adj = abs(lhs - rhs) / max(abs(lhs), 1e-300)

    # ---- Fock-build ms (BASELINE.json metric): eval_rho on every level, Fourier interpolation to the
    #      finest mesh (Eq. 7), restriction of a synthetic fine-grid potential (Eq. 8), eval_mat.  XC and Hartree
    #      are not part of the path: v is synthetic. ----
    fine_shape = (nc,) + tuple(int(x) for x in inp.mesh[0])
    rho_fine = torch.empty(fine_shape, dtype=torch.float64, device="cuda")
    v_fine = torch.randn(fine_shape, dtype=torch.float64, device="cuda", generator=gen)
    v_lev = [torch.empty(s, dtype=torch.float64, device="cuda") for s in shapes]
    v_hartree = torch.empty(fine_shape[1:], dtype=torch.float64, device="cuda")

    def fock_step():
        gpw.gpw_eval_rho(plan, D, deriv, rho)
        gpw.gpw_interp_up(plan, rho, nc, rho_fine)
        gpw.gpw_hartree(plan, rho_fine[0], v_hartree)     # Eq. 5-6: the Hartree potential of the collocated density
        v_fine[0].copy_(v_hartree)                        # components 1.. (the XC side) stay synthetic
        gpw.gpw_restrict_down(plan, v_fine, nc, v_lev)
        gpw.gpw_eval_mat(plan, v_lev, deriv, F)

    fock_step()
    barrier()
    fock_steps = max(2, min(args.steps, 5))
    e0.record()
    for _ in range(fock_steps):
        fock_step()
    e1.record()
    barrier()
    fock_ms = e0.elapsed_time(e1) / fock_steps
    del rho_fine, v_fine, v_lev, v_hartree

    # ---- end to end: host buffers in, host buffers out, copies inside the timed region ----
    Dh = D.cpu().pin_memory()
    vh = [x.cpu().pin_memory() for x in v]
    rho_h = [torch.empty(s, dtype=torch.float64).pin_memory() for s in shapes]
    Fh = torch.empty((inp.nao, inp.nao), dtype=torch.float64).pin_memory()
    h2d = Dh.numel() * 8 + grid_bytes
    d2h = grid_bytes + Fh.numel() * 8

    # the library's host-buffer entry points (include/gpw.h): every array in pinned host memory, uploads, kernels and
    # downloads inside the timed region, overlapped by the library on its own copy streams
    def e2e_step():
        gpw.gpw_eval_rho_host(plan, Dh, deriv, rho_h)
        gpw.gpw_eval_mat_host(plan, vh, deriv, Fh)

    e2e_steps = max(2, min(args.steps, 5))
    e2e_step()
    gpw.gpw_plan_wait(plan)
    barrier()
    e0.record()
    for _ in range(e2e_steps):
        e2e_step()
    gpw.gpw_plan_wait(plan)      # the timing stream waits for the last download
    e1.record()
    barrier()
    step()
    barrier()
    e2e_check = float((Fh - F.cpu()).abs().max() / F.abs().max())   # same result as the resident path
    assert e2e_check <= 1e-12, e2e_check
    e2e_ms = e0.elapsed_time(e1) / e2e_steps
    e2e_ms, _ = reduce_over_ranks(e2e_ms, flops_step, dist, "cuda")
    e2e_value = flops_all / (e2e_ms * 1e-3) / 1e9

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # dominant kernel = the slower of collocation / integration
    dom = "k_integrate" if kt[2] >= kt[1] else "k_collocate"
    dom_ms = float(max(kt[1], kt[2]))
    model_tflops = flops_call / (dom_ms * 1e-3) / 1e12
    # Executed FP64 flops per launch (ncu: 2 DFMA + DADD + DMUL thread instructions), FP64-pipe utilisation and DRAM
    # bytes per launch come from the committed full ncu capture of THIS build (profiles/traffic.json carries the hash
    # of csrc/ it was taken on): a profiler cannot run inside a timed bench.  If the sources changed since, null.
    sha = csrc_sha()
    ncu, ncu_all = {}, {}
    tpath = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(tpath):
        try:
            tj = json.load(open(tpath))
            if tj.get("csrc_sha") == sha:
                ncu_all = tj.get("kernels", {})
                ncu = ncu_all.get(f"{inp.name}:{dom}") or {}
        except Exception:
            ncu, ncu_all = {}, {}
    executed = ncu.get("executed_fp64_flops")
    executed_tflops = (executed / (dom_ms * 1e-3) / 1e12) if executed else None

    def exec_frac(kernel, ms):
        e = (ncu_all.get(f"{inp.name}:{kernel}") or {}).get("executed_fp64_flops")
        return (e / (ms * 1e-3) / 1e12 / NOMINAL_FP64_TFLOPS) if e else None

    # kernels of this repository launched per step (counted from the launch logic of gpw_eval_rho / gpw_eval_mat): the
    # register-form pre/post-pass, the group form when the plan has classes la + lb >= 5 or for deriv = 2, one collocation
    # and one integration launch per class range (two ranges on plans with f shells; collocation splits only for deriv >= 1)
    cls = info["nvisit_class"]
    big = any(int(cls[:, la, lb].sum()) > 0 for la in range(4) for lb in range(4) if la + lb >= 5)
    n_pre = 1 + (1 if (big or deriv == 2) else 0)
    n_col = (2 if (big and deriv >= 1) else 1) + (1 if deriv == 2 else 0)
    n_int = (2 if big else 1) * (2 if deriv == 2 else 1)
    nlaunch = n_pre + n_col + n_int + n_pre
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": W,
        "ms_per_step": ms_step, "ms_per_step_median": float(np.median(per_step)), "ms_per_step_min": float(per_step.min()),
        "higher_is_better": True, "scaling": "strong" if shard else "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": inp.name, "sharded": bool(shard), "nao": inp.nao, "meshes": [int(m[0]) for m in inp.mesh], "deriv": deriv,
                   "tau": inp.tau, "rel_cutoff": inp.rel_cutoff, "hermi": inp.hermi,
                   "pairs": info["ntask"], "block_visits": int(sum(info["nvisit_level"])),
                   "l2": f"inputs+outputs resident {resident_bytes / 1e6:.0f} MB > 126 MB L2, no explicit flush",
                   "flop_model": "SURVEY 8(d): 64*visits*W, W1=4*nca*ncb+10*(nca+ncb)+8 (deriv>=1), W0=2*nca*ncb+2*(nca+ncb)+4; deriv=2: W1+W0"},
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": UNIT, "ms_per_step": e2e_ms, "h2d_bytes_per_step": int(h2d),
                "d2h_bytes_per_step": int(d2h),
                "api": "gpw_eval_rho_host + gpw_eval_mat_host (C ABI, pinned host buffers; copies overlapped on the library's streams)"},
        "gpu_launches": nlaunch * args.steps,
        "roofline": {"bound": "alu", "kernel": dom, "achieved": executed_tflops, "peak": NOMINAL_FP64_TFLOPS,
                     "unit": "TFLOP/s", "frac": (executed_tflops / NOMINAL_FP64_TFLOPS) if executed_tflops else None,
                     "traffic": ncu.get("dram_bytes"),
                     "peak_source": "derived: 148 SMs x 64 FP64 FMA lanes x 2 x 1.965 GHz (MEASURED_PEAKS.json has no FP64 entry)",
                     "peak_measured_dfma": peak_meas, "peak_measured_dmma_m8n8k4": peak_dmma,
                     "peak_measured_dmma_plus_dfma": peak_mixed,
                     "fp64_pipe_pct_ncu": ncu.get("fp64_pipe_pct"), "ncu_capture": ncu.get("capture"), "csrc_sha": sha,
                     "frac_k_collocate": exec_frac("k_collocate", float(kt[1])), "frac_k_integrate": exec_frac("k_integrate", float(kt[2])),
                     "model_tflops": model_tflops,
                     "note": "achieved = FP64 flops the kernel EXECUTES per launch (ncu: 2*DFMA + DADD + DMUL thread instructions, "
                             "from the committed capture of this very build, matched by csrc_sha; null if the sources changed since) "
                             "/ this run's kernel time (CUDA events).  model_tflops = SURVEY 8(d) model flops of one call / the same "
                             "time: the kernels evaluate a cheaper polynomial form than the model charges, so it can exceed the peak "
                             "and is not a roofline fraction (DESIGN.md section 5)"},
        "kernels_ms": {"k_pair_pass_pre": float(kt[0]), "k_collocate": float(kt[1]), "k_integrate": float(kt[2]),
                       "k_pair_pass_post": float(kt[3])},
        "kernels_ms_min": {"k_pair_pass_pre": float(kt_min[0]), "k_collocate": float(kt_min[1]), "k_integrate": float(kt_min[2]),
                           "k_pair_pass_post": float(kt_min[3])},
        "model_gflop_per_call": flops_call / 1e9,
        "eval_rho_tflops_model": flops_call / ((kt[0] + kt[1]) * 1e-3) / 1e12,
        "eval_mat_tflops_model": flops_call / ((kt[2] + kt[3]) * 1e-3) / 1e12,
        "fock_build_ms": fock_ms,
        "fock_build_note": "eval_rho + gpw_interp_up + gpw_hartree (Eq. 5-6) of the interpolated density + gpw_restrict_down of "
                           "[v_H, synthetic N(0,1) XC-side components] + eval_mat; XC functional itself excluded (LibXC)",
        "plan_build_s": build_s, "plan_build_lib_s": float(info["build_seconds"]),   # wall around the call (first use of the
        # library in the process: module loading included) / the library's own clock inside gpw_build_pairs
        "plan_device_bytes": int(info["device_bytes"]),
        "adjointness_rel_err": adj,
    }
    if not args.no_cpu_baseline:
        g, cores, desc, _ = time_oracle_sample(inp, budget_s=20.0)
        line["cpu_baseline"] = {"value": g, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc}
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
