"""Host-side logic of the N > 1 path of bench.py on CPU: two processes over gloo (-m "not gpu").

The path shards as independent workloads per rank (weak scaling, no data-path collective; DESIGN.md
"Multi-GPU"): every rank builds its own plan from its own seed, and the whole-job figures are the flops of
all ranks over the slowest rank's time.  Without a device gpw_build_pairs returns a host-only plan, which is
all this test needs (pair and visit counts -> model flops)."""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    import torch
    import torch.distributed as dist
    import bench
    import paper_2603_24881_b200 as gpw
    from paper_2603_24881_b200 import inputs
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        inp = inputs.make_config(0, seed=bench.rank_seed(0, rank))
        plan = gpw.gpw_build_pairs(*inp.abi_args())
        flops = 2.0 * gpw.model_flops(plan.info, inp.deriv)
        ms = 1.0 + rank                                   # rank 1 is the slow one
        dist.barrier()
        ms_all, flops_all = bench.reduce_over_ranks(ms, flops, dist, "cpu")
        gathered = [torch.zeros(2, dtype=torch.float64) for _ in range(world)]
        dist.all_gather(gathered, torch.tensor([flops, float(inp.seed)], dtype=torch.float64))
        out[rank] = (ms_all, flops_all, [g.tolist() for g in gathered])
    finally:
        dist.destroy_process_group()


def test_two_ranks_gloo_weak_scaling_aggregation():
    import torch.multiprocessing as mp
    world = 2
    with mp.Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_worker, args=(world, _free_port(), out), nprocs=world, join=True)
        res = dict(out)
    assert set(res) == {0, 1}
    (ms0, fl0, g0), (ms1, fl1, g1) = res[0], res[1]
    assert g0 == g1
    per_rank_flops = [g[0] for g in g0]
    seeds = [g[1] for g in g0]
    assert seeds[0] != seeds[1], "ranks must run independent workloads"
    assert all(f > 0 for f in per_rank_flops)
    # every rank sees the same whole-job figures: max of the times, sum of the flops
    assert ms0 == ms1 == 2.0
    assert fl0 == fl1 == pytest.approx(sum(per_rank_flops), rel=1e-15)


def test_rank_seed_convention():
    import bench
    from paper_2603_24881_b200 import inputs
    assert bench.rank_seed(2, 0) is None                  # rank 0 runs the config's own workload
    s = {bench.rank_seed(2, r) for r in range(1, 8)}
    assert len(s) == 7 and all(x != inputs.BASE_SEED + 2 for x in s)
    a = inputs.make_config(0, seed=bench.rank_seed(0, 1))
    b = inputs.make_config(0)
    assert a.nao == b.nao and not np.array_equal(a.prim_exp, b.prim_exp)
