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


def _shard_worker(rank, world, port, out):
    """The sharded mode of the path (gpw_plan_set_partition): every rank builds the SAME plan and owns one n1 slab of
    every level; the only exchange is the sum of the partial F.  Here, without a device, the ranks exchange their slab
    bounds and a stand-in partial F over gloo (the all-reduce bench.py --shard issues over NCCL)."""
    import torch
    import torch.distributed as dist
    import paper_2603_24881_b200 as gpw
    from paper_2603_24881_b200 import inputs
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        inp = inputs.make_small("triclinic")
        plan = gpw.gpw_build_pairs(*inp.abi_args())
        gpw.gpw_plan_set_partition(plan, rank, world)
        bounds = [gpw.gpw_plan_partition_bounds(plan, lev, rank, world) for lev in range(inp.nlevel)]
        mine = torch.tensor(bounds, dtype=torch.int64)
        gathered = [torch.zeros_like(mine) for _ in range(world)]
        dist.all_gather(gathered, mine)
        # stand-in for the partial F of this rank: the number of owned grid planes per level on the diagonal
        F = torch.zeros(inp.nlevel, dtype=torch.float64)
        for lev, (lo, hi) in enumerate(bounds):
            F[lev] = hi - lo
        dist.all_reduce(F, op=dist.ReduceOp.SUM)
        out[rank] = ([g.tolist() for g in gathered], F.tolist(), [int(m[0]) for m in inp.mesh])
    finally:
        dist.destroy_process_group()


def test_two_ranks_gloo_sharded_slabs_tile_every_level():
    import torch.multiprocessing as mp
    world = 2
    with mp.Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_shard_worker, args=(world, _free_port(), out), nprocs=world, join=True)
        res = dict(out)
    assert set(res) == {0, 1}
    gathered, Fsum, n1 = res[0]
    assert res[1][0] == gathered and res[1][1] == Fsum
    for lev, n in enumerate(n1):
        lo0, hi0 = gathered[0][lev]
        lo1, hi1 = gathered[1][lev]
        assert lo0 == 0 and hi0 == lo1 and hi1 == n          # disjoint, contiguous, covering
        assert lo1 % 4 == 0                                   # cut on a block boundary
        assert Fsum[lev] == n                                 # the all-reduce saw every plane once


def test_partition_argument_checks():
    import paper_2603_24881_b200 as gpw
    from paper_2603_24881_b200 import inputs
    plan = gpw.gpw_build_pairs(*inputs.make_small("cubic").abi_args())
    for rank, n in ((2, 2), (-1, 2), (0, 0)):
        with pytest.raises(gpw.GpwError):
            gpw.gpw_plan_set_partition(plan, rank, n)
    # seven ranks on a mesh of few block rows: some slabs are empty, none overlaps
    prev = 0
    for r in range(7):
        lo, hi = gpw.gpw_plan_partition_bounds(plan, 0, r, 7)
        assert lo == prev and hi >= lo
        prev = hi
    assert prev == int(plan.mesh[0][0])
