"""N > 1 host logic on CPU (gloo, world size 2): the path shards by owner with NO data-path collective
(PAPER.md:47, 97), so what there is to test is that each process picks a distinct rank of the plan, that the
resident sets are disjoint and together cover what those ranks own, and that the report reduction (MAX time, SUM
flops) is right."""
import os
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    import paper_2607_05895_b200 as mf
    import workloads
    wl = workloads.get("c5")
    order = bench.rank_order_by_load(mf, wl)
    pr_rank = bench.choose_plan_rank(order, wl.rank, rank, world)
    pr = mf.mfsdp_plan(wl.params, wl.world, wl.policy, wl.metric, pr_rank)
    mats = [pr.desc[i] for i in range(pr.desc._n) if pr.desc[i].role == mf.ROLE_MATRIX]
    f_alg = sum(bench.ns_flops(d.rows, d.cols, 5)[0] for d in mats)
    ids = sorted(d.param_id for d in mats)
    ms_all, _, f_all, launches = bench.reduce_over_ranks(10.0 + rank, 0.0, f_alg, 19, world, "cpu")
    gathered = [None] * world
    dist.all_gather_object(gathered, (pr_rank, ids, f_alg))
    if rank == 0:
        out.put((ms_all, f_all, launches, gathered, order[:world]))
    dist.destroy_process_group()


@pytest.mark.timeout(180)
def test_two_ranks_take_disjoint_resident_sets_and_reduce_report():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    ms_all, f_all, launches, gathered, order = q.get(timeout=150)
    for p in procs:
        p.join(30)
        assert p.exitcode == 0
    assert ms_all == 11.0 and launches == 38
    assert [g[0] for g in gathered] == order and order[0] != order[1]
    assert not set(gathered[0][1]) & set(gathered[1][1]), "two ranks own the same matrix"
    assert f_all == gathered[0][2] + gathered[1][2]
    assert gathered[0][2] >= gathered[1][2]          # heaviest first


def test_single_rank_keeps_workload_choice():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.choose_plan_rank([5, 3, 1], 0, 0, 1) == 0
    assert bench.choose_plan_rank([5, 3, 1], -1, 0, 1) == 5
    assert bench.choose_plan_rank([5, 3, 1], 0, 1, 2) == 3
