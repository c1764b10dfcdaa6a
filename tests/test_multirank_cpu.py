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


# ---- cross-rank validation of the gradient-reduction schedule -------------------------------------------
def _sched_worker(rank, world, port, out, perturb):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import paper_2607_05895_b200 as mf
    from paper_2607_05895_b200 import dist as mdist
    import workloads
    wl = workloads.get("c4")
    params = list(wl.params)
    if perturb and rank == 1:                         # rank 1 believes one matrix is 64 rows taller
        p = params[10]
        params[10] = (p[0], p[1], p[2] + 64, p[3], p[4], p[5])
    pr = mf.mfsdp_plan(params, wl.world, mf.POLICY_COST_AWARE, wl.metric, rank)
    try:
        ops, h = mdist.validated_reduce_schedule(params, wl.world, pr.owner)
        mine = [(o.seq, o.role, o.numel, o.owner_elem_off, o.flag) for o in ops if o.owner == rank]
        out.put((rank, "ok", h, len(ops), mine, [pr.desc[i].elem_off for i in range(pr.desc._n)
                                                 if pr.desc[i].role == mf.ROLE_MATRIX]))
    except mdist.ScheduleMismatch as e:
        out.put((rank, "mismatch", sorted(set(e.hashes)), str(e), None, None))
    dist.destroy_process_group()


def _run_sched(perturb):
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 31500 + os.getpid() % 2000 + (7 if perturb else 0)
    procs = [ctx.Process(target=_sched_worker, args=(r, 2, port, q, perturb)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=150) for _ in range(2))
    for p in procs:
        p.join(30)
        assert p.exitcode == 0
    return res


@pytest.mark.timeout(180)
def test_two_ranks_derive_the_same_reduction_schedule():
    a, b = _run_sched(False)
    assert a[1] == b[1] == "ok" and a[2] == b[2] and a[3] == b[3] == 32 * 8        # 7 matrices + 1 tail per block
    for res in (a, b):                               # the segments a rank receives are its own descriptor table's
        flags = [m for m in res[4] if m[4] >= 0]
        assert sorted(f[4] for f in flags) == list(range(len(res[5])))
        for seq, role, numel, off, flag in flags:
            assert res[5][flag] == off


@pytest.mark.timeout(180)
def test_schedule_mismatch_is_an_explicit_error_on_every_rank():
    a, b = _run_sched(True)
    assert a[1] == b[1] == "mismatch" and a[2] == b[2] and len(a[2]) == 2
    assert "ranks [0]" in a[3] and "ranks [1]" in a[3]


# ---- the exchange steps themselves on CPU (gloo): reduce-to-owner and owner fan-out -------------------------
def _exchange_worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import paper_2607_05895_b200 as mf
    from paper_2607_05895_b200 import dist as mdist
    import workloads
    wl = workloads.get("small")                       # 9 matrices + 3 tails in 3 blocks, planned over 2 ranks
    pr = mf.mfsdp_plan(wl.params, world, mf.POLICY_ROLE_GREEDY, mf.METRIC_NUMEL, rank)
    ops, _ = mdist.validated_reduce_schedule(wl.params, world, pr.owner)
    fwd, _ = mdist.validated_reduce_schedule(wl.params, world, pr.owner, reverse_blocks=False)
    n_mat, n_tail = mf.mfsdp_flat_elems(pr.desc)
    # every rank's full local gradient of role r: seeded by (rank, role), fp32 on CPU
    grads = {op.role: torch.Generator().manual_seed(1000 * rank + op.role) for op in ops}
    grads = {op.role: torch.randn(op.numel, generator=grads[op.role]) for op in ops}
    sent = {r: g.clone() for r, g in grads.items()}
    G, Gt = torch.zeros(max(n_mat, 1)), torch.zeros(max(n_tail, 1))
    mdist.reduce_gradients_to_owners(ops, rank, lambda r: grads[r], G, Gt)
    # expected: sum over ranks of the seeded gradients, only in the segments this rank owns
    ok = True
    for op in ops:
        want = sum(torch.randn(op.numel, generator=torch.Generator().manual_seed(1000 * q + op.role)) for q in range(world))
        flat = G if op.kind == mf.ROLE_MATRIX else Gt
        if op.owner == rank:
            ok &= bool(torch.allclose(flat[op.owner_elem_off:op.owner_elem_off + op.numel], want, rtol=0, atol=1e-6))
    owned = sum(op.numel for op in ops if op.owner == rank)
    nonzero = int((G != 0).sum() + (Gt != 0).sum())
    # fan-out: owners publish "updated weights" = their reduced gradient segments; every rank ends with all of them
    full = {op.role: torch.zeros(op.numel) for op in fwd}
    mdist.fanout_parameters(fwd, rank, G, Gt, lambda r: full[r])
    fan_ok = True
    for op in fwd:
        want = sum(torch.randn(op.numel, generator=torch.Generator().manual_seed(1000 * q + op.role)) for q in range(world))
        fan_ok &= bool(torch.allclose(full[op.role], want, rtol=0, atol=1e-6))
    out.put((rank, ok, owned, nonzero, fan_ok, [op.role for op in ops][:3], [op.role for op in fwd][:3]))
    dist.destroy_process_group()


@pytest.mark.timeout(180)
def test_reduce_to_owner_and_fanout_over_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 33500 + os.getpid() % 2000
    procs = [ctx.Process(target=_exchange_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=150) for _ in range(2))
    for p in procs:
        p.join(30)
        assert p.exitcode == 0
    for rank, ok, owned, nonzero, fan_ok, first_rev, first_fwd in res:
        assert ok, "rank %d: an owned segment is not the sum of the ranks' gradients" % rank
        assert fan_ok, "rank %d: a materialised parameter differs from its owner's segment" % rank
        assert nonzero <= owned and nonzero >= owned - 8      # nothing lands outside owned segments (exact zeros are rare)
    assert res[0][5] == res[1][5] and res[0][6] == res[1][6] and res[0][5] != res[0][6]   # same order on both ranks
