"""Pins for oracle/planner.py: hand traces, brute-force optimum + Graham's LPT bound on tiny
inputs, list-scheduling bound for ROLE_GREEDY, conservation / layout invariants.
The paper prints no assignment, so nothing here is a paper value; the
comparison against the *paper's own* planner stays "parity unpinned"."""
import itertools
import random

import numpy as np
import pytest

from oracle import planner as P
from oracle import planner as oplan


def mat(block, rows, cols, dtype=1, flags=0):
    return (block, 2, rows, cols, dtype, flags)


def vec(block, n, dtype=1, flags=0):
    return (block, 1, n, 1, dtype, flags)


def test_roles_one_per_matrix_one_tail_per_block():
    params = [vec(0, 8), mat(0, 4, 4), vec(0, 3), mat(0, 2, 6), mat(1, 5, 5), vec(2, 7), (2, 3, 6, 2, 1, 0)]
    roles = P.build_roles(params)
    kinds = [(r["kind"], r["block"], r["index"], r["numel"]) for r in roles]
    assert kinds == [(P.ROLE_TAIL, 0, 0, 11), (P.ROLE_MATRIX, 0, 1, 16), (P.ROLE_MATRIX, 0, 3, 12),
                     (P.ROLE_MATRIX, 1, 4, 25), (P.ROLE_TAIL, 2, 5, 19)]
    assert roles[0]["members"] == [0, 2]


def test_skip_flag_removes_parameter():
    params = [mat(0, 4, 4, flags=P.PARAM_SKIP), mat(0, 2, 2), vec(0, 5, flags=P.PARAM_SKIP)]
    roles = P.build_roles(params)
    assert len(roles) == 1 and roles[0]["index"] == 1


def test_seven_equal_roles_two_ranks_hand_trace():
    params = [mat(0, 8, 8) for _ in range(7)]
    for policy in (P.POLICY_ROLE_GREEDY, P.POLICY_SCOPE_GREEDY):
        out = P.plan(params, 2, policy, P.METRIC_NUMEL, rank=0)
        assert out["owner"] == [0, 1, 0, 1, 0, 1, 0]
        assert out["loads"][0] == [256, 192]


def test_role_vs_scope_hand_trace():
    # block 0: 10, 1 ; block 1: 9, 2 ; two ranks, numel metric
    params = [mat(0, 10, 1), mat(0, 1, 1), mat(1, 9, 1), mat(1, 2, 1)]
    role = P.plan(params, 2, P.POLICY_ROLE_GREEDY, P.METRIC_NUMEL)
    # block 0: 10 -> r0, 1 -> r1 ; block 1 (loads 10, 1): 9 -> r1 (10), 2 -> r0 (tie 10/10 -> lowest id)
    assert role["owner"] == [0, 1, 1, 0] and role["loads"][0] == [12, 10]
    scope = P.plan(params, 2, P.POLICY_SCOPE_GREEDY, P.METRIC_NUMEL)
    # pooled: 10 (idx0) -> r0, 9 (idx2) -> r1, 2 (idx3) -> r1 (11), 1 (idx1) -> r0 (11)
    assert scope["owner"] == [0, 0, 1, 1] and scope["loads"][0] == [11, 11]


def test_ns_flops_metric_and_separate_tail_vector():
    params = [vec(0, 100), mat(0, 4, 16), mat(0, 16, 4), mat(0, 8, 8), vec(1, 50), mat(1, 2, 2)]
    out = P.plan(params, 2, P.POLICY_SCOPE_GREEDY, P.METRIC_NS_FLOPS)
    # loads: 4x16 and 16x4 -> 16*(32+4) = 576 ; 8x8 -> 64*24 = 1536 ; 2x2 -> 4*6 = 24
    # sorted: 1536 (idx3) -> r0 ; 576 (idx1) -> r1 ; 576 (idx2) -> r1 (576 < 1536) ; 24 -> r1 (1152 < 1536)
    # tails on their own vector: 100 -> r0 ; 50 -> r1
    assert out["owner"] == [0, 1, 1, 0, 1, 1]
    assert out["loads"] == [[1536, 1176], [100, 50]]


def test_world_one_puts_everything_on_rank_zero():
    params = [vec(0, 3), mat(0, 4, 5), mat(1, 6, 7)]
    out = P.plan(params, 1, P.POLICY_ROLE_GREEDY, P.METRIC_NUMEL)
    assert out["owner"] == [0, 0, 0] and len(out["desc"]) == 3


def test_heaviest_rank_selection_and_tie():
    params = [mat(0, 4, 4), mat(0, 4, 4), mat(0, 2, 2)]
    out = P.plan(params, 2, P.POLICY_SCOPE_GREEDY, P.METRIC_NUMEL, rank=-1)
    # 16 -> r0, 16 -> r1, 4 -> r0 : heaviest is rank 0
    assert out["rank"] == 0
    out = P.plan([mat(0, 4, 4), mat(0, 4, 4)], 3, P.POLICY_SCOPE_GREEDY, P.METRIC_NUMEL, rank=-1)
    assert out["rank"] == 0   # tie between ranks 0 and 1 -> lowest id


def brute_force_makespan(loads, world):
    best = None
    for assign in itertools.product(range(world), repeat=len(loads)):
        per = [0] * world
        for l, r in zip(loads, assign):
            per[r] += l
        mk = max(per)
        best = mk if best is None else min(best, mk)
    return best


@pytest.mark.parametrize("seed", range(25))
def test_scope_greedy_within_graham_lpt_bound(seed):
    rnd = random.Random(seed)
    world = rnd.choice([2, 3])
    n = rnd.randint(1, 8)
    params = [mat(rnd.randint(0, 2), rnd.randint(1, 9), rnd.randint(1, 9)) for _ in range(n)]
    params.sort(key=lambda p: p[0])
    out = P.plan(params, world, P.POLICY_SCOPE_GREEDY, P.METRIC_NUMEL)
    loads = [r["numel"] for r in out["roles"]]
    opt = brute_force_makespan(loads, world)
    assert opt <= max(out["loads"][0])
    assert max(out["loads"][0]) * 3 * world <= (4 * world - 1) * opt      # LPT: <= (4/3 - 1/(3W)) OPT
    # ROLE_GREEDY is list scheduling in some order: <= (2 - 1/W) OPT
    role = P.plan(params, world, P.POLICY_ROLE_GREEDY, P.METRIC_NUMEL)
    assert opt <= max(role["loads"][0])
    assert max(role["loads"][0]) * world <= (2 * world - 1) * opt


@pytest.mark.parametrize("seed", range(10))
@pytest.mark.parametrize("policy", [P.POLICY_ROLE_GREEDY, P.POLICY_SCOPE_GREEDY])
@pytest.mark.parametrize("metric", [P.METRIC_NUMEL, P.METRIC_NS_FLOPS])
def test_invariants_random_models(seed, policy, metric):
    rnd = random.Random(1000 + seed)
    world = rnd.randint(1, 6)
    params = []
    for b in range(rnd.randint(1, 6)):
        for _ in range(rnd.randint(1, 7)):
            if rnd.random() < 0.6:
                params.append(mat(b, rnd.choice([1, 3, 64, 100, 128]), rnd.choice([1, 5, 64, 96, 256])))
            else:
                params.append(vec(b, rnd.randint(1, 300)))
    out = P.plan(params, world, policy, metric, rank=-1)
    roles, owner = out["roles"], out["owner"]
    assert all(0 <= o < world for o in owner)                       # every role exactly one owner
    per = [[0] * world, [0] * world]
    for r, o in zip(roles, owner):
        vecid, load = P.role_load(r, metric)
        per[vecid][o] += load
    assert per == out["loads"]                                      # loads conserved
    covered = sorted(i for r in roles for i in r["members"])
    assert covered == list(range(len(params)))                      # every parameter in exactly one role
    # descriptor tables of all ranks partition the roles; offsets aligned, disjoint, ordered
    seen = 0
    for k in range(world):
        d = P.plan(params, world, policy, metric, rank=k)["desc"]
        seen += len(d)
        P.validate_desc(d)
        assert [x["param_id"] for x in d] == sorted(x["param_id"] for x in d)
        for x in d:
            if x["role"] == P.ROLE_MATRIX:
                assert (x["flags"] & P.DESC_TRANSPOSED) == (1 if x["rows"] > x["cols"] else 0)
            else:
                assert x["cols"] == 1
    assert seen == len(roles)
    assert out["rank"] == max(range(world), key=lambda k: (out["loads"][0][k], -k))


def test_validate_rejects_bad_tables():
    good = [dict(role=0, param_id=0, block_id=0, rows=4, cols=16, dtype=1, flags=0, elem_off=0),
            dict(role=0, param_id=1, block_id=0, rows=4, cols=16, dtype=1, flags=0, elem_off=64)]
    assert P.validate_desc(good)
    for bad in ([dict(good[0], elem_off=8)], [good[0], dict(good[1], elem_off=0)],
                [dict(good[0], rows=0)], [dict(good[0], role=7)]):
        with pytest.raises(ValueError):
            P.validate_desc(bad)


def test_transformer_shaped_balance_is_in_the_papers_range():
    """Sanity only (PAPER.md:174, 219-222 report max/avg 1.02-1.39 on other models)."""
    params = []
    for b in range(16):
        params += [vec(b, 4096), mat(b, 4096, 4096), mat(b, 4096, 4096), mat(b, 4096, 4096), mat(b, 4096, 4096),
                   vec(b, 4096), mat(b, 16384, 4096), mat(b, 4096, 16384)]
    for policy in (P.POLICY_ROLE_GREEDY, P.POLICY_SCOPE_GREEDY):
        out = P.plan(params, 8, policy, P.METRIC_NUMEL)
        assert 1.0 <= P.balance(out["loads"][0]) <= 1.4


# ---- resource scorer and COSTAWARE (Algorithm 1 line 4; reading P5) ---------------------------
def test_score_plan_hand_example():
    """Two blocks, two ranks, bytes by hand.  Block 0: 4x8 bf16 (64 B) on rank 0, 8x2 fp32 (64 B) on rank 1, a tail of
    10 bf16 (20 B) on rank 0; block 1: 16x16 bf16 (512 B) on rank 1."""
    params = [(0, 2, 4, 8, 0, 0), (0, 2, 8, 2, 1, 0), (0, 1, 10, 1, 0, 0), (1, 2, 16, 16, 0, 0)]
    sc = oplan.score_plan(params, 2, [0, 1, 0, 1])
    r0, r1 = sc["rank"]
    assert (r0["param"], r1["param"]) == (84, 576) and (r0["grad"], r1["grad"]) == (84, 576)
    assert (r0["state"], r1["state"]) == (4 * 32 + 8 * 10, 4 * 16 + 4 * 256)
    assert (r0["ws"], r1["ws"]) == (2 * (2 * 32 + 2 * 16), 2 * (2 * 16 + 2 * 4) + 2 * (2 * 256 + 2 * 256))
    assert (r0["comm"], r1["comm"]) == (84, 64 + 512) and (r0["blk"], r1["blk"]) == (84, 512)
    b0, b1 = sc["block"]
    assert (b0["param"], b0["max_owner"]) == (148, 84) and (b1["param"], b1["max_owner"]) == (512, 512)
    assert b0["gamma"] == pytest.approx(84 * 2 / 148, rel=1e-15) and b0["c_fsdp"] == 74.0 and b0["c_owner"] == 84.0
    assert b1["gamma"] == 2.0 and b1["c_fsdp"] == 256.0 and b1["c_owner"] == 512.0


def test_bandwidth_model_closed_forms():
    """"a block with one large owner can be bandwidth-poor (gamma_B ~ W); when the planner spreads matrix and
    tail owners within the block (gamma_B ~ 1), the leading bandwidth term matches ordinary FSDP", and the second
    equality of PAPER.md:79: C_B^owner = gamma_B P_B (W-1)/W."""
    for W in (2, 8, 64):
        one = oplan.score_plan([(0, 2, 32, 32, 0, 0)], W, [W - 1])["block"][0]
        assert one["gamma"] == float(W) and one["c_owner"] == float((W - 1) * 32 * 32 * 2)
        spread = oplan.score_plan([(0, 2, 8, 8, 0, 0)] * W, W, list(range(W)))["block"][0]
        assert spread["gamma"] == 1.0 and spread["c_owner"] == spread["c_fsdp"]
    rng = np.random.default_rng(5)
    for _ in range(50):
        W = int(rng.integers(1, 9))
        params = [(int(b), 2, int(rng.integers(1, 30)), int(rng.integers(1, 30)), int(rng.integers(0, 2)), 0)
                  for b in sorted(rng.integers(0, 4, size=int(rng.integers(1, 12))))]
        owner = [int(rng.integers(0, W)) for _ in params]
        sc = oplan.score_plan(params, W, owner)
        total = sum(r * c * (2, 4)[dt] for (_, _, r, c, dt, _) in params)
        assert sum(x["param"] for x in sc["rank"]) == total == sum(b["param"] for b in sc["block"])
        assert sum(x["comm"] for x in sc["rank"]) == (W - 1) * total
        for b in sc["block"]:
            assert b["c_owner"] == pytest.approx(b["gamma"] * b["c_fsdp"], rel=1e-12) or W == 1
            assert 1.0 - 1e-12 <= b["gamma"] <= W + 1e-12
        for r in range(W):
            assert sc["rank"][r]["blk"] == max([0] + [sum(rr * cc * (2, 4)[dt] for (bb, _, rr, cc, dt, _), o in
                                                         zip(params, owner) if o == r and bb == b)
                                                     for b in {p[0] for p in params}])


def test_cost_aware_hand_traces():
    """Algorithm 1 line 4 (reading P5), world 2, numel metric, bf16 column vectors.
    A: block 0 = {2, 6 elements}, block 1 = {7}.  ROLE: 6 -> r0, 2 -> r1 | 7 -> r1 (lightest): loads (6, 9).  SCOPE:
       7 -> r0, 6 -> r1, 2 -> r1: loads (7, 8) -- flatter, but rank 1 now owns 4 + 12 = 16 B of block 0 against a largest
       owner segment of 14 B under ROLE: 16 * 8 > 9 * 14, the cap is exceeded -> ROLE is used.
    B: block 0 = {2, 4}, block 1 = {8}.  ROLE loads (4, 10), SCOPE (8, 6); the largest owner segment is 16 B either way
       and the step workspace falls (48 -> 36 B) -> SCOPE is used."""
    A = [(0, 2, 2, 1, 0, 0), (0, 2, 6, 1, 0, 0), (1, 2, 7, 1, 0, 0)]
    used, owner, loads = oplan.cost_aware(A, 2)
    assert used == oplan.POLICY_ROLE_GREEDY and owner == [1, 0, 1] and loads[0] == [6, 9]
    assert oplan.plan(A, 2, oplan.POLICY_SCOPE_GREEDY)["owner"] == [1, 1, 0]
    used, owner, loads = oplan.cost_aware(A, 2, caps=dict(owner_num=8, owner_den=7))       # 16 * 7 <= 8 * 14: allowed
    assert used == oplan.POLICY_SCOPE_GREEDY and owner == [1, 1, 0] and loads[0] == [7, 8]
    used, _, _ = oplan.cost_aware(A, 2, caps=dict(owner_num=8, owner_den=7, abs_owner_bytes=15))
    assert used == oplan.POLICY_ROLE_GREEDY                                                  # absolute cap 15 B < 16 B
    B = [(0, 2, 2, 1, 0, 0), (0, 2, 4, 1, 0, 0), (1, 2, 8, 1, 0, 0)]
    used, owner, loads = oplan.cost_aware(B, 2)
    assert used == oplan.POLICY_SCOPE_GREEDY and owner == [1, 1, 0] and loads[0] == [8, 6]
    used, _, _ = oplan.cost_aware(B, 2, caps=dict(abs_ws_bytes=35))                        # scope needs 36 B
    assert used == oplan.POLICY_ROLE_GREEDY
    p = oplan.plan(B, 2, oplan.POLICY_COST_AWARE, rank=1)
    assert p["policy_used"] == oplan.POLICY_SCOPE_GREEDY and [d["rows"] for d in p["desc"]] == [2, 4]


def test_cost_aware_is_one_of_the_two_plans_and_never_worse_balanced_than_role():
    rng = np.random.default_rng(9)
    for _ in range(60):
        W = int(rng.integers(1, 7))
        params = []
        for b in range(int(rng.integers(1, 5))):
            for _ in range(int(rng.integers(1, 6))):
                if rng.random() < 0.7:
                    params.append((b, 2, int(rng.integers(1, 40)), int(rng.integers(1, 40)), 0, 0))
                else:
                    params.append((b, 1, int(rng.integers(1, 200)), 1, 0, 0))
        for metric in (oplan.METRIC_NUMEL, oplan.METRIC_NS_FLOPS):
            role = oplan.plan(params, W, oplan.POLICY_ROLE_GREEDY, metric)
            scope = oplan.plan(params, W, oplan.POLICY_SCOPE_GREEDY, metric)
            cost = oplan.plan(params, W, oplan.POLICY_COST_AWARE, metric)
            assert cost["owner"] in (role["owner"], scope["owner"])
            assert max(cost["loads"][0]) <= max(role["loads"][0])


def test_llama_balance_ratios_in_the_papers_range():
    """Context, not a pin (different model): Table 5 reports r/s/c = 1.07/1.02/1.07 ... 1.27/1.04/1.27;
    on the Llama-3-8B shapes the three policies land in the same range, scope flattest, cost = role or scope."""
    import workloads
    wl = workloads.get("c4")
    for W in (8, 64):
        bal = [oplan.balance(oplan.plan(wl.params, W, pol, wl.metric)["loads"][0]) for pol in (0, 1, 2)]
        assert 1.0 <= bal[1] <= bal[2] <= bal[0] <= 1.4


# ---- gradient-reduction schedule and its validation hash (reading F1) -------------------------------------
def test_fnv1a64_published_vectors():
    """FNV-1a 64 test vectors of the algorithm's reference distribution: "" / "a" / "foobar"."""
    assert oplan.fnv1a64(b"") == 0xCBF29CE484222325
    assert oplan.fnv1a64(b"a") == 0xAF63DC4C8601EC8C
    assert oplan.fnv1a64(b"foobar") == 0x85944171F73967E8


def test_reduce_schedule_hand_trace():
    """Two blocks, world 2.  Block 0: matrix 4x8 (rank 0), tail of 10 (rank 1), matrix 8x4 (rank 0); block 1: matrix
    16x16 (rank 1).  Backward order: block 1 first.  Offsets follow emit_desc (64-element alignment per kind)."""
    params = [(0, 2, 4, 8, 0, 0), (0, 1, 10, 1, 0, 0), (0, 2, 8, 4, 0, 0), (1, 2, 16, 16, 0, 0)]
    ops, h = oplan.reduce_schedule(params, 2, [0, 1, 0, 1])
    assert [(o["role"], o["owner"], o["numel"], o["owner_elem_off"], o["flag"]) for o in ops] == \
        [(3, 1, 256, 0, 0), (0, 0, 32, 0, 0), (1, 1, 10, 0, -1), (2, 0, 32, 64, 1)]
    assert [o["seq"] for o in ops] == [0, 1, 2, 3]
    fwd, h2 = oplan.reduce_schedule(params, 2, [0, 1, 0, 1], reverse_blocks=False)
    assert [o["role"] for o in fwd] == [0, 1, 2, 3] and h2 != h
    # the offsets and flags are the ones of each owner's descriptor table
    for rank in (0, 1):
        desc = oplan.emit_desc(oplan.build_roles(params), [0, 1, 0, 1], rank)
        mats = [d for d in desc if d["role"] == oplan.ROLE_MATRIX]
        for o in ops:
            if o["owner"] == rank and o["kind"] == oplan.ROLE_MATRIX:
                assert mats[o["flag"]]["elem_off"] == o["owner_elem_off"] and mats[o["flag"]]["param_id"] == o["param_id"]


def test_reduce_schedule_hash_detects_any_mismatch():
    import workloads
    wl = workloads.get("c4")
    owner = oplan.plan(wl.params, 8, 0, wl.metric)["owner"]
    ops, h = oplan.reduce_schedule(wl.params, 8, owner)
    assert len(ops) == len(owner) and sorted(o["role"] for o in ops) == list(range(len(owner)))
    assert sum(o["numel"] for o in ops) == sum(r["numel"] for r in oplan.build_roles(wl.params))
    assert oplan.reduce_schedule(wl.params, 8, owner)[1] == h                       # deterministic
    other = list(owner); other[5] = (other[5] + 1) % 8
    assert oplan.reduce_schedule(wl.params, 8, other)[1] != h                       # different owner
    p2 = list(wl.params); p2[3] = p2[3][:2] + (p2[3][2] + 64,) + p2[3][3:]
    assert oplan.reduce_schedule(p2, 8, owner)[1] != h                              # different segment size
    assert oplan.reduce_schedule(wl.params, 8, owner, reverse_blocks=False)[1] != h  # different order
