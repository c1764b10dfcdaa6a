"""Host-side checks that need no GPU: the C-ABI library loads and exports every symbol include/mfsdp.h declares,
the host planner (mfsdp_plan, C++) matches the oracle planner BIT-EXACTLY, layout validation, workspace sizing and
error codes.  No compute entry point is exercised beyond its argument checks."""
import ctypes
import os
import re

import numpy as np
import pytest

import paper_2607_05895_b200 as mf
import workloads
from oracle import planner as oplan

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    header = open(os.path.join(ROOT, "include", "mfsdp.h")).read()
    declared = set(re.findall(r"\b(mfsdp_[a-z_0-9]+)\s*\(", header))
    assert declared, "no declarations found in mfsdp.h"
    lib = ctypes.CDLL(mf.lib_path())
    for name in sorted(declared):
        assert hasattr(lib, name), "libmfsdp.so does not export %s" % name
    assert declared == set(mf.exported_symbols()), "binding and header disagree on the entry points"
    assert mf.mfsdp_version() == 2


def test_struct_sizes_match_header_layout():
    assert ctypes.sizeof(mf.Param) == 24
    assert ctypes.sizeof(mf.Desc) == 40
    assert ctypes.sizeof(mf.MuonHParams) == 7 * 8 + 6 * 4
    assert ctypes.sizeof(mf.AdamWHParams) == 5 * 8 + 8


def _compare_plan(params, world, policy, metric, rank, caps=None):
    want = oplan.plan(params, world, policy, metric, rank, caps=caps)
    if caps is None:
        got = mf.mfsdp_plan(params, world, policy, metric, rank)
        got_ex = mf.mfsdp_plan_ex(params, world, policy, metric, rank)
        assert got_ex.owner == got.owner and got_ex.policy_used == want["policy_used"]
    else:
        got = mf.mfsdp_plan_ex(params, world, policy, metric, rank, mf.Caps(**caps))
        assert got.policy_used == want["policy_used"]
    assert got.n_roles == len(want["roles"])
    assert got.owner == want["owner"]
    assert got.rank == want["rank"]
    assert got.rank_load[:world] == want["loads"][0]
    assert got.rank_load[world:] == want["loads"][1]
    gd = [got.desc[i].as_dict() for i in range(got.desc._n)]
    assert gd == want["desc"]
    return got, want


@pytest.mark.parametrize("name", ["c1", "c2", "c3", "c4", "c5", "small"])
@pytest.mark.parametrize("policy", [mf.POLICY_ROLE_GREEDY, mf.POLICY_SCOPE_GREEDY, mf.POLICY_COST_AWARE])
@pytest.mark.parametrize("metric", [mf.METRIC_NUMEL, mf.METRIC_NS_FLOPS])
def test_planner_matches_oracle_bit_exact_on_configs(name, policy, metric):
    wl = workloads.get(name)
    ranks = sorted({0, wl.world - 1, -1, wl.world // 2})
    for rank in ranks:
        _compare_plan(wl.params, wl.world, policy, metric, rank)


def test_planner_matches_oracle_on_random_models():
    rng = np.random.default_rng(123)
    for trial in range(200):
        n_blocks = int(rng.integers(1, 6))
        params = []
        for b in range(n_blocks):
            for _ in range(int(rng.integers(0, 6))):
                if rng.random() < 0.6:
                    params.append((b, 2, int(rng.integers(1, 40)), int(rng.integers(1, 40)), 0, int(rng.random() < 0.1)))
                else:
                    params.append((b, 1, int(rng.integers(1, 300)), 1, 0, int(rng.random() < 0.1)))
        world = int(rng.integers(1, 7))
        policy = int(rng.integers(0, 3))
        metric = int(rng.integers(0, 2))
        rank = int(rng.integers(-1, world))
        _compare_plan(params, world, policy, metric, rank)
        if policy == mf.POLICY_COST_AWARE and trial % 2:
            caps = dict(owner_num=int(rng.integers(1, 5)), owner_den=int(rng.integers(1, 5)),
                        ws_num=int(rng.integers(1, 5)), ws_den=int(rng.integers(1, 5)),
                        abs_owner_bytes=int(rng.integers(0, 3)) * int(rng.integers(1, 4000)),
                        abs_ws_bytes=int(rng.integers(0, 3)) * int(rng.integers(1, 8000)))
            _compare_plan(params, world, policy, metric, rank, caps=caps)


def _compare_score(params, world, owner):
    want = oplan.score_plan(params, world, owner)
    ranks, blocks = mf.mfsdp_score_plan(params, world, owner)
    assert len(ranks) == world and len(blocks) == len(want["block"])
    for g, w in zip(ranks, want["rank"]):
        assert (g.param_bytes, g.grad_bytes, g.state_bytes, g.comm_bytes, g.workspace_bytes, g.max_block_owner_bytes) == \
            (w["param"], w["grad"], w["state"], w["comm"], w["ws"], w["blk"])
    for g, w in zip(blocks, want["block"]):
        assert (g.block_id, g.param_bytes, g.max_owner_bytes) == (w["block"], w["param"], w["max_owner"])
        assert (g.gamma, g.c_fsdp, g.c_owner) == (w["gamma"], w["c_fsdp"], w["c_owner"])      # same IEEE operations
    return ranks, blocks


def test_score_plan_matches_oracle_bit_exact():
    """mfsdp_score_plan (resource scorer + gamma_B / C_B model) against oracle.planner.score_plan on
    the Llama-shaped plans of C4 / C5 under all three policies and on random models with random owners."""
    for name in ("c2", "c4", "c5"):
        wl = workloads.get(name)
        for policy in (0, 1, 2):
            pr = mf.mfsdp_plan(wl.params, wl.world, policy, wl.metric, 0)
            ranks, blocks = _compare_score(wl.params, wl.world, pr.owner)
            if wl.world > 1:
                assert all(1.0 <= b.gamma <= wl.world for b in blocks)
    rng = np.random.default_rng(77)
    for trial in range(200):
        params = []
        for b in range(int(rng.integers(1, 6))):
            for _ in range(int(rng.integers(0, 6))):
                if rng.random() < 0.6:
                    params.append((b, 2, int(rng.integers(1, 40)), int(rng.integers(1, 40)), int(rng.integers(0, 2)), 0))
                else:
                    params.append((b, 1, int(rng.integers(1, 300)), 1, 0, int(rng.random() < 0.1)))
        world = int(rng.integers(1, 7))
        n_roles = len(oplan.build_roles(params))
        _compare_score(params, world, [int(rng.integers(0, world)) for _ in range(n_roles)])


def test_workspace_estimate_lower_bounds_the_real_workspace():
    """The scorer's unpadded estimate 2 (2 rows cols + 2 d^2) per matrix vs mfsdp_workspace_bytes of the same rank's
    table (adds 1024-byte alignment, row pitches and the norm scratch): never above it, within 2 % on the Llama sets."""
    for name, slack in (("c4", 1.02), ("c5", 1.02), ("c3", 1.6)):
        wl = workloads.get(name)
        pr = mf.mfsdp_plan(wl.params, wl.world, wl.policy, wl.metric, wl.rank)
        ranks, _ = mf.mfsdp_score_plan(wl.params, wl.world, pr.owner)
        est = ranks[pr.rank].workspace_bytes
        real = mf.mfsdp_workspace_bytes(pr.desc, mf.NS_BF16)
        assert est <= real <= slack * est + 65536, (name, est, real)


def test_score_and_plan_ex_errors():
    lib = mf.load()
    P = (mf.Param * 2)(mf.Param(0, 2, 4, 4, 0, 0), mf.Param(1, 2, 8, 4, 0, 0))
    own = (ctypes.c_int32 * 2)(0, 1)
    nb = ctypes.c_size_t(0)
    assert lib.mfsdp_score_plan(P, 2, 2, own, 2, None, None, 0, ctypes.byref(nb)) == 0 and nb.value == 2
    assert lib.mfsdp_score_plan(P, 2, 2, own, 1, None, None, 0, ctypes.byref(nb)) == mf.EINVAL     # n_roles mismatch
    bad = (ctypes.c_int32 * 2)(0, 2)
    assert lib.mfsdp_score_plan(P, 2, 2, bad, 2, None, None, 0, ctypes.byref(nb)) == mf.EINVAL     # owner out of range
    B = (mf.BlockScore * 1)()
    assert lib.mfsdp_score_plan(P, 2, 2, own, 2, None, B, 1, ctypes.byref(nb)) == mf.ECAP
    nd = ctypes.c_size_t(0)
    zero_den = mf.Caps(owner_den=0)
    assert lib.mfsdp_plan_ex(P, 2, 2, mf.POLICY_COST_AWARE, 0, 0, ctypes.byref(zero_den), None, None, None, None, 0,
                             ctypes.byref(nd), None, None) == mf.EINVAL
    assert lib.mfsdp_plan_ex(P, 2, 2, 3, 0, 0, None, None, None, None, None, 0, ctypes.byref(nd), None, None) == mf.EINVAL


def test_configured_resident_sets():
    """The sets bench.py and the GPU tests run (regenerated, not trusted from the survey)."""
    wl = workloads.get("c2")
    got, _ = _compare_plan(wl.params, wl.world, wl.policy, wl.metric, wl.rank)
    assert sum(1 for i in range(got.desc._n) if got.desc[i].role == mf.ROLE_MATRIX) == 48
    assert sum(1 for i in range(got.desc._n) if got.desc[i].role == mf.ROLE_TAIL) == 12
    wl = workloads.get("c5")
    got, want = _compare_plan(wl.params, wl.world, wl.policy, wl.metric, wl.rank)
    loads = want["loads"][0]
    assert loads[got.rank] == max(loads)
    assert 1.0 <= oplan.balance(loads) <= 1.4          # PAPER.md:174, 219-222 sanity range
    wl = workloads.get("c4")
    got, want = _compare_plan(wl.params, wl.world, wl.policy, wl.metric, wl.rank)
    assert 1.0 <= oplan.balance(want["loads"][0]) <= 1.4


def test_plan_errors_and_size_query():
    lib = mf.load()
    n_desc = ctypes.c_size_t(0)
    P = (mf.Param * 2)(mf.Param(0, 2, 4, 4, 0, 0), mf.Param(0, 2, 8, 4, 0, 0))
    assert lib.mfsdp_plan(P, 2, 0, 0, 0, 0, None, None, None, None, 0, ctypes.byref(n_desc), None) == mf.EINVAL
    assert lib.mfsdp_plan(P, 2, 2, 0, 0, 2, None, None, None, None, 0, ctypes.byref(n_desc), None) == mf.EINVAL
    assert lib.mfsdp_plan(P, 2, 1, 7, 0, 0, None, None, None, None, 0, ctypes.byref(n_desc), None) == mf.EINVAL
    assert lib.mfsdp_plan(P, 2, 1, 0, 0, 0, None, None, None, None, 0, ctypes.byref(n_desc), None) == 0
    assert n_desc.value == 2
    D = (mf.Desc * 1)()
    assert lib.mfsdp_plan(P, 2, 1, 0, 0, 0, None, None, None, D, 1, ctypes.byref(n_desc), None) == mf.ECAP
    assert n_desc.value == 2
    bad = (mf.Param * 2)(mf.Param(1, 2, 4, 4, 0, 0), mf.Param(0, 2, 8, 4, 0, 0))      # decreasing block ids
    assert lib.mfsdp_plan(bad, 2, 1, 0, 0, 0, None, None, None, None, 0, ctypes.byref(n_desc), None) == mf.EINVAL
    zero = (mf.Param * 1)(mf.Param(0, 2, 0, 4, 0, 0))
    assert lib.mfsdp_plan(zero, 1, 1, 0, 0, 0, None, None, None, None, 0, ctypes.byref(n_desc), None) == mf.EINVAL


def test_validate_desc_rejects_bad_layouts():
    good = [dict(role=0, param_id=0, block_id=0, rows=8, cols=16, dtype=0, flags=0, elem_off=0),
            dict(role=0, param_id=1, block_id=0, rows=16, cols=8, dtype=0, flags=1, elem_off=128),
            dict(role=1, param_id=2, block_id=0, rows=5, cols=1, dtype=0, flags=0, elem_off=0)]
    assert mf.mfsdp_validate_desc(good) == 0
    overlap = [dict(good[0]), dict(good[1], elem_off=64)]
    assert mf.mfsdp_validate_desc(overlap) == mf.ELAYOUT
    misaligned = [dict(good[0], elem_off=8)]
    assert mf.mfsdp_validate_desc(misaligned) == mf.ELAYOUT
    wrong_flag = [dict(good[1], flags=0, elem_off=0)]
    assert mf.mfsdp_validate_desc(wrong_flag) == mf.ELAYOUT
    assert mf.mfsdp_flat_elems(good) == (256, 64)


def test_workspace_sizing_is_consistent():
    wl = workloads.get("small")
    pr = mf.mfsdp_plan(wl.params, 1)
    for prec, es in ((mf.NS_BF16, 2), (mf.NS_FP32, 4)):
        total = mf.mfsdp_workspace_bytes(pr.desc, prec)
        n_mat = sum(1 for i in range(pr.desc._n) if pr.desc[i].role == mf.ROLE_MATRIX)
        spans = []
        for i in range(n_mat):
            x0, x1, a, p, px, pa = mf.mfsdp_debug_ws_offsets(pr.desc, prec, i)
            d = [pr.desc[j] for j in range(pr.desc._n) if pr.desc[j].role == mf.ROLE_MATRIX][i]
            dmin = min(d.rows, d.cols)
            assert px >= d.cols and pa >= dmin and px % 8 == 0 and pa % 8 == 0
            for off, nbytes in ((x0, d.rows * px * es), (x1, d.rows * px * es), (a, dmin * pa * es), (p, dmin * pa * es)):
                assert off % 1024 == 0 and off + nbytes <= total
                spans.append((off, off + nbytes))
            o_off, o_pitch, ssq_off = mf.mfsdp_workspace_view(pr.desc, prec, 5, i)
            assert o_off == x1 and o_pitch == px and ssq_off == 8 * i          # K = 5 -> O in X buffer 1
        spans.sort()
        for (a0, a1), (b0, b1) in zip(spans, spans[1:]):
            assert a1 <= b0, "workspace buffers overlap"


def test_step_entry_points_reject_bad_arguments_without_a_gpu():
    """Argument checks run before any CUDA call; with valid arguments and no device the answer is MFSDP_EARCH."""
    lib = mf.load()
    wl = workloads.get("c1")
    pr = mf.mfsdp_plan(wl.params, 1)
    hp = mf.MuonHParams(precision=mf.NS_FP32)
    n = pr.desc._n
    assert lib.mfsdp_muon_step(pr.desc, n, None, None, None, None, 0, ctypes.byref(hp), None) == mf.EINVAL
    assert lib.mfsdp_muon_step(pr.desc, n, 1024, 1024, 1024, 1024, 0, None, None) == mf.EINVAL
    bad = mf.MuonHParams(ns_steps=0)
    assert lib.mfsdp_muon_step(pr.desc, n, 1024, 1024, 1024, 1024, 1 << 30, ctypes.byref(bad), None) == mf.EINVAL
    ah = mf.AdamWHParams(step=0)
    assert lib.mfsdp_adamw_tail_step(pr.desc, n, 1024, 1024, 1024, 1024, ctypes.byref(ah), None) == mf.EINVAL
    import torch
    if not torch.cuda.is_available():
        rc = lib.mfsdp_muon_step(pr.desc, n, 1024, 1024, 1024, 1024, 1 << 30, ctypes.byref(hp), None)
        assert rc == mf.EARCH, "no device must mean MFSDP_EARCH, never a CPU fallback"
        assert "no CPU fallback" in mf.mfsdp_strerror(mf.EARCH)


def test_tune_knobs_roundtrip_and_reject_bad_values():
    """mfsdp_tune / mfsdp_get_tune are host-only: defaults, round trip, error codes (no device needed)."""
    knobs = [mf.TUNE_PAIR_MIN_D, mf.TUNE_SYM_BAND, mf.TUNE_SYM_BAND2, mf.TUNE_RECT_GROUP, mf.TUNE_WIDE_MIN_KB,
             mf.TUNE_FUSED_BELOW_D, mf.TUNE_FUSED2_BELOW_D]
    old = [mf.mfsdp_get_tune(k) for k in knobs]
    assert old == [1024, 16, 8, 4, 8, 129, 257]         # the header's defaults; no environment variable can change them
    try:
        for k in knobs:
            mf.mfsdp_tune(k, 3)
            assert mf.mfsdp_get_tune(k) == 3
        for bad in ((-1, 1), (len(knobs), 1), (0, 0), (0, -5)):
            with pytest.raises(mf.MfsdpError) as e:
                mf.mfsdp_tune(*bad)
            assert e.value.code == mf.EINVAL
        with pytest.raises(mf.MfsdpError):
            mf.mfsdp_get_tune(99)
    finally:
        for k, v in zip(knobs, old):
            mf.mfsdp_tune(k, v)


def test_debug_trace_rejects_bad_buffers():
    lib = mf.load()
    assert lib.mfsdp_debug_trace(ctypes.c_void_p(8), 16) == mf.EINVAL       # too small
    assert lib.mfsdp_debug_trace(ctypes.c_void_p(12), 4096) == mf.EINVAL    # not 8-byte aligned
    assert lib.mfsdp_debug_trace(None, 0) == 0                              # off


def test_reduce_schedule_matches_oracle_bit_exact():
    """mfsdp_reduce_schedule (reading F1) against oracle.planner.reduce_schedule: records and the
    FNV-1a validation hash, on the Llama plans and on random models, both block orders."""
    def compare(params, world, owner, rev):
        want, wh = oplan.reduce_schedule(params, world, owner, rev)
        got, gh_ = mf.mfsdp_reduce_schedule(params, world, owner, rev)
        assert gh_ == wh and len(got) == len(want)
        for g, w in zip(got, want):
            assert (g.seq, g.role, g.kind, g.block_id, g.param_id, g.owner, g.dtype, g.flag, g.numel, g.owner_elem_off) == \
                (w["seq"], w["role"], w["kind"], w["block"], w["param_id"], w["owner"], w["dtype"], w["flag"], w["numel"],
                 w["owner_elem_off"])
    for name in ("c2", "c4", "c5"):
        wl = workloads.get(name)
        pr = mf.mfsdp_plan(wl.params, wl.world, wl.policy, wl.metric, 0)
        for rev in (True, False):
            compare(wl.params, wl.world, pr.owner, rev)
    rng = np.random.default_rng(31)
    for trial in range(150):
        params = []
        for b in range(int(rng.integers(1, 6))):
            for _ in range(int(rng.integers(0, 6))):
                if rng.random() < 0.6:
                    params.append((b, 2, int(rng.integers(1, 40)), int(rng.integers(1, 40)), int(rng.integers(0, 2)), 0))
                else:
                    params.append((b, 1, int(rng.integers(1, 300)), 1, 0, int(rng.random() < 0.1)))
        world = int(rng.integers(1, 7))
        n_roles = len(oplan.build_roles(params))
        compare(params, world, [int(rng.integers(0, world)) for _ in range(n_roles)], bool(trial % 2))


def test_gated_step_and_signal_reject_bad_arguments_without_a_gpu():
    lib = mf.load()
    wl = workloads.get("c1")
    pr = mf.mfsdp_plan(wl.params, 1)
    hp = mf.MuonHParams(precision=mf.NS_FP32)
    assert lib.mfsdp_muon_step_gated(pr.desc, pr.desc._n, 1024, 1024, 1024, 1024, 1 << 30, ctypes.byref(hp), None, 1,
                                     None) == mf.EINVAL                      # no flags
    assert lib.mfsdp_muon_step_gated(pr.desc, pr.desc._n, 1024, 1024, 1024, 1024, 1 << 30, ctypes.byref(hp), 1026, 1,
                                     None) == mf.EINVAL                      # misaligned flags
    assert lib.mfsdp_signal_ready(None, 0, 1, None) == mf.EINVAL


def test_shampoo_layout_and_argument_checks_without_a_gpu():
    """mfsdp_shampoo_state_bytes / _workspace_bytes / _view are host-only; the step checks its arguments before any
    CUDA call and answers MFSDP_EARCH without a device (no CPU fallback)."""
    assert ctypes.sizeof(mf.ShampooHParams) == 6 * 8 + 8 + 4 * 4
    lib = mf.load()
    wl = workloads.get("small")
    pr = mf.mfsdp_plan(wl.params, 1)
    n = pr.desc._n
    mats = [pr.desc[j] for j in range(n) if pr.desc[j].role == mf.ROLE_MATRIX]
    total = mf.mfsdp_shampoo_state_bytes(pr.desc)
    spans = []
    for i, d in enumerate(mats):
        v = mf.mfsdp_shampoo_view(pr.desc, mf.SHAMPOO_KEEP_D, i)
        pr_, pc_ = v[4], v[5]
        assert pr_ >= d.rows and pc_ >= d.cols and pr_ % 64 == 0 and pc_ % 64 == 0
        assert v[6] == d.rows * pr_ and v[7] == d.cols * pc_ and v[10] == 64
        for off, nbytes in ((v[0], d.rows * pr_ * 4), (v[1], d.cols * pc_ * 4), (v[2], 3 * v[6] * 2), (v[3], 3 * v[7] * 2)):
            assert off % 1024 == 0 and off + nbytes <= total
            spans.append((off, off + nbytes))
    spans.sort()
    for (a0, a1), (b0, b1) in zip(spans, spans[1:]):
        assert a1 <= b0, "state buffers overlap"
    lo, hi = mf.mfsdp_shampoo_workspace_bytes(pr.desc, 0)
    lo_d, hi_d = mf.mfsdp_shampoo_workspace_bytes(pr.desc, mf.SHAMPOO_KEEP_D)
    dmax = max(max(d.rows, d.cols) for d in mats)
    assert lo < hi and lo_d > lo and hi_d - hi == lo_d - lo
    assert lo >= 7 * 3 * dmax * dmax * 2, "the smallest workspace holds the seven three-plane buffers of the largest root"
    with pytest.raises(mf.MfsdpError):
        mf.mfsdp_shampoo_view(pr.desc, 0, len(mats))
    with pytest.raises(mf.MfsdpError):
        mf.mfsdp_shampoo_workspace_bytes(pr.desc, 2)
    # the step: argument checks first
    ok = mf.ShampooHParams(step=1)
    call = lambda hp, W=1024, G=1024, st=1024, ws=1024: lib.mfsdp_shampoo_step(pr.desc, n, W, G, st, 1 << 40, ws, 1 << 40,
                                                                                 ctypes.byref(hp) if hp else None, None)
    assert call(None) == mf.EINVAL
    for bad in (dict(step=0), dict(root_every=0), dict(beta2=0.0), dict(beta2=1.5), dict(eps=-1.0), dict(eps_floor=-1.0),
                dict(max_root_iters=-1), dict(flags=4)):
        assert call(mf.ShampooHParams(**dict(dict(step=1), **bad))) == mf.EINVAL, bad
    assert call(ok, W=None) == mf.EINVAL and call(ok, st=1000) == mf.EINVAL and call(ok, ws=1032) == mf.EINVAL
    import torch
    if not torch.cuda.is_available():
        assert call(ok) == mf.EARCH
    # a table without matrices is a no-op
    tails = mf.make_desc_array([pr.desc[j] for j in range(n) if pr.desc[j].role == mf.ROLE_TAIL])
    assert lib.mfsdp_shampoo_step(tails, tails._n, None, None, None, 0, None, 0, ctypes.byref(ok), None) == 0
