"""GPU parity at BASELINE.json's full sizes (`-m gpu`), in the launch configuration bench.py times.

C2 and C3 are compared with the full fp64 oracle (C2: every matrix at step 1, one matrix per shape at later steps; M,
||U||^2, the lock-step update and the AdamW tails on everything at every step).  C4 / C5: one matrix per DISTINCT
shape of the resident set gets the full fp64 oracle (4096 x 4096, 1024 x 4096, 14336 x 4096, 4096 x 14336; 8192 x 8192,
1024 x 8192, 28672 x 8192 -- about 4-5 minutes of dgemm on the box's host cores); every matrix gets momentum state,
||U||^2 and the lock-step update from the oracle's elementwise functions, the size-independent probe identities of
gpu_harness.probe_last_iteration (one per GEMM phase + fused epilogue) and a singular-value band check."""
import numpy as np
import pytest
import torch

import paper_2607_05895_b200 as mf
import workloads
from oracle import adamw as oadamw
from oracle import muon as omuon

import gpu_harness as gh
from helpers import rel_fro

pytestmark = pytest.mark.gpu


def _elementwise_checks(sess, i, W_old, M_old):
    """M, ||U||^2 and the lock-step update of matrix i by the oracle's elementwise functions (any size)."""
    d = sess.mats[i]
    hp = sess.hp
    G = sess.seg(sess.hG, d).to(torch.float64).numpy()
    M_ref, U_ref = omuon.momentum_update(M_old, G, hp.momentum, bool(hp.nesterov))
    assert rel_fro(sess.seg64(sess.M, d), M_ref) <= gh.TOL_STATE
    want = float(np.sum(U_ref * U_ref))
    assert abs(sess.read_ssq(i) - want) <= gh.TOL_STATE * want
    del G, M_ref, U_ref
    O_gpu = sess.read_O(i)
    assert np.isfinite(O_gpu).all()
    gh.check_update_lockstep(sess, d, W_old, sess.seg64(sess.W, d), O_gpu, None)
    return O_gpu


def _adamw_check(sess, t, state):
    P_old = [sess.seg64(sess.P, d).reshape(-1) for d in sess.tails]
    sess.adamw_step(t)
    for j, d in enumerate(sess.tails):
        g = sess.seg(sess.hGt, d).to(torch.float64).numpy().reshape(-1)
        m_old, v_old = state.get(j, (np.zeros(d.rows), np.zeros(d.rows)))
        p_ref, m_ref, v_ref = oadamw.adamw_step(P_old[j], g, m_old, v_old, t, **sess.wl.adamw)
        state[j] = (m_ref, v_ref)
        assert rel_fro(sess.seg64(sess.m, d).reshape(-1), m_ref) <= gh.TOL_STATE
        assert rel_fro(sess.seg64(sess.v, d).reshape(-1), v_ref) <= gh.TOL_STATE
        p_gpu = sess.seg64(sess.P, d).reshape(-1)
        assert np.abs(p_gpu - p_ref).max() <= 2.0 ** -8 * np.abs(p_ref).max()     # one bf16 rounding of p


def test_c2_gpt2_small_ten_steps():
    wl = workloads.get("c2")
    sess = gh.Session(wl)
    assert len(sess.mats) == 48 and len(sess.tails) == 12
    M_ref = [np.zeros((d.rows, d.cols)) for d in sess.mats]      # free-running oracle momentum
    adam_state = {}
    worst = 0.0
    for step in range(wl.steps):
        sess.load_grads(step)
        W_old = [sess.seg64(sess.W, d) for d in sess.mats]
        sess.muon_step()
        full = range(len(sess.mats)) if step == 0 else [4 * ((step + k) % 12) + k for k in range(4)]
        for i, d in enumerate(sess.mats):
            if i in full:
                eo, _ = gh.check_matrix_against_oracle(sess, i, W_old[i], M_ref[i])
                worst = max(worst, eo)
            else:
                _elementwise_checks(sess, i, W_old[i], M_ref[i])
            G = sess.seg(sess.hG, d).to(torch.float64).numpy()
            M_ref[i], _ = omuon.momentum_update(M_ref[i], G, sess.hp.momentum, bool(sess.hp.nesterov))
        _adamw_check(sess, step + 1, adam_state)
    assert worst <= 3e-2


def test_c3_ragged_512():
    wl = workloads.get("c3")
    sess = gh.Session(wl)
    assert len(sess.mats) == 512
    sess.load_grads(0)
    W_old = [sess.seg64(sess.W, d) for d in sess.mats]
    sess.muon_step()
    errs = []
    zeros = {}
    for i, d in enumerate(sess.mats):
        z = zeros.setdefault((d.rows, d.cols), np.zeros((d.rows, d.cols)))
        eo, _ = gh.check_matrix_against_oracle(sess, i, W_old[i], z)
        errs.append(eo)
    assert max(errs) <= 3e-2
    n_tall = sum(d.rows > d.cols for d in sess.mats)
    assert 150 <= n_tall <= 280       # the transposed path is really exercised


def test_vocab_embedding_shape():
    """50,257 x 768 (GPT-2 vocabulary embedding on Muon): odd row count, GRAM k loop of 786 blocks, APPLY
    with 197 row blocks; full oracle comparison plus the per-phase probes."""
    wl = workloads.get("vocab")
    sess = gh.Session(wl)
    sess.load_grads(0)
    W_old = [sess.seg64(sess.W, d) for d in sess.mats]
    M_old = [np.zeros((d.rows, d.cols)) for d in sess.mats]
    sess.muon_step()
    rng = np.random.default_rng(3)
    for i in range(len(sess.mats)):
        eo, _ = gh.check_matrix_against_oracle(sess, i, W_old[i], M_old[i])
        assert eo <= 3e-2
        gh.probe_last_iteration(sess, i, rng, 2e-2)


def _band_by_probes(O, rng, lo=0.55, hi=1.35):
    """O has singular values in the quintic's band ([0.68, 1.20] for sigma0 >= 0.002; tiny singular values
    of a heavy-tailed gradient may sit below).  ||O v|| <= sigma_max ||v|| for any v; and ||O||_F^2 / m is the mean
    squared singular value."""
    m, n = min(O.shape), max(O.shape)
    v = rng.standard_normal(O.shape[1])
    assert np.linalg.norm(O @ v) <= hi * np.linalg.norm(v)
    u = rng.standard_normal(O.shape[0])
    assert np.linalg.norm(u @ O) <= hi * np.linalg.norm(u)
    mean_sq = np.sum(O * O) / m
    assert lo ** 2 <= mean_sq <= hi ** 2, mean_sq


def _large_config(name):
    """One full fp64-oracle comparison (M, ||U||^2, O over the whole K-step chain, lock-step update) per DISTINCT shape
    of the resident set -- the 4096- / 8192-row matrices that carry > 99 % of the flops included (north_star: "matching
    the fp64 oracle ... on all five configs") -- and, on every other matrix, the oracle's elementwise functions for M,
    ||U||^2 and the update plus the size-independent probes."""
    wl = workloads.get(name)
    sess = gh.Session(wl)
    sess.load_grads(0)
    rng = np.random.default_rng(11)
    seen = {}
    # W_old / M_old one matrix at a time (host memory): M starts at zero, W_old is the seeded input
    sess.muon_step()
    for i, d in enumerate(sess.mats):
        W_old = sess.seg(sess.hW, d).to(torch.float64).numpy()
        M_old = np.zeros((d.rows, d.cols))
        if (d.rows, d.cols) not in seen:
            eo, _ = gh.check_matrix_against_oracle(sess, i, W_old, M_old)
            seen[(d.rows, d.cols)] = eo
            O = sess.read_O(i)
        else:
            O = _elementwise_checks(sess, i, W_old, M_old)
        _band_by_probes(O, rng)
        del O, W_old, M_old
        gh.probe_last_iteration(sess, i, rng, 2e-2)
    print("%s: relF(O) vs fp64 oracle per distinct shape: %s" % (name, ", ".join(
        "%dx%d %.2e" % (r, c, e) for (r, c), e in seen.items())))
    assert max(seen.values()) <= 3e-2
    state = {}
    _adamw_check(sess, 1, state)
    return sess, seen


def test_c4_llama8b_rank0():
    sess, seen = _large_config("c4")
    assert len(sess.mats) == 30
    assert set(seen) == {(4096, 4096), (1024, 4096), (14336, 4096), (4096, 14336)}


def test_c5_llama70b_heaviest():
    sess, seen = _large_config("c5")
    assert len(sess.mats) == 13
    assert set(seen) == {(8192, 8192), (1024, 8192), (28672, 8192)}
