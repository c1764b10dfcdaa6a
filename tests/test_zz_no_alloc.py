"""mfsdp_momentum_pass_static: the momentum pass for callers that must not allocate on the GPU.

Who needs it: a trainer whose own allocator has already taken the device memory it planned for (a raw cudaMalloc from a
library may fail there, or break the job's memory limit), and code that runs in the step loop while the gradient
reduction is still busy on another stream (cudaMalloc / cudaFree stop the whole device, which is the overlap the owner
layout exists for).  The ordinary entry points build cached launch tables with cudaMalloc on first use and want a
workspace; this one keeps its only scratch -- the per-chunk partial sums of ||U||^2 -- in a fixed 512 KiB array that
is part of the library's device image, so it allocates nothing, and it refuses matrices above 2^30 elements.

What is checked: on the same seeded inputs the new entry point returns the same M, X~ = cast(U) and ||U||^2 as the
existing mfsdp_muon_momentum_pass (which the parity tests tie to the fp64 oracle), bit for bit, on two calls in a row
per matrix -- the second call finds the scratch array as the first one left it, and the momentum carries over.

This file sorts last on purpose (pytest -x stops at the first failure, so a failure here hides nothing), and it holds
no state of its own: it passes alone in a fresh process and after the rest of the suite.
"""
import numpy as np
import pytest
import torch

import paper_2607_05895_b200 as mf
import workloads

import gpu_harness as gh

FAKE = 1 << 20            # a non-null, well-aligned address that is never dereferenced (the call fails before any launch)


def test_rejects_sizes_beyond_the_fixed_scratch():
    """Needs no GPU: the size check comes before anything touches the device."""
    limit = mf.mfsdp_static_max_elems()
    assert limit == 65536 * 16384
    hp = mf.MuonHParams()
    with pytest.raises(mf.MfsdpError) as e:
        mf.mfsdp_momentum_pass_static(65536, 16385, mf.BF16, mf.NS_BF16, FAKE, FAKE, FAKE, FAKE, FAKE, hp, stream=0)
    assert e.value.code == mf.ETOOBIG and "mfsdp_static_max_elems" in str(e.value)
    for bad in (dict(rows=0), dict(dtype=7), dict(precision=5), dict(G=None), dict(M=FAKE + 4), dict(ssq=FAKE + 4)):
        kw = dict(rows=8, cols=8, dtype=mf.BF16, precision=mf.NS_BF16, G=FAKE, M=FAKE, X=FAKE, ssq=FAKE, inv_norm=FAKE)
        kw.update(bad)
        with pytest.raises(mf.MfsdpError) as e:
            mf.mfsdp_momentum_pass_static(hp=hp, stream=0, **kw)
        assert e.value.code == mf.EINVAL, bad


def _existing_path(sess, steps):
    """The table-driven pass, `steps` calls in a row.  Per step and matrix: (M bits, X~ bits, ||U||^2)."""
    out = []
    for step in range(steps):
        sess.load_grads(step)
        mf.mfsdp_muon_momentum_pass(sess.desc, sess.G, sess.M, sess.ws, sess.hp)
        torch.cuda.synchronize()
        rec = []
        for i, d in enumerate(sess.mats):
            x0, _, _, _, px, _ = mf.mfsdp_debug_ws_offsets(sess.desc, sess.precision, i)
            es, dt = (2, torch.bfloat16) if sess.precision == mf.NS_BF16 else (4, torch.float32)
            X = sess.ws[x0:x0 + d.rows * px * es].view(dt).reshape(d.rows, px)[:, :d.cols].clone().contiguous()
            rec.append((sess.seg(sess.M, d).clone(), X, sess.read_ssq(i)))
        out.append(rec)
    return out


@pytest.mark.gpu
@pytest.mark.parametrize("dtype", [mf.BF16, mf.F32])
@pytest.mark.parametrize("precision", [mf.NS_BF16, mf.NS_FP32])
@pytest.mark.parametrize("nesterov", [1, 0])
def test_static_pass_equals_existing_pass_two_calls_in_a_row(dtype, precision, nesterov):
    wl = workloads.medium_ragged(dtype=dtype, precision=precision)     # 4 to 40 chunks per matrix, ragged last chunk
    sess = gh.Session(wl, hp_over=dict(nesterov=nesterov))
    want = _existing_path(sess, 2)
    xdt = torch.bfloat16 if precision == mf.NS_BF16 else torch.float32
    for i, d in enumerate(sess.mats):
        M = torch.zeros(d.rows * d.cols, dtype=torch.float32, device="cuda")
        X = torch.empty(d.rows * d.cols, dtype=xdt, device="cuda")
        ssq = torch.zeros(1, dtype=torch.float64, device="cuda")
        inv = torch.zeros(1, dtype=torch.float32, device="cuda")
        for step in range(2):                                           # second call: scratch as the first left it
            hG = workloads.fill_flat(wl, sess.descs, workloads.KIND_G, step=step)
            G = hG[d.elem_off:d.elem_off + d.rows * d.cols].cuda()
            X.fill_(float("nan"))
            mf.mfsdp_momentum_pass_static(d.rows, d.cols, dtype, precision, G, M, X, ssq, inv, sess.hp)
            torch.cuda.synchronize()
            M_ref, X_ref, ssq_ref = want[step][i]
            assert torch.equal(M.view(torch.int32), M_ref.reshape(-1).view(torch.int32)), (i, step)
            assert torch.equal(X.reshape(d.rows, d.cols), X_ref), (i, step)
            got = float(ssq.item())
            assert got == ssq_ref and got > 0.0, (i, step, got, ssq_ref)
            # 1 / max(||U||, eps), formed in double and rounded once (include/mfsdp.h)
            inv_want = 1.0 / max(np.sqrt(got), sess.hp.eps)
            assert abs(float(inv.item()) - inv_want) <= gh.TOL_STATE * inv_want


@pytest.mark.gpu
def test_static_pass_odd_pitch_and_tiny_shapes():
    """Shapes whose cols are not a multiple of 8 (the table-driven path pads X's row pitch, this one does not), a
    single-element matrix, and a call with a smaller matrix right after a larger one (stale partials beyond its
    chunk count must not leak into its norm)."""
    wl = workloads.small_ragged(dtype=mf.BF16, precision=mf.NS_BF16)
    sess = gh.Session(wl)
    want = _existing_path(sess, 2)
    order = sorted(range(len(sess.mats)), key=lambda i: -sess.mats[i].rows * sess.mats[i].cols)   # large first
    Ms = {i: torch.zeros(sess.mats[i].rows * sess.mats[i].cols, dtype=torch.float32, device="cuda") for i in order}
    ssq = torch.zeros(1, dtype=torch.float64, device="cuda")
    inv = torch.zeros(1, dtype=torch.float32, device="cuda")
    for step in range(2):
        hG = workloads.fill_flat(wl, sess.descs, workloads.KIND_G, step=step)
        for i in order:
            d = sess.mats[i]
            n = d.rows * d.cols
            G = hG[d.elem_off:d.elem_off + n].cuda()
            X = torch.empty(n, dtype=torch.bfloat16, device="cuda")
            mf.mfsdp_momentum_pass_static(d.rows, d.cols, mf.BF16, mf.NS_BF16, G, Ms[i], X, ssq, inv, sess.hp)
            torch.cuda.synchronize()
            M_ref, X_ref, ssq_ref = want[step][i]
            assert torch.equal(Ms[i].view(torch.int32), M_ref.reshape(-1).view(torch.int32)), (i, step)
            assert torch.equal(X.reshape(d.rows, d.cols), X_ref), (i, step)
            assert float(ssq.item()) == ssq_ref, (i, step)
    # 1 x 1
    G = torch.tensor([3.0], dtype=torch.float32, device="cuda")
    M = torch.zeros(1, dtype=torch.float32, device="cuda")
    X = torch.zeros(4, dtype=torch.float32, device="cuda")
    hp = mf.MuonHParams(momentum=0.5, nesterov=0, precision=mf.NS_FP32)
    mf.mfsdp_momentum_pass_static(1, 1, mf.F32, mf.NS_FP32, G, M, X, ssq, inv, hp)
    torch.cuda.synchronize()
    assert M.item() == 1.5 and X[0].item() == 1.5 and ssq.item() == 2.25 and abs(inv.item() - 1 / 1.5) < 1e-7


@pytest.mark.gpu
def test_static_pass_allocates_nothing():
    """Device memory in use (cudaMemGetInfo, which sees every allocation of the process, not only torch's) does not
    move across calls once the first call on the device has done its set-up."""
    n_r, n_c = 1024, 2048
    G = torch.randn(n_r * n_c, device="cuda", dtype=torch.float32, generator=torch.Generator("cuda").manual_seed(3))
    M = torch.zeros_like(G)
    X = torch.empty(n_r * n_c, dtype=torch.bfloat16, device="cuda")
    ssq = torch.zeros(1, dtype=torch.float64, device="cuda")
    inv = torch.zeros(1, dtype=torch.float32, device="cuda")
    hp = mf.MuonHParams()
    mf.mfsdp_momentum_pass_static(n_r, n_c, mf.F32, mf.NS_BF16, G, M, X, ssq, inv, hp)      # set-up call
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(5):
        mf.mfsdp_momentum_pass_static(n_r, n_c, mf.F32, mf.NS_BF16, G, M, X, ssq, inv, hp)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0
