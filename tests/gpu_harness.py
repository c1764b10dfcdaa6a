"""Shared plumbing of the GPU parity tests: plan -> seeded inputs -> device buffers -> C-ABI calls -> read-back.
No method arithmetic here; expected values come from oracle/ only."""
import numpy as np
import torch

import paper_2607_05895_b200 as mf
import workloads
from oracle import adamw as oadamw
from oracle import muon as omuon

from helpers import bf16_rne, bf16_ulp_distance, rel_fro

TOL_O = {mf.NS_BF16: 3e-2, mf.NS_FP32: 1e-4}     # BASELINE.json north_star
TOL_STATE = 1e-6


def aligned_bytes(nbytes, device="cuda", align=1024):
    """uint8 device tensor of nbytes whose data_ptr is `align`-byte aligned (torch only guarantees 512)."""
    raw = torch.empty(nbytes + align, dtype=torch.uint8, device=device)
    off = (-raw.data_ptr()) % align
    out = raw[off:off + nbytes]
    out._keep = raw
    return out


class Session:
    """One resident set on the GPU."""

    def __init__(self, wl, desc=None, precision=None, hp_over=None):
        self.wl = wl
        if desc is None:
            pr = mf.mfsdp_plan(wl.params, wl.world, wl.policy, wl.metric, wl.rank)
            desc = pr.desc
            self.plan = pr
        self.desc = mf.make_desc_array(desc)
        self.n_desc = self.desc._n
        self.descs = [self.desc[i] for i in range(self.n_desc)]
        self.mats = [d for d in self.descs if d.role == mf.ROLE_MATRIX]
        self.tails = [d for d in self.descs if d.role == mf.ROLE_TAIL]
        self.precision = wl.precision if precision is None else precision
        kw = dict(wl.muon)
        kw.update(hp_over or {})
        kw.setdefault("flags", mf.STEP_KEEP_O)       # the tests read O back after the whole step
        self.hp = mf.MuonHParams(precision=self.precision, **kw)
        self.n_mat_el, self.n_tail_el = mf.mfsdp_flat_elems(self.desc)
        self.tdt = workloads.TORCH_DTYPE[wl.dtype]
        self.ws = aligned_bytes(mf.mfsdp_workspace_bytes(self.desc, self.precision))
        self.hW = workloads.fill_flat(wl, self.descs, workloads.KIND_W)
        self.W = self.hW.cuda()
        self.M = torch.zeros(self.n_mat_el, dtype=torch.float32, device="cuda")
        self.hG = None
        self.G = None
        # tails
        self.hP = workloads.fill_flat(wl, self.descs, workloads.KIND_W, role=mf.ROLE_TAIL)
        self.P = self.hP.cuda()
        self.m = torch.zeros(self.n_tail_el, dtype=torch.float32, device="cuda")
        self.v = torch.zeros(self.n_tail_el, dtype=torch.float32, device="cuda")
        self.hGt = None
        self.Gt = None

    def load_grads(self, step):
        self.hG = workloads.fill_flat(self.wl, self.descs, workloads.KIND_G, step=step)
        self.G = self.hG.cuda()
        self.hGt = workloads.fill_flat(self.wl, self.descs, workloads.KIND_G, step=step, role=mf.ROLE_TAIL)
        self.Gt = self.hGt.cuda()

    def muon_step(self):
        mf.mfsdp_muon_step(self.desc, self.W, self.G, self.M, self.ws, self.hp)
        torch.cuda.synchronize()

    def adamw_step(self, t):
        kw = dict(self.wl.adamw)
        mf.mfsdp_adamw_tail_step(self.desc, self.P, self.Gt, self.m, self.v, mf.AdamWHParams(step=t, **kw))
        torch.cuda.synchronize()

    # ---- read-back (numpy float64) -------------------------------------------------------------------------------
    def seg(self, flat, d):
        n = d.rows * d.cols
        return flat[d.elem_off:d.elem_off + n].reshape(d.rows, d.cols)

    def seg64(self, flat, d):
        return self.seg(flat, d).to(torch.float64).cpu().numpy()

    def ws_matrix(self, byte_off, rows, cols, pitch):
        es = 2 if self.precision == mf.NS_BF16 else 4
        dt = torch.bfloat16 if self.precision == mf.NS_BF16 else torch.float32
        raw = self.ws[byte_off:byte_off + rows * pitch * es].view(dt).reshape(rows, pitch)[:, :cols]
        return raw.to(torch.float64).cpu().numpy()

    def read_O(self, i):
        d = self.mats[i]
        o_off, pitch, _ = mf.mfsdp_workspace_view(self.desc, self.precision, self.hp.ns_steps, i)
        return self.ws_matrix(o_off, d.rows, d.cols, pitch)

    def read_ssq(self, i):
        _, _, s_off = mf.mfsdp_workspace_view(self.desc, self.precision, self.hp.ns_steps, i)
        return float(self.ws[s_off:s_off + 8].view(torch.float64).cpu().item())

    def read_ns_buffers(self, i):
        """(X_prev, A, P, X_last) of the LAST iteration, float64."""
        d = self.mats[i]
        x0, x1, a, p, px, pa = mf.mfsdp_debug_ws_offsets(self.desc, self.precision, i)
        k = self.hp.ns_steps
        xs = (x0, x1)
        dmin = min(d.rows, d.cols)
        return (self.ws_matrix(xs[(k - 1) & 1], d.rows, d.cols, px), self.ws_matrix(a, dmin, dmin, pa),
                self.ws_matrix(p, dmin, dmin, pa), self.ws_matrix(xs[k & 1], d.rows, d.cols, px))


def oracle_muon(sess, i, W_old, M_old):
    """fp64 oracle step of matrix i from the stored inputs."""
    d = sess.mats[i]
    hp = sess.hp
    G = sess.seg(sess.hG, d).to(torch.float64).numpy()
    return omuon.muon_step(W_old, G, M_old, lr=hp.lr, weight_decay=hp.weight_decay, momentum=hp.momentum,
                           nesterov=bool(hp.nesterov), ns_steps=hp.ns_steps, coeffs=(hp.a, hp.b, hp.c), eps=hp.eps,
                           scale_mode=hp.scale_mode)


def check_update_lockstep(sess, d, W_old64, W_new_gpu64, O_gpu64, tol_o):
    """SURVEY.md 8(c) "Tolerances" with DESIGN.md reading U1: the oracle's update formula, evaluated in fp64 from the
    GPU's own O, is `want`; the kernel evaluates fma(-fl(lr s), O, fl(1 - lr wd) W) in fp32, i.e. errs by at most
    delta = 4 * 2^-24 * (|W_old| + |lr s O|) per element (relative to the OPERANDS, which may cancel).
    bf16 storage -> W_gpu lies in [rne_bf16(want - delta), rne_bf16(want + delta)] on every element and differs from
    rne_bf16(want) on <= 1e-3 of them; fp32 storage -> |W_gpu - want| <= delta on every element."""
    hp = sess.hp
    s = omuon.update_scale(d.rows, d.cols, hp.scale_mode)
    want = omuon.weight_update(W_old64, O_gpu64, hp.lr, hp.weight_decay, s)
    delta = 4.0 * 2.0 ** -24 * (np.abs(W_old64) + np.abs(hp.lr * s * O_gpu64))
    if sess.wl.dtype == mf.BF16:
        # W_gpu must be the bf16 rounding of some x with |x - want| <= delta.
        lo, hi = bf16_rne(want - delta).astype(np.float64), bf16_rne(want + delta).astype(np.float64)
        bad = (W_new_gpu64 < lo) | (W_new_gpu64 > hi)
        assert not bad.any(), "update outside the fp32 rounding interval on %d elements" % bad.sum()
        off = W_new_gpu64 != bf16_rne(want).astype(np.float64)
        assert off.mean() <= 1e-3, "%.2e of elements differ from the fp64 rounding" % off.mean()
    else:
        bad = np.abs(W_new_gpu64 - want) > delta
        assert not bad.any(), "fp32 update outside the fp32 rounding bound on %d elements" % bad.sum()


def check_matrix_against_oracle(sess, i, W_old64, M_old64, tol_o=None, check_O=True):
    """Full comparison of matrix i after one GPU step.  Returns (errO, errM)."""
    d = sess.mats[i]
    tol_o = TOL_O[sess.precision] if tol_o is None else tol_o
    ref = oracle_muon(sess, i, W_old64, M_old64) if check_O else None
    M_gpu = sess.seg64(sess.M, d)
    O_gpu = sess.read_O(i)
    W_gpu = sess.seg64(sess.W, d)
    assert np.isfinite(O_gpu).all()
    err_o = err_m = None
    if check_O:
        err_m = rel_fro(M_gpu, ref["M"])
        assert err_m <= TOL_STATE, "momentum relF %.3e (matrix %d %dx%d)" % (err_m, i, d.rows, d.cols)
        ssq = sess.read_ssq(i)
        assert abs(ssq - ref["ssq"]) <= TOL_STATE * ref["ssq"], "ssq %r vs %r" % (ssq, ref["ssq"])
        err_o = rel_fro(O_gpu, ref["O"])
        assert err_o <= tol_o, "O relF %.3e > %.1e (matrix %d %dx%d)" % (err_o, tol_o, i, d.rows, d.cols)
        if sess.wl.dtype == mf.F32:
            err_w = rel_fro(W_gpu - W_old64, ref["W"] - W_old64)
            assert err_w <= tol_o, "W update relF %.3e" % err_w
    check_update_lockstep(sess, d, W_old64, W_gpu, O_gpu, tol_o)
    return err_o, err_m


def probe_last_iteration(sess, i, rng, tol):
    """Size-independent property of the tensor-core phases, checked on the workspace the step leaves behind:
    with random probe vectors v (fp64 matvecs, O(mn) each), for the last iteration
        A v == Y (Y^T v),   P v == a v + b A v + c A (A v),   X_last-side product == P applied to Y
    where Y is the wide view of X_prev.  Each identity tests one GEMM phase + its fused epilogue."""
    d = sess.mats[i]
    hp = sess.hp
    if sess.precision == mf.NS_BF16 and mf.mfsdp_ns_class(d.rows, d.cols) == 0:
        return                 # whole-matrix kernel: A and P never leave the SM (nothing to probe; O is oracle-checked)
    Xp, A, P, Xl = sess.read_ns_buffers(i)
    tall = d.rows > d.cols
    Y = Xp.T if tall else Xp
    Yl = Xl.T if tall else Xl
    dmin, nlong = Y.shape
    first = hp.ns_steps == 1
    if first:
        return
    v = rng.standard_normal(dmin)
    Av = Y @ (Y.T @ v)
    e1 = np.linalg.norm(A @ v - Av) / np.linalg.norm(Av)
    Pv = hp.a * v + hp.b * (A @ v) + hp.c * (A @ (A @ v))
    e2 = np.linalg.norm(P @ v - Pv) / np.linalg.norm(Pv)
    u = rng.standard_normal(nlong)
    want = P @ (Y @ u)
    e3 = np.linalg.norm(Yl @ u - want) / np.linalg.norm(want)
    assert max(e1, e2, e3) <= tol, "probe errors %.2e %.2e %.2e (matrix %d %dx%d)" % (e1, e2, e3, i, d.rows, d.cols)
    assert np.abs(A - A.T).max() == 0.0 and np.abs(P - P.T).max() == 0.0, "mirrored write not symmetric"


def oracle_adamw_all(sess, t, P_old, m_old, v_old):
    out = []
    for j, d in enumerate(sess.tails):
        g = sess.seg(sess.hGt, d).to(torch.float64).numpy().reshape(-1)
        kw = dict(sess.wl.adamw)
        out.append(oadamw.adamw_step(P_old[j], g, m_old[j], v_old[j], t, **kw))
    return out
