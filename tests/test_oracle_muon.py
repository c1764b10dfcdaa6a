"""Pins for oracle/muon.py: closed forms, library routines (LAPACK SVD, torch.optim.Muon),
special matrices and invariants.  None of them re-types the oracle's own formula: the
momentum pins use the geometric closed form, the NS pins use the SVD form of the iteration
(scalar polynomial on singular values) or hand-worked matrices, the update pins are hand
numbers.  SURVEY.md 8(c) "What pins the oracle"."""
import os

import numpy as np
import pytest

from oracle import muon

RNG = np.random.default_rng(20260705895)
A_, B_, C_ = muon.NS_COEFFS


def load_table(path):
    rows = []
    for line in open(path):
        if line.startswith("#") or not line.strip():
            continue
        rows.append(line.split())
    return rows


def fk(x, k):
    """scalar quintic in Horner form on singular values (SVD form of the NS iteration)."""
    x = np.asarray(x, dtype=np.float64)
    for _ in range(k):
        x2 = x * x
        x = x * (A_ + x2 * (B_ + C_ * x2))
    return x


# ------------------------------------------------------------------ momentum

def test_momentum_constant_gradient_closed_form(golden_dir):
    table = load_table(os.path.join(golden_dir, "momentum_constant_grad.txt"))
    G = RNG.standard_normal((5, 7))
    M = np.zeros_like(G)
    for k, mk, uk in table:
        M, U = muon.momentum_update(M, G, 0.95, nesterov=True)
        np.testing.assert_allclose(M, float(mk) * G, rtol=1e-14, atol=0)
        np.testing.assert_allclose(U, float(uk) * G, rtol=1e-14, atol=0)


def test_momentum_general_sum_form():
    mu = 0.9
    Gs = [RNG.standard_normal((4, 3)) for _ in range(6)]
    M = np.zeros((4, 3))
    for k, G in enumerate(Gs, start=1):
        M, U = muon.momentum_update(M, G, mu, nesterov=True)
        expect = (1 - mu) * sum(mu ** (k - j) * Gs[j - 1] for j in range(1, k + 1))
        np.testing.assert_allclose(M, expect, rtol=1e-13, atol=1e-16)
        np.testing.assert_allclose(U, (1 - mu) * G + mu * expect, rtol=1e-13, atol=1e-16)


def test_momentum_without_nesterov_is_the_buffer():
    G = RNG.standard_normal((3, 3))
    M0 = RNG.standard_normal((3, 3))
    M, U = muon.momentum_update(M0, G, 0.5, nesterov=False)
    np.testing.assert_array_equal(M, U)
    np.testing.assert_allclose(M, 0.5 * M0 + 0.5 * G, rtol=1e-15)


def test_momentum_convention_switch_leaves_O_unchanged():
    # reading M1: classic buffers are the EMA buffers / (1 - mu); U is proportional; O identical.
    mu = 0.95
    Gs = [RNG.standard_normal((6, 10)) for _ in range(3)]
    Me = Mc = np.zeros((6, 10))
    for G in Gs:
        Me, Ue = muon.momentum_update(Me, G, mu, True)
        Mc, Uc = muon.momentum_update(Mc, G, mu, True, classic=True)
        np.testing.assert_allclose(Mc, Me / (1 - mu), rtol=1e-13)
        np.testing.assert_allclose(Uc, Ue / (1 - mu), rtol=1e-13)
        np.testing.assert_allclose(muon.newton_schulz(Uc), muon.newton_schulz(Ue), rtol=0, atol=1e-13)


# ------------------------------------------------------------------ Newton-Schulz

def test_quintic_scalars_match_golden(golden_dir):
    # pins the helper used by the SVD-form tests below to exact arithmetic
    for x0, k, val in load_table(os.path.join(golden_dir, "ns_quintic_scalars.txt")):
        x = np.sqrt(0.5) if x0 == "sqrt(1/2)" else float(x0)
        assert abs(fk(x, int(k)) - float(val)) <= 2e-13 * abs(float(val))


@pytest.mark.parametrize("shape", [(4, 8), (8, 4), (16, 16), (33, 70), (70, 33), (128, 512), (96, 64)])
@pytest.mark.parametrize("steps", [1, 2, 5])
def test_ns_equals_svd_form(shape, steps):
    """O = U diag(f^K(sigma_i / ||G||_F)) V^T  -- LAPACK SVD + scalar polynomial."""
    G = RNG.standard_normal(shape) * np.exp(0.5 * RNG.standard_normal((shape[0], 1)))
    Us, s, Vt = np.linalg.svd(G, full_matrices=False)
    expect = (Us * fk(s / np.linalg.norm(G), steps)) @ Vt
    O = muon.newton_schulz(G, steps=steps)
    assert O.shape == G.shape
    assert np.linalg.norm(O - expect) <= 1e-12 * np.linalg.norm(expect)
    # singular vectors: U^T O V is diagonal
    D = Us.T @ O @ Vt.T
    off = D - np.diag(np.diag(D))
    assert np.abs(off).max() <= 1e-12


def test_ns_output_band_and_not_polar_factor():
    G = RNG.standard_normal((48, 96))
    O = muon.newton_schulz(G)
    s = np.linalg.svd(O, compute_uv=False)
    # sigma0 = s_i/||G||_F in [0.01, 1] here -> invariant band's image (SURVEY.md 8(c) band pin)
    s0 = np.linalg.svd(G, compute_uv=False) / np.linalg.norm(G)
    assert s0.min() > 0.01
    assert s.min() >= 0.681831 - 1e-6 and s.max() <= 1.134357 + 1e-6
    Us, _, Vt = np.linalg.svd(G, full_matrices=False)
    polar = Us @ Vt
    rel = np.linalg.norm(O - polar) / np.linalg.norm(polar)
    assert 0.05 < rel < 0.4          # close in direction, not in norm: it is a band, not convergence
    cos = np.sum(O * polar) / (np.linalg.norm(O) * np.linalg.norm(polar))
    assert cos > 0.97


def test_quintic_band_on_a_grid():
    x = np.linspace(1e-6, 1.0, 200001)
    y = fk(x, 1)
    assert y.max() <= 1.202369 + 1e-6            # local max 1.202369 at x = 0.554529
    i = np.argmax(y)
    assert abs(x[i] - 0.554529) < 1e-4
    xr = np.linspace(0.9, 1.21, 310001)           # iterates can exceed 1 (up to 1.2024): local min at x = 1.050136
    yr = fk(xr, 1)
    assert abs(yr.min() - 0.681831) < 1e-5
    assert abs(xr[np.argmin(yr)] - 1.050136) < 1e-4
    assert abs(fk(1.0, 1) - 0.701) < 1e-15
    y5 = fk(np.linspace(0.002, 1.0, 100001), 5)
    assert y5.min() >= 0.681831 - 1e-6 and y5.max() <= 1.202369 + 1e-6


def test_ns_special_matrices(golden_dir):
    tab = {(r[0], int(r[1])): float(r[2]) for r in load_table(os.path.join(golden_dir, "ns_quintic_scalars.txt"))}
    # diag(3, 4): ||G|| = 5 -> O = diag(f5(0.6), f5(0.8))
    O = muon.newton_schulz(np.diag([3.0, 4.0]))
    np.testing.assert_allclose(O, np.diag([tab[("0.6", 5)], tab[("0.8", 5)]]), rtol=1e-12, atol=1e-15)
    # orthogonal Q (m x m): all singular values 1/sqrt(m)
    Q, _ = np.linalg.qr(RNG.standard_normal((2, 2)))
    np.testing.assert_allclose(muon.newton_schulz(Q), tab[("sqrt(1/2)", 5)] * Q, rtol=1e-11, atol=1e-14)
    Q100, _ = np.linalg.qr(RNG.standard_normal((100, 100)))
    np.testing.assert_allclose(muon.newton_schulz(Q100), tab[("0.1", 5)] * Q100, rtol=1e-10, atol=1e-13)
    # rank one
    u, v = RNG.standard_normal(5), RNG.standard_normal(9)
    expect = tab[("1", 5)] * np.outer(u / np.linalg.norm(u), v / np.linalg.norm(v))
    np.testing.assert_allclose(muon.newton_schulz(np.outer(u, v)), expect, rtol=1e-11, atol=1e-14)
    np.testing.assert_allclose(muon.newton_schulz(np.outer(v, u)), expect.T, rtol=1e-11, atol=1e-14)
    # K = 2 (the paper's own setting)
    np.testing.assert_allclose(muon.newton_schulz(np.outer(u, v), steps=2),
                               tab[("1", 2)] * np.outer(u / np.linalg.norm(u), v / np.linalg.norm(v)),
                               rtol=1e-12, atol=1e-15)
    # zero gradient: exactly zero, no NaN (reading M3)
    Z = muon.newton_schulz(np.zeros((3, 5)))
    assert np.all(Z == 0.0)


def test_ns_eps_is_a_clamp_not_an_addend(golden_dir):
    tab = {(r[0], int(r[1])): float(r[2]) for r in load_table(os.path.join(golden_dir, "ns_quintic_scalars.txt"))}
    u = np.array([1.0, 0.0, 0.0]); v = np.array([0.0, 1.0, 0.0, 0.0])
    # ||G|| = 1e-7 exactly: clamp -> sigma0 = 1 -> f5(1); the additive form would give f5(0.5)
    O = muon.newton_schulz(1e-7 * np.outer(u, v))
    assert abs(O[0, 1] - tab[("1", 5)]) < 1e-9
    # ||G|| = 5e-8 < eps: X0 = G / eps -> sigma0 = 0.5
    O = muon.newton_schulz(5e-8 * np.outer(u, v))
    assert abs(O[0, 1] - tab[("0.5", 5)]) < 1e-9


def test_ns_first_iterate_brute_force():
    """X1 = a X + b (X X^T) X + c (X X^T)^2 X by explicit loops on a tiny matrix; also pins that
    the iteration acts from the left on the wide orientation (transposed operand would change A's shape)."""
    G = RNG.standard_normal((3, 5))
    X = G / np.sqrt(sum(G[i, j] ** 2 for i in range(3) for j in range(5)))
    S = [[sum(X[i, k] * X[j, k] for k in range(5)) for j in range(3)] for i in range(3)]
    S2 = [[sum(S[i][k] * S[k][j] for k in range(3)) for j in range(3)] for i in range(3)]
    X1 = np.zeros((3, 5))
    for i in range(3):
        for j in range(5):
            X1[i, j] = A_ * X[i, j] + sum((B_ * S[i][k] + C_ * S2[i][k]) * X[k, j] for k in range(3))
    O, its = muon.newton_schulz(G, steps=1, return_iterates=True)
    np.testing.assert_allclose(its[0], X, rtol=1e-14)
    np.testing.assert_allclose(O, X1, rtol=1e-13, atol=1e-15)


def test_ns_invariances():
    G = RNG.standard_normal((12, 20))
    O = muon.newton_schulz(G)
    # positive scaling
    np.testing.assert_allclose(muon.newton_schulz(37.5 * G), O, rtol=0, atol=1e-13)
    np.testing.assert_allclose(muon.newton_schulz(1e-3 * G), O, rtol=0, atol=1e-13)
    # transpose symmetry (also pins the tall-matrix rule)
    np.testing.assert_allclose(muon.newton_schulz(G.T), O.T, rtol=0, atol=1e-13)
    # orthogonal equivariance
    Q1, _ = np.linalg.qr(RNG.standard_normal((12, 12)))
    Q2, _ = np.linalg.qr(RNG.standard_normal((20, 20)))
    np.testing.assert_allclose(muon.newton_schulz(Q1 @ G @ Q2), Q1 @ O @ Q2, rtol=0, atol=1e-12)
    # permutation equivariance
    pr, pc = RNG.permutation(12), RNG.permutation(20)
    np.testing.assert_allclose(muon.newton_schulz(G[pr][:, pc]), O[pr][:, pc], rtol=0, atol=1e-13)
    # sign
    np.testing.assert_allclose(muon.newton_schulz(-G), -O, rtol=0, atol=1e-15)


def test_ns_tall_equals_in_place_right_iteration():
    """Reading M6: transposing a tall matrix is the same as iterating X <- aX + X(bA' + cA'^2), A' = X^T X."""
    G = RNG.standard_normal((40, 12))
    X = G / np.linalg.norm(G)
    for _ in range(5):
        Ap = X.T @ X
        X = A_ * X + X @ (B_ * Ap + C_ * Ap @ Ap)
    np.testing.assert_allclose(muon.newton_schulz(G), X, rtol=0, atol=1e-13)


def test_ns_square_is_not_transposed_but_it_would_not_matter():
    G = RNG.standard_normal((9, 9))
    np.testing.assert_allclose(muon.newton_schulz(G), muon.newton_schulz(G.T).T, rtol=0, atol=1e-13)


# ------------------------------------------------------------------ update

def test_update_scale_values():
    assert muon.update_scale(256, 256) == pytest.approx(3.2, rel=1e-15)
    assert muon.update_scale(256, 1024) == pytest.approx(6.4, rel=1e-15)
    assert muon.update_scale(1024, 256) == pytest.approx(6.4, rel=1e-15)
    assert muon.update_scale(28672, 8192) == pytest.approx(33.8656168, rel=1e-8)   # 0.2*sqrt(28672) = 0.2*169.3280839...
    assert muon.update_scale(64, 256, muon.SCALE_ORIGINAL) == 1.0
    assert muon.update_scale(256, 64, muon.SCALE_ORIGINAL) == 2.0
    assert muon.update_scale(5, 7, muon.SCALE_NONE) == 1.0


def test_weight_update_hand_example(golden_dir):
    tab = {(r[0], int(r[1])): float(r[2]) for r in load_table(os.path.join(golden_dir, "ns_quintic_scalars.txt"))}
    out = muon.muon_step(np.eye(2), np.diag([3.0, 4.0]), np.zeros((2, 2)), lr=0.02, weight_decay=0.01,
                         momentum=0.95, nesterov=True, scale_mode=muon.SCALE_ORIGINAL)
    # U = 0.0975 G -> same direction -> O = diag(f5(.6), f5(.8)); W' = 0.9998 I - 0.02 O
    expect = 0.9998 * np.eye(2) - 0.02 * np.diag([tab[("0.6", 5)], tab[("0.8", 5)]])
    np.testing.assert_allclose(out["W"], expect, rtol=1e-13, atol=1e-16)
    np.testing.assert_allclose(out["M"], 0.05 * np.diag([3.0, 4.0]), rtol=1e-15)
    assert out["ssq"] == pytest.approx(0.0975 ** 2 * 25.0, rel=1e-14)
    # decay uses the unadjusted lr: with match_rms the decay factor is still 1 - lr*wd
    out2 = muon.muon_step(np.eye(2), np.diag([3.0, 4.0]), np.zeros((2, 2)), lr=0.02, weight_decay=0.01)
    s = 0.2 * np.sqrt(2.0)
    np.testing.assert_allclose(out2["W"], 0.9998 * np.eye(2) - 0.02 * s * np.diag([tab[("0.6", 5)], tab[("0.8", 5)]]),
                               rtol=1e-13, atol=1e-16)


# ------------------------------------------------------------------ the optimizer the paper names

@pytest.mark.parametrize("shape", [(64, 256), (256, 64), (96, 96)])
def test_against_torch_optim_muon(shape):
    """the paper's runs use torch.optim.Muon.  Black-box call of the installed one
    (a library routine): its momentum buffer must equal the oracle's (EMA form, reading M1) and its
    weight update must agree up to its internal bf16 Newton-Schulz (reading M4)."""
    torch = pytest.importorskip("torch")
    if not hasattr(torch.optim, "Muon"):
        pytest.skip("torch.optim.Muon not in this torch")
    g = torch.Generator().manual_seed(7)
    W0 = (0.02 * torch.randn(shape, generator=g, dtype=torch.float64))
    p = torch.nn.Parameter(W0.clone())
    opt = torch.optim.Muon([p], lr=0.02, weight_decay=0.01, momentum=0.95, nesterov=True,
                           ns_steps=5, adjust_lr_fn="match_rms_adamw")
    W = W0.numpy().copy()
    M = np.zeros(shape)
    for step in range(2):
        G = 1e-3 * torch.randn(shape, generator=g, dtype=torch.float64)
        p.grad = G.clone()
        opt.step()
        out = muon.muon_step(W, G.numpy(), M, lr=0.02, weight_decay=0.01, momentum=0.95, nesterov=True,
                             scale_mode=muon.SCALE_MATCH_RMS_ADAMW)
        W_prev, W, M = W, out["W"], out["M"]
        buf = opt.state[p]["momentum_buffer"].numpy()
        assert np.linalg.norm(buf - M) <= 1e-12 * np.linalg.norm(M)
        dW_t = p.detach().numpy() - W_prev
        dW_o = W - W_prev
        assert np.linalg.norm(dW_t - dW_o) <= 3e-2 * np.linalg.norm(dW_o)
        # keep the two trajectories in lock step so step 2 compares a single step again
        with torch.no_grad():
            p.copy_(torch.from_numpy(W))


def test_against_torch_optim_muon_original_scale():
    torch = pytest.importorskip("torch")
    if not hasattr(torch.optim, "Muon"):
        pytest.skip("torch.optim.Muon not in this torch")
    g = torch.Generator().manual_seed(11)
    shape = (128, 32)
    W0 = 0.02 * torch.randn(shape, generator=g, dtype=torch.float64)
    G = 1e-3 * torch.randn(shape, generator=g, dtype=torch.float64)
    p = torch.nn.Parameter(W0.clone())
    opt = torch.optim.Muon([p], lr=0.02, weight_decay=0.01, momentum=0.5, nesterov=False, ns_steps=2,
                           adjust_lr_fn="original")
    p.grad = G.clone()
    opt.step()
    out = muon.muon_step(W0.numpy(), G.numpy(), np.zeros(shape), lr=0.02, weight_decay=0.01, momentum=0.5,
                         nesterov=False, ns_steps=2, scale_mode=muon.SCALE_ORIGINAL)
    dW_t = p.detach().numpy() - W0.numpy()
    dW_o = out["W"] - W0.numpy()
    assert np.linalg.norm(dW_t - dW_o) <= 3e-2 * np.linalg.norm(dW_o)
