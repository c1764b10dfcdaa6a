"""Pins for oracle/shampoo.py ("Shampoo (full L/R preconditioners with inverse fourth root)").

The paper prints no Shampoo number, so every pin is a closed form, a defining property, a textbook special case or an
independent library route:
  * hand example G = diag(3, 4), eps = 0: L = R = diag(9, 16), roots diag(1/sqrt 3, 1/2), D = I;
  * diagonal G with the ridge written out; orthogonal G;
  * SVD form of the first step: D = U diag(s (s^2 + rho_L)^{-1/4} (s^2 + rho_R)^{-1/4}) V^T through LAPACK's SVD (not the
    eigendecomposition the oracle uses), and its eps -> 0 limit, the polar factor U V^T (what Muon's Newton-Schulz
    approximates -- the known identity "Shampoo without accumulation = orthogonalisation");
  * the defining property P^4 (S + rho I) = I and scipy's Schur-Pade fractional_matrix_power (another algorithm);
  * statistics: constant gradient closed forms for the running sum and the moving average, brute-force triple loops;
  * invariances: scale of G at step 1, transposition; stale roots under root_every; zero gradient.
A plausible mistake -- G^T G for L, exponent -1/2, ridge not scaled by the trace, w = 1 under a moving average, roots
taken before the statistics see G_t, P_R applied on the left -- fails at least one of them.
"""
import numpy as np
import pytest

from oracle import shampoo


def _rng(seed):
    return np.random.default_rng(seed)


def test_hand_example_diag_3_4():
    G = np.diag([3.0, 4.0])
    out = shampoo.shampoo_step(np.eye(2), G, np.zeros((2, 2)), np.zeros((2, 2)), None, None, 1, lr=0.5, eps=0.0)
    np.testing.assert_allclose(out["L"], np.diag([9.0, 16.0]), rtol=0, atol=0)
    np.testing.assert_allclose(out["R"], np.diag([9.0, 16.0]), rtol=0, atol=0)
    np.testing.assert_allclose(out["P_L"], np.diag([1 / np.sqrt(3.0), 0.5]), rtol=1e-15, atol=1e-16)
    np.testing.assert_allclose(out["D"], np.eye(2), rtol=1e-15, atol=1e-15)
    np.testing.assert_allclose(out["W"], 0.5 * np.eye(2), rtol=1e-15, atol=1e-15)


def test_diagonal_with_ridge_closed_form():
    g = np.array([0.5, -2.0, 3.0, 0.25])
    eps = 1e-2
    rho = eps * np.sum(g * g) / 4
    D = shampoo.shampoo_step(np.zeros((4, 4)), np.diag(g), np.zeros((4, 4)), np.zeros((4, 4)), None, None, 1,
                             eps=eps)["D"]
    np.testing.assert_allclose(D, np.diag(g / np.sqrt(g * g + rho)), rtol=1e-14, atol=1e-15)


def test_rectangular_ridges_differ():
    # 2 x 3, only two non-zero entries: L = diag(4, 9), R = diag(4, 9, 0); rho_L = eps 13/2, rho_R = eps 13/3
    G = np.array([[2.0, 0, 0], [0, 3.0, 0]])
    eps = 0.1
    out = shampoo.shampoo_step(np.zeros((2, 3)), G, np.zeros((2, 2)), np.zeros((3, 3)), None, None, 1, eps=eps)
    rl, rr = eps * 13 / 2, eps * 13 / 3
    want = np.zeros((2, 3))
    want[0, 0] = 2 * (4 + rl) ** -0.25 * (4 + rr) ** -0.25
    want[1, 1] = 3 * (9 + rl) ** -0.25 * (9 + rr) ** -0.25
    np.testing.assert_allclose(out["D"], want, rtol=1e-14, atol=1e-15)
    np.testing.assert_allclose(out["P_R"][2, 2], rr ** -0.25, rtol=1e-14)


def test_orthogonal_gradient():
    Q, _ = np.linalg.qr(_rng(0).standard_normal((6, 6)))
    eps = 1e-3
    out = shampoo.shampoo_step(np.zeros((6, 6)), Q, np.zeros((6, 6)), np.zeros((6, 6)), None, None, 1, eps=eps)
    np.testing.assert_allclose(out["D"], Q / np.sqrt(1 + eps), rtol=1e-12, atol=1e-13)


@pytest.mark.parametrize("shape", [(5, 5), (4, 9), (12, 3), (32, 96)])
def test_first_step_svd_form_and_polar_limit(shape):
    m, n = shape
    G = _rng(1).standard_normal(shape)
    U, s, Vt = np.linalg.svd(G, full_matrices=False)
    for eps in (1e-2, 1e-6):
        rl, rr = eps * np.sum(s * s) / m, eps * np.sum(s * s) / n
        want = (U * (s * (s * s + rl) ** -0.25 * (s * s + rr) ** -0.25)) @ Vt
        D = shampoo.shampoo_step(np.zeros(shape), G, np.zeros((m, m)), np.zeros((n, n)), None, None, 1, eps=eps)["D"]
        np.testing.assert_allclose(D, want, rtol=1e-9, atol=1e-11)
    D0 = shampoo.shampoo_step(np.zeros(shape), G, np.zeros((m, m)), np.zeros((n, n)), None, None, 1, eps=1e-14)["D"]
    np.testing.assert_allclose(D0, U @ Vt, rtol=0, atol=1e-6)       # polar factor: singular values all 1


def test_root_defining_property_and_scipy():
    scipy_linalg = pytest.importorskip("scipy.linalg")
    X = _rng(2).standard_normal((7, 20))
    S = X @ X.T
    eps = 1e-4
    P = shampoo.inverse_root(S, eps)
    St = S + eps * np.trace(S) / 7 * np.eye(7)
    np.testing.assert_allclose(P @ P @ P @ P @ St, np.eye(7), rtol=0, atol=1e-10)
    np.testing.assert_allclose(P, P.T, rtol=0, atol=1e-14)
    assert np.linalg.eigvalsh(P).min() > 0                           # the principal (positive definite) root
    np.testing.assert_allclose(P, scipy_linalg.fractional_matrix_power(St, -0.25).real, rtol=1e-9, atol=1e-12)
    # other orders: p = 2 is the inverse square root
    P2 = shampoo.inverse_root(S, eps, p=2)
    np.testing.assert_allclose(P2 @ P2 @ St, np.eye(7), rtol=0, atol=1e-10)


def test_rank_deficient_statistic_uses_the_ridge():
    # R = G^T G of a wide G has n - m zero eigenvalues; on that null space the root is rho^{-1/4}
    G = _rng(3).standard_normal((3, 8))
    eps = 1e-3
    P = shampoo.inverse_root(G.T @ G, eps)
    rho = eps * np.sum(G * G) / 8
    lam = np.sort(np.linalg.eigvalsh(P))
    np.testing.assert_allclose(lam[-5:], rho ** -0.25, rtol=1e-8)


def test_statistics_brute_force_and_orientation():
    G = _rng(4).standard_normal((3, 5))
    L0, R0 = _rng(5).standard_normal((3, 3)), _rng(6).standard_normal((5, 5))
    L, R = shampoo.statistics_update(L0, R0, G, beta2=0.9)
    for i in range(3):
        for j in range(3):
            assert L[i, j] == pytest.approx(0.9 * L0[i, j] + 0.1 * sum(G[i, k] * G[j, k] for k in range(5)), rel=1e-13)
    for i in range(5):
        for j in range(5):
            assert R[i, j] == pytest.approx(0.9 * R0[i, j] + 0.1 * sum(G[k, i] * G[k, j] for k in range(3)), rel=1e-13)
    L, R = shampoo.statistics_update(L0, R0, G, beta2=1.0)           # Gupta et al.: a running sum
    np.testing.assert_allclose(L, L0 + G @ G.T, rtol=1e-14)
    np.testing.assert_allclose(R, R0 + G.T @ G, rtol=1e-14)


@pytest.mark.parametrize("beta2", [1.0, 0.95])
def test_constant_gradient_closed_form(beta2):
    # L_t = c_t G G^T with c_t = t (sum) or 1 - beta2^t (average); the relative ridge makes D_t = D_1' / sqrt(c_t)
    # where D_1' is the first step's direction computed from the unweighted G G^T
    G = _rng(7).standard_normal((6, 10))
    eps = 1e-5
    base = shampoo.shampoo_step(np.zeros((6, 10)), G, np.zeros((6, 6)), np.zeros((10, 10)), None, None, 1, eps=eps,
                                beta2=1.0)["D"]
    L, R, PL, PR = np.zeros((6, 6)), np.zeros((10, 10)), None, None
    for t in range(1, 5):
        out = shampoo.shampoo_step(np.zeros((6, 10)), G, L, R, PL, PR, t, eps=eps, beta2=beta2)
        L, R, PL, PR = out["L"], out["R"], out["P_L"], out["P_R"]
        c = float(t) if beta2 == 1.0 else 1.0 - beta2 ** t
        np.testing.assert_allclose(L, c * (G @ G.T), rtol=1e-12)
        np.testing.assert_allclose(out["D"], base / np.sqrt(c), rtol=1e-9, atol=1e-12)


def test_scale_and_transpose_invariance():
    G = _rng(8).standard_normal((5, 9))
    z = lambda a, b: np.zeros((a, b))
    D = shampoo.shampoo_step(z(5, 9), G, z(5, 5), z(9, 9), None, None, 1, eps=1e-4)["D"]
    Dc = shampoo.shampoo_step(z(5, 9), 37.5 * G, z(5, 5), z(9, 9), None, None, 1, eps=1e-4)["D"]
    np.testing.assert_allclose(Dc, D, rtol=1e-10, atol=1e-13)
    Dt = shampoo.shampoo_step(z(9, 5), G.T, z(9, 9), z(5, 5), None, None, 1, eps=1e-4)["D"]
    np.testing.assert_allclose(Dt, D.T, rtol=1e-10, atol=1e-13)
    # left and right preconditioners are not interchangeable
    L, R = shampoo.statistics_update(z(5, 5), z(9, 9), G)
    assert L.shape == (5, 5) and R.shape == (9, 9)


def test_stale_roots_and_update():
    rng = _rng(9)
    G1, G2 = rng.standard_normal((4, 6)), rng.standard_normal((4, 6))
    W0 = rng.standard_normal((4, 6))
    s1 = shampoo.shampoo_step(W0, G1, np.zeros((4, 4)), np.zeros((6, 6)), None, None, 1, lr=0.1, weight_decay=0.5,
                              root_every=2)
    s2 = shampoo.shampoo_step(s1["W"], G2, s1["L"], s1["R"], s1["P_L"], s1["P_R"], 2, lr=0.1, weight_decay=0.5,
                              root_every=2)
    np.testing.assert_array_equal(s2["P_L"], s1["P_L"])              # step 2 reuses the roots of step 1 ...
    np.testing.assert_allclose(s2["L"], G1 @ G1.T + G2 @ G2.T, rtol=1e-13)   # ... while the statistics keep moving
    np.testing.assert_allclose(s2["D"], s1["P_L"] @ G2 @ s1["P_R"], rtol=1e-13)
    np.testing.assert_allclose(s2["W"], s1["W"] * (1 - 0.05) - 0.1 * s2["D"], rtol=1e-13)
    s3 = shampoo.shampoo_step(s2["W"], G1, s2["L"], s2["R"], s2["P_L"], s2["P_R"], 3, root_every=2)
    assert np.abs(s3["P_L"] - s2["P_L"]).max() > 1e-3                # step 3 refreshes, from statistics that include G_3
    np.testing.assert_allclose(s3["P_L"], shampoo.inverse_root(2 * G1 @ G1.T + G2 @ G2.T), rtol=1e-10)


def test_zero_gradient_only_decays():
    W0 = _rng(10).standard_normal((3, 4))
    out = shampoo.shampoo_step(W0, np.zeros((3, 4)), np.zeros((3, 3)), np.zeros((4, 4)), None, None, 1, lr=0.1,
                               weight_decay=0.1)
    np.testing.assert_array_equal(out["D"], np.zeros((3, 4)))
    np.testing.assert_array_equal(out["P_L"], np.eye(3))
    np.testing.assert_allclose(out["W"], W0 * 0.99, rtol=1e-15)


def test_ridge_floor_closed_form_and_switch():
    # reading S7: rho = max(eps tr S / d, eps_floor ||S||_F).  S = diag(9, 16, 0): tr / d = 25 / 3, ||S||_F = sqrt(337)
    S = np.diag([9.0, 16.0, 0.0])
    eps, fl = 1e-3, 1e-2
    rho_s2, rho_s7 = eps * 25 / 3, fl * np.sqrt(337.0)
    assert rho_s7 > rho_s2
    P = shampoo.inverse_root(S, eps, eps_floor=fl)
    np.testing.assert_allclose(P, np.diag([(9 + rho_s7) ** -0.25, (16 + rho_s7) ** -0.25, rho_s7 ** -0.25]), rtol=1e-14)
    # the floor is inactive when the S2 ridge is the larger one, and off by default
    P2 = shampoo.inverse_root(S, eps, eps_floor=1e-6)
    np.testing.assert_allclose(P2, np.diag([(9 + rho_s2) ** -0.25, (16 + rho_s2) ** -0.25, rho_s2 ** -0.25]), rtol=1e-14)
    np.testing.assert_array_equal(shampoo.inverse_root(S, eps), P2)
    # the step passes it to both roots
    G = np.array([[2.0, 0, 0], [0, 3.0, 0]])
    out = shampoo.shampoo_step(np.zeros((2, 3)), G, np.zeros((2, 2)), np.zeros((3, 3)), None, None, 1, eps=0.0,
                               eps_floor=0.1)
    rl = rr = 0.1 * np.sqrt(16.0 + 81.0)
    np.testing.assert_allclose(out["D"][0, 0], 2 * (4 + rl) ** -0.25 * (4 + rr) ** -0.25, rtol=1e-14)
    np.testing.assert_allclose(out["P_R"][2, 2], rr ** -0.25, rtol=1e-14)
