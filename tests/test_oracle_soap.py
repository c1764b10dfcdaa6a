"""Pins of oracle/soap.py (`-m "not gpu"`): the SOAP oracle against things other than itself -- the AdamW oracle (itself
pinned by a 50-digit golden) on inputs where the eigenbasis is a permutation, LAPACK's SVD (first step = polar factor),
exact equivariance under orthogonal changes of basis, a hand example, brute-force loops for the rotations, uniqueness
of the sign-fixed QR, convergence of the refresh rule to the eigendecomposition.  Readings SO1-SO7: DESIGN.md section 4.
No CUDA path for SOAP exists yet; these pins come first."""
import numpy as np
import pytest

from oracle import adamw as oadamw
from oracle import soap as osoap

KW = dict(lr=1e-2, beta1=0.9, beta2=0.95, shampoo_beta=0.9, eps=1e-8, weight_decay=0.1)


def _run(W, grads, refresh_every, **kw):
    args = dict(KW)
    args.update(kw)
    st = osoap.soap_init(*W.shape)
    out = []
    for t, G in enumerate(grads, 1):
        W, st, N = osoap.soap_step(W, G, st, t, refresh_every=refresh_every, **args)
        out.append((W, N, st))
    return out


def test_hand_example_diag_3_4():
    """G = diag(3, 4): L = R = (1 - b_s) diag(9, 16); descending eigenvalues put e_2 first, so Q = [[0, 1], [1, 0]] and
    G' = diag(4, 3).  Step 1: m^ = g', v^ = g'^2, N' = g' / (|g'| + eps) -> N = diag(3 / (3 + eps), 4 / (4 + eps))."""
    W = np.array([[1.0, 2.0], [3.0, 4.0]])
    G = np.diag([3.0, 4.0])
    Wn, st, N = osoap.soap_step(W, G, osoap.soap_init(2, 2), 1, lr=0.5, beta1=0.9, beta2=0.95, shampoo_beta=0.75,
                                eps=1e-8, weight_decay=0.1, refresh_every=1)
    assert np.array_equal(st["L"], 0.25 * np.diag([9.0, 16.0])) and np.array_equal(st["R"], st["L"])
    assert np.array_equal(st["Q_L"], np.array([[0.0, 1.0], [1.0, 0.0]])) and np.array_equal(st["Q_R"], st["Q_L"])
    want_N = np.diag([3.0 / (3.0 + 1e-8), 4.0 / (4.0 + 1e-8)])
    assert np.allclose(N, want_N, rtol=0, atol=1e-15)
    assert np.allclose(Wn, W * 0.95 - 0.5 * want_N, rtol=0, atol=1e-15)
    assert np.allclose(st["V"], 0.05 * np.diag([16.0, 9.0]), rtol=1e-15) and np.allclose(st["M"], 0.1 * G, rtol=1e-15)


@pytest.mark.parametrize("refresh_every", [1, 2, 5])
def test_diagonal_gradients_reduce_to_adamw(refresh_every):
    """Diagonal gradients with distinct magnitudes keep L and R diagonal, so every basis (eigh at the first refresh,
    power iteration + QR later) is a permutation matrix and Adam in that basis is Adam: W must follow oracle.adamw
    element by element over six steps (the off-diagonal weights see a zero gradient: decay only)."""
    rng = np.random.default_rng(0)
    n = 5
    W = rng.standard_normal((n, n))
    grads = [np.diag(rng.uniform(0.5, 2.0, n) * rng.choice([-1.0, 1.0], n) * (1 + np.arange(n))) for _ in range(6)]
    got = _run(W, grads, refresh_every)
    p, m, v = W.reshape(-1), np.zeros(n * n), np.zeros(n * n)
    for t, G in enumerate(grads, 1):
        p, m, v = oadamw.adamw_step(p, G.reshape(-1), m, v, t, lr=KW["lr"], beta1=KW["beta1"], beta2=KW["beta2"],
                                    eps=KW["eps"], weight_decay=KW["weight_decay"])
        Q = got[t - 1][2]["Q_L"]
        assert np.allclose(np.abs(Q).max(axis=0), 1.0, atol=1e-12) and np.count_nonzero(np.abs(Q) > 1e-12) == n   # a permutation
        assert np.allclose(got[t - 1][0].reshape(-1), p, rtol=0, atol=1e-8), t      # rounding dust / eps = 1e-16 / 1e-8, times lr


@pytest.mark.parametrize("shape", [(6, 6), (4, 9), (9, 4)])
def test_first_step_is_the_polar_factor(shape):
    """Step 1 with a fresh eigh basis: Q_L, Q_R are the singular vectors of G, G' = diag(sigma) (up to signs and
    zero padding), m^ / (sqrt(v^) + eps) = sign(sigma) on the diagonal and 0 elsewhere, so N = U V^T, the polar factor
    of G (what Newton-Schulz approximates) -- through LAPACK's SVD, to about eps / sigma_min."""
    rng = np.random.default_rng(1)
    G = rng.standard_normal(shape)
    _, _, N = osoap.soap_step(np.zeros(shape), G, osoap.soap_init(*shape), 1, refresh_every=1, **KW)
    U, s, Vt = np.linalg.svd(G, full_matrices=False)
    assert np.abs(N - U @ Vt).max() <= 1e-6
    assert np.allclose(np.linalg.svd(N, compute_uv=False), 1.0, atol=1e-6)


@pytest.mark.parametrize("refresh_every", [1, 3])
def test_equivariance_under_orthogonal_changes_of_basis(refresh_every):
    """SOAP(A W B^T; A G_t B^T) = A SOAP(W; G_t) B^T for orthogonal A, B, at every step: the statistics, both kinds of
    refresh (the sign rules flip columns of Q consistently, and nothing in the update depends on a column's sign), the
    rotated second moment.  A transposed operand, a basis applied on the wrong side or a re-projected V fails here."""
    rng = np.random.default_rng(2)
    m, n = 6, 6       # square: both statistics have full rank and distinct eigenvalues from the first step on (see below)
    A, _ = np.linalg.qr(rng.standard_normal((m, m)))
    B, _ = np.linalg.qr(rng.standard_normal((n, n)))
    W = rng.standard_normal((m, n))
    grads = [rng.standard_normal((m, n)) for _ in range(7)]
    a = _run(W, grads, refresh_every)
    b = _run(A @ W @ B.T, [A @ G @ B.T for G in grads], refresh_every)
    for t in range(7):
        assert np.abs(b[t][0] - A @ a[t][0] @ B.T).max() <= 1e-7, t      # a wrong side or a transposed operand is O(lr) = 1e-2
        assert np.abs(b[t][2]["V"] - a[t][2]["V"]).max() <= 1e-7 * np.abs(a[t][2]["V"]).max(), t


def test_rectangular_equivariance_holds_at_the_first_step_only():
    """For a 5 x 7 matrix R = G^T G has a two-dimensional null space at step 1; eigh's basis INSIDE it is arbitrary (any
    rotation of it is an eigenbasis), and Adam is not rotation-invariant.  Step 1 does not see the choice (G' vanishes
    there); later steps do, until the statistic has full rank and a refresh has happened.  Recorded as a property of the
    method -- a GPU comparison must fix that sub-basis (take it from this oracle) or compare what does not depend on it."""
    rng = np.random.default_rng(9)
    m, n = 5, 7
    A, _ = np.linalg.qr(rng.standard_normal((m, m)))
    B, _ = np.linalg.qr(rng.standard_normal((n, n)))
    W = rng.standard_normal((m, n))
    grads = [rng.standard_normal((m, n)) for _ in range(2)]
    a = _run(W, grads, 5)
    b = _run(A @ W @ B.T, [A @ G @ B.T for G in grads], 5)
    assert np.abs(b[0][0] - A @ a[0][0] @ B.T).max() <= 1e-7
    assert np.abs(b[1][0] - A @ a[1][0] @ B.T).max() > 1e-6


def test_transpose_symmetry():
    """SOAP(W^T; G_t^T) = SOAP(W; G_t)^T: L and R, Q_L and Q_R swap roles."""
    rng = np.random.default_rng(3)
    W = rng.standard_normal((4, 6))
    grads = [rng.standard_normal((4, 6)) for _ in range(5)]
    a = _run(W, grads, 2)
    b = _run(W.T, [G.T for G in grads], 2)
    for t in range(5):
        assert np.abs(b[t][0] - a[t][0].T).max() <= 1e-8


def test_rotations_against_brute_force_loops():
    rng = np.random.default_rng(4)
    m, n = 3, 4
    QL, _ = np.linalg.qr(rng.standard_normal((m, m)))
    QR, _ = np.linalg.qr(rng.standard_normal((n, n)))
    X = rng.standard_normal((m, n))
    fwd = np.zeros((m, n))
    back = np.zeros((m, n))
    for i in range(m):
        for j in range(n):
            for k in range(m):
                for l in range(n):
                    fwd[i, j] += QL[k, i] * X[k, l] * QR[l, j]        # (Q_L^T X Q_R)_ij
                    back[i, j] += QL[i, k] * X[k, l] * QR[j, l]       # (Q_L X Q_R^T)_ij
    assert np.allclose(osoap.rotate(QL, X, QR), fwd, atol=1e-14)
    assert np.allclose(osoap.rotate_back(QL, X, QR), back, atol=1e-14)
    assert np.allclose(osoap.rotate_back(QL, osoap.rotate(QL, X, QR), QR), X, atol=1e-14)


def test_sign_fixed_qr_is_unique_and_keeps_column_identity():
    """eigenbasis_refresh is a function of span and order only: flipping columns of the incoming Q flips the same
    columns of the outgoing one; the result is orthogonal and spans S Q column by column (R upper triangular, diag > 0)."""
    rng = np.random.default_rng(5)
    n = 6
    X = rng.standard_normal((n, 3 * n))
    S = X @ X.T
    Q0, _ = np.linalg.qr(rng.standard_normal((n, n)))
    Q1 = osoap.eigenbasis_refresh(S, Q0)
    assert np.allclose(Q1.T @ Q1, np.eye(n), atol=1e-13)
    Rr = Q1.T @ (S @ Q0)
    assert np.all(np.diag(Rr) > 0) and np.abs(np.tril(Rr, -1)).max() <= 1e-10 * np.abs(Rr).max()
    D = np.diag([1.0, -1.0, 1.0, -1.0, -1.0, 1.0])
    assert np.allclose(osoap.eigenbasis_refresh(S, Q0 @ D), Q1 @ D, atol=1e-12)


def test_refresh_rule_converges_to_the_eigendecomposition():
    """Repeated refreshes on a fixed statistic are orthogonal (subspace) iteration: started from the eigh basis they stay
    there (a fixed point, columns and signs included); started from a perturbed basis they return to it."""
    rng = np.random.default_rng(6)
    n = 5
    V, _ = np.linalg.qr(rng.standard_normal((n, n)))
    S = (V * np.array([16.0, 8.0, 4.0, 2.0, 1.0])) @ V.T
    Q = osoap.eigenbasis_init(S)
    assert np.allclose(np.diag(Q.T @ S @ Q), [16.0, 8.0, 4.0, 2.0, 1.0], rtol=1e-12)
    assert all(Q[np.argmax(np.abs(Q[:, j])), j] > 0 for j in range(n))
    assert np.allclose(osoap.eigenbasis_refresh(S, Q), Q, atol=1e-12)
    P, _ = np.linalg.qr(Q + 0.05 * rng.standard_normal((n, n)))
    P = P * np.sign(np.sum(P * Q, axis=0))[None, :]
    for _ in range(60):
        P = osoap.eigenbasis_refresh(S, P)
    assert np.abs(P - Q).max() <= 1e-9


def test_stale_basis_schedule_and_second_moment_kept_across_a_refresh():
    """refresh_every = 3: steps 2, 3 reuse step 1's bases bit for bit, step 4 changes them; V is carried over as it is
    (SO4): V_4 = b2 V_3 + (1 - b2) G'_4^2 with G'_4 in the NEW basis."""
    rng = np.random.default_rng(7)
    W = rng.standard_normal((4, 5))
    grads = [rng.standard_normal((4, 5)) for _ in range(4)]
    r = _run(W, grads, 3)
    for t in (1, 2):
        assert np.array_equal(r[t][2]["Q_L"], r[0][2]["Q_L"]) and np.array_equal(r[t][2]["Q_R"], r[0][2]["Q_R"])
    assert np.abs(r[3][2]["Q_L"] - r[0][2]["Q_L"]).max() > 1e-3
    Gp = r[3][2]["Q_L"].T @ grads[3] @ r[3][2]["Q_R"]
    assert np.allclose(r[3][2]["V"], KW["beta2"] * r[2][2]["V"] + (1 - KW["beta2"]) * Gp * Gp, rtol=1e-13, atol=0)


def test_memoryless_limit_is_a_sign_update_in_the_eigenbasis():
    """b1 = b2 = 0: N' = g' / (|g'| + eps) at every step, i.e. N = Q_L sign(G') Q_R^T wherever |g'| >> eps; singular values
    of N are then NOT all one after the first step (the basis is stale relative to G_t), but |N'| <= 1 entrywise."""
    rng = np.random.default_rng(8)
    W = rng.standard_normal((4, 4))
    grads = [rng.standard_normal((4, 4)) for _ in range(3)]
    r = _run(W, grads, 1, beta1=0.0, beta2=0.0)
    for t in range(3):
        st = r[t][2]
        Gp = st["Q_L"].T @ grads[t] @ st["Q_R"]
        Np = st["Q_L"].T @ r[t][1] @ st["Q_R"]
        big = np.abs(Gp) > 1e-3
        assert np.allclose(Np[big], np.sign(Gp[big]), atol=1e-4) and np.abs(Np).max() <= 1.0


def test_zero_gradient_only_decays():
    W = np.arange(6.0).reshape(2, 3)
    Wn, st, N = osoap.soap_step(W, np.zeros((2, 3)), osoap.soap_init(2, 3), 1, refresh_every=1, **KW)
    assert np.array_equal(N, np.zeros((2, 3))) and np.allclose(Wn, W * (1 - KW["lr"] * KW["weight_decay"]))
    assert np.allclose(st["Q_L"].T @ st["Q_L"], np.eye(2)) and np.allclose(st["Q_R"].T @ st["Q_R"], np.eye(3))
