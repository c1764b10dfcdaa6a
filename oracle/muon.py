"""fp64 oracle of the owner-local Muon step (TEST INFRASTRUCTURE -- see oracle/__init__.py).

What the paper fixes (PAPER.md = /root/reference/PAPER.md):
  * PAPER.md:7   "Muon orthogonalizes momentum-smoothed updates with Newton-Schulz and
                  therefore requires each complete 2D matrix as optimizer input."
  * PAPER.md:37  "For a 2D weight with momentum-buffered gradient G, Muon applies a
                  Newton-Schulz orthogonalization whose steps are built from products
                  such as X X^T."
  * PAPER.md:47  "The owner applies the Newton-Schulz update to the full matrix and
                  updates its local parameter and Muon state".
  * PAPER.md:121 hyper-parameters of the paper's runs: lr 1e-3, weight decay 1e-2,
                  momentum 0.5, 2 NS steps, match_rms_adamw (torch.optim.Muon).
The paper never prints the formulas; BASELINE.json's north_star does ("Nesterov
momentum, Frobenius normalisation, a 5-step quintic Newton-Schulz orthogonalisation
(A = X X^T, B = bA + cA^2, X <- aX + B X, transposing tall matrices) and the scaled,
weight-decayed weight update", fallback coefficients (3.4445, -4.7750, 2.0315)).
The readings taken where both are silent are SURVEY.md section 8(c) M1-M11 and are
listed in DESIGN.md section 4.

Everything is numpy float64, one statement per formula, in the order of SURVEY.md
8(c) O-2.  `@` (BLAS dgemm) is the only library primitive used as a step.
"""
import numpy as np

# north_star fallback coefficients (the paper gives none).
NS_COEFFS = (3.4445, -4.7750, 2.0315)
NS_EPS = 1e-7

SCALE_MATCH_RMS_ADAMW = 0
SCALE_ORIGINAL = 1
SCALE_NONE = 2


def momentum_update(M, G, mu, nesterov=True, classic=False):
    """O-2 steps 1-2 (reading M1: EMA form).

    M <- mu*M + (1-mu)*G ;  U = (1-mu)*G + mu*M  (Nesterov)  or  U = M.
    classic=True is the other public convention (M <- mu*M + G ; U = G + mu*M), kept
    only so a test can check that O is unchanged and M differs by 1/(1-mu).
    Returns (M_new, U), both float64.
    """
    M = np.asarray(M, dtype=np.float64)
    G = np.asarray(G, dtype=np.float64)
    if classic:
        M_new = mu * M + G
        U = G + mu * M_new if nesterov else M_new
    else:
        M_new = mu * M + (1.0 - mu) * G
        U = (1.0 - mu) * G + mu * M_new if nesterov else M_new
    return M_new, U


def newton_schulz(U, steps=5, coeffs=NS_COEFFS, eps=NS_EPS, return_iterates=False):
    """O-2 steps 3-6: transpose tall, Frobenius-normalise, K quintic iterations, transpose back.

    X0 = U / max(||U||_F, eps)                       (reading M3: clamp form, eps = 1e-7)
    repeat K times:  A = X X^T ; B = b A + c A A ; X <- a X + B X
    Tall matrices (rows > cols) are transposed first and the result transposed back
    (north_star; reading M6: square matrices are not transposed).
    """
    a, b, c = coeffs
    U = np.asarray(U, dtype=np.float64)
    rows, cols = U.shape
    transposed = rows > cols
    X = U.T.copy() if transposed else U.copy()
    norm = np.sqrt(np.sum(X * X))
    X = X / max(norm, eps)
    iterates = [X.copy()] if return_iterates else None
    for _ in range(steps):
        A = X @ X.T
        B = b * A + c * (A @ A)
        X = a * X + B @ X
        if return_iterates:
            iterates.append(X.copy())
    O = X.T.copy() if transposed else X
    if return_iterates:
        return O, iterates
    return O


def update_scale(rows, cols, mode=SCALE_MATCH_RMS_ADAMW):
    """O-2 step 7 scale s(rows, cols) (reading M7).

    match_rms_adamw (the paper's setting): 0.2*sqrt(max(rows, cols));
    original: sqrt(max(1, rows/cols)); none: 1.
    """
    if mode == SCALE_MATCH_RMS_ADAMW:
        return 0.2 * np.sqrt(float(max(rows, cols)))
    if mode == SCALE_ORIGINAL:
        return np.sqrt(max(1.0, float(rows) / float(cols)))
    if mode == SCALE_NONE:
        return 1.0
    raise ValueError("unknown scale mode %r" % (mode,))


def weight_update(W, O, lr, weight_decay, scale):
    """O-2 step 7: W <- W*(1 - lr*wd) - lr*s*O  (decoupled decay with the unadjusted lr, reading M8)."""
    W = np.asarray(W, dtype=np.float64)
    O = np.asarray(O, dtype=np.float64)
    return W * (1.0 - lr * weight_decay) - lr * scale * O


def muon_step(W, G, M, lr=0.02, weight_decay=0.01, momentum=0.95, nesterov=True,
              ns_steps=5, coeffs=NS_COEFFS, eps=NS_EPS, scale_mode=SCALE_MATCH_RMS_ADAMW):
    """One whole owner-local Muon step for one matrix, O-2 steps 1-7.

    Inputs are the *stored* values (bf16/fp32 values are exactly representable in fp64).
    Returns dict(W=, M=, ssq=, O=) in float64; storage rounding is the comparison's business.
    """
    M_new, U = momentum_update(M, G, momentum, nesterov)
    ssq = float(np.sum(U * U))
    O = newton_schulz(U, ns_steps, coeffs, eps)
    rows, cols = U.shape
    W_new = weight_update(W, O, lr, weight_decay, update_scale(rows, cols, scale_mode))
    return {"W": W_new, "M": M_new, "ssq": ssq, "O": O}

