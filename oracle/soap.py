"""fp64 oracle of owner-local SOAP (TEST INFRASTRUCTURE -- see oracle/__init__.py).

STATUS: oracle and pins only.  No CUDA path for SOAP exists yet (row f4); this file is committed,
pinned, BEFORE any kernel that it will judge.

What the paper fixes (PAPER.md = /root/reference/PAPER.md):
  * PAPER.md:182 "... swapping owner-Muon for Shampoo (full L/R preconditioners with inverse fourth root) and SOAP
                  (Adam in the Shampoo eigenbasis) ..." -- owner-placed against a gathered reference, float32.
  * PAPER.md:7, 13, 31, 37 name SOAP beside Muon and Shampoo as a whole-matrix optimizer.
That one parenthesis is all the paper says.  What is computed here is the published algorithm (Vyas et al., 2024,
"SOAP: Improving and stabilizing Shampoo using Adam", Algorithm 3) restated under the readings SO1-SO7 of DESIGN.md
section 4, one statement per formula:
  SO1 statistics   L <- b_s L + (1 - b_s) G G^T,  R <- b_s R + (1 - b_s) G^T G  (reading S1 with a moving average;
                   b_s = "shampoo beta"; b_s = 1 gives the running sum); L_0 = R_0 = 0.
  SO2 basis        Q_L, Q_R orthogonal, columns = eigenvectors of L, R.  At the FIRST refresh: numpy.linalg.eigh (the
                   library primitive of this step), columns in order of DESCENDING eigenvalue, each column's sign chosen
                   so that its entry of largest magnitude is positive (first such entry on ties).  At every LATER
                   refresh: one step of power iteration followed by a QR factorisation, Q <- qr(S Q).Q, with the signs
                   fixed so that diag(R) > 0 -- for S Q of full column rank that factorisation is unique, so the basis
                   is a function of (S, previous Q) and column j keeps its identity from refresh to refresh.  Columns are
                   never re-sorted.
  SO3 schedule     as reading S5: the statistics take in G_t first; the bases are refreshed at steps t (1-based) with
                   (t - 1) % refresh_every == 0, from statistics that include G_t; other steps reuse the stored bases.
                   (The published algorithm refreshes after the step, from the basis of the previous gradient; S5 was
                   fixed for Shampoo first and SOAP follows it, so that both optimizers share one schedule.)
  SO4 moments      first moment M in the ORIGINAL space, M <- b1 M + (1 - b1) G, rotated when used, M' = Q_L^T M Q_R:
                   it needs no re-projection when the basis changes.  Second moment V in the ROTATED space,
                   V <- b2 V + (1 - b2) (G' * G'), G' = Q_L^T G Q_R; at a refresh V is kept as it is (not re-projected,
                   not permuted: SO2 keeps the columns' identity).  M_0 = V_0 = 0.
  SO5 Adam step    bias correction on, eps outside the square root and added after bias correction (reading A1):
                   N' = (M' / (1 - b1^t)) / (sqrt(V / (1 - b2^t)) + eps),  N = Q_L N' Q_R^T.
  SO6 update       W <- W (1 - eta lambda) - eta N  (decoupled decay, as for Muon, Shampoo and AdamW here).
  SO7 both sides   both dimensions are always preconditioned (no one-sided variant, no dimension cap, no merging of
                   small dimensions): the paper's runs place whole 2D matrices.

Everything is numpy float64.
"""
import numpy as np

from .shampoo import statistics_update


def eigenbasis_init(S):
    """SO2, first refresh: eigenvectors of the symmetric S, descending eigenvalues, largest-magnitude entry positive."""
    S = np.asarray(S, dtype=np.float64)
    lam, Q = np.linalg.eigh(S)
    Q = Q[:, ::-1].copy()
    for j in range(Q.shape[1]):
        i = int(np.argmax(np.abs(Q[:, j])))
        if Q[i, j] < 0.0:
            Q[:, j] = -Q[:, j]
    return Q


def eigenbasis_refresh(S, Q):
    """SO2, later refreshes: one power-iteration step and the QR factorisation with diag(R) > 0."""
    S = np.asarray(S, dtype=np.float64)
    Q = np.asarray(Q, dtype=np.float64)
    Z = S @ Q
    Q_new, R = np.linalg.qr(Z)
    sign = np.where(np.diag(R) < 0.0, -1.0, 1.0)
    return Q_new * sign[None, :]


def rotate(Q_L, X, Q_R):
    """X' = Q_L^T X Q_R."""
    return Q_L.T @ np.asarray(X, dtype=np.float64) @ Q_R


def rotate_back(Q_L, X, Q_R):
    """X = Q_L X' Q_R^T."""
    return Q_L @ np.asarray(X, dtype=np.float64) @ Q_R.T


def soap_init(rows, cols):
    """State before the first step (SO1, SO4): zero statistics and moments, no basis yet."""
    return dict(L=np.zeros((rows, rows)), R=np.zeros((cols, cols)), Q_L=None, Q_R=None,
                M=np.zeros((rows, cols)), V=np.zeros((rows, cols)))


def soap_step(W, G, state, step, lr=1e-3, beta1=0.9, beta2=0.95, shampoo_beta=0.95, eps=1e-8, weight_decay=0.01,
              refresh_every=10):
    """One SOAP step of one matrix, float64.  `step` is 1-based.  Returns (W_new, state_new, N)."""
    W = np.asarray(W, dtype=np.float64)
    G = np.asarray(G, dtype=np.float64)
    L, R = statistics_update(state["L"], state["R"], G, shampoo_beta)             # SO1
    Q_L, Q_R = state["Q_L"], state["Q_R"]
    if (step - 1) % refresh_every == 0:                                           # SO3
        if Q_L is None:
            Q_L, Q_R = eigenbasis_init(L), eigenbasis_init(R)                     # SO2, first refresh
        else:
            Q_L, Q_R = eigenbasis_refresh(L, Q_L), eigenbasis_refresh(R, Q_R)     # SO2, later refreshes
    M = beta1 * np.asarray(state["M"], dtype=np.float64) + (1.0 - beta1) * G      # SO4, original space
    G_rot = rotate(Q_L, G, Q_R)
    V = beta2 * np.asarray(state["V"], dtype=np.float64) + (1.0 - beta2) * G_rot * G_rot   # SO4, rotated space
    M_rot = rotate(Q_L, M, Q_R)
    m_hat = M_rot / (1.0 - beta1 ** step)                                         # SO5
    v_hat = V / (1.0 - beta2 ** step)
    N_rot = m_hat / (np.sqrt(v_hat) + eps)
    N = rotate_back(Q_L, N_rot, Q_R)
    W_new = W * (1.0 - lr * weight_decay) - lr * N                                # SO6
    return W_new, dict(L=L, R=R, Q_L=Q_L, Q_R=Q_R, M=M, V=V), N
