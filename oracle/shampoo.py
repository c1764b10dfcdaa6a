"""fp64 oracle of owner-local Shampoo (TEST INFRASTRUCTURE -- see oracle/__init__.py).

What the paper fixes (PAPER.md = /root/reference/PAPER.md):
  * PAPER.md:182 "The owner-placement runtime is optimizer-agnostic: each 2D matrix is whole on
                  its owner, so any single-device matrix optimizer runs there with no gather and
                  no distributed variant.  We verify this by swapping owner-Muon for Shampoo
                  (full L/R preconditioners with inverse fourth root) ... float32".
  * PAPER.md:13, 37 name the algorithm: Shampoo (Gupta et al., 2018; Anil et al., 2020), whose
                  "preconditioners are also whole-matrix operators".
The paper prints neither the formulas nor any hyper-parameter of its Shampoo run.  What is
computed here is Algorithm 1 of Gupta et al. for order-2 tensors, restated:
    L_t = L_{t-1} + G_t G_t^T ;  R_t = R_{t-1} + G_t^T G_t ;  W_{t+1} = W_t - eta L_t^{-1/4} G_t R_t^{-1/4},
under the readings S1-S5, S7 of DESIGN.md section 4 (every place the paper is silent):
  S1  statistics  L <- beta2 L + w G G^T, R <- beta2 R + w G^T G, w = 1 (beta2 = 1, Gupta et al.: a
      running sum) or w = 1 - beta2 (beta2 < 1, the moving average of Anil et al.); L_0 = R_0 = 0.
  S2  ridge       relative to the mean eigenvalue: L~ = L + eps (tr L / m) I (Anil et al. scale the
      ridge by lambda_max; the trace is exact and needs no power iteration).  tr L = 0 (no gradient
      seen yet) -> the preconditioner is I.
  S3  root        P_L = L~^{-1/4}: the DEFINITION through the symmetric eigendecomposition,
      Q diag(lambda^{-1/4}) Q^T (numpy.linalg.eigh is the library primitive of this step).  The GPU
      reaches it with a coupled Newton iteration; that is an approximation of this definition.
  S4  update      D = P_L G P_R ; W <- W (1 - eta lambda) - eta D (decoupled decay as for Muon;
      no momentum, no grafting: neither is in Gupta et al.'s Algorithm 1).
  S7  float32 floor of the ridge (optional, eps_floor = 0 switches it off): rho = max(eps tr S / d, eps_floor ||S||_F).
      PAPER.md:182 runs Shampoo in "float32": a statistic held in float32 carries rounding noise of order 2^-23 ||S||_F,
      and a ridge below that noise leaves S~ indefinite for every rank-deficient statistic (G G^T of a tall G), where
      S~^{-1/4} does not exist in that arithmetic.  The floor is part of the method's definition here (both this file
      and the CUDA path apply the same formula), not a tolerance.
  S5  schedule    the roots are recomputed at steps t with (t - 1) % root_every == 0 (t is 1-based),
      from the statistics that already include G_t; other steps reuse the stored P_L, P_R.

Everything is numpy float64, one statement per formula.
"""
import numpy as np


def statistics_update(L, R, G, beta2=1.0):
    """S1.  Returns (L_new, R_new)."""
    L = np.asarray(L, dtype=np.float64)
    R = np.asarray(R, dtype=np.float64)
    G = np.asarray(G, dtype=np.float64)
    w = 1.0 if beta2 == 1.0 else 1.0 - beta2
    L_new = beta2 * L + w * (G @ G.T)
    R_new = beta2 * R + w * (G.T @ G)
    return L_new, R_new


def inverse_root(S, eps=1e-6, p=4, eps_floor=0.0):
    """S2 + S7 + S3: (S + rho I)^{-1/p}, rho = max(eps tr S / d, eps_floor ||S||_F), of a symmetric positive
    semi-definite S by eigendecomposition."""
    S = np.asarray(S, dtype=np.float64)
    d = S.shape[0]
    tr = float(np.trace(S))
    if tr <= 0.0:
        return np.eye(d)
    ridge = max(eps * tr / d, eps_floor * float(np.sqrt(np.sum(S * S))))
    lam, Q = np.linalg.eigh(S + ridge * np.eye(d))
    return (Q * lam ** (-1.0 / p)) @ Q.T


def precondition(G, P_L, P_R):
    """S4, first half: D = P_L G P_R."""
    return P_L @ np.asarray(G, dtype=np.float64) @ P_R


def weight_update(W, D, lr, weight_decay):
    """S4, second half: W <- W (1 - lr wd) - lr D."""
    return np.asarray(W, dtype=np.float64) * (1.0 - lr * weight_decay) - lr * np.asarray(D, dtype=np.float64)


def shampoo_step(W, G, L, R, P_L, P_R, step, lr=1e-3, weight_decay=0.0, beta2=1.0, eps=1e-6, root_every=1,
                 eps_floor=0.0):
    """One whole owner-local Shampoo step for one matrix (S1-S5).  `step` is 1-based; P_L / P_R are the stored
    roots (ignored at a refresh step, may then be None).  Returns dict(W=, L=, R=, P_L=, P_R=, D=)."""
    L_new, R_new = statistics_update(L, R, G, beta2)
    if (step - 1) % root_every == 0:
        P_L = inverse_root(L_new, eps, eps_floor=eps_floor)
        P_R = inverse_root(R_new, eps, eps_floor=eps_floor)
    D = precondition(G, P_L, P_R)
    W_new = weight_update(W, D, lr, weight_decay)
    return {"W": W_new, "L": L_new, "R": R_new, "P_L": P_L, "P_R": P_R, "D": D}
