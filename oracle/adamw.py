"""fp64 oracle of AdamW on packed non-matrix tails (TEST INFRASTRUCTURE -- see oracle/__init__.py).

PAPER.md:45  "The non-2D tensors in the same FSDP unit are packed into a tail role and
              assigned whole to a tail owner, where they remain on the AdamW path."
PAPER.md:47  "Tail owners apply AdamW to their packed non-matrix tensors."
PAPER.md:121 "AdamW uses ln 10^-3 [garbled: lr 1e-3], weight decay 10^-2, betas (0.9, 0.999),
              eps 10^-8"; BASELINE.json config 1 binds betas = (0.9, 0.95), eps = 1e-8.
The update rule itself is the one of Loshchilov & Hutter, reading A1 of
SURVEY.md 8(c): decoupled decay, bias correction on, eps outside the square root and
added after bias correction, no amsgrad.  SURVEY.md 8(c) O-3, one statement per formula.
"""
import numpy as np


def adamw_step(p, g, m, v, step, lr=1e-3, beta1=0.9, beta2=0.95, eps=1e-8, weight_decay=0.01):
    """One AdamW step, element-wise, float64.  `step` is 1-based.  Returns (p, m, v)."""
    p = np.asarray(p, dtype=np.float64)
    g = np.asarray(g, dtype=np.float64)
    m = np.asarray(m, dtype=np.float64)
    v = np.asarray(v, dtype=np.float64)
    p = p * (1.0 - lr * weight_decay)
    m = beta1 * m + (1.0 - beta1) * g
    v = beta2 * v + (1.0 - beta2) * g * g
    m_hat = m / (1.0 - beta1 ** step)
    v_hat = v / (1.0 - beta2 ** step)
    p = p - lr * m_hat / (np.sqrt(v_hat) + eps)
    return p, m, v
