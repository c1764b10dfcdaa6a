"""Regenerates the text fixtures in this directory with exact / 50-digit arithmetic.

Uses only the Python standard library (fractions, decimal): it imports neither `oracle/`
nor the CUDA package, so the fixtures are independent of both.  Nothing here comes from
the paper (it prints no worked example); each fixture is the closed
form of a definition, worked by exact arithmetic, and says so in its header.

    python tests/golden/make_golden.py
"""
import os
from decimal import Decimal, getcontext
from fractions import Fraction

HERE = os.path.dirname(os.path.abspath(__file__))
getcontext().prec = 50

A, B, C = Fraction("3.4445"), Fraction("-4.7750"), Fraction("2.0315")


def f(x):
    return A * x + B * x ** 3 + C * x ** 5


def fk(x, k):
    # exact rationals explode in size; re-round to 60 significant digits each step
    for _ in range(k):
        x = f(x)
        x = Fraction(Decimal(x.numerator) / Decimal(x.denominator))
    return x


def dec(fr, digits=18):
    d = Decimal(fr.numerator) / Decimal(fr.denominator)
    return format(d, ".%de" % digits)


def ns_scalars():
    lines = [
        "# Quintic Newton-Schulz polynomial f(x) = a x + b x^3 + c x^5 iterated k times on a scalar.",
        "# (a, b, c) = (3.4445, -4.7750, 2.0315): BASELINE.json north_star fallback coefficients",
        "# (the paper gives none; PAPER.md:37 only says NS steps are 'built from products such as XX^T').",
        "# Each singular value of X0 = U/||U||_F is mapped by f^k (SVD form of the iteration).",
        "# Computed by tests/golden/make_golden.py with 50-digit decimal arithmetic.",
        "# columns: x0  k  f^k(x0)",
    ]
    sqrt_half = Fraction(Decimal(2).sqrt() / 2)
    for x0, name in [(Fraction(1), "1"), (Fraction("0.8"), "0.8"), (Fraction("0.6"), "0.6"),
                     (Fraction("0.5"), "0.5"), (sqrt_half, "sqrt(1/2)"), (Fraction("0.1"), "0.1"),
                     (Fraction("0.01"), "0.01"), (Fraction("0.001"), "0.001")]:
        for k in (1, 2, 5):
            lines.append("%s %d %s" % (name, k, dec(fk(x0, k))))
    open(os.path.join(HERE, "ns_quintic_scalars.txt"), "w").write("\n".join(lines) + "\n")


def adamw_two_step():
    # SURVEY.md 8(c) O-3 / Loshchilov & Hutter; hyper-parameters: PAPER.md:121
    # (lr 1e-3, wd 1e-2, eps 1e-8) and BASELINE.json config 1 (betas (0.9, 0.95)).
    D = Decimal
    p, m, v = D("0.5"), D(0), D(0)
    lr, b1, b2, eps, wd = D("0.001"), D("0.9"), D("0.95"), D("1e-8"), D("0.01")
    lines = [
        "# AdamW, scalar, two steps, worked by hand in 50-digit decimal arithmetic",
        "# (tests/golden/make_golden.py).  Rule: SURVEY.md 8(c) O-3 (decoupled decay, bias correction,",
        "# eps added to sqrt(v_hat)); hyper-parameters PAPER.md:121 + BASELINE.json config 1.",
        "# p0 = 0.5, g1 = 0.25, g2 = -0.125, lr = 1e-3, betas = (0.9, 0.95), eps = 1e-8, wd = 0.01",
        "# columns: step  m  v  m_hat  v_hat  p",
    ]
    for t, g in ((1, D("0.25")), (2, D("-0.125"))):
        p = p * (1 - lr * wd)
        m = b1 * m + (1 - b1) * g
        v = b2 * v + (1 - b2) * g * g
        mh = m / (1 - b1 ** t)
        vh = v / (1 - b2 ** t)
        p = p - lr * mh / (vh.sqrt() + eps)
        lines.append("%d %s %s %s %s %s" % (t, format(m, ".20e"), format(v, ".20e"), format(mh, ".20e"),
                                             format(vh, ".20e"), format(p, ".20e")))
    open(os.path.join(HERE, "adamw_two_step.txt"), "w").write("\n".join(lines) + "\n")


def momentum_closed_form():
    # constant gradient g for k steps, M0 = 0:  M_k = (1 - mu^k) g ;  Nesterov U_k = (1 - mu^(k+1)) g
    mu = Fraction("0.95")
    lines = [
        "# EMA momentum with a constant gradient, M0 = 0 (SURVEY.md 8(c) O-2.1-2, reading M1):",
        "# M_k = (1 - mu^k) g ;  Nesterov U_k = (1 - mu) g + mu M_k = (1 - mu^(k+1)) g ; mu = 0.95.",
        "# Exact rationals (tests/golden/make_golden.py).  columns: k  M_k/g  U_k/g",
    ]
    for k in range(1, 6):
        lines.append("%d %s %s" % (k, dec(1 - mu ** k, 17), dec(1 - mu ** (k + 1), 17)))
    open(os.path.join(HERE, "momentum_constant_grad.txt"), "w").write("\n".join(lines) + "\n")


if __name__ == "__main__":
    ns_scalars()
    adamw_two_step()
    momentum_closed_form()
