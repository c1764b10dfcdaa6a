"""Comparison helpers for the tests (numpy only).  No method arithmetic, with one labelled exception at the end: a
model of WHERE the bf16 mode stores bf16, used to explain its error on ill-conditioned inputs."""
import numpy as np


def rel_fro(x, y):
    """||x - y||_F / ||y||_F with y the oracle (SURVEY.md 8(c) "Tolerances")."""
    x = np.asarray(x, dtype=np.float64)
    y = np.asarray(y, dtype=np.float64)
    den = np.sqrt(np.sum(y * y))
    num = np.sqrt(np.sum((x - y) ** 2))
    if den == 0.0:
        return 0.0 if num == 0.0 else np.inf
    return num / den


def bf16_rne(x):
    """Round float64/float32 values to the nearest bfloat16 (ties to even); returns float32
    holding exactly representable bf16 values.  Goes through float32 first, like storage does."""
    f = np.ascontiguousarray(np.asarray(x, dtype=np.float32))
    u = f.view(np.uint32).astype(np.uint64)
    lsb = (u >> 16) & 1
    r = ((u + 0x7FFF + lsb) >> 16) << 16
    out = r.astype(np.uint32).view(np.float32)
    nan = np.isnan(f)
    if nan.any():
        out = out.copy()
        out[nan] = np.nan
    return out.reshape(np.shape(x))


def bf16_bits(x):
    """bfloat16 bit patterns (uint16) of values already representable in bf16."""
    f = np.ascontiguousarray(np.asarray(x, dtype=np.float32))
    return (f.view(np.uint32) >> 16).astype(np.uint16).reshape(np.shape(x))


def bf16_ulp_distance(a, b):
    """Distance in bf16 ulps between two arrays of bf16-representable values (monotone integer map)."""
    def key(x):
        u = bf16_bits(x).astype(np.int32)
        return np.where(u & 0x8000, 0x8000 - u, u)
    return np.abs(key(a) - key(b))


def ns_bf16_storage_model(U, steps, coeffs, eps):
    """NOT the oracle and not a definition of anything: the north_star's iteration evaluated in fp64 with a rounding to
    bf16 at the places where the bf16 mode keeps bf16 (the cast X~ = bf16(U); A, P and every X_k as stored operands of
    the next product; the normalisation folded into the first iteration as include/mfsdp.h describes it).  It separates
    "what storing bf16 costs on this input" (model vs oracle) from "what else the kernels do differently" (GPU vs
    model: fp32 accumulation order).  DESIGN.md section 4, tolerance T-ill."""
    a, b, c = coeffs
    U = np.asarray(U, dtype=np.float64)
    tall = U.shape[0] > U.shape[1]
    X = bf16_rne(U.T if tall else U).astype(np.float64)
    inv = 1.0 / max(np.sqrt(np.sum(U * U)), eps)
    eye = np.eye(X.shape[0])
    for k in range(steps):
        s2, s1 = (inv * inv, inv) if k == 0 else (1.0, 1.0)
        A = bf16_rne((X @ X.T) * s2).astype(np.float64)
        P = bf16_rne(a * eye + b * A + c * (A @ A)).astype(np.float64)
        X = bf16_rne((P @ X) * s1).astype(np.float64)
    return X.T if tall else X
