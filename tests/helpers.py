"""Comparison helpers for the tests (numpy only; no method arithmetic)."""
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
