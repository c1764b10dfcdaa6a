"""Pins for oracle/adamw.py: hand-computed two-step example (50-digit decimal fixture),
first-step sign property, zero-gradient special case, torch.optim.AdamW in fp64 (library)."""
import os

import numpy as np
import pytest

from oracle import adamw


def test_two_step_hand_example(golden_dir):
    rows = [l.split() for l in open(os.path.join(golden_dir, "adamw_two_step.txt")) if not l.startswith("#")]
    p, m, v = np.array([0.5]), np.zeros(1), np.zeros(1)
    for (t, gm, gv, _, _, gp), g in zip(rows, (0.25, -0.125)):
        p, m, v = adamw.adamw_step(p, np.array([g]), m, v, int(t), lr=1e-3, beta1=0.9, beta2=0.95,
                                   eps=1e-8, weight_decay=0.01)
        assert m[0] == pytest.approx(float(gm), rel=1e-14)
        assert v[0] == pytest.approx(float(gv), rel=1e-14)
        assert p[0] == pytest.approx(float(gp), rel=1e-14)


def test_first_step_is_a_sign_step():
    rng = np.random.default_rng(3)
    p0 = rng.standard_normal(100)
    g = rng.standard_normal(100) * 1e-3
    p, m, v = adamw.adamw_step(p0, g, np.zeros(100), np.zeros(100), 1, lr=1e-3, weight_decay=0.01)
    expect = p0 * (1 - 1e-5) - 1e-3 * np.sign(g)
    assert np.abs(p - expect).max() < 1e-3 * 1e-8 / np.abs(g).min() * 1.01


def test_zero_gradient_only_decays():
    p0 = np.array([1.0, -2.0])
    p, m, v = adamw.adamw_step(p0, np.zeros(2), np.zeros(2), np.zeros(2), 1, lr=1e-3, weight_decay=0.01)
    np.testing.assert_allclose(p, p0 * (1 - 1e-5), rtol=1e-15)
    assert np.all(m == 0) and np.all(v == 0)


def test_against_torch_adamw_fp64():
    torch = pytest.importorskip("torch")
    g = torch.Generator().manual_seed(5)
    p0 = 0.02 * torch.randn(257, generator=g, dtype=torch.float64)
    par = torch.nn.Parameter(p0.clone())
    opt = torch.optim.AdamW([par], lr=1e-3, betas=(0.9, 0.95), eps=1e-8, weight_decay=0.01)
    p, m, v = p0.numpy().copy(), np.zeros(257), np.zeros(257)
    for t in range(1, 6):
        grad = 1e-3 * torch.randn(257, generator=g, dtype=torch.float64)
        par.grad = grad.clone()
        opt.step()
        p, m, v = adamw.adamw_step(p, grad.numpy(), m, v, t, lr=1e-3, beta1=0.9, beta2=0.95, eps=1e-8,
                                   weight_decay=0.01)
        np.testing.assert_allclose(par.detach().numpy(), p, rtol=1e-12, atol=1e-15)
        np.testing.assert_allclose(opt.state[par]["exp_avg"].numpy(), m, rtol=1e-12, atol=1e-18)
        np.testing.assert_allclose(opt.state[par]["exp_avg_sq"].numpy(), v, rtol=1e-12, atol=1e-20)
