"""Pins for the oracle's training-step plumbing (Adam with lr 1e-3 and betas
(0.9, 0.999); adaptive density control statistics): a library routine (torch.optim.Adam on the CPU), closed forms and
brute force."""
import numpy as np
import pytest


def test_adam_matches_torch_optim_adam(oracle):
    torch = pytest.importorskip("torch")
    rng = np.random.default_rng(0)
    p0 = rng.standard_normal(257)
    pt = torch.tensor(p0, dtype=torch.float64, requires_grad=True)
    opt = torch.optim.Adam([pt], lr=1e-3, betas=(0.9, 0.999), eps=1e-8)
    p, m, v = p0.copy(), np.zeros(257), np.zeros(257)
    for step in range(1, 8):
        g = rng.standard_normal(257) * 10.0 ** rng.integers(-4, 3)
        pt.grad = torch.tensor(g, dtype=torch.float64)
        opt.step()
        p, m, v = oracle.adam_step(p, g, m, v, 1e-3, 0.9, 0.999, 1e-8, step)
        assert np.allclose(p, pt.detach().numpy(), rtol=1e-13, atol=1e-15), step


def test_adam_closed_forms(oracle):
    g = np.array([3.0, -0.25, 1e-6, 0.0])
    p0 = np.array([1.0, 2.0, 3.0, 4.0])
    # first step from zero state: m^ = g, v^ = g^2  =>  p1 = p0 - lr g / (|g| + eps)
    p, m, v = oracle.adam_step(p0, g, np.zeros(4), np.zeros(4), 1e-3, 0.9, 0.999, 1e-8, 1)
    assert np.allclose(p, p0 - 1e-3 * g / (np.abs(g) + 1e-8), rtol=1e-14)
    assert np.allclose(m, 0.1 * g) and np.allclose(v, 0.001 * g * g)
    assert p[3] == 4.0                                        # zero gradient, zero state: untouched
    # a constant gradient keeps m^ = g and v^ = g^2 at every step: the same update every time
    for step in range(2, 6):
        q, m, v = oracle.adam_step(p, g, m, v, 1e-3, 0.9, 0.999, 1e-8, step)
        assert np.allclose(q - p, -1e-3 * g / (np.abs(g) + 1e-8), rtol=1e-12)
        p = q


def test_density_stats_brute_force(oracle):
    rng = np.random.default_rng(1)
    n = 100
    d = rng.standard_normal((n, 2))
    radius = rng.integers(0, 5, n).astype(np.int32)          # 0 = culled in this view
    ga0, dn0, mr0 = rng.uniform(0, 1, n), rng.integers(0, 3, n).astype(np.uint32), rng.integers(0, 4, n).astype(np.int32)
    ga, dn, mr = oracle.density_stats(d, radius, ga0, dn0, mr0)
    for i in range(n):
        if radius[i] > 0:
            assert ga[i] == pytest.approx(ga0[i] + np.hypot(d[i, 0], d[i, 1]), rel=1e-14)
            assert dn[i] == dn0[i] + 1 and mr[i] == max(mr0[i], radius[i])
        else:
            assert ga[i] == ga0[i] and dn[i] == dn0[i] and mr[i] == mr0[i]
