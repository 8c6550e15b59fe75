"""Pins of oracle.semantic_loss (Eq. 8-12) against things other than itself: closed forms, an independent
scipy evaluation of the loss value, central finite differences of that scipy value for every gradient, and invariants."""
import numpy as np
import pytest
from scipy.special import log_softmax

from oracle import legs_oracle as oracle


@pytest.fixture(scope="module", autouse=True)
def _built():
    oracle.build()


def make(P=40, dims=(8, 16, 12), seed=0, three=False):
    rng = np.random.default_rng(seed)
    dims = list(dims) if not three else [8, 10, 14, 12]
    W = [rng.normal(0, 0.7, (o, i)) for i, o in zip(dims[:-1], dims[1:])]
    b = [rng.normal(0, 0.3, o) for o in dims[1:]]
    x = rng.normal(0, 1, (P, dims[0]))
    u = rng.uniform(0, 1, P)
    m = rng.integers(0, dims[-1], P)
    return x, u, m, W, b


def scipy_loss(x, u, m, W, b, lce, lu):
    """Independent evaluation: numpy matmuls + scipy log_softmax (no code shared with the oracle)."""
    h = x
    for l, (w, bb) in enumerate(zip(W, b)):
        h = h @ w.T + bb
        if l + 1 < len(W):
            h = np.maximum(h, 0.0)
    ce = -log_softmax(h, axis=1)[np.arange(x.shape[0]), m]
    l_ce = float((ce * (1 - u)).mean())
    l_u = float(u.mean())
    return l_ce, l_u, lce * l_ce + lu * l_u


@pytest.mark.parametrize("three", [False, True])
def test_loss_value_matches_scipy(three):
    x, u, m, W, b = make(three=three)
    r = oracle.semantic_loss(x, u, m, W, b, 1.3, 0.2)
    assert np.allclose(r["loss"], scipy_loss(x, u, m, W, b, 1.3, 0.2), rtol=1e-12, atol=1e-14)


def test_closed_forms():
    # zero weights and biases: uniform distribution, CE = log K for every pixel (Eq. 9), weighted by (1 - u) (Eq. 10)
    P, K = 17, 12
    x, u, m, W, b = make(P=P)
    W0 = [np.zeros_like(w) for w in W]
    b0 = [np.zeros_like(v) for v in b]
    r = oracle.semantic_loss(x, u, m, W0, b0, 1.0, 0.5)
    assert r["loss"][0] == pytest.approx(np.log(K) * (1 - u).mean(), rel=1e-13)
    assert r["loss"][1] == pytest.approx(u.mean(), rel=1e-13)                     # Eq. 11
    assert r["loss"][2] == pytest.approx(r["loss"][0] + 0.5 * r["loss"][1], rel=1e-13)   # Eq. 12
    # dL/dR_u = (-lambda_ce CE + lambda_u) / P: here CE = log K everywhere
    assert np.allclose(r["du"], (-np.log(K) + 0.5) / P)
    # the last layer's bias gradient is sum_p coef_p (p - onehot): uniform p = 1/K
    coef = (1 - u) / P
    expect = np.array([(coef * (1.0 / K - (m == k))).sum() for k in range(K)])
    assert np.allclose(r["db"][-1], expect, atol=1e-15)
    # a saturated correct prediction has zero CE and zero logit gradient
    bs = [np.zeros_like(v) for v in b]
    bs[-1][3] = 500.0
    r = oracle.semantic_loss(x, u, np.full(P, 3), W0, bs, 1.0, 0.0)
    assert r["loss"][0] == pytest.approx(0.0, abs=1e-12) and np.abs(r["db"][-1]).max() < 1e-12


def test_invariants():
    x, u, m, W, b = make()
    r = oracle.semantic_loss(x, u, m, W, b, 1.0, 0.1)
    assert abs(r["db"][-1].sum()) < 1e-14          # softmax minus one-hot sums to zero over the codes, pixel by pixel
    # u = 1 everywhere: the CE term and every decoder / feature gradient vanish (Eq. 10), L_u = 1
    r1 = oracle.semantic_loss(x, np.ones_like(u), m, W, b, 1.0, 0.1)
    assert r1["loss"][0] == 0.0 and r1["loss"][1] == 1.0
    assert all(np.abs(g).max() == 0.0 for g in r1["dW"]) and np.abs(r1["dx"]).max() == 0.0
    # shifting the last bias by a constant changes nothing (softmax shift invariance)
    b2 = [v.copy() for v in b]
    b2[-1] += 7.5
    r2 = oracle.semantic_loss(x, u, m, W, b2, 1.0, 0.1)
    assert np.allclose(r2["loss"], r["loss"], rtol=1e-12) and np.allclose(r2["dx"], r["dx"], rtol=1e-9, atol=1e-15)
    # pixels are independent: gradient of pixel subsets adds up (after the 1/P normalisation is undone)
    half = x.shape[0] // 2
    ra = oracle.semantic_loss(x[:half], u[:half], m[:half], W, b, 1.0, 0.1)
    rb = oracle.semantic_loss(x[half:], u[half:], m[half:], W, b, 1.0, 0.1)
    P = x.shape[0]
    assert np.allclose(r["dW"][0] * P, ra["dW"][0] * half + rb["dW"][0] * (P - half), rtol=1e-10, atol=1e-14)


@pytest.mark.parametrize("three", [False, True])
def test_gradients_match_central_differences_of_the_scipy_loss(three):
    x, u, m, W, b = make(P=12, three=three, seed=3)
    lce, lu = 0.9, 0.3
    r = oracle.semantic_loss(x, u, m, W, b, lce, lu)
    f = lambda X, U, WW, BB: scipy_loss(X, U, m, WW, BB, lce, lu)[2]
    eps = 1e-6
    rng = np.random.default_rng(5)

    def fd(arr, rebuild, n=25):
        flat = arr.reshape(-1)
        out = []
        for i in rng.choice(flat.size, min(n, flat.size), replace=False):
            a1, a2 = arr.copy(), arr.copy()
            a1.reshape(-1)[i] += eps
            a2.reshape(-1)[i] -= eps
            out.append((i, (rebuild(a1) - rebuild(a2)) / (2 * eps)))
        return out

    for i, g in fd(x, lambda a: f(a, u, W, b)):
        assert r["dx"].reshape(-1)[i] == pytest.approx(g, rel=2e-5, abs=1e-9)
    for i, g in fd(u, lambda a: f(x, a, W, b)):
        assert r["du"][i] == pytest.approx(g, rel=2e-5, abs=1e-9)
    for l in range(len(W)):
        for i, g in fd(W[l], lambda a: f(x, u, W[:l] + [a] + W[l + 1:], b)):
            assert r["dW"][l].reshape(-1)[i] == pytest.approx(g, rel=2e-5, abs=1e-9)
        for i, g in fd(b[l], lambda a: f(x, u, W, b[:l] + [a] + b[l + 1:])):
            assert r["db"][l][i] == pytest.approx(g, rel=2e-5, abs=1e-9)
