"""Pins for the oracle's adaptive spatial smoothing (Eq. 13-14, Table 4):
an independent numpy evaluation of the loss with the stop-gradient copies as separate arguments, closed forms, and
central finite differences of that numpy loss for every gradient."""
import numpy as np
import pytest


def mlp_numpy(p, Ws, bs):
    h = p
    for l, (W, b) in enumerate(zip(Ws, bs)):
        h = h @ W.T + b
        if l + 1 < len(Ws):
            h = np.maximum(h, 0.0)
    return h


def loss_numpy(p, Ws, bs, s, u, w_s, s_sg=None, smlp_sg=None):
    """Eq. 14 with the stop-gradient copies passed separately: term 1 uses (MLP(W), s_sg), term 2 uses (smlp_sg, s)."""
    smlp = mlp_numpy(p, Ws, bs)
    s_sg = s if s_sg is None else s_sg
    smlp_sg = smlp if smlp_sg is None else smlp_sg
    t1 = np.linalg.norm(smlp - s_sg, axis=1)
    t2 = np.maximum(u, w_s) * np.linalg.norm(smlp_sg - s, axis=1)
    return float((t1 + t2).mean())


def make(n=40, dims=(3, 16, 16, 16, 8), seed=0):
    rng = np.random.default_rng(seed)
    p = rng.standard_normal((n, dims[0]))
    s = rng.standard_normal((n, dims[-1]))
    u = rng.uniform(0, 1, n)
    u[::3] = 0.02                                    # below w_s: the floor is active
    Ws = [rng.uniform(-1, 1, (o, i)) * np.sqrt(6.0 / i) for i, o in zip(dims[:-1], dims[1:])]
    bs = [0.1 * rng.standard_normal(o) for o in dims[1:]]
    return p, s, u, Ws, bs


def test_loss_and_smoothed_features_against_numpy(oracle):
    p, s, u, Ws, bs = make()
    o = oracle.smooth_loss(p, s, u, Ws, bs, 0.1)
    assert np.allclose(o["s_mlp"], mlp_numpy(p, Ws, bs), atol=1e-12)      # Eq. 13, Table 4 shape (narrower hidden layers)
    assert o["loss"] == pytest.approx(loss_numpy(p, Ws, bs, s, u, 0.1), rel=1e-13)


def test_closed_forms(oracle):
    p, s, u, Ws, bs = make()
    Wz = [np.zeros_like(w) for w in Ws]
    o = oracle.smooth_loss(p, s, u, Wz, bs, 0.1)
    # zero weights: s_MLP = b_last for every Gaussian  =>  L = mean (1 + max(u, w_s)) |b_last - s|
    want = ((1 + np.maximum(u, 0.1)) * np.linalg.norm(bs[-1] - s, axis=1)).mean()
    assert o["loss"] == pytest.approx(want, rel=1e-13)
    # ds = -max(u, w_s) (s_MLP - s) / (n |s_MLP - s|): unit direction scaled by the adaptive weight (floor w_s = 0.1 active)
    e = bs[-1] - s
    assert np.allclose(o["ds"], -np.maximum(u, 0.1)[:, None] * e / np.linalg.norm(e, axis=1, keepdims=True) / len(u), atol=1e-15)
    assert np.allclose(np.linalg.norm(o["ds"], axis=1) * len(u), np.maximum(u, 0.1), atol=1e-13)
    # the last bias gradient is the mean unit direction; hidden-layer weight gradients vanish with zero weights downstream
    assert np.allclose(o["db"][-1], (e / np.linalg.norm(e, axis=1, keepdims=True)).mean(0), atol=1e-14)
    assert all(np.abs(g).max() == 0 for g in o["dW"][:-1])
    # s exactly equal to s_MLP (zero weights, s = b_last): the loss is 0 and every gradient is 0 (sub-gradient at the kink)
    o0 = oracle.smooth_loss(p, np.tile(bs[-1], (len(u), 1)), u, Wz, bs, 0.1)
    assert o0["loss"] == 0.0 and np.abs(o0["ds"]).max() == 0 and np.abs(o0["db"][-1]).max() == 0


@pytest.mark.parametrize("dims", [(3, 16, 16, 16, 8), (3, 12, 8)])
def test_gradients_against_central_differences(oracle, dims):
    p, s, u, Ws, bs = make(n=25, dims=dims, seed=1)
    o = oracle.smooth_loss(p, s, u, Ws, bs, 0.1)
    smlp0 = mlp_numpy(p, Ws, bs)
    h = 1e-6
    rng = np.random.default_rng(2)
    # weights and biases: only the first term moves (the second sees the stop-gradient copy of s_MLP)
    for l in range(len(Ws)):
        for _ in range(6):
            i, j = rng.integers(0, Ws[l].shape[0]), rng.integers(0, Ws[l].shape[1])
            Wp = [w.copy() for w in Ws]; Wm = [w.copy() for w in Ws]
            Wp[l][i, j] += h; Wm[l][i, j] -= h
            fd = (loss_numpy(p, Wp, bs, s, u, 0.1, smlp_sg=smlp0) - loss_numpy(p, Wm, bs, s, u, 0.1, smlp_sg=smlp0)) / (2 * h)
            assert o["dW"][l][i, j] == pytest.approx(fd, rel=2e-5, abs=1e-9), (l, i, j)
        i = rng.integers(0, bs[l].shape[0])
        bp = [b.copy() for b in bs]; bm = [b.copy() for b in bs]
        bp[l][i] += h; bm[l][i] -= h
        fd = (loss_numpy(p, Ws, bp, s, u, 0.1, smlp_sg=smlp0) - loss_numpy(p, Ws, bm, s, u, 0.1, smlp_sg=smlp0)) / (2 * h)
        assert o["db"][l][i] == pytest.approx(fd, rel=2e-5, abs=1e-9), (l, i)
    # compact features: only the second term moves (the first sees the stop-gradient copy of s)
    for _ in range(10):
        i, f = rng.integers(0, s.shape[0]), rng.integers(0, s.shape[1])
        sp, sm = s.copy(), s.copy()
        sp[i, f] += h; sm[i, f] -= h
        fd = (loss_numpy(p, Ws, bs, sp, u, 0.1, s_sg=s) - loss_numpy(p, Ws, bs, sm, u, 0.1, s_sg=s)) / (2 * h)
        assert o["ds"][i, f] == pytest.approx(fd, rel=2e-5, abs=1e-10), (i, f)


def test_gradients_add_over_subsets(oracle):
    # n L is a sum over Gaussians: the weight gradients of two halves add up to those of the whole (scaled by the sizes)
    p, s, u, Ws, bs = make(n=30, seed=3)
    a = oracle.smooth_loss(p[:10], s[:10], u[:10], Ws, bs, 0.1)
    b = oracle.smooth_loss(p[10:], s[10:], u[10:], Ws, bs, 0.1)
    c = oracle.smooth_loss(p, s, u, Ws, bs, 0.1)
    for l in range(len(Ws)):
        assert np.allclose(30 * c["dW"][l], 10 * a["dW"][l] + 20 * b["dW"][l], atol=1e-12)
    assert 30 * c["loss"] == pytest.approx(10 * a["loss"] + 20 * b["loss"], rel=1e-13)
