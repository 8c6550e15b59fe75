"""Pins for the oracle's quantisation search and codebook losses (Eq. 3-7 and
:310-329 Eq. 16-20): library routines (numpy matmul / argmax, scipy softmax), closed forms and invariants."""
import numpy as np
import pytest
from scipy.special import softmax


def _data(P=300, N=16, d=40, d_clip=24, seed=0):
    rng = np.random.default_rng(seed)
    return rng.standard_normal((P, d)), rng.standard_normal((N, d)), d_clip


def _scores_numpy(F, S, d_clip, lam):
    n = lambda a: a / np.linalg.norm(a, axis=1, keepdims=True)
    return n(F[:, :d_clip]) @ n(S[:, :d_clip]).T + lam * (n(F[:, d_clip:]) @ n(S[:, d_clip:]).T)


def test_scores_argmax_and_losses_against_numpy(oracle):
    F, S, dc = _data()
    lam = 0.5
    o = oracle.quantize(F, S, dc, lam, 1.0, 0.5, want_scores=True)
    D = _scores_numpy(F, S, dc, lam)                       # Eq. 4 with library matmuls
    assert np.allclose(o["scores"], D, atol=1e-12)
    m = D.argmax(1)
    assert np.array_equal(o["index"], m)                   # Eq. 16
    r = np.bincount(m, minlength=S.shape[0]) / F.shape[0]  # Eq. 17
    p = softmax(D, axis=1).mean(0)                         # Eq. 18-19
    assert np.allclose(o["r"], r, atol=1e-15) and np.allclose(o["p"], p, atol=1e-13)
    assert o["loss"][1] == pytest.approx(float((r * p).sum()), rel=1e-12)          # Eq. 20
    n = lambda a: a / np.linalg.norm(a, axis=1, keepdims=True)
    cc = (n(F[:, :dc]) * n(S[m][:, :dc])).sum(1)
    cd = (n(F[:, dc:]) * n(S[m][:, dc:])).sum(1)
    lcos = ((1 - cc) + lam * (1 - cd)).mean()                                       # Eq. 5 on the selected codes
    assert o["loss"][0] == pytest.approx(lcos, rel=1e-12)
    assert o["loss"][2] == pytest.approx(1.0 * lcos + 0.5 * float((r * p).sum()), rel=1e-12)   # Eq. 7
    srt = np.sort(D, axis=1)
    assert np.allclose(o["gap"], srt[:, -1] - srt[:, -2], atol=1e-12)


def test_features_equal_to_codes_are_quantised_exactly(oracle):
    # Eq. 3: F = c * f_m (any positive scale) selects m, with cosine 1 in both parts: L_cos = 0; an even assignment gives
    # r_i = 1/N, hence L_lb = sum_i p_i / N = 1/N whatever p is
    _, S, dc = _data(N=8)
    rng = np.random.default_rng(1)
    m = np.repeat(np.arange(8), 5)
    F = S[m] * rng.uniform(0.5, 3.0, (40, 1))
    o = oracle.quantize(F, S, dc, 0.5)
    assert np.array_equal(o["index"], m)
    assert abs(o["loss"][0]) < 1e-14
    assert np.allclose(o["r"], 1 / 8) and o["loss"][1] == pytest.approx(1 / 8, rel=1e-13)
    assert o["p"].sum() == pytest.approx(1.0, rel=1e-13)


def test_ties_go_to_the_lowest_index_and_collapse_loss(oracle):
    F, S, dc = _data(P=50, N=6)
    S[4] = S[1]                                   # identical codes: equal scores, the lower index wins (reading C-28)
    o = oracle.quantize(F, S, dc, 0.5)
    assert not (o["index"] == 4).any()
    tied = o["index"] == 1
    assert tied.any() and (o["gap"][tied] == 0).all()
    # collapse: every feature is code 0 => r = e_0 and L_lb = p_0
    F0 = np.tile(S[0], (20, 1))
    o0 = oracle.quantize(F0, S, dc, 0.5)
    assert (o0["index"] == 0).all() and o0["loss"][1] == pytest.approx(o0["p"][0], rel=1e-14)


def test_scale_invariance_and_lambda_dino(oracle):
    F, S, dc = _data(seed=3)
    a = oracle.quantize(F, S, dc, 0.5, want_scores=True)
    b = oracle.quantize(F * 7.5, S * 0.1, dc, 0.5, want_scores=True)   # cosines ignore the scale of either side
    assert np.allclose(a["scores"], b["scores"], atol=1e-12) and np.array_equal(a["index"], b["index"])
    c = oracle.quantize(F, S, dc, 0.0, want_scores=True)              # lambda_DINO = 0: the DINO part is ignored
    F2 = F.copy(); F2[:, dc:] = np.random.default_rng(9).standard_normal(F2[:, dc:].shape)
    d = oracle.quantize(F2, S, dc, 0.0, want_scores=True)
    assert np.allclose(c["scores"], d["scores"], atol=1e-12)
    assert (np.abs(a["scores"]) <= 1.5 + 1e-12).all()                  # |cos| <= 1 in both parts
