"""Pins for the oracle's decode (Eq. 21-22, Table 3; Eq. 3 at :76-81; relevancy :360 read as a
plain cosine, C-21): library matmul, softmax invariants, the one-hot special case and the Gram shortcut."""
import numpy as np
import pytest

from paper_2311_18482_b200 import inputs


def as_f(di):
    f = inputs.bf16_bits_to_f32
    return f(di.feat), [f(w) for w in di.weights], di.biases, f(di.codebook), f(di.queries)


@pytest.mark.parametrize("hidden,K", [((64,), 128), ((128, 256), 128), ((64,), 32)])
def test_decode_against_library_matmul(oracle, hidden, K):
    di = inputs.decode_inputs(P=300, hidden=hidden, n_codes=K, bias_sigma=0.1)
    x, Ws, bs, cb, q = as_f(di)
    r = oracle.decode(x, Ws, bs, cb, di.d_clip, q)
    h = x.astype(np.float64)
    for l, (W, b) in enumerate(zip(Ws, bs)):
        h = h @ W.astype(np.float64).T + b
        if l + 1 < len(Ws):
            h = np.maximum(h, 0)
    import scipy.special as sp
    probs = sp.softmax(h, axis=1)
    assert np.allclose(r["probs"], probs, atol=1e-14)
    assert np.allclose(r["probs"].sum(1), 1.0, atol=1e-14)          # a distribution
    dec = probs @ cb.astype(np.float64)
    assert np.allclose(r["decoded"], dec, atol=1e-14)                # Eq. 22
    fc = dec[:, :512]
    ref = (fc @ q.astype(np.float64).T) / np.linalg.norm(fc, axis=1, keepdims=True) / np.linalg.norm(q.astype(np.float64), axis=1)
    assert np.allclose(r["rel"], ref, atol=1e-13)


def test_one_hot_distribution_returns_codebook_row(oracle):
    # Eq. 3 as a special case of Eq. 22: saturated logits => decoded == codebook row m exactly
    di = inputs.decode_inputs(P=64, hidden=(64,), n_codes=128)
    x, Ws, bs, cb, q = as_f(di)
    Ws[-1] = Ws[-1] * 4000.0
    r = oracle.decode(x, Ws, bs, cb, di.d_clip, q)
    m = r["probs"].argmax(1)
    sat = r["probs"].max(1) > 1 - 1e-12
    assert sat.sum() > 32
    assert np.allclose(r["decoded"][sat], cb[m[sat]].astype(np.float64), atol=1e-10)
    # relevancy is 1 when the query equals the normalised CLIP part of the decoded row
    q2 = cb[m[sat]][:, :512].astype(np.float64)
    r2 = oracle.decode(x[sat], Ws, bs, cb, di.d_clip, q2, want=("rel",))
    assert np.allclose(np.diag(r2["rel"]), 1.0, atol=1e-9)


def test_gram_shortcut_equals_direct_norm(oracle):
    # |F_clip|^2 = p^T (S_clip S_clip^T) p ;  F_clip . q = p^T (S_clip q)
    di = inputs.decode_inputs(P=200, hidden=(64,), n_codes=128)
    x, Ws, bs, cb, q = as_f(di)
    r = oracle.decode(x, Ws, bs, cb, di.d_clip, q)
    Sc = cb[:, :512].astype(np.float64)
    gram = Sc @ Sc.T
    p = r["probs"]
    n2 = np.einsum("pk,kl,pl->p", p, gram, p)
    assert np.allclose(n2, (r["decoded"][:, :512] ** 2).sum(1), rtol=1e-12)
    rel = (p @ (Sc @ q.astype(np.float64).T)) / np.sqrt(n2)[:, None] / np.linalg.norm(q.astype(np.float64), axis=1)
    assert np.allclose(rel, r["rel"], atol=1e-12)


def test_bf16_round_trip_helpers():
    a = np.array([1.0, 1.00390625, 1.005859375, -2.5, 3.1415927, 1e-20, 65504.0], np.float32)
    b = inputs.bf16_bits_to_f32(inputs.to_bf16_bits(a))
    import torch
    ref = torch.from_numpy(a).to(torch.bfloat16).to(torch.float32).numpy()  # library rounding (RNE)
    assert np.array_equal(b, ref)


def test_lerf_relevancy_against_scipy_softmax_and_special_cases(oracle):
    # PAPER.md:360 cites LERF [18] for the relevancy; the formula is not in the paper ("parity unpinned" by the paper,
    # DESIGN.md C-21b). What the mathematics fixes: the score is the first entry of a 2-way softmax, minimised over negatives.
    import scipy.special as sp
    rng = np.random.default_rng(3)
    P, Q, n_pos, tau = 200, 7, 3, 10.0
    c = rng.uniform(-1, 1, (P, Q))
    r = oracle.relevancy_lerf(c, n_pos, tau)
    ref = np.full((P, n_pos), 2.0)
    for j in range(n_pos):
        for i in range(n_pos, Q):
            pair = sp.softmax(tau * np.stack([c[:, j], c[:, i]], 1), axis=1)[:, 0]
            ref[:, j] = np.minimum(ref[:, j], pair)
    assert np.allclose(r, ref, rtol=1e-13)
    # the binding negative is the one with the LARGEST cosine; equal cosines give exactly 1/2; tau = 0 gives 1/2 everywhere
    worst = c[:, n_pos:].max(1)
    assert np.allclose(r, 1.0 / (1.0 + np.exp(tau * (worst[:, None] - c[:, :n_pos]))), rtol=1e-13)
    c2 = c.copy()
    c2[:, n_pos:] = c2[:, [0]]
    assert np.array_equal(oracle.relevancy_lerf(c2, n_pos, tau)[:, 0], np.full(P, 0.5))
    assert np.array_equal(oracle.relevancy_lerf(c, n_pos, 0.0), np.full((P, n_pos), 0.5))
    # monotone: raising a query's cosine raises its score, raising a negative's cannot raise any score
    c3 = c.copy(); c3[:, 0] += 0.1
    assert (oracle.relevancy_lerf(c3, n_pos, tau)[:, 0] > r[:, 0]).all()
    c4 = c.copy(); c4[:, n_pos] += 0.1
    assert (oracle.relevancy_lerf(c4, n_pos, tau) <= r).all()


def test_relevancy_of_a_given_map(oracle):
    # PAPER.md:360 / C-21 for a caller-supplied map F (SURVEY.md 8(b) input_is_probs = 0). Pins: numpy/scipy cosine; the pinned
    # oracle.decode's rel when F is its decoded map; scale invariance in F and in q; orthogonal and parallel special cases;
    # columns beyond d_clip are ignored; a zero row gives 0
    from scipy.spatial.distance import cdist
    rng = np.random.default_rng(5)
    P, d, dc, Q = 37, 96, 40, 5
    F = rng.standard_normal((P, d))
    q = rng.standard_normal((Q, dc)) * rng.uniform(0.5, 3.0, (Q, 1))
    r = oracle.relevancy_map(F, dc, q)
    assert np.allclose(r, 1.0 - cdist(F[:, :dc], q, metric="cosine"), atol=1e-13)
    assert np.allclose(oracle.relevancy_map(F * rng.uniform(0.1, 9.0, (P, 1)), dc, q * 7.0), r, atol=1e-13)
    F2 = F.copy()
    F2[:, dc:] = 1e6
    assert np.array_equal(oracle.relevancy_map(F2, dc, q), r)
    e = np.zeros((3, d))
    e[0, 0], e[1, 1], e[2, 0] = 2.0, 3.0, -4.0
    qe = np.zeros((1, dc))
    qe[0, 0] = 5.0
    assert np.array_equal(oracle.relevancy_map(e, dc, qe)[:, 0], [1.0, 0.0, -1.0])
    assert np.array_equal(oracle.relevancy_map(np.zeros((2, d)), dc, q), np.zeros((2, Q)))
    di = inputs.decode_inputs(P=64, seed=2)
    f = inputs.bf16_bits_to_f32
    full = oracle.decode(f(di.feat), [f(w) for w in di.weights], di.biases, f(di.codebook), di.d_clip, f(di.queries))
    assert np.allclose(oracle.relevancy_map(full["decoded"], di.d_clip, f(di.queries)), full["rel"], atol=1e-13)
