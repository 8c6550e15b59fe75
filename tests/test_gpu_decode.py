"""GPU parity of the tcgen05 decode (legs_decode_semantics, legs_relevancy) against the fp64 oracle.
Tolerances: BASELINE.json north_star — 2e-2 abs on probabilities, cosine >= 0.999 on decoded rows; relevancy 2e-2 abs
(G-5: it is a cosine of the same decoded rows)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from paper_2311_18482_b200 import inputs  # noqa: E402


@pytest.fixture(scope="module")
def legs():
    from paper_2311_18482_b200 import binding
    assert torch.cuda.is_available()
    binding.lib()
    return binding


@pytest.fixture(scope="module")
def ctx(legs):
    return legs.Context(0)


def bf16_tensor(bits):
    return torch.from_numpy(bits.view(np.int16)).cuda().view(torch.bfloat16)


def run_decode(legs, ctx, di, want_probs=True, want_decoded=True):
    P, K, d = di.feat.shape[0], di.dims[-1], di.codebook.shape[1]
    feat, cb = bf16_tensor(di.feat), bf16_tensor(di.codebook)
    ws_ = [bf16_tensor(w) for w in di.weights]
    bs_ = [torch.from_numpy(b).cuda() for b in di.biases]
    dec = legs.make_decoder(ws_, bs_)
    ws = torch.empty(legs.legs_decode_workspace_bytes(dec, d), dtype=torch.uint8, device="cuda")
    probs = torch.zeros((P, K), dtype=torch.bfloat16, device="cuda") if want_probs else None
    decoded = torch.zeros((P, d), dtype=torch.bfloat16, device="cuda") if want_decoded else None
    legs.legs_decode_semantics(ctx, feat, dec, cb, probs, decoded, ws)
    torch.cuda.synchronize()
    return probs, decoded, cb


def oracle_decode(oracle, di):
    f = inputs.bf16_bits_to_f32
    return oracle.decode(f(di.feat), [f(w) for w in di.weights], di.biases, f(di.codebook), di.d_clip, f(di.queries))


CASES = {
    "configs3_shape": dict(P=4000 + 77, in_dim=8, hidden=(64,), n_codes=128, bias_sigma=0.0),
    "table3_shape": dict(P=1500 + 5, in_dim=8, hidden=(128, 256), n_codes=128, bias_sigma=0.1),
    "k64_in16": dict(P=900, in_dim=16, hidden=(64,), n_codes=64, bias_sigma=0.1),
    "k32": dict(P=333, in_dim=8, hidden=(32,), n_codes=32, bias_sigma=0.05),
    "one_tile_ragged": dict(P=17, in_dim=8, hidden=(64,), n_codes=128, bias_sigma=0.0),
}


@pytest.mark.parametrize("name", list(CASES.keys()))
def test_decode_matches_oracle(legs, ctx, oracle, name):
    di = inputs.decode_inputs(seed=1, **CASES[name])
    probs, decoded, cb = run_decode(legs, ctx, di)
    ref = oracle_decode(oracle, di)
    p = probs.float().cpu().numpy().astype(np.float64)
    assert np.abs(p - ref["probs"]).max() <= 2e-2
    assert np.abs(p.sum(1) - 1).max() <= 2e-2
    dec = decoded.float().cpu().numpy().astype(np.float64)
    cos = (dec * ref["decoded"]).sum(1) / (np.linalg.norm(dec, axis=1) * np.linalg.norm(ref["decoded"], axis=1))
    assert cos.min() >= 0.999
    assert np.abs(dec - ref["decoded"]).max() <= 2e-2
    # relevancy from the GPU probabilities
    q = bf16_tensor(di.queries)
    rel = torch.zeros((p.shape[0], di.queries.shape[0]), dtype=torch.float32, device="cuda")
    ws = torch.empty(legs.legs_relevancy_workspace_bytes(di.dims[-1], di.queries.shape[0]), dtype=torch.uint8, device="cuda")
    legs.legs_relevancy(ctx, probs, cb, di.d_clip, q, rel, ws)
    torch.cuda.synchronize()
    assert np.abs(rel.cpu().numpy() - ref["rel"]).max() <= 2e-2


@pytest.mark.parametrize("name,kw", [
    ("configs3_shape", dict(P=148 * 128 * 4 + 333, in_dim=8, hidden=(64,), n_codes=128, bias_sigma=0.0)),
    ("configs3_full_size", dict(P=1920 * 1080, in_dim=8, hidden=(64,), n_codes=128, bias_sigma=0.0)),   # BASELINE configs[3]
    ("table3_shape", dict(P=148 * 128 * 3 + 64, in_dim=8, hidden=(128, 256), n_codes=128, bias_sigma=0.1)),
    ("d832_k64", dict(P=148 * 128 * 3 + 1, in_dim=16, hidden=(64,), n_codes=64, bias_sigma=0.1, d=832, d_clip=512)),
])
def test_decode_persistent_pipeline_sampled_rows(legs, ctx, oracle, name, kw):
    """Several 128-row tiles per CTA (the persistent loop: double-buffered probabilities, next tile's MLP slotted
    into this tile's decode, alternating store slabs). The oracle is evaluated on sampled rows, tile heads and tails
    and the ragged last tile included; the decode is row-wise independent."""
    di = inputs.decode_inputs(seed=1, **kw)
    probs, decoded, _ = run_decode(legs, ctx, di)
    P = di.feat.shape[0]
    rng = np.random.default_rng(7)
    rows = np.unique(np.concatenate([rng.integers(0, P, 3000), np.arange(0, 300), np.arange(P - 300, P),
                                     np.arange(148 * 128 - 130, 148 * 128 + 130)]))
    f = inputs.bf16_bits_to_f32
    ref = oracle.decode(f(di.feat[rows]), [f(w) for w in di.weights], di.biases, f(di.codebook), di.d_clip, f(di.queries))
    idx = torch.from_numpy(rows).cuda()
    p = probs[idx].float().cpu().numpy().astype(np.float64)
    assert np.abs(p - ref["probs"]).max() <= 2e-2
    dec = decoded[idx].float().cpu().numpy().astype(np.float64)
    cos = (dec * ref["decoded"]).sum(1) / (np.linalg.norm(dec, axis=1) * np.linalg.norm(ref["decoded"], axis=1))
    assert cos.min() >= 0.999
    assert np.abs(dec - ref["decoded"]).max() <= 2e-2
    # relevancy over the same rows (persistent kernel: TMA ring of probability tiles, two accumulator buffers)
    K, Q = di.dims[-1], di.queries.shape[0]
    rel = torch.full((P, Q), float("nan"), dtype=torch.float32, device="cuda")
    ws = torch.empty(legs.legs_relevancy_workspace_bytes(K, Q), dtype=torch.uint8, device="cuda")
    legs.legs_relevancy(ctx, probs, bf16_tensor(di.codebook), di.d_clip, bf16_tensor(di.queries), rel, ws)
    torch.cuda.synchronize()
    assert not torch.isnan(rel).any().item()
    assert np.abs(rel[idx].cpu().numpy() - ref["rel"]).max() <= 2e-2
    # every row was written: probabilities sum to one everywhere, no decoded row is left at its zero fill
    assert (probs.float().sum(1) - 1).abs().max().item() <= 2e-2
    assert (decoded.float().abs().sum(1) > 0).all().item()


def test_decode_optional_outputs(legs, ctx):
    di = inputs.decode_inputs(seed=1, **CASES["configs3_shape"])
    probs, decoded, _ = run_decode(legs, ctx, di)
    p_only, none_dec, _ = run_decode(legs, ctx, di, want_decoded=False)
    none_p, d_only, _ = run_decode(legs, ctx, di, want_probs=False)
    assert none_dec is None and none_p is None
    assert torch.equal(p_only.view(torch.int16), probs.view(torch.int16))
    assert torch.equal(d_only.view(torch.int16), decoded.view(torch.int16))


def test_decode_saturated_logits_return_codebook_rows(legs, ctx):
    # Eq. 3 as a special case of Eq. 22: one-hot probabilities reproduce codebook row m exactly
    di = inputs.decode_inputs(seed=1, P=256, hidden=(64,), n_codes=128)
    w_last = inputs.bf16_bits_to_f32(di.weights[-1]) * 16384.0
    di.weights[-1] = inputs.to_bf16_bits(w_last)
    probs, decoded, cb = run_decode(legs, ctx, di)
    p = probs.float().cpu().numpy()
    sat = (p.max(1) == 1.0) & ((p > 0).sum(1) == 1)   # exactly one-hot in bf16
    assert sat.sum() > 100
    m = p.argmax(1)
    assert torch.equal(decoded[torch.from_numpy(sat).cuda()].view(torch.int16),
                       cb[torch.from_numpy(m[sat]).cuda()].view(torch.int16))


def test_prepare_then_packed_equals_one_call(legs, ctx):
    """legs_decode_prepare + legs_decode_semantics_packed (and the relevancy pair) give bit-identical outputs to the
    one-call forms: the packing is the same launch, only hoisted out of the per-frame path."""
    di = inputs.decode_inputs(P=1000, seed=1)
    bf = lambda bits: torch.from_numpy(bits.view(np.int16)).cuda().view(torch.bfloat16)
    dec = legs.make_decoder([bf(w) for w in di.weights], [torch.from_numpy(b).cuda() for b in di.biases])
    cb, feat, q = bf(di.codebook), bf(di.feat), bf(di.queries)
    P = feat.shape[0]
    out = []
    for packed in (False, True):
        probs = torch.zeros((P, 128), dtype=torch.bfloat16, device="cuda")
        decoded = torch.zeros((P, 896), dtype=torch.bfloat16, device="cuda")
        rel = torch.zeros((P, 4), dtype=torch.float32, device="cuda")
        ws = torch.empty(legs.legs_decode_workspace_bytes(dec, 896), dtype=torch.uint8, device="cuda")
        rws = torch.empty(legs.legs_relevancy_workspace_bytes(128, 4), dtype=torch.uint8, device="cuda")
        if packed:
            legs.legs_decode_prepare(ctx, dec, cb, ws)
            legs.legs_relevancy_prepare(ctx, cb, 512, q, rws)
            for _ in range(2):      # the prepared workspace serves any number of frames
                legs.legs_decode_semantics_packed(ctx, feat, dec, 896, probs, decoded, ws)
                legs.legs_relevancy_packed(ctx, probs, 128, 4, rel, rws)
        else:
            legs.legs_decode_semantics(ctx, feat, dec, cb, probs, decoded, ws)
            legs.legs_relevancy(ctx, probs, cb, 512, q, rel, rws)
        torch.cuda.synchronize()
        out.append((probs.view(torch.int16).cpu().numpy(), decoded.view(torch.int16).cpu().numpy(), rel.cpu().numpy()))
    for a, b in zip(out[0], out[1]):
        assert np.array_equal(a, b)
    # d_clip beyond the pack kernel's 1024-float row buffer is an argument error, not a shared-memory overrun
    big = torch.zeros((128, 2048), dtype=torch.bfloat16, device="cuda")
    qb = torch.zeros((4, 1536), dtype=torch.bfloat16, device="cuda")
    with pytest.raises(legs.LegsError) as e:
        legs.legs_relevancy_prepare(ctx, big, 1536, qb, rws)
    assert e.value.status == -3


@pytest.mark.parametrize("P,Q,n_pos,tau", [(5000 + 3, 4, 1, 10.0), (777, 16, 5, 10.0), (1, 2, 1, 1.0), (1920 * 1080, 4, 2, 10.0)])
def test_lerf_relevancy_matches_oracle(legs, ctx, oracle, P, Q, n_pos, tau):
    # LERF-style score from a cosine map (reading C-21b): the fp32 exponential is good to ~2 ulp
    # of a value in [0, 1]; tolerance 2e-6 absolute
    rng = np.random.default_rng(11)
    c = rng.uniform(-1, 1, (P, Q)).astype(np.float32)
    out = torch.full((P, n_pos), float("nan"), dtype=torch.float32, device="cuda")
    legs.legs_relevancy_lerf(ctx, torch.from_numpy(c).cuda(), n_pos, tau, out)
    torch.cuda.synchronize()
    ref = oracle.relevancy_lerf(c.astype(np.float64), n_pos, tau)
    assert np.abs(out.cpu().numpy() - ref).max() <= 2e-6


def test_lerf_relevancy_after_the_cosine_kernel(legs, ctx, oracle):
    # the chain a user runs: probabilities -> cosines against [queries | canonical negatives] -> LERF score
    di = inputs.decode_inputs(seed=1, **CASES["configs3_shape"])
    probs, _, cb = run_decode(legs, ctx, di)
    P, Q = probs.shape[0], di.queries.shape[0]
    rel = torch.zeros((P, Q), dtype=torch.float32, device="cuda")
    ws = torch.empty(legs.legs_relevancy_workspace_bytes(di.dims[-1], Q), dtype=torch.uint8, device="cuda")
    legs.legs_relevancy(ctx, probs, cb, di.d_clip, bf16_tensor(di.queries), rel, ws)
    out = torch.zeros((P, 1), dtype=torch.float32, device="cuda")
    legs.legs_relevancy_lerf(ctx, rel, 1, 10.0, out)
    torch.cuda.synchronize()
    ref = oracle.relevancy_lerf(oracle_decode(oracle, di)["rel"], 1, 10.0)
    # cosines within 2e-2 (G-5); d score / d cosine <= tau / 4 per cosine, two cosines enter
    assert np.abs(out.cpu().numpy() - ref).max() <= 2 * 2e-2 * 10.0 / 4
    with pytest.raises(RuntimeError):
        legs.legs_relevancy_lerf(ctx, rel, Q, 10.0, out)     # no negatives left


@pytest.mark.parametrize("P,d,d_clip,Q", [(148 * 8 * 16 * 2 + 13, 896, 512, 4), (1000, 896, 512, 16), (77, 64, 40, 1),
                                          (4096 + 5, 1024, 1024, 9), (16, 128, 8, 3)])
def test_relevancy_from_a_decoded_map(legs, ctx, oracle, P, d, d_clip, Q):
    """legs_relevancy_decoded (SURVEY.md 8(b) input_is_probs = 0): cosine of a given bf16 map F against the
    queries. Both sides read the same bf16 values, so only the fp32 accumulation differs: 1e-5 abs (the north_star tolerance
    for relevancy against the full decode is 2e-2, G-5). Ragged row counts, a partial 32-column block (d_clip = 40, 8), both
    query tile counts, unnormalised queries, and an all-zero row."""
    rng = np.random.default_rng(P + Q)
    F = inputs.to_bf16_bits((rng.standard_normal((P, d)) * rng.uniform(0.05, 4.0, (P, 1))).astype(np.float32))
    F[P // 2] = 0
    q = inputs.to_bf16_bits((rng.standard_normal((Q, d_clip)) * rng.uniform(0.5, 2.0, (Q, 1))).astype(np.float32))
    rel = torch.full((P, Q), float("nan"), dtype=torch.float32, device="cuda")
    legs.legs_relevancy_decoded(ctx, bf16_tensor(F), d_clip, bf16_tensor(q), rel)
    torch.cuda.synchronize()
    got = rel.cpu().numpy()
    assert not np.isnan(got).any()
    ref = oracle.relevancy_map(inputs.bf16_bits_to_f32(F), d_clip, inputs.bf16_bits_to_f32(q))
    assert np.abs(ref).max() > 0.05 and np.array_equal(got[P // 2], np.zeros(Q))
    assert np.abs(got - ref).max() <= 1e-5


def test_relevancy_from_decoded_agrees_with_relevancy_from_probabilities(legs, ctx, oracle):
    """The two routes to S11 on one frame: probabilities (Gram shortcut) and the decoded map the same call produced. Both
    within 2e-2 of the oracle's cosine (G-5); the decoded route sees F after its bf16 rounding."""
    di = inputs.decode_inputs(seed=1, **CASES["configs3_shape"])
    probs, decoded, cb = run_decode(legs, ctx, di)
    P, Q = probs.shape[0], di.queries.shape[0]
    q = bf16_tensor(di.queries)
    rel_p = torch.zeros((P, Q), dtype=torch.float32, device="cuda")
    rel_f = torch.zeros((P, Q), dtype=torch.float32, device="cuda")
    ws = torch.empty(legs.legs_relevancy_workspace_bytes(di.dims[-1], Q), dtype=torch.uint8, device="cuda")
    legs.legs_relevancy(ctx, probs, cb, di.d_clip, q, rel_p, ws)
    legs.legs_relevancy_decoded(ctx, decoded, di.d_clip, q, rel_f)
    torch.cuda.synchronize()
    f = inputs.bf16_bits_to_f32
    rows = np.arange(0, P, 37)
    ref = oracle.decode(f(di.feat[rows]), [f(w) for w in di.weights], di.biases, f(di.codebook), di.d_clip, f(di.queries))["rel"]
    assert np.abs(rel_f.cpu().numpy()[rows] - ref).max() <= 2e-2
    assert np.abs(rel_p.cpu().numpy()[rows] - ref).max() <= 2e-2
    assert (rel_f - rel_p).abs().max().item() <= 2e-2
    with pytest.raises(legs.LegsError):
        legs.legs_relevancy_decoded(ctx, decoded, 516, q, rel_f)      # d_clip not a multiple of 8
