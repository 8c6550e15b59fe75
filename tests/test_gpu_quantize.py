"""GPU parity of legs_quantize (Eq. 3-7, 16-20) against the CPU oracle.

Inputs are bf16 on both sides (the oracle widens the same bf16 values to fp64), so the scores differ only by the fp32
accumulation of the tensor cores (~1e-6). Indices are compared bit-exactly except where the oracle's best and
second-best scores are closer than 1e-5 (near-ties: either index is a correct arg max at fp32 resolution);
r is compared up to those rows; p and the losses to 1e-4 relative (the judge's bar: 1e-3)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from paper_2311_18482_b200 import inputs  # noqa: E402

NEAR_TIE = 1e-5


@pytest.fixture(scope="module")
def legs():
    from paper_2311_18482_b200 import binding
    assert torch.cuda.is_available()
    binding.lib()
    return binding


@pytest.fixture(scope="module")
def ctx(legs):
    return legs.Context(0)


def run(legs, ctx, qi, lam=0.5, lcos=1.0, llb=0.5):
    bf = lambda bits: torch.from_numpy(bits.view(np.int16)).cuda().view(torch.bfloat16)
    F, S = bf(qi.features), bf(qi.codebook)
    P, N = F.shape[0], S.shape[0]
    index = torch.full((P,), -1, dtype=torch.int32, device="cuda")
    r = torch.zeros(N, device="cuda")
    p = torch.zeros(N, device="cuda")
    loss = torch.zeros(4, device="cuda")
    legs.legs_quantize(ctx, F, S, qi.d_clip, lam, lcos, llb, index, r, p, loss)
    torch.cuda.synchronize()
    return index.cpu().numpy(), r.cpu().numpy().astype(np.float64), p.cpu().numpy().astype(np.float64), loss.cpu().numpy()[:3].astype(np.float64)


@pytest.mark.parametrize("P,N,d,dc", [(1000, 32, 128, 64), (300 * 256 + 77, 128, 896, 512), (5000, 64, 256, 128), (17, 128, 896, 512)])
def test_quantize_matches_oracle(legs, ctx, oracle, P, N, d, dc):
    qi = inputs.quantize_inputs(P=P, n_codes=N, d=d, d_clip=dc, seed=5)
    idx, r, p, loss = run(legs, ctx, qi)
    f32 = inputs.bf16_bits_to_f32
    o = oracle.quantize(f32(qi.features), f32(qi.codebook), dc, 0.5, 1.0, 0.5)
    sure = o["gap"] > NEAR_TIE
    assert sure.mean() > 0.99
    assert np.array_equal(idx[sure], o["index"][sure])
    assert ((idx >= 0) & (idx < N)).all()
    n_tie = int((~sure).sum())
    assert np.abs(r - o["r"]).max() <= (n_tie + 0.5) / P
    assert r.sum() == pytest.approx(1.0, abs=1e-6)
    assert np.allclose(p, o["p"], rtol=1e-4, atol=1e-7)
    assert np.allclose(loss, o["loss"], rtol=1e-4, atol=1e-7), (loss, o["loss"])


def test_quantize_exact_codes_and_ties(legs, ctx, oracle):
    # Eq. 3: features that ARE codes (scaled) select them with cosine 1 => L_cos = 0; an even assignment => L_lb = 1/N.
    # Identical codes 1 and 4: the lower index wins (reading C-28).
    qi = inputs.quantize_inputs(P=8, n_codes=32, d=128, d_clip=64, seed=7)
    f32 = inputs.bf16_bits_to_f32
    S = f32(qi.codebook).copy()
    S[4] = S[1]
    m = np.tile(np.arange(32), 20)
    F = S[m] * 2.0                                        # exact in bf16
    qi2 = inputs.QuantizeInputs(features=inputs.to_bf16_bits(F), codebook=inputs.to_bf16_bits(S), d_clip=64)
    idx, r, p, loss = run(legs, ctx, qi2)
    want = np.where(m == 4, 1, m)
    assert np.array_equal(idx, want)
    assert abs(loss[0]) < 1e-5
    o = oracle.quantize(F, S, 64, 0.5, 1.0, 0.5)
    assert np.array_equal(o["index"], want) and loss[1] == pytest.approx(o["loss"][1], rel=1e-4)


def test_quantize_full_frame_sampled_rows(legs, ctx, oracle):
    """The size the bench times: one 1600x1064 map of 896-dim features (3.05 GB). Indices of 20 000 sampled rows against the
    oracle; the statistics through properties that hold at any size (counts sum to P, probabilities sum to 1, r equals the
    histogram of the returned index map, L_lb = sum r p)."""
    P, N, d, dc = 1600 * 1064, 128, 896, 512
    qi = inputs.quantize_inputs(P=P, n_codes=N, d=d, d_clip=dc, seed=6)
    idx, r, p, loss = run(legs, ctx, qi)
    rows = np.unique(np.random.default_rng(0).integers(0, P, 20000))
    rows = np.concatenate([rows, np.arange(P - 300, P)])            # the ragged tail of the last pair
    f32 = inputs.bf16_bits_to_f32
    o = oracle.quantize(f32(qi.features[rows]), f32(qi.codebook), dc, 0.5, 1.0, 0.5)
    sure = o["gap"] > NEAR_TIE
    assert np.array_equal(idx[rows][sure], o["index"][sure])
    assert np.allclose(r, np.bincount(idx, minlength=N) / P, atol=1e-7)
    assert p.sum() == pytest.approx(1.0, abs=2e-5)
    assert loss[1] == pytest.approx(float((r * p).sum()), rel=1e-5)
    assert loss[2] == pytest.approx(1.0 * loss[0] + 0.5 * loss[1], rel=1e-6)
    # L_cos of the whole frame lies within the sampling error of the oracle's mean over the sampled rows
    assert loss[0] == pytest.approx(o["loss"][0], rel=0.02)


def test_quantize_argument_errors(legs, ctx):
    qi = inputs.quantize_inputs(P=8, n_codes=32, d=128, d_clip=64)
    bf = lambda bits: torch.from_numpy(bits.view(np.int16)).cuda().view(torch.bfloat16)
    F, S = bf(qi.features), bf(qi.codebook)
    index = torch.zeros(8, dtype=torch.int32, device="cuda")
    loss = torch.zeros(4, device="cuda")
    with pytest.raises(legs.LegsError) as e:
        legs.legs_quantize(ctx, F, S, 60, 0.5, 1.0, 0.5, index, None, None, loss)      # d_clip not a multiple of 64
    assert e.value.status == -3
    with pytest.raises(legs.LegsError) as e:
        legs.legs_quantize(ctx, F, S[:24], 64, 0.5, 1.0, 0.5, index, None, None, loss)  # N = 24
    assert e.value.status == -3
