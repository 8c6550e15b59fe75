"""GPU parity of the semantic loss head (legs_semantic_loss, Eq. 8-12) against the fp64 oracle.
Tolerances (G-6): the hidden activations, dz and dpre enter the tensor cores as bf16 (relative rounding 2^-9),
accumulation is fp32. Losses: 2e-3 relative. dL/dR_u = (lambda_u - lambda_ce CE) / P: the logits carry the bf16 rounding of
the 64 hidden activations, |dz| <= 2^-9 sum_j |W1_kj h_j| ~ 4e-2 at these weight scales, so 4e-2 lambda_ce / P absolute. dL/dR_s rows and the weight
gradients: 2e-2 of the largest magnitude of the row / matrix (+ a 1e-7 floor)."""
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


CASES = {
    "configs3_shape": dict(P=3000 + 77, in_dim=8, hidden=(64,), n_codes=128, bias_sigma=0.1),
    "persistent": dict(P=148 * 128 * 3 + 5, in_dim=8, hidden=(64,), n_codes=128, bias_sigma=0.1),
    "f16_k64_h32": dict(P=2000, in_dim=16, hidden=(32,), n_codes=64, bias_sigma=0.1),
    "k32_ragged": dict(P=17, in_dim=8, hidden=(32,), n_codes=32, bias_sigma=0.0),
}


@pytest.mark.parametrize("name", list(CASES.keys()))
def test_semantic_loss_matches_oracle(legs, ctx, oracle, name):
    kw = CASES[name]
    di = inputs.decode_inputs(seed=1, d=64, d_clip=32, **kw)
    P, F, K = kw["P"], kw["in_dim"], kw["n_codes"]
    CH = inputs.channels(F)
    rng = np.random.Generator(np.random.PCG64(7))
    pixels = rng.standard_normal((P, CH)).astype(np.float32)          # R_s in slots 4..4+F-1
    pixels[:, 4 + F] = rng.uniform(0, 1, P).astype(np.float32)        # R_u
    index = rng.integers(0, K, P).astype(np.int32)
    lce, lu = 1.0, 0.25
    ws_ = [bf16_tensor(w) for w in di.weights]
    bs_ = [torch.from_numpy(b).cuda() for b in di.biases]
    dec = legs.make_decoder(ws_, bs_)
    dL = torch.full((P, CH), 7.0, dtype=torch.float32, device="cuda")
    dw = [torch.zeros(w.shape, dtype=torch.float32, device="cuda") for w in ws_]
    db = [torch.zeros(b.shape, dtype=torch.float32, device="cuda") for b in bs_]
    loss = torch.zeros(3, dtype=torch.float32, device="cuda")
    ws = torch.empty(legs.legs_loss_workspace_bytes(dec), dtype=torch.uint8, device="cuda")
    legs.legs_semantic_loss(ctx, torch.from_numpy(pixels).cuda(), torch.from_numpy(index).cuda(), dec, lce, lu, dL, dw, db, loss, ws)
    torch.cuda.synchronize()
    f = inputs.bf16_bits_to_f32
    ref = oracle.semantic_loss(pixels[:, 4:4 + F], pixels[:, 4 + F], index, [f(w) for w in di.weights], di.biases, lce, lu)
    assert np.allclose(loss.cpu().numpy(), ref["loss"], rtol=2e-3, atol=1e-6), (loss.cpu().numpy(), ref["loss"])
    g = dL.cpu().numpy()
    keep = np.ones(CH, bool); keep[4:5 + F] = False
    assert (g[:, keep] == 7.0).all()                                   # other slots untouched
    assert np.abs(g[:, 4 + F] - ref["du"]).max() <= 4e-2 * lce / P
    dx = g[:, 4:4 + F].astype(np.float64)
    tol = 2e-2 * np.abs(ref["dx"]).max(1, keepdims=True) + 1e-7 / P
    assert (np.abs(dx - ref["dx"]) <= tol).all(), np.abs(dx - ref["dx"]).max()
    for l in range(2):
        a, b = dw[l].cpu().numpy().astype(np.float64), ref["dW"][l]
        assert np.abs(a - b).max() <= 2e-2 * np.abs(b).max() + 1e-7, (l, np.abs(a - b).max(), np.abs(b).max())
        a, b = db[l].cpu().numpy().astype(np.float64), ref["db"][l]
        assert np.abs(a - b).max() <= 2e-2 * np.abs(b).max() + 1e-7, (l, "bias", np.abs(a - b).max(), np.abs(b).max())
