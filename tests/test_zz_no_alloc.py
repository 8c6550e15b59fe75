"""legs_relevancy_static: the relevancy map for callers that cannot allocate device memory.

Who needs it: a viewer or serving loop that carved up a fixed memory pool at start-up and may not call cudaMalloc inside
the frame loop (an allocation can synchronise the device and stall every stream), or a plugin that is only handed the host
application's input and output buffers. Every other legs call takes its scratch as a `workspace` argument; this one keeps
the 64 KB it needs (Gram matrix of the codebook + projected queries) in an array inside liblegs.so, up to K = 128 codes.

The array is shared by all calls on a device and keeps the last call's contents, so the test makes two calls in a row with
different codebooks, query sets and sizes (K = 128 then K = 32): if the second call did not clear and repack the array, it
would score against the first call's Gram matrix. Each result is compared with legs_relevancy on a caller-owned workspace
(the existing path), within the 2e-2 the relevancy parity tests use; the kernels are the same, so the difference is in fact 0.

This file sorts last on purpose (pytest -x stops at the first failure: a failure here must not hide the parity tests), and
it must pass alone in a fresh process (the first call on the device looks up the array's address) as well as after the
others (the library is already loaded and used by then)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from paper_2311_18482_b200 import inputs  # noqa: E402

REL_TOL = 2e-2   # tests/test_gpu_decode.py, G-5


def bf16_tensor(bits):
    return torch.from_numpy(bits.view(np.int16)).cuda().view(torch.bfloat16)


def probabilities(P, K, seed):
    g = torch.Generator(device="cpu").manual_seed(seed)
    logits = torch.randn((P, K), generator=g) * 3.0
    return torch.softmax(logits, dim=1).to(torch.bfloat16).cuda()


def test_static_scratch_relevancy_matches_workspace_path_on_two_calls_in_a_row():
    from paper_2311_18482_b200 import binding as legs
    assert torch.cuda.is_available()
    ctx = legs.Context(0)
    assert legs.legs_relevancy_static_max_codes() == 128
    assert legs.legs_relevancy_static_bytes() == legs.legs_relevancy_workspace_bytes(128, 16) == 65536

    # (K, Q, d, d_clip, P): several 128-pixel tiles per CTA and a ragged tail; the second call is smaller in every respect
    cases = [dict(n_codes=128, n_queries=4, d=896, d_clip=512, P=148 * 128 * 2 + 77, seed=3),
             dict(n_codes=32, n_queries=3, d=256, d_clip=128, P=5 * 128 + 19, seed=4)]
    static_out, expected = [], []
    for c in cases:                                     # the two static calls back to back, nothing in between
        di = inputs.decode_inputs(seed=c["seed"], P=256, hidden=(64,), n_codes=c["n_codes"], d=c["d"], d_clip=c["d_clip"],
                                  n_queries=c["n_queries"])
        c["cb"], c["q"] = bf16_tensor(di.codebook), bf16_tensor(di.queries)
        c["probs"] = probabilities(c["P"], c["n_codes"], c["seed"])
        rel = torch.full((c["P"], c["n_queries"]), float("nan"), dtype=torch.float32, device="cuda")
        legs.legs_relevancy_static(ctx, c["probs"], c["cb"], c["d_clip"], c["q"], rel)
        static_out.append(rel)
    torch.cuda.synchronize()
    for c in cases:                                     # the existing path, on a workspace the caller allocates
        rel = torch.full((c["P"], c["n_queries"]), float("nan"), dtype=torch.float32, device="cuda")
        ws = torch.empty(legs.legs_relevancy_workspace_bytes(c["n_codes"], c["n_queries"]), dtype=torch.uint8, device="cuda")
        legs.legs_relevancy(ctx, c["probs"], c["cb"], c["d_clip"], c["q"], rel, ws)
        expected.append(rel)
    torch.cuda.synchronize()
    for got, want in zip(static_out, expected):
        assert not torch.isnan(want).any().item() and not torch.isnan(got).any().item()
        assert (want.abs().max().item() > 0.01)                       # a real map, not zeros against zeros
        assert (got - want).abs().max().item() <= REL_TOL
        assert torch.equal(got, want)                                 # same kernels on the same packed operands

    # sizes the fixed array cannot serve are refused up front (LEGS_ERR_DIM = -3), and the next call still works
    big_cb = torch.zeros((256, 896), dtype=torch.bfloat16, device="cuda")
    big_p = torch.zeros((128, 256), dtype=torch.bfloat16, device="cuda")
    rel = torch.zeros((128, 4), dtype=torch.float32, device="cuda")
    with pytest.raises(legs.LegsError) as e:
        legs.legs_relevancy_static(ctx, big_p, big_cb, 512, cases[0]["q"], rel)
    assert e.value.status == -3
    c = cases[0]
    again = torch.full((c["P"], c["n_queries"]), float("nan"), dtype=torch.float32, device="cuda")
    legs.legs_relevancy_static(ctx, c["probs"], c["cb"], c["d_clip"], c["q"], again)
    torch.cuda.synchronize()
    assert torch.equal(again, expected[0])
