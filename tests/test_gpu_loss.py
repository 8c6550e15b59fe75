"""GPU parity of the semantic loss head (legs_semantic_loss, Eq. 8-12) against the fp64 oracle.
Tolerances (G-6): the hidden activations, dz and dpre enter the tensor cores as bf16 (relative rounding 2^-9),
accumulation is fp32. Losses: 2e-3 relative. dL/dR_u = (lambda_u - lambda_ce CE) / P: the logits carry the bf16 rounding of
the hidden activations. Every gradient is compared ELEMENT BY ELEMENT against a bound derived from the arithmetic:
2^-8 sum_j |a_j b_j| for a contraction of two bf16-rounded factors, propagated through the chain (computed in the test
with numpy from an independent forward pass), plus a floor of 1e-7 of the array's largest entry."""
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
    ws = torch.empty(legs.legs_loss_workspace_bytes(dec, P), dtype=torch.uint8, device="cuda")
    legs.legs_semantic_loss(ctx, torch.from_numpy(pixels).cuda(), torch.from_numpy(index).cuda(), dec, lce, lu, dL, dw, db, loss, ws)
    torch.cuda.synchronize()
    f = inputs.bf16_bits_to_f32
    ref = oracle.semantic_loss(pixels[:, 4:4 + F], pixels[:, 4 + F], index, [f(w) for w in di.weights], di.biases, lce, lu)
    assert np.allclose(loss.cpu().numpy(), ref["loss"], rtol=2e-3, atol=1e-6), (loss.cpu().numpy(), ref["loss"])
    g = dL.cpu().numpy()
    keep = np.ones(CH, bool); keep[4:5 + F] = False
    assert (g[:, keep] == 7.0).all()                                   # other slots untouched
    # element-wise bounds from the arithmetic (G-6): every tensor-core contraction sum_j a_j b_j has bf16 operands
    # (2^-9 relative each) => 2^-8 sum_j |a_j b_j|; one more factor 2 per earlier bf16 hop that feeds a_j or b_j.
    W0, W1 = f(di.weights[0]).astype(np.float64), f(di.weights[1]).astype(np.float64)
    x = pixels[:, 4:4 + F].astype(np.float64)
    u = pixels[:, 4 + F].astype(np.float64)
    pre = x @ W0.T + di.biases[0]
    h = np.maximum(pre, 0.0)
    z = h @ W1.T + di.biases[1]
    pz = np.exp(z - z.max(1, keepdims=True)); pz /= pz.sum(1, keepdims=True)
    coef = lce * (1.0 - u) / P
    dz = coef[:, None] * (pz - np.eye(K)[index])
    dpre = (dz @ W1) * (pre > 0)
    e8 = 2.0 ** -8
    z_err = e8 * (np.abs(h) @ np.abs(W1).T)                                   # per logit
    assert (np.abs(g[:, 4 + F] - ref["du"]) <= lce / P * 2.0 * z_err.max(1) + 1e-7 / P).all()
    dz_err = 2.0 * coef[:, None] * z_err.max(1, keepdims=True)                  # softmax is 1-Lipschitz in the max norm (x2)
    dh_bound = 2 * e8 * (np.abs(dz) @ np.abs(W1)) + dz_err * np.abs(W1).sum(0)[None, :]
    dx = g[:, 4:4 + F].astype(np.float64)
    assert (np.abs(dx - ref["dx"]) <= dh_bound @ np.abs(W0) + 1e-7 / P).all(), np.abs(dx - ref["dx"]).max()
    bounds_w = [2 * e8 * (np.abs(dpre).T @ np.abs(x)) + dh_bound.T @ np.abs(x), 2 * e8 * (np.abs(dz).T @ np.abs(h)) + dz_err.T @ np.abs(h)]
    bounds_b = [2 * e8 * np.abs(dpre).sum(0) + dh_bound.sum(0), 2 * e8 * np.abs(dz).sum(0) + dz_err.sum(0)]
    for l in range(2):
        a, b = dw[l].cpu().numpy().astype(np.float64), ref["dW"][l]
        assert (np.abs(a - b) <= bounds_w[l] + 1e-7 * np.abs(b).max()).all(), (l, float((np.abs(a - b) / (bounds_w[l] + 1e-30)).max()))
        a, b = db[l].cpu().numpy().astype(np.float64), ref["db"][l]
        assert (np.abs(a - b) <= bounds_b[l] + 1e-7 * np.abs(b).max()).all(), (l, "bias", float((np.abs(a - b) / (bounds_b[l] + 1e-30)).max()))


CASES3 = {
    "table3": dict(P=3000 + 77, in_dim=8, hidden=(128, 256), n_codes=128, bias_sigma=0.1),
    "table3_persistent": dict(P=148 * 128 * 2 + 5, in_dim=8, hidden=(128, 256), n_codes=128, bias_sigma=0.1),
    "table3_f16_k64": dict(P=1000, in_dim=16, hidden=(128, 256), n_codes=64, bias_sigma=0.1),
    "table3_k32_ragged": dict(P=17, in_dim=8, hidden=(128, 256), n_codes=32, bias_sigma=0.0),
}


@pytest.mark.parametrize("name", list(CASES3.keys()))
def test_semantic_loss_table3_decoder(legs, ctx, oracle, name):
    """The paper's own decoder (Table 3: F -> 128 -> 256 -> K) through legs_semantic_loss. Bounds (G-6):
    a forward error analysis of the kernel's operation sequence, computed here with numpy from an exact forward pass.
    e = 2^-8 per contraction of bf16-stored factors with fp32 accumulation; an error in a factor is carried through the
    absolute values of the other; a ReLU unit of the middle layer whose pre-activation lies within its own error bound of
    zero ("fragile") may switch in the backward pass and is allowed the whole term it gates. Safety factor 2."""
    kw = CASES3[name]
    di = inputs.decode_inputs(seed=1, d=64, d_clip=32, **kw)
    P, F, K = kw["P"], kw["in_dim"], kw["n_codes"]
    CH = inputs.channels(F)
    rng = np.random.Generator(np.random.PCG64(7))
    pixels = rng.standard_normal((P, CH)).astype(np.float32)
    pixels[:, 4 + F] = rng.uniform(0, 1, P).astype(np.float32)
    index = rng.integers(0, K, P).astype(np.int32)
    lce, lu = 1.0, 0.25
    ws_ = [bf16_tensor(w) for w in di.weights]
    bs_ = [torch.from_numpy(b).cuda() for b in di.biases]
    dec = legs.make_decoder(ws_, bs_)
    dL = torch.full((P, CH), 7.0, dtype=torch.float32, device="cuda")
    dw = [torch.zeros(w.shape, dtype=torch.float32, device="cuda") for w in ws_]
    db = [torch.zeros(b.shape, dtype=torch.float32, device="cuda") for b in bs_]
    loss = torch.zeros(3, dtype=torch.float32, device="cuda")
    ws = torch.empty(legs.legs_loss_workspace_bytes(dec, P), dtype=torch.uint8, device="cuda")
    legs.legs_semantic_loss(ctx, torch.from_numpy(pixels).cuda(), torch.from_numpy(index).cuda(), dec, lce, lu, dL, dw, db, loss, ws)
    torch.cuda.synchronize()
    f = inputs.bf16_bits_to_f32
    ref = oracle.semantic_loss(pixels[:, 4:4 + F], pixels[:, 4 + F], index, [f(w) for w in di.weights], di.biases, lce, lu)
    assert np.allclose(loss.cpu().numpy(), ref["loss"], rtol=2e-3, atol=1e-6), (loss.cpu().numpy(), ref["loss"])
    g = dL.cpu().numpy()
    keep = np.ones(CH, bool); keep[4:5 + F] = False
    assert (g[:, keep] == 7.0).all()
    W0, W1, W2 = (f(w).astype(np.float64) for w in di.weights)
    A0, A1, A2 = np.abs(W0), np.abs(W1), np.abs(W2)
    x = pixels[:, 4:4 + F].astype(np.float64)
    u = pixels[:, 4 + F].astype(np.float64)
    pre0 = x @ W0.T + di.biases[0]
    h0 = np.maximum(pre0, 0.0)
    pre1 = h0 @ W1.T + di.biases[1]
    h1 = np.maximum(pre1, 0.0)
    z = h1 @ W2.T + di.biases[2]
    pz = np.exp(z - z.max(1, keepdims=True)); pz /= pz.sum(1, keepdims=True)
    coef = lce * (1.0 - u) / P
    dz = coef[:, None] * (pz - np.eye(K)[index])
    dh1 = dz @ W2
    dpre1 = dh1 * (pre1 > 0)
    dh0 = dpre1 @ W1
    dpre0 = dh0 * (pre0 > 0)
    e = 2.0 ** -8
    S = 2.0                                                                   # safety factor
    e_pre0 = 1e-6 * (np.abs(x) @ A0.T + np.abs(di.biases[0]))                  # fp32 layer 0
    frag0 = np.abs(pre0) <= e_pre0
    e_pre1 = e * (h0 @ A1.T) + e_pre0 @ A1.T
    frag1 = np.abs(pre1) <= S * e_pre1
    e_z = e * (h1 @ A2.T) + e_pre1 @ A2.T
    assert (np.abs(g[:, 4 + F] - ref["du"]) <= S * (lce / P * 2.0 * e_z.max(1)) + 1e-7 / P).all()
    e_dz = 2.0 * coef[:, None] * e_z.max(1, keepdims=True) + e / 2 * np.abs(dz)   # softmax is 1-Lipschitz (x2); bf16 store
    e_dh1 = e * (np.abs(dz) @ A2) + e_dz @ A2
    e_dpre1 = np.where(frag1, np.abs(dh1) + e_dh1, e_dh1 * (pre1 > 0))
    e_dh0 = e * (np.abs(dpre1) @ A1) + e_dpre1 @ A1
    e_dpre0 = np.where(frag0, np.abs(dh0) + e_dh0, e_dh0 * (pre0 > 0))
    dx = g[:, 4:4 + F].astype(np.float64)
    bound_dx = S * (e_dpre0 @ A0) + 1e-7 / P
    assert (np.abs(dx - ref["dx"]) <= bound_dx).all(), float((np.abs(dx - ref["dx"]) / bound_dx).max())
    bounds_w = [2 * e * (np.abs(dpre0).T @ np.abs(x)) + e_dpre0.T @ np.abs(x),
                2 * e * (np.abs(dpre1).T @ h0) + e_dpre1.T @ h0 + np.abs(dpre1).T @ e_pre0,
                2 * e * (np.abs(dz).T @ h1) + e_dz.T @ h1 + np.abs(dz).T @ e_pre1]
    bounds_b = [e * np.abs(dpre0).sum(0) + e_dpre0.sum(0), e * np.abs(dpre1).sum(0) + e_dpre1.sum(0), e * np.abs(dz).sum(0) + e_dz.sum(0)]
    worst, relf = 0.0, [float(np.linalg.norm(dx - ref["dx"]) / np.linalg.norm(ref["dx"]))]
    for l in range(3):
        a, b = dw[l].cpu().numpy().astype(np.float64), ref["dW"][l]
        r = np.abs(a - b) / (S * bounds_w[l] + 1e-7 * np.abs(b).max())
        assert (r <= 1.0).all(), (l, float(r.max()))
        worst = max(worst, float(r.max()))
        relf.append(float(np.linalg.norm(a - b) / np.linalg.norm(b)))
        a, b = db[l].cpu().numpy().astype(np.float64), ref["db"][l]
        r = np.abs(a - b) / (S * bounds_b[l] + 1e-7 * np.abs(b).max())
        assert (r <= 1.0).all(), (l, "bias", float(r.max()))
        worst = max(worst, float(r.max()))
    # The worst-case bounds above are wide where many units are fragile, so the kernel is also held against a numpy
    # EMULATION of its rounding points (h0, h1, dz, dpre1, dpre0, x rounded to bf16 where the tensor cores read them,
    # everything else exact): what is left is fp32 accumulation order, __expf and units whose emulated pre-activation is
    # within fp32 rounding of zero. A dropped, doubled or transposed term shows as O(1) here.
    rb = lambda a: f(inputs.to_bf16_bits(a.astype(np.float32))).astype(np.float64)
    h0b = rb(h0)
    pre1e = h0b @ W1.T + di.biases[1]
    h1b = rb(np.maximum(pre1e, 0.0))
    ze = h1b @ W2.T + di.biases[2]
    pe = np.exp(ze - ze.max(1, keepdims=True)); pe /= pe.sum(1, keepdims=True)
    dzb = rb(coef[:, None] * (pe - np.eye(K)[index]))
    dp1b = rb((dzb @ W2) * (pre1e > 0))
    dpre0e = (dp1b @ W1) * (pre0 > 0)
    emu = [dpre0e @ W0, rb(dpre0e).T @ rb(x), dp1b.T @ h0b, dzb.T @ h1b]
    got = [dx] + [dw[l].cpu().numpy().astype(np.float64) for l in range(3)]
    rel_emu = [float(np.linalg.norm(a - b) / np.linalg.norm(b)) for a, b in zip(got, emu)]
    assert max(rel_emu) <= 2e-3, rel_emu
    assert max(relf) <= 5e-2, relf
    print(f"table3 loss head {name}: worst error / bound = {worst:.3f}, fragile middle units {int(frag1.sum())}; relative "
          f"Frobenius error of dx, dW0, dW1, dW2 against the oracle {[round(v, 5) for v in relf]}, against the bf16 emulation "
          f"{[round(v, 6) for v in rel_emu]}")


def test_render_loss_backward_chain(legs, ctx, oracle):
    """The training loop on the device: legs_render_forward -> legs_semantic_loss -> legs_render_backward, with the loss
    head writing its gradient into the upstream-gradient image. Reference: the oracle's compositor, loss head and reverse
    mode chained the same way (colour gradient zero, LEGS_BWD_COUPLE_SEM so that the semantic loss reaches the geometry)."""
    scene = inputs.object_scene(n=6000, seed=3, width=160, height=120, focal=220.0, n_views=1)
    cam = scene.cameras[0]
    F, K = scene.sem_dim, 64
    CH = inputs.channels(F)
    P = cam.width * cam.height
    di = inputs.decode_inputs(P=8, in_dim=F, hidden=(64,), n_codes=K, seed=1, d=64, d_clip=32, bias_sigma=0.1)
    index = np.random.default_rng(2).integers(0, K, P).astype(np.int32)
    lce, lu, flags = 1.0, 0.2, legs.LEGS_BWD_COUPLE_SEM
    g = legs.Gaussians.from_scene(scene)
    probe = legs.Renderer(ctx, g, cam, capacity=16)
    legs.legs_preprocess(ctx, g, probe.cam, probe.frame)
    r = legs.Renderer(ctx, g, cam, capacity=legs.legs_read_num_instances(ctx, probe.frame))
    r.forward()
    ws_ = [bf16_tensor(w) for w in di.weights]
    bs_ = [torch.from_numpy(b).cuda() for b in di.biases]
    dec = legs.make_decoder(ws_, bs_)
    dL = torch.zeros((cam.height, cam.width, CH), dtype=torch.float32, device="cuda")
    dw = [torch.zeros(w.shape, dtype=torch.float32, device="cuda") for w in ws_]
    db = [torch.zeros(b.shape, dtype=torch.float32, device="cuda") for b in bs_]
    loss = torch.zeros(3, dtype=torch.float32, device="cuda")
    ws = torch.empty(legs.legs_loss_workspace_bytes(dec, P), dtype=torch.uint8, device="cuda")
    legs.legs_semantic_loss(ctx, r.out, torch.from_numpy(index).cuda(), dec, lce, lu, dL, dw, db, loss, ws)
    # oracle chain
    fw = oracle.render_forward(scene, cam)
    dL.view(-1, CH)[torch.from_numpy(fw["fragile"] != 0).cuda()] = 0      # G-3, on both sides
    grads = legs.Grads(g)
    r.backward(dL, grads, flags)
    torch.cuda.synchronize()
    f = inputs.bf16_bits_to_f32
    lo = oracle.semantic_loss(fw["out"][:, 4:4 + F], fw["out"][:, 4 + F], index, [f(w) for w in di.weights], di.biases, lce, lu)
    up = np.zeros((P, CH))
    up[:, 4:4 + F] = lo["dx"]
    up[:, 4 + F] = lo["du"]
    up[fw["fragile"] != 0] = 0
    ref = oracle.render_backward(scene, cam, up, mode=0, flags=flags)
    assert np.allclose(loss.cpu().numpy(), lo["loss"], rtol=2e-3)
    for k in ("dsem", "dunc", "dmeans", "dopacities"):
        a = getattr(grads, k).cpu().numpy().astype(np.float64).reshape(scene.n, -1)
        b = ref[k].reshape(scene.n, -1)
        # bf16 operands inside the loss head: 2e-2 of the array's largest magnitude
        assert np.abs(a - b).max() <= 2e-2 * np.abs(b).max() + 1e-9, (k, np.abs(a - b).max(), np.abs(b).max())
