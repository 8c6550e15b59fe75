"""GPU parity of the training-step plumbing against the CPU oracle.

Tolerances (derived from the arithmetic): m and v are two and three fp32 roundings (3e-7, 5e-7); the
update lr m^ / (sqrt(v^) + eps) is five fp32 operations (<= 2^-21 relative, asserted at 1e-6) and the new parameter
carries one more rounding of p itself (2^-24 |p|)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def legs():
    from paper_2311_18482_b200 import binding
    assert torch.cuda.is_available()
    binding.lib()
    return binding


@pytest.fixture(scope="module")
def ctx(legs):
    return legs.Context(0)


def test_adam_multi_tensor_against_oracle(legs, ctx, oracle):
    rng = np.random.default_rng(0)
    n = 4099                                                        # odd: the tails are not multiples of four floats
    shapes = [(n, 3), (n, 3), (n, 4), (n,), (n, 16, 3), (n, 8), (n,), (5,), (1,)]   # means .. unc + two tiny tensors
    p0 = [rng.standard_normal(s).astype(np.float32) for s in shapes]
    P = [torch.from_numpy(a.copy()).cuda() for a in p0]
    M = [torch.zeros_like(t) for t in P]
    V = [torch.zeros_like(t) for t in P]
    ref = [(a.astype(np.float64).reshape(-1), np.zeros(a.size), np.zeros(a.size)) for a in p0]
    # the hyper-parameters reach the kernel as fp32: the oracle gets the same (rounded) values
    lr, b1, b2, eps = (float(np.float32(x)) for x in (1e-3, 0.9, 0.999, 1e-8))
    for step in range(1, 6):
        g = [(rng.standard_normal(s) * 10.0 ** rng.integers(-5, 2)).astype(np.float32) for s in shapes]
        g[3][::7] = 0.0                                             # exact zeros among the gradients
        G = [torch.from_numpy(a).cuda() for a in g]
        before = [t.cpu().numpy().astype(np.float64).reshape(-1) for t in P]
        legs.legs_adam_step(ctx, P, G, M, V, step)
        torch.cuda.synchronize()
        for k in range(len(shapes)):
            # the oracle steps from the GPU's own fp32 state of the previous step, so one step is compared at a time
            pr, mr, vr = oracle.adam_step(before[k], g[k], ref[k][1], ref[k][2], lr, b1, b2, eps, step)
            pg = P[k].cpu().numpy().astype(np.float64).reshape(-1)
            mg = M[k].cpu().numpy().astype(np.float64).reshape(-1)
            vg = V[k].cpu().numpy().astype(np.float64).reshape(-1)
            # m = b1 m + (1-b1) g may cancel: the rounding bound is relative to the terms, not to their sum
            gk = g[k].astype(np.float64).reshape(-1)
            assert (np.abs(mg - mr) <= 3e-7 * (np.abs(ref[k][1]) + np.abs(gk)) + 1e-30).all(), (k, step)
            assert np.allclose(vg, vr, rtol=5e-7, atol=1e-30), (k, step)
            upd_g, upd_r = pg - before[k], pr - before[k]
            # the update inherits m's bound, scaled like the update itself: |upd| |dm| / |m|
            dm = 3e-7 * (np.abs(ref[k][1]) + np.abs(gk))
            scale = np.abs(upd_r) / np.maximum(np.abs(mr), 1e-300)
            assert (np.abs(upd_g - upd_r) <= 1e-6 * np.abs(upd_r) + scale * dm + 2.0 ** -23 * np.abs(before[k]) + 1e-12).all(), (k, step)
            ref[k] = (pr, mg.copy(), vg.copy())


def test_adam_argument_errors(legs, ctx):
    t = torch.zeros(8, device="cuda")
    with pytest.raises(legs.LegsError) as e:
        legs.legs_adam_step(ctx, [t], [t], [t], [t], 0)
    assert e.value.status == -3
    with pytest.raises(legs.LegsError) as e:
        legs.legs_adam_step(ctx, [t[1:]], [t[1:]], [t[1:]], [t[1:]], 1)
    assert e.value.status == -2


def test_density_stats_against_oracle(legs, ctx, oracle):
    rng = np.random.default_rng(1)
    n = 10007
    d = rng.standard_normal((n, 2)).astype(np.float32)
    radius = rng.integers(0, 6, n).astype(np.int32)
    ga0 = rng.uniform(0, 2, n).astype(np.float32)
    dn0 = rng.integers(0, 4, n).astype(np.uint32)
    mr0 = rng.integers(0, 5, n).astype(np.int32)
    ga, dn, mr = (torch.from_numpy(ga0.copy()).cuda(), torch.from_numpy(dn0.astype(np.int32)).cuda(), torch.from_numpy(mr0.copy()).cuda())
    legs.legs_density_stats(ctx, torch.from_numpy(d).cuda(), torch.from_numpy(radius).cuda(), ga, dn, mr)
    torch.cuda.synchronize()
    rga, rdn, rmr = oracle.density_stats(d, radius, ga0, dn0, mr0)
    assert np.allclose(ga.cpu().numpy(), rga, rtol=3e-7)
    assert np.array_equal(dn.cpu().numpy().view(np.uint32), rdn) and np.array_equal(mr.cpu().numpy(), rmr)
    untouched = radius == 0
    assert np.array_equal(ga.cpu().numpy()[untouched], ga0[untouched])
