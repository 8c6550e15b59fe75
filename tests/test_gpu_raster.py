"""GPU parity tests (run with -m gpu on the B200 box): the CUDA path through the C-ABI against the CPU oracle, element
by element on the same seeded inputs. Tolerances are BASELINE.json north_star's: tile lists / keys / ranges bit-exact,
forward images 1e-4 abs (depth: 1e-4 relative to max(1,|z|), G-2), gradients 1e-3 rel with a 1e-5 abs floor
or the conditioning term of tests/gradcheck.py (G-4) for 100 % of the elements, outside the oracle's fragile mask (G-3)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from paper_2311_18482_b200 import inputs  # noqa: E402


@pytest.fixture(scope="module")
def legs():
    from paper_2311_18482_b200 import binding
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    binding.lib()  # fails loudly if liblegs.so is missing: there is no fallback
    return binding


@pytest.fixture(scope="module")
def ctx(legs):
    return legs.Context(0)


def scenes():
    return {
        "tiny": lambda: inputs.tiny_scene(),                                                    # configs[0]
        "tiny_ragged": lambda: inputs.tiny_scene(n=700, seed=5, width=75, height=53),
        "object_small": lambda: inputs.object_scene(n=20000, seed=1, width=328, height=250, focal=450.0, n_views=2),
        "unbounded_small": lambda: inputs.unbounded_scene(n=40000, seed=2, width=400, height=266, focal=287.5),
        "large_small": lambda: inputs.large_scene(n=30000, seed=4, width=240, height=136, focal=144.0, n_views=1),
    }


def run_gpu(legs, ctx, scene, cam, want_keys=True, capacity=None, flags=None, upstream=None, tile_order=False):
    g = legs.Gaussians.from_scene(scene)
    probe = legs.Renderer(ctx, g, cam, capacity=16)
    legs.legs_preprocess(ctx, g, probe.cam, probe.frame)
    D = legs.legs_read_num_instances(ctx, probe.frame)
    r = legs.Renderer(ctx, g, cam, capacity=max(D, 1) if capacity is None else capacity, want_keys=want_keys, want_bf16=True)
    if tile_order:
        r.use_tile_order()      # legs_tile_order + the *_ordered render calls: heavy tiles first
    r.forward()
    torch.cuda.synchronize()
    res = dict(D=D, renderer=r, g=g)
    f = r.frame
    res["frame"] = {k: getattr(f, k).cpu().numpy() for k in
                    ("depth", "radius", "rect", "mean2d", "conic_opacity", "rgb", "clamped", "tiles_touched")}
    res["vals"] = r.vals_sorted[:D].cpu().numpy().view(np.uint32)
    res["ranges"] = r.ranges.cpu().numpy().view(np.uint32)
    if want_keys:
        res["keys"] = r.keys_sorted[:D].cpu().numpy().view(np.uint64)
    res["out"] = r.out.cpu().numpy()
    res["n_contrib"] = r.n_contrib.cpu().numpy().view(np.uint32)
    res["sem_bf16"] = r.sem_bf16.view(torch.int16).cpu().numpy().view(np.uint16)
    if upstream is not None:
        grads = legs.Grads(g)
        r.backward(torch.from_numpy(upstream).cuda(), grads, flags or 0)
        torch.cuda.synchronize()
        res["grads"] = {k: getattr(grads, k).cpu().numpy() for k in
                        ("dmeans", "dscales", "dquats", "dopacities", "dsh", "dsem", "dunc", "dmean2d")}
    return res


def bits(a):
    return np.ascontiguousarray(a, dtype=np.float32).view(np.uint32)


def check_preprocess(res, proj):
    fr = res["frame"]
    assert np.array_equal(fr["tiles_touched"].view(np.uint32), proj["tiles_touched"])
    assert np.array_equal(fr["radius"], proj["radius"])
    assert np.array_equal(fr["rect"], proj["rect"])
    assert np.array_equal(fr["clamped"], proj["clamped"])
    assert np.array_equal(bits(fr["depth"]), bits(proj["depth"]))
    for k in ("mean2d", "conic_opacity", "rgb"):
        assert np.array_equal(bits(fr[k]), bits(proj[k])), k  # rule P-0: same fp32 operation sequence on both sides


def check_tile_lists(res, tl):
    assert res["D"] == tl["D"]
    assert np.array_equal(res["vals"], tl["vals"])
    assert np.array_equal(res["ranges"], tl["ranges"])
    if "keys" in res:
        assert np.array_equal(res["keys"], tl["keys"])


def forward_errors(out_gpu, ref, F):
    """abs error per channel; depth (slot 3) relative to max(1, |z|)."""
    err = np.abs(out_gpu.astype(np.float64) - ref)
    err[:, 3] /= np.maximum(1.0, np.abs(ref[:, 3]))
    return err[:, :6 + F]


def check_forward(res, ora, F, tol=1e-4):
    H, W, CH = res["out"].shape
    out = res["out"].reshape(-1, CH)
    ok = ora["fragile"] == 0
    err = forward_errors(out, ora["out"], F)
    assert err[ok].max() <= tol, f"max forward error {err[ok].max()} at channel {np.unravel_index(err[ok].argmax(), err[ok].shape)}"
    assert np.array_equal(res["n_contrib"].reshape(-1)[ok], ora["n_contrib"][ok])
    assert np.allclose(out[ok, 6 + F], 1.0 - ora["out"][ok, 5 + F], atol=1e-6)   # stored final transmittance
    assert (~ok).mean() < 2e-3
    return float(err[ok].max()), float((~ok).mean())


@pytest.mark.parametrize("name", list(scenes().keys()))
def test_forward_path_matches_oracle(legs, ctx, oracle, name):
    scene = scenes()[name]()
    cam = scene.cameras[0]
    res = run_gpu(legs, ctx, scene, cam)
    proj = oracle.project(scene, cam, 0)
    check_preprocess(res, proj)
    check_tile_lists(res, oracle.tile_lists(proj, cam))
    ora = oracle.composite_forward(proj, scene.sem, scene.unc, cam)
    check_forward(res, ora, scene.sem_dim)
    # the bf16 copy of the semantic channels is the fp32 result rounded to nearest even
    sem32 = res["out"].reshape(-1, res["out"].shape[2])[:, 4:4 + scene.sem_dim]
    assert np.array_equal(res["sem_bf16"], inputs.to_bf16_bits(sem32))


@pytest.mark.parametrize("width,height", [(2304, 48), (48, 4160), (2100, 333), (32, 12000), (12000, 32)])
def test_tile_lists_on_extreme_grids(legs, ctx, oracle, width, height):
    """Tile grids outside the benchmark's shape: more than 128 tile columns (the expansion walks the column windows four
    at a time), more than 256 tile rows (nine groups of 32 rows in the ranked row emission), a grid whose rows are much
    shorter than an expansion chunk (many rows per chunk), 750 tile rows (the emission's per-row tables need more than
    48 KB of shared memory) and 750 tile columns (24 column windows). Tile lists, keys and ranges stay bit-exact; the
    image is compared too."""
    scene = inputs.tiny_scene(n=6000, seed=11, width=64, height=64)
    # stretch the tiny scene over the whole image: x, y in [-1, 1] at depth z in [2, 6]
    fx, fy = 0.9 * width, 0.9 * height
    cam = inputs.identity_camera(width, height, fx, fy, width / 2.0, height / 2.0)
    res = run_gpu(legs, ctx, scene, cam)
    proj = oracle.project(scene, cam, 0)
    check_preprocess(res, proj)
    check_tile_lists(res, oracle.tile_lists(proj, cam))
    assert res["D"] > 20000
    ora = oracle.composite_forward(proj, scene.sem, scene.unc, cam)
    check_forward(res, ora, scene.sem_dim)


from gradcheck import GRAD_KEYS, check_grads  # noqa: E402  (the one gradient check, shared with __graft_entry__.smoke)


@pytest.mark.parametrize("flags", [0, 2])
@pytest.mark.parametrize("name", ["tiny", "tiny_ragged", "object_small", "unbounded_small", "large_small"])
def test_backward_matches_oracle(legs, ctx, oracle, name, flags):
    scene = scenes()[name]()
    cam = scene.cameras[0]
    up = inputs.upstream_gradient(scene, 0)
    # G-3: at fragile pixels a correct fp32 implementation may take the other branch of a threshold test, so their
    # upstream gradient is zeroed on both sides (the oracle's mask also flags alpha within 1e-5 of the 0.99 clamp)
    fragile = oracle.render_forward(scene, cam)["fragile"].reshape(cam.height, cam.width) != 0
    assert fragile.mean() < 2e-3
    up[fragile] = 0
    res = run_gpu(legs, ctx, scene, cam, upstream=up, flags=flags)
    ref = oracle.render_backward(scene, cam, up.reshape(-1, up.shape[2]), mode=0, flags=flags, with_abs=True)
    report = check_grads(res["grads"], ref)
    print(name, flags, report)


@pytest.mark.parametrize("flags", [8, 10])
@pytest.mark.parametrize("name", ["tiny", "tiny_ragged", "object_small", "unbounded_small", "large_small"])
def test_backward_with_depth_and_alpha_upstream(legs, ctx, oracle, name, flags):
    # LEGS_BWD_DEPTH_ALPHA (reading C-17b): upstream gradients on the depth and alpha images too;
    # same element-wise check as above (north_star tolerance + the one conditioning term, tests/gradcheck.py)
    scene = scenes()[name]()
    cam = scene.cameras[0]
    up = inputs.upstream_gradient(scene, 0, depth_alpha=True)
    fragile = oracle.render_forward(scene, cam)["fragile"].reshape(cam.height, cam.width) != 0
    up[fragile] = 0
    res = run_gpu(legs, ctx, scene, cam, upstream=up, flags=flags)
    ref = oracle.render_backward(scene, cam, up.reshape(-1, up.shape[2]), mode=0, flags=(flags & 2) | 4, with_abs=True)
    report = check_grads(res["grads"], ref)
    print(name, flags, report)
    # the depth / alpha upstream really reached the geometry
    base = oracle.render_backward(scene, cam, up.reshape(-1, up.shape[2]), mode=0, flags=flags & 2)
    assert not np.allclose(base["dmeans"], ref["dmeans"], rtol=1e-2)


def sample_pixels(cam, rng, n_random=2400):
    W, H = cam.width, cam.height
    tile = np.array([(H // 2 + j) * W + W // 2 + i for j in range(16) for i in range(16)])
    strip = np.arange(W) + (H - 1) * W
    return np.unique(np.concatenate([tile, strip[::4], rng.choice(W * H, n_random, replace=False)])).astype(np.int64)


def full_size_views(legs, ctx, oracle, scene, views, min_D, want_keys=False):
    """Full-size scene in the launch configuration bench.py times. Per view: tile lists bit-exact against the oracle;
    forward on ~3000 sampled pixels (a whole tile, an image-border strip and random pixels). Gradients: the upstream
    gradient is nonzero on the sampled pixels only, so the oracle's per-pixel reverse mode over those pixels is the
    complete reference; several views accumulate into one gradient set (LEGS_BWD_ACCUMULATE), as configs[4] prescribes."""
    F = scene.sem_dim
    rng = np.random.default_rng(3)
    g = legs.Gaussians.from_scene(scene)
    grads = legs.Grads(g)
    ref = ref_abs = None
    r = None
    for vi, view in enumerate(views):
        cam = scene.cameras[view]
        W, H = cam.width, cam.height
        pix = sample_pixels(cam, rng)
        proj = oracle.project(scene, cam, 0)
        fwd = oracle.composite_forward(proj, scene.sem, scene.unc, cam, pix)
        G = np.zeros((pix.shape[0], inputs.channels(F)))
        G[:, 0:3] = rng.standard_normal((pix.shape[0], 3))
        G[:, 4:5 + F] = rng.standard_normal((pix.shape[0], F + 1))
        G[fwd["fragile"] != 0] = 0                      # G-3
        up = np.zeros((H, W, inputs.channels(F)), dtype=np.float32)
        up.reshape(-1, up.shape[2])[pix] = G.astype(np.float32)
        if r is None:
            probe = legs.Renderer(ctx, g, cam, capacity=16)
            legs.legs_preprocess(ctx, g, probe.cam, probe.frame)
            D0 = legs.legs_read_num_instances(ctx, probe.frame)
            r = legs.Renderer(ctx, g, cam, capacity=int(1.5 * D0) + 1024, want_keys=want_keys, want_bf16=True)
        r.set_camera(cam)
        r.forward()
        D = legs.legs_read_num_instances(ctx, r.frame)
        r.backward(torch.from_numpy(up).cuda(), grads, legs.LEGS_BWD_ACCUMULATE if vi else 0)
        torch.cuda.synchronize()
        res = dict(D=D, frame={k: getattr(r.frame, k).cpu().numpy() for k in
                               ("depth", "radius", "rect", "mean2d", "conic_opacity", "rgb", "clamped", "tiles_touched")},
                   vals=r.vals_sorted[:D].cpu().numpy().view(np.uint32), ranges=r.ranges.cpu().numpy().view(np.uint32))
        check_preprocess(res, proj)
        tl = oracle.tile_lists(proj, cam)
        assert res["D"] == tl["D"] > min_D
        assert np.array_equal(res["vals"], tl["vals"]) and np.array_equal(res["ranges"], tl["ranges"])
        if want_keys:   # the 64-bit (tile << 32 | depth bits) keys at full size, all D of them
            assert np.array_equal(r.keys_sorted[:D].cpu().numpy().view(np.uint64), tl["keys"])
        out = r.out.cpu().numpy().reshape(-1, r.CH)[pix]
        ok = fwd["fragile"] == 0
        assert forward_errors(out, fwd["out"], F)[ok].max() <= 1e-4
        assert np.array_equal(r.n_contrib.cpu().numpy().view(np.uint32).reshape(-1)[pix][ok], fwd["n_contrib"][ok])
        g2d = oracle.composite_backward(proj, scene.sem, scene.unc, cam, G.astype(np.float32).astype(np.float64), pix, flags=0,
                                        with_abs=True)
        g3d = oracle.project_backward(scene, cam, g2d, 0)
        one = dict(dmeans=g3d["dmeans"], dscales=g3d["dscales"], dquats=g3d["dquats"], dopacities=g2d["dopac"],
                   dsh=g3d["dsh"], dsem=g2d["dsem"], dunc=g2d["dunc"], dmean2d=g2d["dmean2d"])
        one_abs = oracle.gradient_abs(scene, cam, g2d["abs"], 0)
        ref = one if ref is None else {k: ref[k] + one[k] for k in ref}
        ref_abs = one_abs if ref_abs is None else {k: ref_abs[k] + one_abs[k] for k in ref_abs}
    ref["abs"] = ref_abs
    print(check_grads({k: getattr(grads, k).cpu().numpy() for k in GRAD_KEYS}, ref))
    return r


def test_full_size_configs2_sampled_pixels(legs, ctx, oracle):
    """BASELINE.json configs[2]: 1M Gaussians, 1600x1064 (the benchmarked workload)."""
    full_size_views(legs, ctx, oracle, inputs.unbounded_scene(), [0], 25_000_000, want_keys=True)


def test_full_size_configs1_sampled_pixels(legs, ctx, oracle):
    """BASELINE.json configs[1]: 100k Gaussians, 800x800, gradients accumulated over three of the eight views."""
    full_size_views(legs, ctx, oracle, inputs.object_scene(), [0, 3, 7], 300_000)


def test_full_size_configs4_sampled_pixels(legs, ctx, oracle):
    """BASELINE.json configs[4]: 3M Gaussians in 200 clusters, F = 16, 1920x1080, gradients accumulated over two of the
    four views; then the decode (16 -> 64 -> 128, 128 x 896 codebook) of the last view's rendered semantic map, checked
    on sampled rows."""
    scene = inputs.large_scene()
    r = full_size_views(legs, ctx, oracle, scene, [0, 2], 1_000_000)
    di = inputs.decode_inputs(P=8, in_dim=16, hidden=(64,), n_codes=128, seed=1)
    bf = lambda bits: torch.from_numpy(bits.view(np.int16)).cuda().view(torch.bfloat16)
    dec = legs.make_decoder([bf(w) for w in di.weights], [torch.from_numpy(b).cuda() for b in di.biases])
    cb = bf(di.codebook)
    P = r.sem_bf16.shape[0]
    probs = torch.zeros((P, 128), dtype=torch.bfloat16, device="cuda")
    decoded = torch.zeros((P, 896), dtype=torch.bfloat16, device="cuda")
    ws = torch.empty(legs.legs_decode_workspace_bytes(dec, 896), dtype=torch.uint8, device="cuda")
    legs.legs_decode_semantics(ctx, r.sem_bf16, dec, cb, probs, decoded, ws)
    torch.cuda.synchronize()
    rows = np.unique(np.random.default_rng(5).integers(0, P, 3000))
    idx = torch.from_numpy(rows).cuda()
    f32 = inputs.bf16_bits_to_f32
    x = f32(r.sem_bf16[idx].view(torch.int16).cpu().numpy().view(np.uint16))
    o = oracle.decode(x, [f32(w) for w in di.weights], di.biases, f32(di.codebook), 512, f32(di.queries))
    assert np.abs(probs[idx].float().cpu().numpy() - o["probs"]).max() <= 2e-2
    d = decoded[idx].float().cpu().numpy().astype(np.float64)
    cos = (d * o["decoded"]).sum(1) / (np.linalg.norm(d, axis=1) * np.linalg.norm(o["decoded"], axis=1))
    assert cos.min() >= 0.999 and np.abs(d - o["decoded"]).max() <= 2e-2


def test_backward_accumulate_flag(legs, ctx):
    scene = inputs.tiny_scene()
    cam = scene.cameras[0]
    up = inputs.upstream_gradient(scene, 0)
    a = run_gpu(legs, ctx, scene, cam, upstream=up, flags=0)
    r, g = a["renderer"], a["g"]
    grads = legs.Grads(g)
    upt = torch.from_numpy(up).cuda()
    r.backward(upt, grads, 0)
    r.backward(upt, grads, legs.LEGS_BWD_ACCUMULATE)
    torch.cuda.synchronize()
    for k in ("dmeans", "dsh", "dsem", "dmean2d", "dopacities"):
        assert np.allclose(getattr(grads, k).cpu().numpy(), 2 * a["grads"][k], rtol=2e-4, atol=1e-6), k


def test_step_is_cuda_graph_capturable(legs, ctx):
    """Every call enqueues on the caller's stream and never synchronises (include/legs.h), so a whole step can be captured
    into a CUDA graph and replayed: same tile lists and image, gradients equal up to the order of the atomics."""
    scene = inputs.object_scene(n=20000, seed=1, width=328, height=250, focal=450.0, n_views=1)
    cam = scene.cameras[0]
    a = run_gpu(legs, ctx, scene, cam, upstream=inputs.upstream_gradient(scene, 0), flags=0)
    r, g = a["renderer"], a["g"]
    grads = legs.Grads(g)
    up = torch.from_numpy(inputs.upstream_gradient(scene, 0)).cuda()

    def step():
        r.forward()
        r.backward(up, grads, 0)

    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        step()
    torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=side):
        step()
    r.out.zero_(); r.vals_sorted.zero_(); grads.dmeans.zero_()
    graph.replay()
    torch.cuda.synchronize()
    assert np.array_equal(r.vals_sorted[:a["D"]].cpu().numpy().view(np.uint32), a["vals"])
    assert np.array_equal(r.out.cpu().numpy(), a["out"])
    for k in ("dmeans", "dsh", "dsem", "dopacities"):
        assert np.allclose(getattr(grads, k).cpu().numpy(), a["grads"][k], rtol=1e-3, atol=1e-5), k


def test_edge_cases(legs, ctx, oracle):
    # every Gaussian culled (behind the camera): empty lists, background-only image
    scene = inputs.tiny_scene(n=64, seed=9)
    scene.means[:, 2] = -scene.means[:, 2]
    cam = inputs.identity_camera(64, 64, 64, 64, 32, 32, bg=(0.25, 0.5, 0.75))
    res = run_gpu(legs, ctx, scene, cam)
    assert res["D"] == 0 and (res["ranges"] == 0).all() and (res["n_contrib"] == 0).all()
    assert np.allclose(res["out"][..., 0:3], [0.25, 0.5, 0.75]) and (res["out"][..., 3:14] == 0).all()
    # a single huge Gaussian covering every tile
    from test_oracle_projection import mk_scene
    one = mk_scene([[0, 0, 1.0]], [[2.0, 2.0, 2.0]], [[1, 0, 0, 0]], opac=[0.7])
    one.sem = np.ones((1, 8)); one.unc = np.array([0.5])
    for k in ("means", "scales", "quats", "opacities", "sh", "sem", "unc"):
        setattr(one, k, np.ascontiguousarray(getattr(one, k), dtype=np.float32))
    cam2 = inputs.identity_camera(100, 60, 80, 80, 50, 30)
    res = run_gpu(legs, ctx, one, cam2)
    assert res["D"] == 7 * 4 and (res["vals"] == 0).all()
    ora = oracle.render_forward(one, cam2)
    check_forward(res, ora, 8)


def test_capacity_overflow_is_reported(legs, ctx):
    scene = inputs.tiny_scene()
    cam = scene.cameras[0]
    g = legs.Gaussians.from_scene(scene)
    r = legs.Renderer(ctx, g, cam, capacity=100)
    r.ranges.fill_(7)
    legs.legs_preprocess(ctx, g, r.cam, r.frame)
    legs.legs_bin_and_sort(ctx, r.frame, r.cam, g.n, r.capacity, None, r.vals_sorted, r.ranges, r.sort_ws)
    with pytest.raises(legs.LegsError) as e:
        legs.legs_read_num_instances(ctx, r.frame)
    assert e.value.status == -4
    assert (r.ranges.cpu().numpy() == 0).all()  # nothing written, every tile empty


def test_argument_errors(legs, ctx):
    scene = inputs.tiny_scene(n=32)
    g = legs.Gaussians.from_scene(scene)
    r = legs.Renderer(ctx, g, scene.cameras[0], capacity=64)
    small = torch.empty(16, dtype=torch.uint8, device="cuda")
    with pytest.raises(legs.LegsError) as e:
        legs.legs_bin_and_sort(ctx, r.frame, r.cam, g.n, r.capacity, None, r.vals_sorted, r.ranges, small)
    assert e.value.status == -5
    with pytest.raises(legs.LegsError) as e:
        legs.legs_bin_and_sort(ctx, r.frame, r.cam, g.n, r.capacity, None, None, r.ranges, r.sort_ws)
    assert e.value.status == -1
    mis = r.sort_ws[4:]
    with pytest.raises(legs.LegsError) as e:
        legs.legs_bin_and_sort(ctx, r.frame, r.cam, g.n, r.capacity, None, r.vals_sorted, r.ranges, mis)
    assert e.value.status == -2


def test_overflow_beyond_2_pow_32_instances_is_detected(legs, ctx):
    """70 000 screen-filling Gaussians on a 256 x 256 tile grid make D = 4.6e9 > 2^32. The overflow test uses
    the exact 64-bit count of legs_preprocess, so the capacity error is reported (and nothing is written) instead of a
    wrapped 32-bit count slipping under the capacity."""
    n = 70_000
    z = lambda *s: torch.zeros(s, dtype=torch.float32, device="cuda")
    means = z(n, 3); means[:, 2] = 1.0
    scales = torch.full((n, 3), 50.0, device="cuda")
    quats = z(n, 4); quats[:, 0] = 1.0
    g = legs.Gaussians(means, scales, quats, torch.full((n,), 0.5, device="cuda"), z(n, 1, 3), z(n, 8), z(n), 0)
    cam = inputs.identity_camera(4096, 4096, 2048.0, 2048.0, 2048.0, 2048.0)
    r = legs.Renderer(ctx, g, cam, capacity=1 << 20)
    r.ranges.fill_(7)
    legs.legs_preprocess(ctx, g, r.cam, r.frame)
    assert legs.legs_read_num_instances(ctx, r.frame) == n * 65536          # > 2^32, exact
    legs.legs_bin_and_sort(ctx, r.frame, r.cam, g.n, r.capacity, None, r.vals_sorted, r.ranges, r.sort_ws)
    with pytest.raises(legs.LegsError) as e:
        legs.legs_read_num_instances(ctx, r.frame)
    assert e.value.status == -4
    assert (r.ranges.cpu().numpy() == 0).all()


def test_backward_with_and_without_forward_block_masks(legs, ctx):
    """legs_render_backward recomputes the per-entry warp-block masks when the caller does not hand over the ones
    legs_render_forward wrote: same gradients either way (up to the order of the atomics)."""
    scene = inputs.unbounded_scene(n=40000, seed=2, width=400, height=266, focal=287.5)
    cam = scene.cameras[0]
    up = inputs.upstream_gradient(scene, 0)
    a = run_gpu(legs, ctx, scene, cam, upstream=up, flags=0)           # Renderer hands the masks over
    r, g = a["renderer"], a["g"]
    grads = legs.Grads(g)
    legs.legs_render_backward(ctx, g, r.cam, r.frame, r.vals_sorted, r.ranges, r.out, r.n_contrib, torch.from_numpy(up).cuda(), 0,
                              grads, r.bwd_ws, None)
    torch.cuda.synchronize()
    for k in GRAD_KEYS:
        x, y = getattr(grads, k).cpu().numpy(), a["grads"][k]
        assert np.allclose(x, y, rtol=1e-4, atol=1e-6 * max(1.0, float(np.abs(y).max()))), k


@pytest.mark.parametrize("name", ["tiny_ragged", "large_small", "unbounded_small"])
def test_heavy_tiles_first_order_changes_the_schedule_not_the_results(legs, ctx, oracle, name):
    """legs_tile_order + legs_render_forward_ordered / legs_render_backward_ordered: the order is a permutation of the tiles
    with the long lists first (four buckets per octave: an entry is never followed by one more than 5/4 as long, +1); the
    forward images, n_contrib and the bf16 copy are bit-identical to the row-major launch; the gradients pass the same
    element-wise check against the oracle (the atomics' order differs, the sums do not)."""
    scene = scenes()[name]()
    cam = scene.cameras[0]
    up = inputs.upstream_gradient(scene, 0)
    fragile = oracle.render_forward(scene, cam)["fragile"].reshape(cam.height, cam.width) != 0
    up[fragile] = 0
    plain = run_gpu(legs, ctx, scene, cam, upstream=up, flags=0)
    res = run_gpu(legs, ctx, scene, cam, upstream=up, flags=0, tile_order=True)
    order = res["renderer"].tile_order.cpu().numpy().view(np.uint32).astype(np.int64)
    ntiles = res["ranges"].shape[0]
    assert np.array_equal(np.sort(order), np.arange(ntiles))
    count = (res["ranges"][:, 1].astype(np.int64) - res["ranges"][:, 0].astype(np.int64))[order]
    suffix_max = np.maximum.accumulate(count[::-1])[::-1]
    assert (count * 5 // 4 + 1 >= suffix_max).all() and count[0] * 5 // 4 + 1 >= count.max()
    assert np.array_equal(bits(res["out"]), bits(plain["out"]))
    assert np.array_equal(res["n_contrib"], plain["n_contrib"]) and np.array_equal(res["sem_bf16"], plain["sem_bf16"])
    ref = oracle.render_backward(scene, cam, up.reshape(-1, up.shape[2]), mode=0, flags=0, with_abs=True)
    check_grads(res["grads"], ref)
