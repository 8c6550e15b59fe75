"""Pins for the oracle's reverse-mode gradients ("differentiable rendering and gradient descent",
:182 "does not affect original reconstruction quality"): central finite differences in the fp64 mode on tiny
scenes, and the isolation-flag identities (reading C-14)."""
from types import SimpleNamespace

import numpy as np
import pytest

from paper_2311_18482_b200 import inputs


def small_scene(n=24, seed=0, size=32, sh_degree=3, F=8):
    rng = np.random.default_rng(seed)
    means = np.concatenate([rng.uniform(-0.6, 0.6, (n, 2)), rng.uniform(2.0, 4.0, (n, 1))], 1)
    scales = np.exp(rng.normal(-2.0, 0.4, (n, 3)))
    q = rng.standard_normal((n, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    opac = 1 / (1 + np.exp(-rng.normal(0, 1, n)))
    K = (sh_degree + 1) ** 2
    sh = rng.normal(0, 0.3, (n, K, 3))
    sc = SimpleNamespace(means=means, scales=scales, quats=q, opacities=opac, sh=sh, sem=rng.standard_normal((n, F)),
                         unc=rng.uniform(0, 1, n), sh_degree=sh_degree)
    cam = inputs.look_at_camera([0.4, -0.3, -1.0], size, size, 40.0, 44.0, size / 2.0, size / 2.0, bg=(0.2, 0.4, 0.6))
    sc.means = sc.means - np.array([0, 0, 3.0])  # centre the blob around the look-at point
    G = np.zeros((size * size, inputs.channels(F)))
    G[:, 0:3] = rng.standard_normal((size * size, 3))
    G[:, 4:4 + F + 1] = rng.standard_normal((size * size, F + 1))
    return sc, cam, G


def loss(oracle, sc, cam, G):
    return float((oracle.render_forward(sc, cam, mode=1, fragile_rel=1e-4)["out"] * G).sum())


FIELDS = [("means", "dmeans"), ("scales", "dscales"), ("quats", "dquats"), ("opacities", "dopacities"), ("sh", "dsh"),
          ("sem", "dsem"), ("unc", "dunc")]


@pytest.mark.parametrize("flags", [2])
@pytest.mark.parametrize("seed,sh_degree", [(0, 3), (1, 1), (2, 0)])
def test_full_reverse_mode_matches_central_differences(oracle, seed, sh_degree, flags):
    # flags bit1: full reverse mode (every channel's upstream gradient reaches geometry) == d(loss)/d(param)
    sc, cam, G = small_scene(seed=seed, sh_degree=sh_degree)
    fw = oracle.render_forward(sc, cam, mode=1, fragile_rel=1e-4)
    assert fw["fragile"].sum() == 0 and fw["blended"] > 2000
    g = oracle.render_backward(sc, cam, G, mode=1, flags=flags)
    rng = np.random.default_rng(100 + seed)
    worst = 0.0
    for name, gname in FIELDS:
        arr = getattr(sc, name)
        flat = arr.reshape(-1)
        ana = g[gname].reshape(-1)
        idx = rng.choice(flat.size, size=min(60, flat.size), replace=False)
        for i in idx:
            h = 1e-6 * max(1.0, abs(flat[i])) if name != "scales" else 1e-6 * flat[i]
            old = flat[i]
            flat[i] = old + h
            lp = loss(oracle, sc, cam, G)
            flat[i] = old - h
            lm = loss(oracle, sc, cam, G)
            flat[i] = old
            fd = (lp - lm) / (2 * h)
            err = abs(fd - ana[i]) / max(1e-3, abs(fd), abs(ana[i]))
            worst = max(worst, err)
            assert err < 2e-5, (name, int(i), fd, ana[i])
    assert worst < 2e-5


def test_rgb_only_loss_matches_default_flag(oracle):
    # with upstream gradient on rgb only, default (isolated) mode is the exact derivative too
    sc, cam, G = small_scene(seed=3)
    G[:, 3:] = 0
    g = oracle.render_backward(sc, cam, G, mode=1, flags=0)
    rng = np.random.default_rng(5)
    for name, gname in FIELDS[:5]:
        flat = getattr(sc, name).reshape(-1)
        ana = g[gname].reshape(-1)
        for i in rng.choice(flat.size, size=12, replace=False):
            h = 1e-6 * max(1.0, abs(flat[i]))
            old = flat[i]
            flat[i] = old + h
            lp = loss(oracle, sc, cam, G)
            flat[i] = old - h
            lm = loss(oracle, sc, cam, G)
            flat[i] = old
            fd = (lp - lm) / (2 * h)
            assert abs(fd - ana[i]) <= 2e-5 * max(1e-3, abs(fd)), (name, int(i), fd, ana[i])


def test_isolation_flag_identities(oracle):
    # C-14: flag off == flag on with sem/unc upstream zeroed, for geometry/colour/opacity; dsem, dunc identical in both
    sc, cam, G = small_scene(seed=4)
    off = oracle.render_backward(sc, cam, G, mode=0, flags=0)
    on = oracle.render_backward(sc, cam, G, mode=0, flags=2)
    G0 = G.copy()
    G0[:, 4:] = 0
    on0 = oracle.render_backward(sc, cam, G0, mode=0, flags=2)
    for k in ("dmeans", "dscales", "dquats", "dopacities", "dsh", "dmean2d"):
        assert np.allclose(off[k], on0[k], rtol=1e-12, atol=1e-15), k
        if k != "dsh":  # dL/dc = w*G never involves alpha, so it is the same in both modes
            assert not np.allclose(off[k], on[k], rtol=1e-3), k  # the coupling is real when switched on
    for k in ("dsem", "dunc"):
        assert np.allclose(off[k], on[k], rtol=1e-12, atol=1e-15), k
    assert np.abs(on0["dsem"]).max() == 0 and np.abs(on0["dunc"]).max() == 0


def test_jacobian_clamp_and_colour_clamp_derivatives(oracle):
    # a wide Gaussian far off-axis (Jacobian clamp active) and a negative colour (clamped at 0): true derivative (C-15)
    sc, cam, G = small_scene(n=6, seed=6, sh_degree=0)
    W = cam.world_to_cam.astype(np.float64).reshape(3, 4)
    sc.means[0] = W[:, :3].T @ (np.array([0.8, 0.05, 1.2]) - W[:, 3])  # view-space x/z = 0.67 > 1.3 * tan(half fov) = 0.52
    sc.scales[0] = [0.5, 0.4, 0.45]
    sc.sh[1, 0] = [-4.0, 0.3, -4.0]
    p = oracle.project(sc, cam, 1)
    assert p["clamped"][0] & 8 and p["tiles_touched"][0] > 0
    assert p["clamped"][1] & 7 == 5
    fw = oracle.render_forward(sc, cam, mode=1, fragile_rel=1e-4)
    assert fw["fragile"].sum() == 0
    g = oracle.render_backward(sc, cam, G, mode=1, flags=2)
    assert np.abs(g["dsh"][1, 0, [0, 2]]).max() == 0 and abs(g["dsh"][1, 0, 1]) > 0
    for name, gname, i in [("means", "dmeans", 0), ("means", "dmeans", 1), ("means", "dmeans", 2), ("scales", "dscales", 0),
                           ("scales", "dscales", 2), ("quats", "dquats", 1)]:
        flat = getattr(sc, name).reshape(-1)
        h = 1e-6
        old = flat[i]
        flat[i] = old + h
        lp = loss(oracle, sc, cam, G)
        flat[i] = old - h
        lm = loss(oracle, sc, cam, G)
        flat[i] = old
        fd = (lp - lm) / (2 * h)
        assert abs(fd - g[gname].reshape(-1)[i]) <= 5e-5 * max(1e-3, abs(fd)), (name, i, fd, g[gname].reshape(-1)[i])


def test_saturated_alpha_has_zero_geometry_gradient(oracle):
    # one Gaussian whose o*exp(power) > 0.99 everywhere it matters on a pixel: alpha is the constant 0.99 there
    sc, cam, G = small_scene(n=1, seed=7, sh_degree=0)
    sc.opacities[:] = 0.999
    sc.scales[:] = 40.0
    fw = oracle.render_forward(sc, cam, mode=1)
    assert np.allclose(fw["out"][:, 13], 0.99)
    g = oracle.render_backward(sc, cam, G, mode=1, flags=2)
    assert np.abs(g["dopacities"]).max() == 0 and np.abs(g["dmean2d"]).max() == 0 and np.abs(g["dscales"]).max() == 0
    assert np.abs(g["dsem"]).max() > 0


# ---- reading C-17b: upstream gradients for the depth image (slot 3) and the alpha image (slot 5+F), flags bit 2
def geo_upstream(G, F, seed):
    rng = np.random.default_rng(900 + seed)
    G = G.copy()
    G[:, 3] = rng.standard_normal(G.shape[0])
    G[:, 5 + F] = rng.standard_normal(G.shape[0])
    return G


@pytest.mark.parametrize("seed,sh_degree,flags", [(0, 3, 6), (1, 1, 4), (2, 0, 6)])
def test_depth_alpha_upstream_matches_central_differences(oracle, seed, sh_degree, flags):
    # loss = <out, G> with G nonzero on EVERY slot the forward writes, incl. depth and alpha = 1 - T_final
    sc, cam, G = small_scene(seed=seed, sh_degree=sh_degree)
    G = geo_upstream(G, 8, seed)
    if not (flags & 2):
        G[:, 4:13] = 0          # without the coupling flag sem / unc do not reach geometry: leave them out of the loss
    g = oracle.render_backward(sc, cam, G, mode=1, flags=flags)
    rng = np.random.default_rng(300 + seed)
    for name, gname in FIELDS:
        flat = getattr(sc, name).reshape(-1)
        ana = g[gname].reshape(-1)
        for i in rng.choice(flat.size, size=min(40, flat.size), replace=False):
            h = 1e-6 * max(1.0, abs(flat[i])) if name != "scales" else 1e-6 * flat[i]
            old = flat[i]
            flat[i] = old + h
            lp = loss(oracle, sc, cam, G)
            flat[i] = old - h
            lm = loss(oracle, sc, cam, G)
            flat[i] = old
            fd = (lp - lm) / (2 * h)
            assert abs(fd - ana[i]) / max(1e-3, abs(fd), abs(ana[i])) < 2e-5, (name, int(i), fd, ana[i])


def test_depth_alpha_flag_identities(oracle):
    sc, cam, G = small_scene(seed=8)
    Gg = geo_upstream(G, 8, 8)
    base = oracle.render_backward(sc, cam, G, mode=0, flags=0)
    # the flag with zero depth / alpha upstream changes nothing; without the flag those slots are ignored
    same = oracle.render_backward(sc, cam, G, mode=0, flags=4)
    ignored = oracle.render_backward(sc, cam, Gg, mode=0, flags=0)
    with_geo = oracle.render_backward(sc, cam, Gg, mode=0, flags=4)
    for k in ("dmeans", "dscales", "dquats", "dopacities", "dsh", "dsem", "dunc", "dmean2d"):
        # (the oracle's OpenMP atomics add in a thread-dependent order: equal up to fp64 rounding)
        assert np.allclose(base[k], same[k], rtol=1e-12, atol=1e-15) and np.allclose(base[k], ignored[k], rtol=1e-12, atol=1e-15), k
    for k in ("dmeans", "dscales", "dquats", "dopacities", "dmean2d"):
        assert not np.allclose(base[k], with_geo[k], rtol=1e-3), k
    for k in ("dsh", "dsem", "dunc"):          # w G of the other channels never sees the depth / alpha upstream
        assert np.allclose(base[k], with_geo[k], rtol=1e-12, atol=1e-15), k
    # linearity in the upstream gradient: grad(G + Gd) = grad(G) + grad(Gd only)
    Gd = Gg - G
    only = oracle.render_backward(sc, cam, Gd, mode=0, flags=4)
    for k in ("dmeans", "dscales", "dquats", "dopacities", "dmean2d"):
        assert np.allclose(with_geo[k], base[k] + only[k], rtol=1e-10, atol=1e-13), k


def test_depth_alpha_single_gaussian_closed_form(oracle):
    # one isotropic Gaussian on the optical axis, identity camera: at the centre pixel power = 0, so alpha = o there;
    # alpha_out = o exp(power) and depth_out = alpha_out z at every pixel:
    #   d<alpha_out, Ga>/do = sum_p Ga_p exp(power_p);  d<depth_out, Gd>/dz (through the blended VALUE only) = sum_p Gd_p alpha_p
    n, F, size = 1, 8, 16
    sc = SimpleNamespace(means=np.array([[0.0, 0.0, 4.0]]), scales=np.full((1, 3), 0.3), quats=np.array([[1.0, 0, 0, 0]]),
                         opacities=np.array([0.6]), sh=np.zeros((1, 1, 3)), sem=np.zeros((1, F)), unc=np.zeros(1), sh_degree=0)
    cam = inputs.identity_camera(size, size, 20.0, 20.0, 8.5, 8.5)
    fw = oracle.render_forward(sc, cam, mode=1)
    a = fw["out"][:, 5 + F]
    sig2 = (20.0 * 0.3 / 4.0) ** 2 + 0.3
    yy, xx = np.mgrid[0:size, 0:size]
    expect = 0.6 * np.exp(-0.5 * ((xx - 8.0) ** 2 + (yy - 8.0) ** 2) / sig2).reshape(-1)
    expect[expect < 1 / 255] = 0
    assert np.allclose(a, expect, rtol=1e-12, atol=1e-15) and abs(a[8 * size + 8] - 0.6) < 1e-15
    assert np.allclose(fw["out"][:, 3], 4.0 * a, rtol=1e-12)
    rng = np.random.default_rng(1)
    G = np.zeros((size * size, inputs.channels(F)))
    G[:, 5 + F] = rng.standard_normal(size * size)
    g = oracle.render_backward(sc, cam, G, mode=1, flags=4)
    assert abs(g["dopacities"][0] - (G[:, 5 + F] * a / 0.6).sum()) < 1e-12
    G[:] = 0
    G[:, 3] = rng.standard_normal(size * size)
    g = oracle.render_backward(sc, cam, G, mode=1, flags=4)
    assert abs(g["ddepth"][0] - (G[:, 3] * a).sum()) < 1e-12
    assert abs(g["dopacities"][0] - (G[:, 3] * 4.0 * a / 0.6).sum()) < 1e-11
