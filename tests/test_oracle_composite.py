"""Pins for the oracle's per-pixel compositing ("rasterization and alpha blending" of s_G, Eq. 8;
:138 R_u) and its brute-force tile lists (BASELINE.json north_star (2)). Closed forms and invariants only."""
from types import SimpleNamespace

import numpy as np
import pytest

from paper_2311_18482_b200 import inputs
from test_oracle_projection import cam64, mk_scene


def test_single_isotropic_alpha_closed_form(oracle):
    # north_star: a single isotropic Gaussian's rendered alpha equals opacity * exp(-1/2 d^T Sigma'^-1 d)
    sigma, z, f, o = 0.3, 3.0, 64.0, 0.8
    cam = cam64(64, 64, f, f)
    sc = mk_scene([[0.1, -0.05, z]], [[sigma] * 3], [[1, 0, 0, 0]], opac=[o])
    r = oracle.render_forward(sc, cam, mode=1)
    alpha = r["out"][:, 5 + 8].reshape(64, 64)
    x, y = 0.1, -0.05
    a = sigma ** 2 * (f / z) ** 2 * (1 + x * x / z ** 2) + 0.3
    c = sigma ** 2 * (f / z) ** 2 * (1 + y * y / z ** 2) + 0.3
    b = sigma ** 2 * f * f * x * y / z ** 4
    inv = np.linalg.inv([[a, b], [b, c]])
    mu = np.array([f * x / z + 32 - 0.5, f * y / z + 32 - 0.5])
    jj, ii = np.mgrid[0:64, 0:64]
    d = np.stack([ii - mu[0], jj - mu[1]], -1)
    ref = o * np.exp(-0.5 * np.einsum("...i,ij,...j", d, inv, d))
    ref = np.where(ref < 1 / 255, 0.0, np.minimum(ref, 0.99))
    assert np.allclose(alpha, ref, atol=1e-12)
    assert (ref > 0).sum() > 300 and ref.max() < 0.99


def test_alpha_clamp_at_099(oracle):
    sc = mk_scene([[0, 0, 3.0]], [[0.5] * 3], [[1, 0, 0, 0]], opac=[0.999])
    r = oracle.render_forward(sc, cam64(), mode=1)
    assert r["out"][:, 13].max() == pytest.approx(0.99, abs=1e-15)


def _scene(n=300, seed=7):
    return inputs.tiny_scene(n=n, seed=seed)


def test_weights_plus_final_T_sum_to_one_and_ru_range(oracle):
    s = _scene()
    s.unc = np.ones_like(s.unc)            # R_u then equals sum of weights
    s.sem = np.ones_like(s.sem)
    r = oracle.render_forward(s, s.cameras[0])
    out = r["out"]
    assert np.allclose(out[:, 4 + 8], out[:, 5 + 8], atol=1e-13)          # sum w = 1 - T_final
    assert np.allclose(out[:, 4], out[:, 5 + 8], atol=1e-13)
    assert (out[:, 13] >= 0).all() and (out[:, 13] <= 1 - 1e-4 + 1e-12).all()  # stops before T < 1e-4
    s2 = _scene()
    r2 = oracle.render_forward(s2, s2.cameras[0])
    ru = r2["out"][:, 12]
    assert (ru >= 0).all() and (ru <= 1).all()                              # convex blend of u in [0,1]
    # background: rgb = blended + T_final * bg, nothing on sem/unc/depth
    cam_bg = inputs.identity_camera(64, 64, 64, 64, 32, 32, bg=(0.2, 0.5, 0.9))
    r3 = oracle.render_forward(s2, cam_bg)
    T = 1 - r2["out"][:, 13]
    assert np.allclose(r3["out"][:, 0:3], r2["out"][:, 0:3] + T[:, None] * np.array([0.2, 0.5, 0.9]), atol=1e-13)
    assert np.array_equal(r3["out"][:, 3:], r2["out"][:, 3:])


def test_transmittance_monotone_over_depth_prefixes(oracle):
    s = _scene(n=120, seed=11)
    cam = s.cameras[0]
    order = np.argsort(s.means[:, 2], kind="stable")
    prev = np.zeros(64 * 64)
    for k in (10, 40, 80, 120):
        keep = order[:k]
        sub = SimpleNamespace(means=s.means[keep], scales=s.scales[keep], quats=s.quats[keep], opacities=s.opacities[keep],
                              sh=s.sh[keep], sem=s.sem[keep], unc=s.unc[keep], sh_degree=0)
        a = oracle.render_forward(sub, cam)["out"][:, 13]
        assert (a >= prev - 1e-15).all()  # adding farther Gaussians never raises T
        prev = a


def test_input_permutation_invariance(oracle):
    s = _scene(n=250, seed=13)
    cam = s.cameras[0]
    a = oracle.render_forward(s, cam)
    perm = np.random.default_rng(0).permutation(s.n)
    sp = SimpleNamespace(means=s.means[perm], scales=s.scales[perm], quats=s.quats[perm], opacities=s.opacities[perm],
                         sh=s.sh[perm], sem=s.sem[perm], unc=s.unc[perm], sh_degree=0)
    b = oracle.render_forward(sp, cam)
    assert np.allclose(a["out"], b["out"], atol=1e-14)  # depths are distinct, so the order is unique
    assert np.array_equal(a["n_contrib"], b["n_contrib"])


def test_non_overlapping_gaussians_are_depth_independent(oracle):
    # four small well-separated blobs: swapping their depths (with scale ~ z so footprints stay equal) changes nothing
    cam = cam64()
    xs = np.array([[-0.25, -0.25], [0.25, -0.25], [-0.25, 0.25], [0.25, 0.25]])
    def build(z):
        means = np.concatenate([xs * z[:, None], z[:, None]], 1)
        return mk_scene(means, np.repeat(0.01 * z[:, None], 3, 1), [[1, 0, 0, 0]] * 4, opac=[0.9, 0.8, 0.7, 0.6])
    a = build(np.array([2.0, 3.0, 4.0, 5.0]))
    b = build(np.array([5.0, 2.0, 3.0, 4.0]))
    for sc in (a, b):
        sc.sem = np.arange(32, dtype=np.float64).reshape(4, 8)
        sc.unc = np.array([0.1, 0.2, 0.3, 0.4])
    ra, rb = oracle.render_forward(a, cam, mode=1)["out"], oracle.render_forward(b, cam, mode=1)["out"]
    keep = [c for c in range(16) if c != 3]  # every channel except depth itself
    assert np.allclose(ra[:, keep], rb[:, keep], atol=1e-9)
    assert ra[:, 13].max() > 0.5


def test_tile_lists_brute_force(oracle):
    s = _scene(n=400, seed=17)
    cam = inputs.identity_camera(72, 56, 64, 64, 36, 28)  # ragged: 72x56 -> 5x4 tiles
    p = oracle.project(s, cam, 0)
    tl = oracle.tile_lists(p, cam)
    gx, gy = 5, 4
    depth_bits = p["depth"].astype(np.float32).view(np.uint32)
    pos = 0
    for t in range(gx * gy):
        tx, ty = t % gx, t // gx
        members = [i for i in range(s.n) if p["tiles_touched"][i] and p["rect"][i, 0] <= tx < p["rect"][i, 2]
                   and p["rect"][i, 1] <= ty < p["rect"][i, 3]]
        members.sort(key=lambda i: (int(depth_bits[i]), i))
        lo, hi = tl["ranges"][t]
        if not members:
            assert (lo, hi) == (0, 0)
            continue
        assert (lo, hi) == (pos, pos + len(members))
        assert list(tl["vals"][lo:hi]) == members
        assert (tl["keys"][lo:hi] >> np.uint64(32) == t).all()
        assert list(tl["keys"][lo:hi] & np.uint64(0xFFFFFFFF)) == [int(depth_bits[i]) for i in members]
        pos = hi
    assert pos == tl["D"] == int(p["tiles_touched"].sum())
    assert (np.diff(tl["keys"].astype(np.uint64)) >= 0).all()


def test_n_contrib_is_position_in_tile_list(oracle):
    s = _scene(n=400, seed=19)
    cam = s.cameras[0]
    r = oracle.render_forward(s, cam)
    tl = oracle.tile_lists(r["proj"], cam)
    nc = r["n_contrib"].reshape(64, 64)
    for ty in range(4):
        for tx in range(4):
            lo, hi = tl["ranges"][ty * 4 + tx]
            blk = nc[ty * 16:(ty + 1) * 16, tx * 16:(tx + 1) * 16]
            assert blk.max() <= hi - lo
    assert nc.max() > 0


def test_forward_linearity_links_forward_and_backward(oracle):
    # out . G = sum_k (dL/dv_k . v_k) + T_final * bg . G  (compositing is linear in the blended values)
    s = _scene(n=200, seed=23)
    cam = inputs.identity_camera(64, 64, 64, 64, 32, 32, bg=(0.3, 0.1, 0.7))
    G = inputs.upstream_gradient(s, 0).reshape(-1, 16).astype(np.float64)
    r = oracle.render_forward(s, cam)
    g = oracle.composite_backward(r["proj"], s.sem, s.unc, cam, G)
    lhs = (r["out"] * G).sum()
    T = 1 - r["out"][:, 13]
    rhs = (g["drgb"] * r["proj"]["rgb"]).sum() + (g["dsem"] * s.sem).sum() + (g["dunc"] * s.unc).sum() \
        + (T[:, None] * np.array([0.3, 0.1, 0.7]) * G[:, 0:3]).sum()
    assert lhs == pytest.approx(rhs, rel=1e-12)
