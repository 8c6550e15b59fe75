"""Pins for the oracle's CONDITIONING outputs (reading G-4): composite_backward_abs / project_backward_abs /
gradient_abs give, for every gradient element, the sum of the absolute values of the single products behind it. They are
not part of the method (PAPER.md has no such quantity), but tests/gradcheck.py turns them into the third arm of the gradient
parity bound, so a slip there (a missing fabs, a suffix added twice, a wrong |J| column) would loosen every gradient test
without failing anything. Pinned here against what the mathematics fixes:

  (a) triangle inequality: abs >= |gradient| for every element of every array, every flag combination;
  (b) equality where every product has one sign (one Gaussian, non-negative upstream gradient and values, black background);
  (c) an explicit expansion in numpy, product by product, on an 8-Gaussian 16x16 scene (own walk over the contributors from
      the projected 2D quantities: no call into the oracle's compositor);
  (d) project_backward_abs = |J| abs2d with J the Jacobian of the (linear) projection backward taken by central differences
      around a random point."""
from types import SimpleNamespace

import numpy as np
import pytest

from paper_2311_18482_b200 import inputs

KEYS8 = ("dmeans", "dscales", "dquats", "dopacities", "dsh", "dsem", "dunc", "dmean2d")


def scene_of(n, seed, size, sh_degree=1, F=8, bg=(0.2, 0.4, 0.6), focal=None, log_scale=-2.0):
    rng = np.random.default_rng(seed)
    means = np.concatenate([rng.uniform(-0.5, 0.5, (n, 2)), rng.uniform(-0.8, 0.8, (n, 1))], 1)
    q = rng.standard_normal((n, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    K = (sh_degree + 1) ** 2
    sc = SimpleNamespace(means=means, scales=np.exp(rng.normal(log_scale, 0.4, (n, 3))), quats=q,
                         opacities=1 / (1 + np.exp(-rng.normal(0.5, 1, n))), sh=rng.normal(0, 0.3, (n, K, 3)),
                         sem=rng.standard_normal((n, F)), unc=rng.uniform(0, 1, n), sh_degree=sh_degree)
    f = focal if focal is not None else 1.3 * size
    cam = inputs.look_at_camera([0.4, -0.3, -3.0], size, size, f, 1.1 * f, size / 2.0, size / 2.0, bg=bg)
    return sc, cam, rng


def upstream(rng, npix, F, depth_alpha):
    G = np.zeros((npix, inputs.channels(F)))
    G[:, 0:3] = rng.standard_normal((npix, 3))
    G[:, 4:4 + F + 1] = rng.standard_normal((npix, F + 1))
    if depth_alpha:
        G[:, 3] = rng.standard_normal(npix)
        G[:, 5 + F] = rng.standard_normal(npix)
    return G


@pytest.mark.parametrize("flags", [0, 2, 4, 6])
def test_abs_sums_dominate_the_gradients(oracle, flags):
    # (a) |sum of terms| <= sum of |terms|, for all eight arrays the GPU parity check uses and the 2D intermediates
    sc, cam, rng = scene_of(40, seed=flags, size=32, sh_degree=3)
    G = upstream(rng, 32 * 32, 8, depth_alpha=bool(flags & 4))
    res = oracle.render_backward(sc, cam, G, mode=0, flags=flags, with_abs=True)
    assert sum(np.abs(res[k]).sum() > 0 for k in KEYS8) == 8
    for k in KEYS8:
        g, a = np.abs(res[k]), res["abs"][k]
        assert g.shape == a.shape
        assert (a >= g * (1 - 1e-12)).all(), k
        assert (a[g > 0] > 0).all(), k
    g2 = oracle.composite_backward(res["proj"], sc.sem, sc.unc, cam, G, flags=flags, with_abs=True)
    for k in ("dopac", "dconic", "dmean2d", "drgb", "dsem", "dunc", "ddepth"):
        assert (g2["abs"][k] >= np.abs(g2[k]) * (1 - 1e-12)).all(), k
    # some cancellation really happens in this scene (else (a) would not distinguish abs from |gradient|)
    assert (g2["abs"]["dmean2d"] > 1.5 * np.abs(g2["dmean2d"])).any()


def test_abs_sums_equal_the_gradients_when_no_term_cancels(oracle):
    # (b) one Gaussian, black background, upstream gradient >= 0 on every channel, values >= 0: with nothing behind it the
    # suffix is zero, dL/dalpha = sum_ch G_ch T v_ch >= 0, and every product of dopac, drgb, dsem, dunc, dconic_xx, dconic_yy
    # has one sign over all pixels. (dconic_xy and dmean2d change sign with dx, dy: there abs > |gradient|.)
    sc, cam, rng = scene_of(1, seed=11, size=32, sh_degree=0, bg=(0.0, 0.0, 0.0), log_scale=-1.6)
    sc.means[:] = [[0.05, -0.03, 0.0]]
    sc.sh[:] = 0.8            # rgb = 0.5 + Y0 * 0.8 > 0
    sc.sem = np.abs(sc.sem)
    sc.opacities[:] = 0.7
    G = np.abs(upstream(rng, 32 * 32, 8, depth_alpha=False))
    proj = oracle.project(sc, cam, 0)
    assert proj["tiles_touched"][0] > 0
    for flags in (0, 2):
        g = oracle.composite_backward(proj, sc.sem, sc.unc, cam, G, flags=flags, with_abs=True)
        a = g["abs"]
        assert g["dopac"][0] > 0
        for k in ("dopac", "drgb", "dsem", "dunc"):
            np.testing.assert_allclose(a[k], np.abs(g[k]), rtol=1e-12, atol=0)
        np.testing.assert_allclose(a["dconic"][:, [0, 2]], np.abs(g["dconic"][:, [0, 2]]), rtol=1e-12, atol=0)
        assert a["dconic"][0, 1] > 1.5 * abs(g["dconic"][0, 1])
        assert (a["dmean2d"][0] > 1.5 * np.abs(g["dmean2d"][0])).all()


def expand_abs(proj, sem, unc, cam, G, flags):
    """Every product of the compositor's reverse mode, written out one by one, by absolute value (SURVEY.md 8(c) forward
    walk + "Backward"). One tile: every visible Gaussian is a member of every pixel's list."""
    n, F = sem.shape
    couple, geo = bool(flags & 2), bool(flags & 4)
    vis = np.flatnonzero(proj["tiles_touched"] > 0)
    order = vis[np.lexsort((vis, proj["depth"][vis]))]
    out = dict(dopac=np.zeros(n), dconic=np.zeros((n, 3)), dmean2d=np.zeros((n, 2)), drgb=np.zeros((n, 3)),
               dsem=np.zeros((n, F)), dunc=np.zeros(n), ddepth=np.zeros(n))
    bg = np.asarray(cam.background, dtype=np.float64)
    # channel table: (slot in G, per-Gaussian value array, background) for every channel whose gradient reaches alpha
    for py in range(cam.height):
        for px in range(cam.width):
            g_up = G[py * cam.width + px]
            T, rec = 1.0, []
            for g in order:
                A, B, C, o = proj["conic_opacity"][g]
                dx, dy = px - proj["mean2d"][g, 0], py - proj["mean2d"][g, 1]
                power = -0.5 * (A * dx * dx + C * dy * dy) - B * dx * dy
                if power > 0:
                    continue
                gauss = np.exp(power)
                alpha = min(0.99, o * gauss)
                if alpha < 1.0 / 255.0:
                    continue
                if T * (1 - alpha) < 1e-4:
                    break
                rec.append((g, alpha, T, gauss, dx, dy, o * gauss > 0.99))
                T = T * (1 - alpha)
            T_final = T
            chans = [(c, proj["rgb"][:, c], bg[c]) for c in range(3)]
            if couple:
                chans += [(4 + f, sem[:, f], 0.0) for f in range(F)] + [(4 + F, unc, 0.0)]
            if geo:
                chans += [(3, proj["depth"], 0.0), (5 + F, np.zeros(n), -1.0)]
            for m, (g, alpha, Tk, gauss, dx, dy, clamped) in enumerate(rec):
                w = alpha * Tk
                for c in range(3):
                    out["drgb"][g, c] += abs(w * g_up[c])
                for f in range(F):
                    out["dsem"][g, f] += abs(w * g_up[4 + f])
                out["dunc"][g] += abs(w * g_up[4 + F])
                if geo:
                    out["ddepth"][g] += abs(w * g_up[3])
                if clamped:
                    continue
                products = []
                for slot, val, back in chans:
                    products.append(g_up[slot] * Tk * val[g])
                    for (gj, aj, Tj, *_rest) in rec[m + 1:]:
                        products.append(-g_up[slot] * (aj * Tj) * val[gj] / (1 - alpha))
                    products.append(-g_up[slot] * T_final * back / (1 - alpha))
                A, B, C, o = proj["conic_opacity"][g]
                for pr in products:
                    out["dopac"][g] += abs(gauss * pr)
                    dpow = o * gauss * pr
                    out["dconic"][g] += np.abs([dpow * 0.5 * dx * dx, dpow * dx * dy, dpow * 0.5 * dy * dy])
                    out["dmean2d"][g, 0] += abs(dpow * A * dx) + abs(dpow * B * dy)
                    out["dmean2d"][g, 1] += abs(dpow * C * dy) + abs(dpow * B * dx)
    return out


@pytest.mark.parametrize("flags", [0, 2, 6])
def test_abs_sums_equal_an_explicit_expansion(oracle, flags):
    # (c) 8 Gaussians on one 16x16 tile, several contributors per pixel (suffix terms), a coloured background
    sc, cam, rng = scene_of(8, seed=21, size=16, sh_degree=1, log_scale=-1.7)
    G = upstream(rng, 16 * 16, 8, depth_alpha=bool(flags & 4))
    proj = oracle.project(sc, cam, 0)
    fw = oracle.composite_forward(proj, sc.sem, sc.unc, cam)
    assert (proj["tiles_touched"] > 0).sum() >= 6 and fw["n_contrib"].max() >= 4
    got = oracle.composite_backward_abs(proj, sc.sem, sc.unc, cam, G, flags=flags)
    want = expand_abs(proj, np.asarray(sc.sem, float), np.asarray(sc.unc, float), cam, G, flags)
    for k in want:
        if k == "ddepth" and not flags & 4:
            continue
        assert want[k].sum() > 0, k
        np.testing.assert_allclose(got[k], want[k], rtol=1e-10, atol=1e-300, err_msg=k)


def test_projection_abs_is_the_absolute_jacobian_times_abs2d(oracle):
    # (d) the projection backward is linear in (dconic, dmean2d, drgb, ddepth) per Gaussian: its Jacobian by central
    # differences around a random point, then |J| abs2d, against project_backward_abs
    sc, cam, rng = scene_of(3, seed=31, size=32, sh_degree=2)
    n = 3
    base = dict(dconic=rng.standard_normal((n, 3)), dmean2d=rng.standard_normal((n, 2)), drgb=rng.standard_normal((n, 3)),
                ddepth=rng.standard_normal(n))
    abs2d = dict(dconic=rng.uniform(0.5, 2, (n, 3)), dmean2d=rng.uniform(0.5, 2, (n, 2)), drgb=rng.uniform(0.5, 2, (n, 3)),
                 ddepth=rng.uniform(0.5, 2, n))
    want = None
    h = 0.25
    for key, width in (("dconic", 3), ("dmean2d", 2), ("drgb", 3), ("ddepth", 1)):
        for j in range(width):
            hi = {k: v.copy() for k, v in base.items()}
            lo = {k: v.copy() for k, v in base.items()}
            hi[key].reshape(n, -1)[:, j] += h
            lo[key].reshape(n, -1)[:, j] -= h
            fh, fl = oracle.project_backward(sc, cam, hi, 0), oracle.project_backward(sc, cam, lo, 0)
            col = {k: (fh[k] - fl[k]) / (2 * h) for k in fh}
            if want is None:
                want = {k: np.zeros_like(v) for k, v in col.items()}
            a = abs2d[key].reshape(n, -1)[:, j]
            for k in want:
                want[k] += np.abs(col[k]) * a.reshape((n,) + (1,) * (want[k].ndim - 1))
    got = oracle.project_backward_abs(sc, cam, abs2d, 0)
    for k in ("dmeans", "dscales", "dquats", "dsh"):
        assert want[k].sum() > 0
        np.testing.assert_allclose(got[k], want[k], rtol=1e-8, atol=1e-12, err_msg=k)
    # and gradient_abs passes the 2D sums through unchanged where no projection is involved
    a2 = dict(abs2d, dopac=rng.uniform(0.5, 2, n), dsem=rng.uniform(0.5, 2, (n, 8)), dunc=rng.uniform(0.5, 2, n))
    full = oracle.gradient_abs(sc, cam, a2, 0)
    for k8, k2 in (("dopacities", "dopac"), ("dsem", "dsem"), ("dunc", "dunc"), ("dmean2d", "dmean2d")):
        assert np.array_equal(full[k8], a2[k2])
    for k in ("dmeans", "dscales", "dquats", "dsh"):
        assert np.array_equal(full[k], got[k])
