"""Pins for the oracle's per-Gaussian projection (steps 1-8) — closed forms, invariants and library
routines; nothing here re-types the oracle's own formula sequence.

PAPER.md:56-58 (Eq. 1: position p, covariance Sigma, colour c, opacity alpha; camera pose) names the quantities;
the EWA reading (C-1..C-11) fixes the constants (0.3 dilation, 3-sigma radius, 16x16 tiles)."""
import math
from types import SimpleNamespace

import numpy as np
import pytest
from scipy.spatial.transform import Rotation

from paper_2311_18482_b200 import inputs


def mk_scene(means, scales, quats, opac=None, sh=None, sh_degree=0, F=8):
    n = len(means)
    K = (sh_degree + 1) ** 2
    return SimpleNamespace(
        means=np.asarray(means, np.float64).reshape(n, 3), scales=np.asarray(scales, np.float64).reshape(n, 3),
        quats=np.asarray(quats, np.float64).reshape(n, 4),
        opacities=np.full(n, 0.5) if opac is None else np.asarray(opac, np.float64),
        sh=np.zeros((n, K, 3)) if sh is None else np.asarray(sh, np.float64).reshape(n, K, 3),
        sem=np.zeros((n, F)), unc=np.zeros(n), sh_degree=sh_degree)


def cam64(W=64, H=64, fx=64.0, fy=64.0):
    return inputs.identity_camera(W, H, fx, fy, W / 2.0, H / 2.0)


@pytest.mark.parametrize("mode,tol", [(0, 2e-6), (1, 1e-13)])
def test_isotropic_on_axis_closed_form(oracle, mode, tol):
    # isotropic Gaussian on the optical axis: Sigma' = diag((fx s/z)^2 + 0.3, (fy s/z)^2 + 0.3)
    sigma, z, fx, fy = 0.05, 3.0, 80.0, 60.0
    cam = cam64(64, 48, fx, fy)
    p = oracle.project(mk_scene([[0, 0, z]], [[sigma] * 3], [[1, 0, 0, 0]]), cam, mode)
    a, c = (fx * sigma / z) ** 2 + 0.3, (fy * sigma / z) ** 2 + 0.3
    A, B, C, o = p["conic_opacity"][0]
    assert A == pytest.approx(1 / a, rel=tol) and C == pytest.approx(1 / c, rel=tol) and abs(B) < 1e-12
    assert p["radius"][0] == math.ceil(3 * math.sqrt(max(a, c)))
    assert p["mean2d"][0] == pytest.approx([32 - 0.5, 24 - 0.5], abs=1e-6)
    assert p["depth"][0] == z and o == 0.5


@pytest.mark.parametrize("mode,tol", [(0, 3e-5), (1, 1e-12)])
def test_isotropic_off_axis_closed_form(oracle, mode, tol):
    # Sigma' = s^2 J J^T + 0.3 I,  JJ^T_00 = (fx/z)^2 (1 + x^2/z^2), JJ^T_01 = fx fy x y / z^4
    s, fx, fy = 0.04, 70.0, 90.0
    x, y, z = 0.5, -0.3, 2.5
    cam = cam64(96, 96, fx, fy)
    p = oracle.project(mk_scene([[x, y, z]], [[s] * 3], [[1, 0, 0, 0]]), cam, mode)
    a = s * s * (fx / z) ** 2 * (1 + x * x / z ** 2) + 0.3
    c = s * s * (fy / z) ** 2 * (1 + y * y / z ** 2) + 0.3
    b = s * s * fx * fy * x * y / z ** 4
    inv = np.linalg.inv(np.array([[a, b], [b, c]]))
    A, B, C, _ = p["conic_opacity"][0]
    assert [A, B, C] == pytest.approx([inv[0, 0], inv[0, 1], inv[1, 1]], rel=tol)
    lam = 0.5 * (a + c) + math.sqrt(max(0.1, (0.5 * (a + c)) ** 2 - (a * c - b * b)))
    assert p["radius"][0] == math.ceil(3 * math.sqrt(lam))
    assert p["mean2d"][0] == pytest.approx([fx * x / z + 48 - 0.5, fy * y / z + 48 - 0.5], rel=1e-6)


def test_isotropic_rotation_invariance(oracle):
    rng = np.random.default_rng(0)
    q = rng.standard_normal((16, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    q[0] = [1, 0, 0, 0]
    means = np.tile([[0.3, 0.2, 3.0]], (16, 1))
    p = oracle.project(mk_scene(means, np.full((16, 3), 0.07), q), cam64(), 1)
    assert np.allclose(p["conic_opacity"], p["conic_opacity"][0], rtol=1e-12)
    assert (p["radius"] == p["radius"][0]).all()


@pytest.mark.parametrize("mode,tol", [(0, 2e-4), (1, 1e-11)])
def test_anisotropic_against_library_rotation(oracle, mode, tol):
    # Sigma = R S S^T R^T with R from scipy (library routine), general camera pose
    rng = np.random.default_rng(1)
    n = 64
    q = rng.standard_normal((n, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    s = np.exp(rng.normal(-2.5, 0.5, (n, 3)))
    means = rng.normal(0, 0.4, (n, 3))
    cam = inputs.look_at_camera([1.0, 2.0, -3.0], 128, 96, 150.0, 140.0, 64.0, 48.0)
    sc = mk_scene(np.float32(means), np.float32(s), q)  # q unit in fp64 (mode 0 rounds it to fp32 itself)
    p = oracle.project(sc, cam, mode)
    W = cam.world_to_cam.astype(np.float64).reshape(3, 4)
    Rm = Rotation.from_quat(q[:, [1, 2, 3, 0]]).as_matrix()  # scipy wants x,y,z,w
    for i in range(n):
        t = W[:, :3] @ sc.means[i] + W[:, 3]
        Sig = Rm[i] @ np.diag(sc.scales[i] ** 2) @ Rm[i].T
        J = np.array([[cam.fx / t[2], 0, -cam.fx * t[0] / t[2] ** 2], [0, cam.fy / t[2], -cam.fy * t[1] / t[2] ** 2]])
        cov = J @ W[:, :3] @ Sig @ W[:, :3].T @ J.T + 0.3 * np.eye(2)
        inv = np.linalg.inv(cov)
        A, B, C, _ = p["conic_opacity"][i]
        assert [A, B, C] == pytest.approx([inv[0, 0], inv[0, 1], inv[1, 1]], rel=tol,
                                          abs=tol * max(abs(inv[0, 0]), abs(inv[1, 1])))
        assert p["depth"][i] == pytest.approx(t[2], rel=1e-6)


def test_rigid_motion_invariance(oracle):
    # moving world and camera together leaves every projected quantity unchanged
    s = inputs.tiny_scene(n=200, seed=3)
    cam0 = s.cameras[0]
    Rg = Rotation.from_rotvec([0.3, -0.5, 0.2]).as_matrix()
    tg = np.array([0.4, -1.0, 2.0])
    means1 = s.means.astype(np.float64) @ Rg.T + tg
    qg = Rotation.from_matrix(Rg)
    s.quats = s.quats.astype(np.float64)
    s.quats /= np.linalg.norm(s.quats, axis=1, keepdims=True)  # unit in fp64: the library rotation normalises, the oracle does not (C-2)
    q0 = Rotation.from_quat(s.quats[:, [1, 2, 3, 0]])
    q1 = (qg * q0).as_quat()[:, [3, 0, 1, 2]]
    W0 = cam0.world_to_cam.astype(np.float64).reshape(3, 4)
    R1 = W0[:, :3] @ Rg.T
    t1 = W0[:, 3] - R1 @ tg
    cam1 = SimpleNamespace(width=cam0.width, height=cam0.height, fx=cam0.fx, fy=cam0.fy, cx=cam0.cx, cy=cam0.cy,
                           background=cam0.background,
                           as_vector=lambda: np.concatenate([[cam0.fx, cam0.fy, cam0.cx, cam0.cy],
                                                             np.concatenate([R1, t1[:, None]], 1).reshape(12),
                                                             [0.2, 0, 0, 0]]))
    a = oracle.project(s, cam0, 1)
    s1 = SimpleNamespace(means=means1, scales=s.scales, quats=q1, opacities=s.opacities, sh=s.sh, sem=s.sem, unc=s.unc,
                         sh_degree=0)
    b = oracle.project(s1, cam1, 1)
    assert np.allclose(a["conic_opacity"], b["conic_opacity"], rtol=1e-9, atol=1e-12)
    assert np.allclose(a["mean2d"], b["mean2d"], atol=1e-9)
    assert (a["rect"] == b["rect"]).all() and (a["radius"] == b["radius"]).all()


def test_culling_and_rect(oracle):
    cam = cam64()
    means = [[0, 0, 0.2], [0, 0, 0.2001], [0, 0, -1.0], [50.0, 0, 3.0], [0, 0, 3.0]]
    p = oracle.project(mk_scene(means, np.full((5, 3), 0.01), np.tile([[1, 0, 0, 0]], (5, 1))), cam, 0)
    assert list(p["tiles_touched"] > 0) == [False, True, False, False, True]  # z<=near, behind, off-screen culled
    # rect is the conservative AABB of the 3-sigma disc in 16-pixel tiles, clamped to the grid
    r = p["radius"][4]
    mx, my = p["mean2d"][4]
    x0, y0, x1, y1 = p["rect"][4]
    assert x0 == max(0, math.floor((mx - r) / 16)) and x1 == min(4, math.floor((mx + r + 15) / 16))
    assert y0 == max(0, math.floor((my - r) / 16)) and y1 == min(4, math.floor((my + r + 15) / 16))
    assert p["tiles_touched"][4] == (x1 - x0) * (y1 - y0)


def _complex_sph_harm(l, m, polar, azim):
    import scipy.special as sp
    if hasattr(sp, "sph_harm_y"):
        return sp.sph_harm_y(l, m, polar, azim)
    return sp.sph_harm(m, l, azim, polar)


def test_sh_basis_against_scipy(oracle):
    # real basis = sqrt2*Im(Y_l^|m|) (m<0), Y_l^0, sqrt2*Re(Y_l^m) (m>0) of the Condon-Shortley complex harmonics
    rng = np.random.default_rng(2)
    d = rng.standard_normal((50, 3))
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    polar, azim = np.arccos(d[:, 2]), np.arctan2(d[:, 1], d[:, 0])
    b = oracle.sh_basis(d, 3)
    k = 0
    for l in range(4):
        for m in range(-l, l + 1):
            Y = _complex_sph_harm(l, abs(m), polar, azim)
            ref = math.sqrt(2) * Y.imag if m < 0 else (Y.real if m == 0 else math.sqrt(2) * Y.real)
            assert np.allclose(b[:, k], ref, atol=1e-12), (l, m)
            k += 1


def test_sh_gram_matrix_by_quadrature(oracle):
    # orthonormality on the sphere: Gauss-Legendre in cos(polar) x uniform azimuth (exact for degree <= 6 products)
    x, wx = np.polynomial.legendre.leggauss(16)
    na = 32
    az = 2 * np.pi * np.arange(na) / na
    ct, ph = np.meshgrid(x, az, indexing="ij")
    st = np.sqrt(1 - ct ** 2)
    d = np.stack([st * np.cos(ph), st * np.sin(ph), ct], -1).reshape(-1, 3)
    w = (wx[:, None] * np.full(na, 2 * np.pi / na)[None, :]).reshape(-1)
    b = oracle.sh_basis(d, 3)
    gram = (b * w[:, None]).T @ b
    assert np.allclose(gram, np.eye(16), atol=1e-12)


def test_degree0_colour_is_view_independent(oracle):
    s = inputs.tiny_scene(n=50, seed=5)
    c0 = oracle.project(s, s.cameras[0], 0)["rgb"]
    cam1 = inputs.look_at_camera([0.5, 0.5, -2.0], 64, 64, 64, 64, 32, 32)
    c1 = oracle.project(s, cam1, 0)["rgb"]
    vis = (oracle.project(s, cam1, 0)["tiles_touched"] > 0) & (oracle.project(s, s.cameras[0], 0)["tiles_touched"] > 0)
    assert vis.sum() > 5 and np.array_equal(c0[vis], c1[vis])
    # reading C-12: the DC coefficient stores (rgb - 0.5)/Y0, so the colour is 0.5 + Y0*c
    assert np.allclose(c0[vis], 0.5 + 0.28209479177387814 * s.sh[vis, 0, :], atol=1e-6)


def test_colour_clamp_flags(oracle):
    sh = np.zeros((2, 1, 3))
    sh[0, 0] = [-3.0, 0.0, 1.0]
    sh[1, 0] = [0.5, -2.0, -2.0]
    p = oracle.project(mk_scene([[0, 0, 3.0], [0.1, 0, 3.0]], np.full((2, 3), 0.05), [[1, 0, 0, 0]] * 2, sh=sh), cam64(), 0)
    assert list(p["clamped"] & 7) == [1, 6]
    assert p["rgb"][0][0] == 0 and p["rgb"][1][1] == 0 and p["rgb"][1][2] == 0
