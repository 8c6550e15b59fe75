"""ctypes wrapper around oracle/legs_oracle.cpp — TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
It imports nothing from the CUDA package; scenes and cameras are duck-typed (attributes means, scales, quats,
opacities, sh, sem, unc, sh_degree / width, height, as_vector()).
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "legs_oracle.cpp")
_LIB = os.path.join(_HERE, "liblegs_oracle.so")
_lib = None

FRAGILE_REL = 1e-5  # DESIGN.md reading G-3


def build(force: bool = False) -> str:
    """g++ -O2 -ffp-contract=off (rule P-0: no FMA contraction, no fast-math), OpenMP over pixels."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-o", _LIB, _SRC]
        subprocess.run(cmd, check=True)
    return _LIB


def _c(a, dtype):
    return np.ascontiguousarray(a, dtype=dtype)


def _p(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_LIB)
        _lib.oracle_tile_lists.restype = ctypes.c_int64
    return _lib


def channels(F: int) -> int:
    return (3 + 1 + F + 1 + 1 + 3) // 4 * 4


def cam_vector(cam) -> np.ndarray:
    return _c(cam.as_vector(), np.float64)


def project(scene, cam, mode: int = 0) -> dict:
    """Steps 1-8 for every Gaussian. mode 0: rule P-0 fp32 (values exactly representable in float32)."""
    n = scene.means.shape[0]
    K = scene.sh.shape[1]
    out = dict(
        depth=np.zeros(n), radius=np.zeros(n, np.int32), rect=np.zeros((n, 4), np.int32), mean2d=np.zeros((n, 2)),
        conic_opacity=np.zeros((n, 4)), rgb=np.zeros((n, 3)), clamped=np.zeros(n, np.uint8),
        tiles_touched=np.zeros(n, np.uint32))
    means, scales, quats = _c(scene.means, np.float64), _c(scene.scales, np.float64), _c(scene.quats, np.float64)
    opac, sh = _c(scene.opacities, np.float64), _c(scene.sh, np.float64)
    cv = cam_vector(cam)
    rc = lib().oracle_project(ctypes.c_int(mode), ctypes.c_int64(n), ctypes.c_int(scene.sh_degree), ctypes.c_int(K),
                              _p(means), _p(scales), _p(quats), _p(opac), _p(sh), _p(cv), ctypes.c_int(cam.width),
                              ctypes.c_int(cam.height), _p(out["depth"]), _p(out["radius"]), _p(out["rect"]),
                              _p(out["mean2d"]), _p(out["conic_opacity"]), _p(out["rgb"]), _p(out["clamped"]),
                              _p(out["tiles_touched"]))
    assert rc == 0
    return out


def tile_grid(cam):
    return (cam.width + 15) // 16, (cam.height + 15) // 16


def tile_lists(proj: dict, cam) -> dict:
    gx, gy = tile_grid(cam)
    n = proj["depth"].shape[0]
    args = (ctypes.c_int64(n), _p(proj["depth"]), _p(proj["rect"]), _p(proj["tiles_touched"]), ctypes.c_int(gx),
            ctypes.c_int(gx * gy))
    D = lib().oracle_tile_lists(*args, None, None, None)
    keys, vals = np.zeros(D, np.uint64), np.zeros(D, np.uint32)
    ranges = np.zeros((gx * gy, 2), np.uint32)
    D2 = lib().oracle_tile_lists(*args, _p(keys), _p(vals), _p(ranges))
    assert D2 == D
    return dict(D=int(D), keys=keys, vals=vals, ranges=ranges)


def _pix(pix, cam):
    if pix is None:
        return None, cam.width * cam.height
    pix = _c(pix, np.int64)
    return pix, pix.shape[0]


def composite_forward(proj: dict, sem, unc, cam, pix=None, fragile_rel: float = FRAGILE_REL) -> dict:
    sem, unc = _c(sem, np.float64), _c(unc, np.float64)
    n, F = sem.shape
    CH = channels(F)
    pix, npix = _pix(pix, cam)
    out = np.zeros((npix, CH))
    n_contrib, n_walked = np.zeros(npix, np.uint32), np.zeros(npix, np.uint32)
    fragile, counters = np.zeros(npix, np.uint8), np.zeros(2, np.uint64)
    bg = _c(cam.background, np.float64)
    rc = lib().oracle_composite_forward(
        ctypes.c_int64(n), ctypes.c_int(F), _p(proj["depth"]), _p(proj["rect"]), _p(proj["tiles_touched"]),
        _p(proj["mean2d"]), _p(proj["conic_opacity"]), _p(proj["rgb"]), _p(sem), _p(unc), ctypes.c_int(cam.width),
        ctypes.c_int(cam.height), _p(bg), ctypes.c_int64(npix), _p(pix), ctypes.c_double(fragile_rel), _p(out),
        _p(n_contrib), _p(n_walked), _p(fragile), _p(counters))
    assert rc == 0
    return dict(out=out, n_contrib=n_contrib, n_walked=n_walked, fragile=fragile, examined=int(counters[0]),
                blended=int(counters[1]))


def composite_backward(proj: dict, sem, unc, cam, dL_dpix, pix=None, flags: int = 0, with_abs: bool = False) -> dict:
    """Plain reverse mode over the recorded contributors (SURVEY.md 8(c) "Backward").
    with_abs: also return `abs` = composite_backward_abs(...) (the conditioning of every sum, reading G-4; a function of
    its own, not part of the method)."""
    sem, unc = _c(sem, np.float64), _c(unc, np.float64)
    n, F = sem.shape
    CH = channels(F)
    pix, npix = _pix(pix, cam)
    g = _c(dL_dpix, np.float64).reshape(npix, CH)
    out = dict(dopac=np.zeros(n), dconic=np.zeros((n, 3)), dmean2d=np.zeros((n, 2)), drgb=np.zeros((n, 3)),
               dsem=np.zeros((n, F)), dunc=np.zeros(n), ddepth=np.zeros(n))
    bg = _c(cam.background, np.float64)
    rc = lib().oracle_composite_backward(
        ctypes.c_int64(n), ctypes.c_int(F), _p(proj["depth"]), _p(proj["rect"]), _p(proj["tiles_touched"]),
        _p(proj["mean2d"]), _p(proj["conic_opacity"]), _p(proj["rgb"]), _p(sem), _p(unc), ctypes.c_int(cam.width),
        ctypes.c_int(cam.height), _p(bg), ctypes.c_int64(npix), _p(pix), _p(g), ctypes.c_int(flags), _p(out["dopac"]),
        _p(out["dconic"]), _p(out["dmean2d"]), _p(out["drgb"]), _p(out["dsem"]), _p(out["dunc"]), _p(out["ddepth"]))
    assert rc == 0
    if with_abs:
        out["abs"] = composite_backward_abs(proj, sem, unc, cam, dL_dpix, pix, flags)
    return out


def composite_backward_abs(proj: dict, sem, unc, cam, dL_dpix, pix=None, flags: int = 0) -> dict:
    """For every sum composite_backward forms (same keys), the sum of the absolute values of the single products it expands
    into: the conditioning that the gradient parity bound uses (reading G-4). Pinned in tests/test_oracle_conditioning.py."""
    sem, unc = _c(sem, np.float64), _c(unc, np.float64)
    n, F = sem.shape
    CH = channels(F)
    pix, npix = _pix(pix, cam)
    g = _c(dL_dpix, np.float64).reshape(npix, CH)
    geo = (flags & 4) != 0      # depth / alpha upstream gradients (flags bit 2)
    abs_sums = np.zeros((n, 10 + F + (1 if geo else 0)))
    bg = _c(cam.background, np.float64)
    rc = lib().oracle_composite_backward_abs(
        ctypes.c_int64(n), ctypes.c_int(F), _p(proj["depth"]), _p(proj["rect"]), _p(proj["tiles_touched"]),
        _p(proj["mean2d"]), _p(proj["conic_opacity"]), _p(proj["rgb"]), _p(sem), _p(unc), ctypes.c_int(cam.width),
        ctypes.c_int(cam.height), _p(bg), ctypes.c_int64(npix), _p(pix), _p(g), ctypes.c_int(flags), _p(abs_sums))
    assert rc == 0
    return dict(dopac=abs_sums[:, 0].copy(), dconic=abs_sums[:, 1:4].copy(), dmean2d=abs_sums[:, 4:6].copy(),
                drgb=abs_sums[:, 6:9].copy(), dsem=abs_sums[:, 9:9 + F].copy(), dunc=abs_sums[:, 9 + F].copy(),
                ddepth=abs_sums[:, 10 + F].copy() if geo else np.zeros(n))


def project_backward(scene, cam, g2d: dict, mode: int = 0) -> dict:
    n = scene.means.shape[0]
    K = scene.sh.shape[1]
    means, scales, quats = _c(scene.means, np.float64), _c(scene.scales, np.float64), _c(scene.quats, np.float64)
    sh = _c(scene.sh, np.float64)
    cv = cam_vector(cam)
    out = dict(dmeans=np.zeros((n, 3)), dscales=np.zeros((n, 3)), dquats=np.zeros((n, 4)), dsh=np.zeros((n, K, 3)))
    rc = lib().oracle_project_backward(
        ctypes.c_int(mode), ctypes.c_int64(n), ctypes.c_int(scene.sh_degree), ctypes.c_int(K), _p(means), _p(scales),
        _p(quats), _p(sh), _p(cv), ctypes.c_int(cam.width), ctypes.c_int(cam.height), _p(g2d["dconic"]),
        _p(g2d["dmean2d"]), _p(g2d["drgb"]), _p(out["dmeans"]), _p(out["dscales"]), _p(out["dquats"]), _p(out["dsh"]),
        _p(_c(g2d["ddepth"], np.float64)) if g2d.get("ddepth") is not None else None)
    assert rc == 0
    return out


def render_forward(scene, cam, mode: int = 0, pix=None, fragile_rel: float = FRAGILE_REL) -> dict:
    proj = project(scene, cam, mode)
    res = composite_forward(proj, scene.sem, scene.unc, cam, pix, fragile_rel)
    res["proj"] = proj
    return res


def project_backward_abs(scene, cam, abs2d: dict, mode: int = 0) -> dict:
    """Conditioning of the 3D gradients: the per-Gaussian projection backward is a LINEAR map J of (dconic, dmean2d,
    drgb); the absolute sums of the 2D gradients are pushed through |J|, column by column (eight calls of
    project_backward with unit inputs give the columns of J for every Gaussian at once)."""
    n = scene.means.shape[0]
    K = scene.sh.shape[1]
    out = dict(dmeans=np.zeros((n, 3)), dscales=np.zeros((n, 3)), dquats=np.zeros((n, 4)), dsh=np.zeros((n, K, 3)))
    for key, width in (("dconic", 3), ("dmean2d", 2), ("drgb", 3), ("ddepth", 1)):
        for j in range(width):
            unit = dict(dconic=np.zeros((n, 3)), dmean2d=np.zeros((n, 2)), drgb=np.zeros((n, 3)), ddepth=np.zeros((n, 1)))
            unit[key][:, j] = 1.0
            unit["ddepth"] = unit["ddepth"][:, 0].copy()
            col = project_backward(scene, cam, unit, mode)
            a = abs2d[key].reshape(n, -1)[:, j]
            for k in out:
                out[k] += np.abs(col[k]) * a.reshape((n,) + (1,) * (out[k].ndim - 1))
    return out


def render_backward(scene, cam, dL_dpix, mode: int = 0, pix=None, flags: int = 0, with_abs: bool = False) -> dict:
    """Full reverse-mode: pixels -> 2D per-Gaussian gradients -> 3D parameters.
    Returns dmeans, dscales, dquats, dopacities, dsh, dsem, dunc, dmean2d (+ the intermediate dconic, drgb).
    with_abs: also `abs`, the same eight arrays holding the sum of absolute terms behind every element (G-4)."""
    proj = project(scene, cam, mode)
    g2d = composite_backward(proj, scene.sem, scene.unc, cam, dL_dpix, pix, flags, with_abs)
    g3d = project_backward(scene, cam, g2d, mode)
    res = dict(dmeans=g3d["dmeans"], dscales=g3d["dscales"], dquats=g3d["dquats"], dopacities=g2d["dopac"],
               dsh=g3d["dsh"], dsem=g2d["dsem"], dunc=g2d["dunc"], dmean2d=g2d["dmean2d"], dconic=g2d["dconic"],
               drgb=g2d["drgb"], ddepth=g2d["ddepth"], proj=proj)
    if with_abs:
        res["abs"] = gradient_abs(scene, cam, g2d["abs"], mode)
    return res


def gradient_abs(scene, cam, abs2d: dict, mode: int = 0) -> dict:
    a3 = project_backward_abs(scene, cam, abs2d, mode)
    return dict(dmeans=a3["dmeans"], dscales=a3["dscales"], dquats=a3["dquats"], dopacities=abs2d["dopac"],
                dsh=a3["dsh"], dsem=abs2d["dsem"], dunc=abs2d["dunc"], dmean2d=abs2d["dmean2d"])


def sh_basis(dirs: np.ndarray, degree: int = 3) -> np.ndarray:
    dirs = _c(dirs, np.float64).reshape(-1, 3)
    out = np.zeros((dirs.shape[0], 16))
    tmp = np.zeros(16)
    for i in range(dirs.shape[0]):
        lib().oracle_sh_basis(_p(dirs[i]), ctypes.c_int(degree), _p(tmp))
        out[i] = tmp
    return out


def decode(x, weights, biases, codebook, d_clip: int, queries, want=("probs", "decoded", "rel")) -> dict:
    """x [P,in] and all weights are float arrays holding the (already bf16-rounded) values."""
    x = _c(x, np.float64)
    P = x.shape[0]
    Ws = [_c(w, np.float64) for w in weights]
    bs = [None if b is None else _c(b, np.float64) for b in biases]
    L = len(Ws)
    dims = np.array([Ws[0].shape[1]] + [w.shape[0] for w in Ws], np.int32)
    K = int(dims[-1])
    cb = _c(codebook, np.float64)
    d = cb.shape[1]
    q = _c(queries, np.float64)
    Q = q.shape[0]
    Wp = (ctypes.c_void_p * L)(*[w.ctypes.data for w in Ws])
    bp = (ctypes.c_void_p * L)(*[None if b is None else b.ctypes.data for b in bs])
    probs = np.zeros((P, K)) if "probs" in want else None
    decoded = np.zeros((P, d)) if "decoded" in want else None
    rel = np.zeros((P, Q)) if "rel" in want else None
    rc = lib().oracle_decode(ctypes.c_int64(P), ctypes.c_int(L), _p(dims), _p(x), Wp, bp, _p(cb), ctypes.c_int(d),
                             ctypes.c_int(d_clip), _p(q), ctypes.c_int(Q), _p(probs), _p(decoded), _p(rel))
    assert rc == 0
    return dict(probs=probs, decoded=decoded, rel=rel)


def relevancy_map(F, d_clip: int, queries) -> np.ndarray:
    """PAPER.md:360 (reading C-21): cosine of the first d_clip dims of every row of F [P,d] against each query [Q,d_clip]."""
    F = _c(F, np.float64)
    q = _c(queries, np.float64)
    P, d = F.shape
    Q = q.shape[0]
    rel = np.zeros((P, Q))
    rc = lib().oracle_relevancy_map(ctypes.c_int64(P), ctypes.c_int(d), ctypes.c_int(d_clip), _p(F), _p(q), ctypes.c_int(Q), _p(rel))
    assert rc == 0
    return rel


def semantic_loss(x, u, index, weights, biases, lambda_ce: float = 1.0, lambda_u: float = 0.1) -> dict:
    """PAPER.md Eq. 8-12 forward + reverse mode in fp64. x [P,in] rendered compact features, u [P] rendered uncertainty,
    index [P] int. Returns loss = (L_CE, L_u, L_s), dx, du, dW (list), db (list)."""
    x, u = _c(x, np.float64), _c(u, np.float64)
    idx = _c(index, np.int32)
    P = x.shape[0]
    Ws = [_c(w, np.float64) for w in weights]
    bs = [None if b is None else _c(b, np.float64) for b in biases]
    L = len(Ws)
    dims = np.array([Ws[0].shape[1]] + [w.shape[0] for w in Ws], np.int32)
    dW = [np.zeros_like(w) for w in Ws]
    db = [None if b is None else np.zeros_like(b) for b in bs]
    arr = lambda lst: (ctypes.c_void_p * L)(*[None if a is None else a.ctypes.data for a in lst])
    loss, dx, du = np.zeros(3), np.zeros_like(x), np.zeros(P)
    rc = lib().oracle_semantic_loss(ctypes.c_int64(P), ctypes.c_int(L), _p(dims), _p(x), _p(u), _p(idx), arr(Ws), arr(bs),
                                    ctypes.c_double(lambda_ce), ctypes.c_double(lambda_u), _p(loss), _p(dx), _p(du), arr(dW),
                                    arr(db))
    assert rc == 0, rc
    return dict(loss=loss, dx=dx, du=du, dW=dW, db=db)


def adam_step(p, g, m, v, lr=1e-3, beta1=0.9, beta2=0.999, eps=1e-8, step=1):
    """PAPER.md:182 Adam step in fp64; returns new (p, m, v) copies."""
    p, m, v = (np.array(a, dtype=np.float64, copy=True).reshape(-1) for a in (p, m, v))
    g = _c(np.asarray(g, dtype=np.float64).reshape(-1), np.float64)
    rc = lib().oracle_adam_step(ctypes.c_int64(p.size), _p(p), _p(g), _p(m), _p(v), ctypes.c_double(lr),
                                ctypes.c_double(beta1), ctypes.c_double(beta2), ctypes.c_double(eps), ctypes.c_int(step))
    assert rc == 0
    return p, m, v


def density_stats(dmean2d, radius, grad_accum, denom, max_radius):
    """Density-control statistics of one view (reading C-27); returns updated copies (grad_accum, denom, max_radius)."""
    d = _c(dmean2d, np.float64).reshape(-1, 2)
    n = d.shape[0]
    r = _c(radius, np.int32)
    ga = np.array(grad_accum, dtype=np.float64, copy=True)
    dn = np.array(denom, dtype=np.uint32, copy=True)
    mr = np.array(max_radius, dtype=np.int32, copy=True)
    rc = lib().oracle_density_stats(ctypes.c_int64(n), _p(d), _p(r), _p(ga), _p(dn), _p(mr))
    assert rc == 0
    return ga, dn, mr


def relevancy_lerf(cosines, n_pos: int, tau: float = 10.0) -> np.ndarray:
    """LERF-style relevancy from a cosine map [P,Q] (columns 0..n_pos-1 positive queries, the rest canonical negatives):
    min over the negatives of the pairwise softmax at scale tau. Formula absent from PAPER.md (:360 cites LERF [18])."""
    c = _c(cosines, np.float64)
    P, Q = c.shape
    out = np.zeros((P, n_pos))
    rc = lib().oracle_relevancy_lerf(ctypes.c_int64(P), ctypes.c_int(Q), ctypes.c_int(n_pos), ctypes.c_double(tau), _p(c), _p(out))
    assert rc == 0
    return out


def quantize(F, S, d_clip: int, lambda_dino: float = 0.5, lambda_cos: float = 1.0, lambda_lb: float = 0.5,
             want_scores: bool = False) -> dict:
    """PAPER.md Eq. 3-7, 16-20 in fp64. F [P,d] features, S [N,d] codebook. Returns index [P], gap [P] (best minus
    second-best score), r [N], p [N], loss = (L_cos, L_lb, L_q) and optionally the scores D [P,N]."""
    F, S = _c(F, np.float64), _c(S, np.float64)
    P, d = F.shape
    N = S.shape[0]
    index, gap = np.zeros(P, np.int32), np.zeros(P)
    r, p, loss = np.zeros(N), np.zeros(N), np.zeros(3)
    scores = np.zeros((P, N)) if want_scores else None
    rc = lib().oracle_quantize(ctypes.c_int64(P), ctypes.c_int(N), ctypes.c_int(d), ctypes.c_int(d_clip), _p(F), _p(S),
                               ctypes.c_double(lambda_dino), ctypes.c_double(lambda_cos), ctypes.c_double(lambda_lb),
                               _p(index), _p(gap), _p(r), _p(p), _p(loss), _p(scores))
    assert rc == 0
    return dict(index=index, gap=gap, r=r, p=p, loss=loss, scores=scores)


def smooth_loss(p, s, u, weights, biases, w_s: float = 0.1) -> dict:
    """PAPER.md Eq. 13-14 (reading C-25) forward + reverse mode in fp64. p [n,3] positions, s [n,F] compact features,
    u [n] uncertainties. Returns loss (L_smo), s_mlp [n,F], ds [n,F], dW (list), db (list)."""
    p, s, u = _c(p, np.float64), _c(s, np.float64), _c(u, np.float64)
    n = p.shape[0]
    Ws = [_c(w, np.float64) for w in weights]
    bs = [None if b is None else _c(b, np.float64) for b in biases]
    L = len(Ws)
    dims = np.array([Ws[0].shape[1]] + [w.shape[0] for w in Ws], np.int32)
    dW = [np.zeros_like(w) for w in Ws]
    db = [None if b is None else np.zeros_like(b) for b in bs]
    arr = lambda lst: (ctypes.c_void_p * L)(*[None if a is None else a.ctypes.data for a in lst])
    loss, s_mlp, ds = np.zeros(1), np.zeros_like(s), np.zeros_like(s)
    rc = lib().oracle_smooth_loss(ctypes.c_int64(n), ctypes.c_int(L), _p(dims), _p(p), _p(s), _p(u), arr(Ws), arr(bs),
                                  ctypes.c_double(w_s), _p(loss), _p(s_mlp), _p(ds), arr(dW), arr(db))
    assert rc == 0, rc
    return dict(loss=float(loss[0]), s_mlp=s_mlp, ds=ds, dW=dW, db=db)
