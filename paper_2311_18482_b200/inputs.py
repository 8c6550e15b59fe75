"""Seeded synthetic inputs for the LEGS hot path (shared by the oracle tests and the CUDA tests/bench).

This module holds NONE of the method's arithmetic: it only draws random numbers, applies the
activations that BASELINE.json's configs list as generator steps (exp on log-scales, sigmoid on opacity
logits, quaternion normalisation, look-at camera matrices) and rounds decode inputs to bf16 storage.
It imports neither `oracle/` nor the CUDA binding.

Recipe: numpy.random.Generator(PCG64(seed)), float64 draws cast to float32,
fixed draw order  means, log_scales, quats, opacity_logits, sh, sem, unc  (scene generator), then cameras
from PCG64(seed + 100), upstream gradients from PCG64(seed + 200 + view).

The scenes stand in for the paper's Mip-NeRF360 workloads ("six scenes of Mip-NeRF360"),
which are not available here; shapes/sizes/distributions follow BASELINE.json configs[0..4].
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

SH_C0 = 0.28209479177387814  # only used to turn an rgb draw into a DC coefficient (configs[0], reading C-12)


@dataclass
class Camera:
    width: int
    height: int
    fx: float
    fy: float
    cx: float
    cy: float
    world_to_cam: np.ndarray  # [12] float32, row-major 3x4 [R|t]
    near_plane: float = 0.2
    background: tuple = (0.0, 0.0, 0.0)

    def as_vector(self) -> np.ndarray:
        """fx, fy, cx, cy, w2c[12], near, bg[3]  (float32[20])."""
        v = np.zeros(20, dtype=np.float32)
        v[0:4] = (self.fx, self.fy, self.cx, self.cy)
        v[4:16] = self.world_to_cam
        v[16] = self.near_plane
        v[17:20] = self.background
        return v


@dataclass
class Scene:
    name: str
    means: np.ndarray       # [N,3] f32 world
    scales: np.ndarray      # [N,3] f32, already exp()
    quats: np.ndarray       # [N,4] f32 (w,x,y,z), normalised
    opacities: np.ndarray   # [N]   f32, already sigmoid()
    sh: np.ndarray          # [N,K,3] f32, K = (deg+1)^2
    sem: np.ndarray         # [N,F] f32
    unc: np.ndarray         # [N]   f32 in [0,1]
    sh_degree: int
    cameras: list = field(default_factory=list)
    seed: int = 0

    @property
    def n(self) -> int:
        return int(self.means.shape[0])

    @property
    def sem_dim(self) -> int:
        return int(self.sem.shape[1])


def _f32(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64).astype(np.float32))


def look_at_camera(cam_pos, width, height, fx, fy, cx, cy, up=(0.0, 1.0, 0.0), near=0.2, bg=(0.0, 0.0, 0.0)) -> Camera:
    """Camera at cam_pos looking at the origin: f = -c/|c|, r = normalise(up x f), u' = f x r,
    rows of R_wc = (r, u', f), t = -R_wc c  (camera looks down +z, x right, y down)."""
    c = np.asarray(cam_pos, dtype=np.float64)
    f = -c / np.linalg.norm(c)
    r = np.cross(np.asarray(up, dtype=np.float64), f)
    r /= np.linalg.norm(r)
    u = np.cross(f, r)
    R = np.stack([r, u, f])
    t = -R @ c
    w2c = np.concatenate([R, t[:, None]], axis=1).reshape(12)
    return Camera(width, height, float(fx), float(fy), float(cx), float(cy), _f32(w2c), near, tuple(bg))


def identity_camera(width, height, fx, fy, cx, cy, near=0.2, bg=(0.0, 0.0, 0.0)) -> Camera:
    w2c = np.array([1, 0, 0, 0, 0, 1, 0, 0, 0, 0, 1, 0], dtype=np.float32)
    return Camera(width, height, float(fx), float(fy), float(cx), float(cy), w2c, near, tuple(bg))


def _sphere_dirs(rng, k):
    v = rng.standard_normal((k, 3))
    return v / np.linalg.norm(v, axis=1, keepdims=True)


def _common_attributes(rng, n, log_scale_mu, log_scale_sigma, opacity_sigma, sh_degree, sem_dim, sh_sigma=0.2,
                       rgb_uniform=False):
    """Draw order after means: log_scales, quats, opacity_logits, sh, sem, unc."""
    log_scales = log_scale_mu + log_scale_sigma * rng.standard_normal((n, 3))
    q = rng.standard_normal((n, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    logits = opacity_sigma * rng.standard_normal(n)
    K = (sh_degree + 1) ** 2
    if rgb_uniform:
        rgb = rng.uniform(0.0, 1.0, (n, 1, 3))
        sh = (rgb - 0.5) / SH_C0
    else:
        sh = sh_sigma * rng.standard_normal((n, K, 3))
    sem = rng.standard_normal((n, sem_dim))
    unc = rng.uniform(0.0, 1.0, n)
    return dict(scales=_f32(np.exp(log_scales)), quats=_f32(q), opacities=_f32(1.0 / (1.0 + np.exp(-logits))),
                sh=_f32(sh), sem=_f32(sem), unc=_f32(unc))


def tiny_scene(n=1000, seed=0, width=64, height=64, sem_dim=8) -> Scene:
    """BASELINE.json configs[0]."""
    rng = np.random.Generator(np.random.PCG64(seed))
    xy = rng.uniform(-1.0, 1.0, (n, 2))
    z = rng.uniform(2.0, 6.0, (n, 1))
    means = np.concatenate([xy, z], axis=1)
    a = _common_attributes(rng, n, -3.0, 0.3, 1.0, 0, sem_dim, rgb_uniform=True)
    cam = identity_camera(width, height, 64.0 * width / 64.0, 64.0 * width / 64.0, width / 2.0, height / 2.0)
    return Scene("tiny", _f32(means), sh_degree=0, cameras=[cam], seed=seed, **a)


def object_scene(n=100_000, seed=1, width=800, height=800, focal=1111.0, n_views=8, sem_dim=8, sh_degree=3,
                 cam_radius=4.0) -> Scene:
    """BASELINE.json configs[1]."""
    rng = np.random.Generator(np.random.PCG64(seed))
    means = 0.5 * rng.standard_normal((n, 3))
    a = _common_attributes(rng, n, -4.5, 0.5, 1.5, sh_degree, sem_dim)
    crng = np.random.Generator(np.random.PCG64(seed + 100))
    dirs = _sphere_dirs(crng, n_views)
    cams = [look_at_camera(cam_radius * d, width, height, focal, focal, width / 2.0, height / 2.0) for d in dirs]
    return Scene("object", _f32(means), sh_degree=sh_degree, cameras=cams, seed=seed, **a)


def unbounded_scene(n=1_000_000, seed=2, width=1600, height=1064, focal=1150.0, sem_dim=8, sh_degree=3,
                    cam_radius=6.0) -> Scene:
    """BASELINE.json configs[2]: 70% N(0,I3), 30% on a shell of radius 10..50, heavy-tailed footprints."""
    rng = np.random.Generator(np.random.PCG64(seed))
    n_in = int(round(0.7 * n))
    inner = rng.standard_normal((n_in, 3))
    d = _sphere_dirs(rng, n - n_in)
    r = rng.uniform(10.0, 50.0, (n - n_in, 1))
    means = np.concatenate([inner, r * d], axis=0)
    a = _common_attributes(rng, n, -3.5, 0.8, 1.5, sh_degree, sem_dim)
    c = np.array([math.cos(0.35), math.sin(0.35), 0.3])
    c = cam_radius * c / np.linalg.norm(c)
    cam = look_at_camera(c, width, height, focal, focal, width / 2.0, height / 2.0)
    return Scene("unbounded", _f32(means), sh_degree=sh_degree, cameras=[cam], seed=seed, **a)


def large_scene(n=3_000_000, seed=4, width=1920, height=1080, focal=1150.0, n_views=4, sem_dim=16, sh_degree=3,
                n_clusters=200, cam_radius=30.0) -> Scene:
    """BASELINE.json configs[4]: mixture of 200 anisotropic clusters."""
    rng = np.random.Generator(np.random.PCG64(seed))
    centres = rng.uniform(-20.0, 20.0, (n_clusters, 3))
    G = rng.standard_normal((n_clusters, 3, 3))
    e = np.exp(-0.5 + 0.5 * rng.standard_normal((n_clusters, 3)))
    A = G * e[:, None, :]
    k = rng.integers(0, n_clusters, n)
    xi = rng.standard_normal((n, 3))
    means = centres[k] + np.einsum("nij,nj->ni", A[k], xi)
    a = _common_attributes(rng, n, -4.0, 0.7, 1.5, sh_degree, sem_dim)
    crng = np.random.Generator(np.random.PCG64(seed + 100))
    dirs = _sphere_dirs(crng, n_views)
    cams = [look_at_camera(cam_radius * d, width, height, focal, focal, width / 2.0, height / 2.0) for d in dirs]
    return Scene("large", _f32(means), sh_degree=sh_degree, cameras=cams, seed=seed, **a)


def channels(sem_dim: int) -> int:
    """CH = roundup4(3 rgb + 1 depth + F sem + 1 unc + 1 alpha)."""
    return (3 + 1 + sem_dim + 1 + 1 + 3) // 4 * 4


def upstream_gradient(scene: Scene, view: int = 0, depth_alpha: bool = False) -> np.ndarray:
    """dL/dpixel [H,W,CH] ~ N(0,1) on the 3+F+1 differentiable channels (rgb, sem, unc); 0 on depth/alpha/pad.
    depth_alpha: also N(0,1) on the depth (3) and alpha (5+F) slots, from a generator of its own (the other draws do not
    change) — the upstream of LEGS_BWD_DEPTH_ALPHA."""
    cam = scene.cameras[view]
    F = scene.sem_dim
    CH = channels(F)
    rng = np.random.Generator(np.random.PCG64(scene.seed + 200 + view))
    g = np.zeros((cam.height, cam.width, CH), dtype=np.float32)
    g[..., 0:3] = rng.standard_normal((cam.height, cam.width, 3))
    g[..., 4:4 + F + 1] = rng.standard_normal((cam.height, cam.width, F + 1))
    if depth_alpha:
        rng2 = np.random.Generator(np.random.PCG64(scene.seed + 300 + view))
        g[..., 3] = rng2.standard_normal((cam.height, cam.width))
        g[..., 5 + F] = rng2.standard_normal((cam.height, cam.width))
    return g


# ---------------------------------------------------------------------------------------------------------
# decode inputs (BASELINE.json configs[3])

def to_bf16_bits(a: np.ndarray) -> np.ndarray:
    """float32 -> bf16 storage (uint16), round-to-nearest-even. A storage-format conversion, not method arithmetic."""
    u = np.ascontiguousarray(a, dtype=np.float32).view(np.uint32)
    rounding = ((u >> 16) & 1) + np.uint32(0x7FFF)
    return ((u + rounding) >> 16).astype(np.uint16)


def bf16_bits_to_f32(b: np.ndarray) -> np.ndarray:
    return (b.astype(np.uint32) << 16).view(np.float32)


@dataclass
class DecodeInputs:
    feat: np.ndarray        # [P,F] uint16 (bf16 bits)
    weights: list           # list of [out,in] uint16 (bf16 bits)
    biases: list            # list of [out] float32
    codebook: np.ndarray    # [K,d] uint16 (bf16 bits)
    queries: np.ndarray     # [Q,d_clip] uint16 (bf16 bits)
    d_clip: int
    dims: list              # [in, hidden..., K]


def decode_inputs(P=1920 * 1080, in_dim=8, hidden=(64,), n_codes=128, d=896, d_clip=512, n_queries=4, seed=1,
                  bias_sigma=0.0) -> DecodeInputs:
    """Draw order: feat, weights layer by layer (Kaiming-uniform U(+-sqrt(6/fan_in))), biases, codebook, queries."""
    rng = np.random.Generator(np.random.PCG64(seed))
    feat = rng.standard_normal((P, in_dim))
    dims = [in_dim, *hidden, n_codes]
    weights, biases = [], []
    for fan_in, fan_out in zip(dims[:-1], dims[1:]):
        bound = math.sqrt(6.0 / fan_in)
        weights.append(rng.uniform(-bound, bound, (fan_out, fan_in)))
    for fan_out in dims[1:]:
        biases.append(bias_sigma * rng.standard_normal(fan_out))
    cb = rng.standard_normal((n_codes, d))
    cb[:, :d_clip] /= np.linalg.norm(cb[:, :d_clip], axis=1, keepdims=True)
    cb[:, d_clip:] /= np.linalg.norm(cb[:, d_clip:], axis=1, keepdims=True)
    q = rng.standard_normal((n_queries, d_clip))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    return DecodeInputs(feat=to_bf16_bits(_f32(feat)), weights=[to_bf16_bits(_f32(w)) for w in weights],
                        biases=[_f32(b) for b in biases], codebook=to_bf16_bits(_f32(cb)),
                        queries=to_bf16_bits(_f32(q)), d_clip=d_clip, dims=dims)


# ---------------------------------------------------------------------------------------------------------
# quantisation inputs: synthetic stand-ins for the dense CLIP + DINO maps of PAPER.md:60-70,
# which need the pretrained models and the datasets.

@dataclass
class QuantizeInputs:
    features: np.ndarray    # [P,d] uint16 (bf16 bits), each part L2-normalised before rounding
    codebook: np.ndarray    # [N,d] uint16 (bf16 bits)
    d_clip: int


def quantize_inputs(P=4096, n_codes=128, d=896, d_clip=512, seed=5, noise=0.6, chunk=65536) -> QuantizeInputs:
    """"Features within a single object share very similar semantics": every pixel feature is one of
    n_codes random centres plus N(0, noise^2) noise, each part (CLIP, DINO) L2-normalised as the extraction step does
    (PAPER.md:64). The codebook is the centres perturbed by N(0, 0.3^2) (a partly trained space S), unnormalised.
    Draw order: centres, codebook perturbation, then per chunk of rows: centre indices, noise."""
    rng = np.random.Generator(np.random.PCG64(seed))
    centres = rng.standard_normal((n_codes, d))
    codebook = centres + 0.3 * rng.standard_normal((n_codes, d))
    feats = np.empty((P, d), dtype=np.uint16)
    for r0 in range(0, P, chunk):
        n = min(chunk, P - r0)
        k = rng.integers(0, n_codes, n)
        f = centres[k] + noise * rng.standard_normal((n, d))
        f[:, :d_clip] /= np.linalg.norm(f[:, :d_clip], axis=1, keepdims=True)
        f[:, d_clip:] /= np.linalg.norm(f[:, d_clip:], axis=1, keepdims=True)
        feats[r0:r0 + n] = to_bf16_bits(_f32(f))
    return QuantizeInputs(features=feats, codebook=to_bf16_bits(_f32(codebook)), d_clip=d_clip)


# ---------------------------------------------------------------------------------------------------------
# smoothing MLP weights (Table 4: 3 -> 128 -> 128 -> 128 -> d_s)

def smooth_mlp_inputs(sem_dim=8, hidden=128, seed=3, bias_sigma=0.05):
    """Kaiming-uniform weights (bf16 storage) and small N(0, bias_sigma^2) biases; draw order: weights layer by layer,
    then biases."""
    rng = np.random.Generator(np.random.PCG64(seed))
    dims = [3, hidden, hidden, hidden, sem_dim]
    weights = [rng.uniform(-math.sqrt(6.0 / i), math.sqrt(6.0 / i), (o, i)) for i, o in zip(dims[:-1], dims[1:])]
    biases = [bias_sigma * rng.standard_normal(o) for o in dims[1:]]
    return [to_bf16_bits(_f32(w)) for w in weights], [_f32(b) for b in biases]
