"""Thin ctypes binding of include/legs.h — argument marshalling only; every step of the path runs in liblegs.so.

PyTorch is used for device memory and streams (torch tensors are passed as raw device pointers, the current torch
CUDA stream as the `stream` argument). There is NO CPU fallback: loading fails loudly if liblegs.so is missing.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "liblegs.so")
_lib = None

STATUS = {0: "LEGS_OK", -1: "LEGS_ERR_NULL", -2: "LEGS_ERR_ALIGN", -3: "LEGS_ERR_DIM", -4: "LEGS_ERR_CAPACITY",
          -5: "LEGS_ERR_WORKSPACE", -6: "LEGS_ERR_CUDA"}
LEGS_BWD_ACCUMULATE = 1
LEGS_BWD_COUPLE_SEM = 2
LEGS_BWD_COMPOSITE_ONLY = 4
LEGS_BWD_DEPTH_ALPHA = 8

EXPORTS = ["legs_create", "legs_destroy", "legs_status_string", "legs_last_cuda_error", "legs_launch_count",
           "legs_record_stride", "legs_pixel_channels", "legs_sort_workspace_bytes", "legs_backward_workspace_bytes",
           "legs_preprocess", "legs_read_num_instances", "legs_bin_and_sort", "legs_render_forward",
           "legs_render_forward_stats", "legs_render_backward", "legs_decode_workspace_bytes", "legs_decode_semantics",
           "legs_relevancy_workspace_bytes", "legs_relevancy", "legs_loss_workspace_bytes", "legs_semantic_loss",
           "legs_peak_kernel", "legs_num_sms", "legs_adam_step", "legs_density_stats",
           "legs_quantize_workspace_bytes", "legs_quantize", "legs_smooth_workspace_bytes", "legs_smooth_loss",
           "legs_decode_prepare", "legs_decode_semantics_packed", "legs_relevancy_prepare", "legs_relevancy_packed",
           "legs_relevancy_lerf", "legs_relevancy_static", "legs_relevancy_static_bytes",
           "legs_relevancy_static_max_codes", "legs_relevancy_decoded", "legs_tile_order",
           "legs_render_forward_ordered", "legs_render_backward_ordered"]


class LegsError(RuntimeError):
    def __init__(self, status, where):
        self.status = status
        super().__init__(f"{where}: {STATUS.get(status, status)}")


class CCamera(C.Structure):
    _fields_ = [("width", C.c_int32), ("height", C.c_int32), ("fx", C.c_float), ("fy", C.c_float), ("cx", C.c_float),
                ("cy", C.c_float), ("world_to_cam", C.c_float * 12), ("near_plane", C.c_float),
                ("background", C.c_float * 3)]


class CGaussians(C.Structure):
    _fields_ = [("n", C.c_int64), ("sh_degree", C.c_int32), ("sh_coefs_stored", C.c_int32), ("sem_dim", C.c_int32),
                ("means", C.c_void_p), ("scales", C.c_void_p), ("quats", C.c_void_p), ("opacities", C.c_void_p),
                ("sh", C.c_void_p), ("sem", C.c_void_p), ("unc", C.c_void_p)]


class CFrame(C.Structure):
    _fields_ = [("depth", C.c_void_p), ("radius", C.c_void_p), ("rect", C.c_void_p), ("mean2d", C.c_void_p),
                ("conic_opacity", C.c_void_p), ("rgb", C.c_void_p), ("clamped", C.c_void_p),
                ("tiles_touched", C.c_void_p), ("record", C.c_void_p), ("num_instances", C.c_void_p)]


class CGrads(C.Structure):
    _fields_ = [("dmeans", C.c_void_p), ("dscales", C.c_void_p), ("dquats", C.c_void_p), ("dopacities", C.c_void_p),
                ("dsh", C.c_void_p), ("dsem", C.c_void_p), ("dunc", C.c_void_p), ("dmean2d", C.c_void_p)]


class CDecoder(C.Structure):
    _fields_ = [("n_layers", C.c_int32), ("in_dim", C.c_int32), ("hidden", C.c_int32 * 2), ("n_codes", C.c_int32),
                ("w", C.c_void_p * 3), ("b", C.c_void_p * 3)]


class CDecoderGrads(C.Structure):
    _fields_ = [("dw", C.c_void_p * 3), ("db", C.c_void_p * 3)]


def lib():
    """Loads liblegs.so; raises if it is missing (the product path never falls back to anything else)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_2311_18482_b200.build` "
                               "(there is no CPU or PyTorch fallback for the legs hot path)")
        L = C.CDLL(LIB_PATH)
        L.legs_status_string.restype = C.c_char_p
        L.legs_launch_count.restype = C.c_uint64
        for f in ("legs_sort_workspace_bytes", "legs_backward_workspace_bytes", "legs_decode_workspace_bytes",
                  "legs_relevancy_workspace_bytes", "legs_loss_workspace_bytes", "legs_quantize_workspace_bytes",
                  "legs_smooth_workspace_bytes", "legs_relevancy_static_bytes"):
            if hasattr(L, f):
                getattr(L, f).restype = C.c_size_t
        _lib = L
    return _lib


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _check(rc, where):
    if rc != 0:
        raise LegsError(rc, where)


def channels(F):
    return int(lib().legs_pixel_channels(C.c_int32(F)))


def record_stride(F):
    return int(lib().legs_record_stride(C.c_int32(F)))


def make_camera(cam) -> CCamera:
    c = CCamera()
    c.width, c.height = int(cam.width), int(cam.height)
    c.fx, c.fy, c.cx, c.cy = float(cam.fx), float(cam.fy), float(cam.cx), float(cam.cy)
    for i in range(12):
        c.world_to_cam[i] = float(cam.world_to_cam[i])
    c.near_plane = float(cam.near_plane)
    for i in range(3):
        c.background[i] = float(cam.background[i])
    return c


class Context:
    def __init__(self, device: int = 0):
        self._h = C.c_void_p()
        _check(lib().legs_create(C.c_int(device), C.byref(self._h)), "legs_create")
        self.device = torch.device("cuda", device)

    def __del__(self):
        if getattr(self, "_h", None) and _lib is not None:
            _lib.legs_destroy(self._h)
            self._h = None

    @property
    def launches(self) -> int:
        return int(lib().legs_launch_count(self._h))

    def last_cuda_error(self) -> int:
        return int(lib().legs_last_cuda_error(self._h))

    @property
    def num_sms(self) -> int:
        return int(lib().legs_num_sms(self._h))


class Gaussians:
    """Device-resident Gaussian set: tensors are float32, contiguous, on the GPU."""

    def __init__(self, means, scales, quats, opacities, sh, sem, unc, sh_degree):
        self.t = dict(means=means, scales=scales, quats=quats, opacities=opacities, sh=sh, sem=sem, unc=unc)
        for k, v in self.t.items():
            assert v.is_cuda and v.dtype == torch.float32 and v.is_contiguous(), k
        self.n = int(means.shape[0])
        self.sh_degree = int(sh_degree)
        self.sh_stored = int(sh.shape[1])
        self.F = int(sem.shape[1])
        c = CGaussians()
        c.n, c.sh_degree, c.sh_coefs_stored, c.sem_dim = self.n, self.sh_degree, self.sh_stored, self.F
        for k, v in self.t.items():
            setattr(c, k, v.data_ptr())
        self.c = c

    @staticmethod
    def from_scene(scene, device="cuda"):
        f = lambda a: torch.from_numpy(a).to(device).contiguous()
        return Gaussians(f(scene.means), f(scene.scales), f(scene.quats), f(scene.opacities), f(scene.sh), f(scene.sem),
                         f(scene.unc), scene.sh_degree)


class Frame:
    """Caller-owned per-view buffers of legs_preprocess (allocated with torch)."""

    def __init__(self, n, F, device="cuda"):
        e = lambda shape, dt: torch.empty(shape, dtype=dt, device=device)
        self.depth = e((n,), torch.float32)
        self.radius = e((n,), torch.int32)
        self.rect = e((n, 4), torch.int32)
        self.mean2d = e((n, 2), torch.float32)
        self.conic_opacity = e((n, 4), torch.float32)
        self.rgb = e((n, 3), torch.float32)
        self.clamped = e((n,), torch.uint8)
        self.tiles_touched = e((n,), torch.int32)
        self.record = e((n, record_stride(F)), torch.float32)
        self.num_instances = torch.zeros((2,), dtype=torch.int64, device=device)
        c = CFrame()
        for name, _ in CFrame._fields_:
            setattr(c, name, getattr(self, name).data_ptr())
        self.c = c


def legs_preprocess(ctx, g: Gaussians, cam: CCamera, frame: Frame):
    _check(lib().legs_preprocess(ctx._h, C.byref(g.c), C.byref(cam), C.byref(frame.c), _stream()), "legs_preprocess")


def legs_read_num_instances(ctx, frame: Frame) -> int:
    out = C.c_uint64(0)
    _check(lib().legs_read_num_instances(ctx._h, C.byref(frame.c), C.byref(out), _stream()), "legs_read_num_instances")
    return int(out.value)


def legs_sort_workspace_bytes(n, capacity, width, height) -> int:
    return int(lib().legs_sort_workspace_bytes(C.c_int64(n), C.c_uint64(capacity), C.c_int32(width), C.c_int32(height)))


def legs_bin_and_sort(ctx, frame: Frame, cam: CCamera, n, capacity, keys_sorted, vals_sorted, ranges, workspace):
    _check(lib().legs_bin_and_sort(ctx._h, C.byref(frame.c), C.byref(cam), C.c_int64(n), C.c_uint64(capacity),
                                   _ptr(keys_sorted), _ptr(vals_sorted), _ptr(ranges), _ptr(workspace),
                                   C.c_size_t(workspace.numel() * workspace.element_size()), _stream()),
           "legs_bin_and_sort")


def legs_tile_order(ctx, ranges, tile_order):
    _check(lib().legs_tile_order(ctx._h, _ptr(ranges), C.c_int32(int(ranges.shape[0])), _ptr(tile_order), _stream()), "legs_tile_order")


def legs_render_forward(ctx, g: Gaussians, cam: CCamera, frame: Frame, vals_sorted, ranges, out_pixels, n_contrib,
                        sem_bf16=None, block_masks=None, tile_order=None):
    if tile_order is not None:
        _check(lib().legs_render_forward_ordered(ctx._h, C.byref(g.c), C.byref(cam), C.byref(frame.c), _ptr(vals_sorted), _ptr(ranges),
                                                 _ptr(out_pixels), _ptr(n_contrib), _ptr(sem_bf16), _ptr(block_masks),
                                                 _ptr(tile_order), _stream()), "legs_render_forward_ordered")
        return
    _check(lib().legs_render_forward(ctx._h, C.byref(g.c), C.byref(cam), C.byref(frame.c), _ptr(vals_sorted), _ptr(ranges),
                                     _ptr(out_pixels), _ptr(n_contrib), _ptr(sem_bf16), _ptr(block_masks), _stream()),
           "legs_render_forward")


def legs_render_forward_stats(ctx, g: Gaussians, cam: CCamera, frame: Frame, vals_sorted, ranges, out_pixels, n_contrib,
                              counters):
    _check(lib().legs_render_forward_stats(ctx._h, C.byref(g.c), C.byref(cam), C.byref(frame.c), _ptr(vals_sorted),
                                           _ptr(ranges), _ptr(out_pixels), _ptr(n_contrib), _ptr(counters), _stream()),
           "legs_render_forward_stats")


def legs_backward_workspace_bytes(n, F) -> int:
    return int(lib().legs_backward_workspace_bytes(C.c_int64(n), C.c_int32(F)))


class Grads:
    """The eight gradient arrays, carved out of ONE flat fp32 buffer (`flat`) so that a multi-GPU by-view split can sum
    them with a single all-reduce; every array starts on a 16-byte boundary."""
    FIELDS = ("dmeans", "dscales", "dquats", "dopacities", "dsh", "dsem", "dunc", "dmean2d")

    def __init__(self, g: Gaussians, device="cuda"):
        shapes = dict(dmeans=(g.n, 3), dscales=(g.n, 3), dquats=(g.n, 4), dopacities=(g.n,), dsh=(g.n, g.sh_stored, 3),
                      dsem=(g.n, g.F), dunc=(g.n,), dmean2d=(g.n, 2))
        offs, total = {}, 0
        for k in self.FIELDS:
            offs[k] = total
            cnt = 1
            for d in shapes[k]:
                cnt *= d
            total += (cnt + 3) // 4 * 4
        self.flat = torch.zeros(max(total, 4), dtype=torch.float32, device=device)
        for k in self.FIELDS:
            cnt = 1
            for d in shapes[k]:
                cnt *= d
            setattr(self, k, self.flat[offs[k]:offs[k] + cnt].view(shapes[k]))
        c = CGrads()
        for name, _ in CGrads._fields_:
            setattr(c, name, getattr(self, name).data_ptr())
        self.c = c


def legs_render_backward(ctx, g: Gaussians, cam: CCamera, frame: Frame, vals_sorted, ranges, out_pixels, n_contrib,
                         dL_dpixels, flags, grads: Grads, workspace, block_masks=None, tile_order=None):
    if tile_order is not None:
        _check(lib().legs_render_backward_ordered(ctx._h, C.byref(g.c), C.byref(cam), C.byref(frame.c), _ptr(vals_sorted),
                                                  _ptr(ranges), _ptr(out_pixels), _ptr(n_contrib), _ptr(dL_dpixels),
                                                  _ptr(block_masks), C.c_int32(flags), C.byref(grads.c), _ptr(workspace),
                                                  C.c_size_t(workspace.numel() * workspace.element_size()), _ptr(tile_order),
                                                  _stream()), "legs_render_backward_ordered")
        return
    _check(lib().legs_render_backward(ctx._h, C.byref(g.c), C.byref(cam), C.byref(frame.c), _ptr(vals_sorted),
                                      _ptr(ranges), _ptr(out_pixels), _ptr(n_contrib), _ptr(dL_dpixels), _ptr(block_masks),
                                      C.c_int32(flags),
                                      C.byref(grads.c), _ptr(workspace),
                                      C.c_size_t(workspace.numel() * workspace.element_size()), _stream()),
           "legs_render_backward")


def make_decoder(weights, biases) -> CDecoder:
    """weights: list of bf16 [out,in] CUDA tensors (2 or 3 layers); biases: list of fp32 [out] tensors or None."""
    d = CDecoder()
    d.n_layers = len(weights)
    d.in_dim = int(weights[0].shape[1])
    d.hidden[0] = int(weights[0].shape[0])
    d.hidden[1] = int(weights[1].shape[0]) if len(weights) == 3 else 0
    d.n_codes = int(weights[-1].shape[0])
    for i, w in enumerate(weights):
        assert w.is_cuda and w.dtype == torch.bfloat16 and w.is_contiguous()
        d.w[i] = w.data_ptr()
        d.b[i] = None if biases is None or biases[i] is None else biases[i].data_ptr()
    d._keep = (weights, biases)
    return d


def legs_decode_workspace_bytes(dec: CDecoder, d: int) -> int:
    return int(lib().legs_decode_workspace_bytes(C.byref(dec), C.c_int32(d)))


def legs_decode_semantics(ctx, feat, dec: CDecoder, codebook, probs, decoded, workspace):
    P, d = int(feat.shape[0]), int(codebook.shape[1])
    _check(lib().legs_decode_semantics(ctx._h, _ptr(feat), C.c_int64(P), C.byref(dec), _ptr(codebook), C.c_int32(d),
                                       _ptr(probs), _ptr(decoded), _ptr(workspace),
                                       C.c_size_t(workspace.numel() * workspace.element_size()), _stream()),
           "legs_decode_semantics")


def legs_decode_prepare(ctx, dec: CDecoder, codebook, workspace):
    d = int(codebook.shape[1])
    _check(lib().legs_decode_prepare(ctx._h, C.byref(dec), _ptr(codebook), C.c_int32(d), _ptr(workspace),
                                     C.c_size_t(workspace.numel() * workspace.element_size()), _stream()), "legs_decode_prepare")


def legs_decode_semantics_packed(ctx, feat, dec: CDecoder, d, probs, decoded, workspace):
    _check(lib().legs_decode_semantics_packed(ctx._h, _ptr(feat), C.c_int64(int(feat.shape[0])), C.byref(dec), C.c_int32(d),
                                              _ptr(probs), _ptr(decoded), _ptr(workspace),
                                              C.c_size_t(workspace.numel() * workspace.element_size()), _stream()),
           "legs_decode_semantics_packed")


def legs_relevancy_prepare(ctx, codebook, d_clip, queries, workspace):
    K, d, Q = int(codebook.shape[0]), int(codebook.shape[1]), int(queries.shape[0])
    _check(lib().legs_relevancy_prepare(ctx._h, _ptr(codebook), C.c_int32(K), C.c_int32(d), C.c_int32(d_clip), _ptr(queries),
                                        C.c_int32(Q), _ptr(workspace), C.c_size_t(workspace.numel() * workspace.element_size()),
                                        _stream()), "legs_relevancy_prepare")


def legs_relevancy_packed(ctx, probs, K, Q, rel, workspace):
    _check(lib().legs_relevancy_packed(ctx._h, _ptr(probs), C.c_int64(int(probs.shape[0])), C.c_int32(K), C.c_int32(Q), _ptr(rel),
                                       _ptr(workspace), C.c_size_t(workspace.numel() * workspace.element_size()), _stream()),
           "legs_relevancy_packed")


def legs_relevancy_lerf(ctx, cosines, n_pos: int, tau: float, out):
    P, Q = int(cosines.shape[0]), int(cosines.shape[1])
    _check(lib().legs_relevancy_lerf(ctx._h, _ptr(cosines), C.c_int64(P), C.c_int32(Q), C.c_int32(n_pos), C.c_float(tau),
                                     _ptr(out), _stream()), "legs_relevancy_lerf")


def legs_relevancy_workspace_bytes(K: int, Q: int) -> int:
    return int(lib().legs_relevancy_workspace_bytes(C.c_int32(K), C.c_int32(Q)))


def legs_relevancy(ctx, probs, codebook, d_clip, queries, rel, workspace):
    P, K, d, Q = int(probs.shape[0]), int(codebook.shape[0]), int(codebook.shape[1]), int(queries.shape[0])
    _check(lib().legs_relevancy(ctx._h, _ptr(probs), C.c_int64(P), _ptr(codebook), C.c_int32(K), C.c_int32(d),
                                C.c_int32(d_clip), _ptr(queries), C.c_int32(Q), _ptr(rel), _ptr(workspace),
                                C.c_size_t(workspace.numel() * workspace.element_size()), _stream()), "legs_relevancy")


def legs_relevancy_decoded(ctx, decoded, d_clip, queries, rel):
    P, d, Q = int(decoded.shape[0]), int(decoded.shape[1]), int(queries.shape[0])
    _check(lib().legs_relevancy_decoded(ctx._h, _ptr(decoded), C.c_int64(P), C.c_int32(d), C.c_int32(d_clip), _ptr(queries),
                                        C.c_int32(Q), _ptr(rel), _stream()), "legs_relevancy_decoded")


def legs_relevancy_static_bytes() -> int:
    return int(lib().legs_relevancy_static_bytes())


def legs_relevancy_static_max_codes() -> int:
    return int(lib().legs_relevancy_static_max_codes())


def legs_relevancy_static(ctx, probs, codebook, d_clip, queries, rel):
    """legs_relevancy for callers that cannot allocate device memory (a frame loop living off a fixed pool, a plugin
    that only gets the host application's buffers): no workspace argument, the scratch is a 64 KB array inside
    liblegs.so. K <= legs_relevancy_static_max_codes(); calls on one device share the array, so keep them ordered on
    the GPU (include/legs.h)."""
    P, K, d, Q = int(probs.shape[0]), int(codebook.shape[0]), int(codebook.shape[1]), int(queries.shape[0])
    _check(lib().legs_relevancy_static(ctx._h, _ptr(probs), C.c_int64(P), _ptr(codebook), C.c_int32(K), C.c_int32(d),
                                       C.c_int32(d_clip), _ptr(queries), C.c_int32(Q), _ptr(rel), _stream()),
           "legs_relevancy_static")


def legs_loss_workspace_bytes(dec: CDecoder, P: int) -> int:
    return int(lib().legs_loss_workspace_bytes(C.byref(dec), C.c_int64(P)))


def legs_semantic_loss(ctx, pixels, index_map, dec: CDecoder, lambda_ce, lambda_u, dL_dpixels, dw, db, loss, workspace):
    """PAPER.md Eq. 8-12 forward + reverse mode. pixels / dL_dpixels [H,W,CH] or [P,CH] fp32; index_map [P] int32;
    dw, db: lists of fp32 tensors per layer (db entries may be None), added to; loss [3] fp32, added to."""
    CH = int(pixels.shape[-1])
    P = pixels.numel() // CH
    g = CDecoderGrads()
    for l, t in enumerate(dw):
        g.dw[l] = t.data_ptr()
    for l, t in enumerate(db):
        g.db[l] = None if t is None else t.data_ptr()
    _check(lib().legs_semantic_loss(ctx._h, _ptr(pixels), C.c_int64(P), C.c_int32(dec.in_dim), _ptr(index_map), C.byref(dec),
                                    C.c_float(lambda_ce), C.c_float(lambda_u), _ptr(dL_dpixels), C.byref(g), _ptr(loss),
                                    _ptr(workspace), C.c_size_t(workspace.numel() * workspace.element_size()), _stream()),
           "legs_semantic_loss")


def legs_quantize(ctx, features, codebook, d_clip, lambda_dino, lambda_cos, lambda_lb, index_map, r, p, loss):
    """PAPER.md Eq. 3-7, 16-20: features [P,d] bf16, codebook [N,d] bf16 -> index_map [P] int32, r / p [N] fp32 (or None),
    loss [3] fp32 (L_cos, L_lb, L_q)."""
    P, d, N = int(features.shape[0]), int(features.shape[1]), int(codebook.shape[0])
    ws = torch.empty(int(lib().legs_quantize_workspace_bytes(C.c_int32(N))), dtype=torch.uint8, device=features.device)
    _check(lib().legs_quantize(ctx._h, _ptr(features), C.c_int64(P), _ptr(codebook), C.c_int32(N), C.c_int32(d),
                               C.c_int32(d_clip), C.c_float(lambda_dino), C.c_float(lambda_cos), C.c_float(lambda_lb),
                               _ptr(index_map), _ptr(r), _ptr(p), _ptr(loss), _ptr(ws),
                               C.c_size_t(ws.numel()), _stream()), "legs_quantize")


class CSmoothMlp(C.Structure):
    _fields_ = [("hidden", C.c_int32), ("w", C.c_void_p * 4), ("b", C.c_void_p * 4)]


class CSmoothGrads(C.Structure):
    _fields_ = [("dw", C.c_void_p * 4), ("db", C.c_void_p * 4)]


def legs_smooth_loss(ctx, means, sem, unc, weights, biases, w_s, lambda_smo, accumulate, dsem, dw, db, loss):
    """PAPER.md Eq. 13-14 forward + reverse mode. weights: 4 bf16 [out,in] CUDA tensors; biases: 4 fp32 tensors or None;
    dw / db: fp32 tensors per layer, added to; dsem [n,F] overwritten (or added to); loss [1] fp32, added to."""
    n, F = int(sem.shape[0]), int(sem.shape[1])
    m, g = CSmoothMlp(), CSmoothGrads()
    m.hidden = int(weights[0].shape[0])
    for l in range(4):
        m.w[l] = weights[l].data_ptr()
        m.b[l] = None if biases is None or biases[l] is None else biases[l].data_ptr()
        g.dw[l] = dw[l].data_ptr()
        g.db[l] = None if db is None or db[l] is None else db[l].data_ptr()
    ws = torch.empty(int(lib().legs_smooth_workspace_bytes(C.c_int32(F))), dtype=torch.uint8, device=sem.device)
    _check(lib().legs_smooth_loss(ctx._h, C.c_int64(n), C.c_int32(F), _ptr(means), _ptr(sem), _ptr(unc), C.byref(m),
                                  C.c_float(w_s), C.c_float(lambda_smo), C.c_int32(1 if accumulate else 0), _ptr(dsem),
                                  C.byref(g), _ptr(loss), _ptr(ws), C.c_size_t(ws.numel()), _stream()), "legs_smooth_loss")


class CAdam(C.Structure):
    _fields_ = [("lr", C.c_float), ("beta1", C.c_float), ("beta2", C.c_float), ("eps", C.c_float), ("step", C.c_int32)]


def legs_adam_step(ctx, params, grads, m, v, step, lr=1e-3, beta1=0.9, beta2=0.999, eps=1e-8):
    """PAPER.md:182 Adam step over a list of fp32 CUDA tensors (in place), one launch."""
    n = len(params)
    arr = lambda ts: (C.c_void_p * n)(*[t.data_ptr() for t in ts])
    counts = (C.c_int64 * n)(*[int(t.numel()) for t in params])
    hp = CAdam(lr, beta1, beta2, eps, int(step))
    _check(lib().legs_adam_step(ctx._h, C.c_int32(n), arr(params), arr(grads), arr(m), arr(v), counts, C.byref(hp), _stream()),
           "legs_adam_step")


def legs_density_stats(ctx, dmean2d, radius, grad_accum, denom, max_radius):
    _check(lib().legs_density_stats(ctx._h, C.c_int64(int(radius.numel())), _ptr(dmean2d), _ptr(radius), _ptr(grad_accum),
                                    _ptr(denom), _ptr(max_radius), _stream()), "legs_density_stats")


def legs_peak_kernel(ctx, kind: int, iters: int, sink) -> int:
    """Launches one micro-benchmark kernel (include/legs.h "measurement"); returns the lane-operations it executes."""
    ops = C.c_uint64(0)
    _check(lib().legs_peak_kernel(ctx._h, C.c_int32(kind), C.c_int32(iters), _ptr(sink), C.byref(ops), _stream()),
           "legs_peak_kernel")
    return int(ops.value)


class Renderer:
    """Convenience owner of the per-view buffers for one (scene size, camera size, capacity): plumbing only."""

    def __init__(self, ctx: Context, g: Gaussians, cam, capacity: int, want_keys: bool = False, want_bf16: bool = False):
        self.ctx, self.g, self.cam = ctx, g, make_camera(cam)
        dev = ctx.device
        W, H, F = int(cam.width), int(cam.height), g.F
        self.W, self.H, self.F, self.CH = W, H, F, channels(F)
        self.capacity = int(capacity)
        self.ntiles = ((W + 15) // 16) * ((H + 15) // 16)
        self.frame = Frame(g.n, F, dev)
        self.vals_sorted = torch.empty(self.capacity, dtype=torch.int32, device=dev)
        self.keys_sorted = torch.empty(self.capacity, dtype=torch.int64, device=dev) if want_keys else None
        self.ranges = torch.empty((self.ntiles, 2), dtype=torch.int32, device=dev)
        self.sort_ws = torch.empty(legs_sort_workspace_bytes(g.n, self.capacity, W, H), dtype=torch.uint8, device=dev)
        self.out = torch.empty((H, W, self.CH), dtype=torch.float32, device=dev)
        self.n_contrib = torch.empty((H, W), dtype=torch.int32, device=dev)
        self.sem_bf16 = torch.empty((H * W, F), dtype=torch.bfloat16, device=dev) if want_bf16 else None
        self.block_masks = torch.empty(self.capacity, dtype=torch.uint8, device=dev)   # forward -> backward hand-over
        self.bwd_ws = None
        self.tile_order = None    # use_tile_order(): heavy tiles first in both compositors

    def use_tile_order(self, on: bool = True):
        self.tile_order = torch.empty(self.ntiles, dtype=torch.int32, device=self.ctx.device) if on else None

    def set_camera(self, cam):
        self.cam = make_camera(cam)

    def forward(self):
        legs_preprocess(self.ctx, self.g, self.cam, self.frame)
        legs_bin_and_sort(self.ctx, self.frame, self.cam, self.g.n, self.capacity, self.keys_sorted, self.vals_sorted,
                          self.ranges, self.sort_ws)
        if self.tile_order is not None:
            legs_tile_order(self.ctx, self.ranges, self.tile_order)
        legs_render_forward(self.ctx, self.g, self.cam, self.frame, self.vals_sorted, self.ranges, self.out,
                            self.n_contrib, self.sem_bf16, self.block_masks, self.tile_order)
        return self.out

    def backward(self, dL_dpixels, grads: Grads, flags: int = 0):
        if self.bwd_ws is None:
            self.bwd_ws = torch.empty(legs_backward_workspace_bytes(self.g.n, self.F), dtype=torch.uint8,
                                      device=self.ctx.device)
        legs_render_backward(self.ctx, self.g, self.cam, self.frame, self.vals_sorted, self.ranges, self.out,
                             self.n_contrib, dL_dpixels, flags, grads, self.bwd_ws, self.block_masks, self.tile_order)
        return grads
