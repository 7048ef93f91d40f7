"""Thin ctypes binding of libmg.so (include/mg.h): argument marshalling only.

Every step of the path runs in the CUDA kernels of csrc/.  torch is used for device memory, streams
and nothing else.  There is no CPU fallback: if libmg.so is missing or a call fails, this raises.
Function names and argument order follow include/mg.h.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmg.so")
_lib = None

MG_OK, MG_ERR_INVALID_ARG, MG_ERR_CAPACITY, MG_ERR_CUDA = 0, -1, -2, -3
TILE = 16


class MgError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libmg error {code}: {msg}")
        self.code = code


class mg_camera(C.Structure):
    _fields_ = [("width", C.c_int32), ("height", C.c_int32), ("fx", C.c_float), ("fy", C.c_float),
                ("cx", C.c_float), ("cy", C.c_float), ("R", C.c_float * 9), ("t", C.c_float * 3),
                ("bg", C.c_float * 3), ("sh_degree", C.c_int32)]


EXPORTS = ["mg_last_error_string", "mg_version", "mg_workspace_bytes", "mg_preprocess", "mg_bin_sort",
           "mg_render_fwd", "mg_render_bwd", "mg_preprocess_bwd", "mg_mask_sample", "mg_mask_sample_bwd", "mg_mask_loss",
           "mg_mask_prune_keep", "mg_compact_workspace_bytes", "mg_compact", "mg_render_loss_workspace_bytes",
           "mg_render_loss", "mg_render_loss_static", "mg_density_stats", "mg_adam_step", "mg_measure_fp32_peak"]


def load_library(path):
    """ctypes handle of a build of the library at `path`, with the return and argument types of include/mg.h set."""
    if not os.path.exists(path):
        raise MgError(MG_ERR_CUDA, f"{path} not built; run python -m paper_2412_20522_b200.build "
                                   "(there is no CPU fallback)")
    L = C.CDLL(path)
    L.mg_last_error_string.restype = C.c_char_p
    L.mg_workspace_bytes.restype = C.c_size_t
    L.mg_workspace_bytes.argtypes = [C.c_int64, C.c_int32, C.c_int32, C.c_uint64]
    L.mg_render_loss_workspace_bytes.restype = C.c_size_t
    L.mg_render_loss_workspace_bytes.argtypes = [C.c_int32, C.c_int32]
    L.mg_compact_workspace_bytes.restype = C.c_size_t
    L.mg_compact_workspace_bytes.argtypes = [C.c_int64]
    for name in EXPORTS[3:]:
        if not name.endswith("_workspace_bytes"):
            getattr(L, name).restype = C.c_int
    return L


def lib():
    """Load libmg.so (built by `python -m paper_2412_20522_b200.build`).  Raises if it is missing."""
    global _lib
    if _lib is None:
        _lib = load_library(LIB_PATH)
    return _lib


def _check(rc):
    if rc != MG_OK:
        raise MgError(rc, lib().mg_last_error_string().decode())


def camera(cam) -> mg_camera:
    """From a scenes.Camera-like object (width, height, fx, fy, cx, cy, R, t, bg, sh_degree)."""
    c = mg_camera()
    c.width, c.height = int(cam.width), int(cam.height)
    c.fx, c.fy, c.cx, c.cy = float(cam.fx), float(cam.fy), float(cam.cx), float(cam.cy)
    for i, v in enumerate(np.asarray(cam.R, np.float64).reshape(-1)):
        c.R[i] = float(v)
    for i, v in enumerate(np.asarray(cam.t, np.float64).reshape(-1)):
        c.t[i] = float(v)
    for i, v in enumerate(cam.bg):
        c.bg[i] = float(v)
    c.sh_degree = int(cam.sh_degree)
    return c


def grid(cam):
    return (cam.width + TILE - 1) // TILE, (cam.height + TILE - 1) // TILE


def _ptr(t, dtype=None, device="cuda"):
    if t is None:
        return C.c_void_p(0)
    assert t.is_contiguous(), "tensor must be contiguous"
    assert t.device.type == device, f"tensor must live on {device}"
    if dtype is not None:
        assert t.dtype == dtype, f"expected {dtype}, got {t.dtype}"
    return C.c_void_p(t.data_ptr())


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


F32, I32, U8 = torch.float32, torch.int32, torch.uint8


def mg_workspace_bytes(N, width, height, R_capacity) -> int:
    return int(lib().mg_workspace_bytes(int(N), int(width), int(height), int(R_capacity)))


def mg_preprocess(cam: mg_camera, means, log_scales, quats, opacity_logits, sh, means2d, depths, conic_opacity, rgb,
                  radii, rects, tiles_touched, clamped, num_rendered=None, num_rendered_host=None):
    N = means.shape[0]
    _check(lib().mg_preprocess(C.byref(cam), C.c_int64(N), _ptr(means, F32), _ptr(log_scales, F32), _ptr(quats, F32),
                               _ptr(opacity_logits, F32), _ptr(sh, F32), _ptr(means2d, F32), _ptr(depths, F32),
                               _ptr(conic_opacity, F32), _ptr(rgb, F32), _ptr(radii, I32), _ptr(rects, I32),
                               _ptr(tiles_touched, I32), _ptr(clamped, U8), _ptr(num_rendered, torch.int64),
                               _ptr(num_rendered_host, torch.int64, "cpu"), _stream()))


def mg_bin_sort(cam: mg_camera, depths, rects, tiles_touched, R_capacity, workspace, sorted_ids, tile_ranges,
                R_out_host=None, tile_order=None):
    N = depths.shape[0]
    _check(lib().mg_bin_sort(C.byref(cam), C.c_int64(N), _ptr(depths, F32), _ptr(rects, I32), _ptr(tiles_touched, I32),
                             C.c_uint64(int(R_capacity)), _ptr(workspace, U8), C.c_size_t(workspace.numel()),
                             _ptr(sorted_ids, I32), _ptr(tile_ranges, I32), _ptr(tile_order, I32),
                             _ptr(R_out_host, torch.int64, "cpu"), _stream()))


def mg_render_fwd(cam: mg_camera, sorted_ids, tile_ranges, means2d, conic_opacity, rgb, masks, image, final_T,
                  n_contrib, tile_order=None):
    _check(lib().mg_render_fwd(C.byref(cam), _ptr(sorted_ids, I32), _ptr(tile_ranges, I32), _ptr(tile_order, I32),
                               _ptr(means2d, F32),
                               _ptr(conic_opacity, F32), _ptr(rgb, F32), _ptr(masks, F32), _ptr(image, F32),
                               _ptr(final_T, F32), _ptr(n_contrib, I32), _stream()))


def mg_render_bwd(cam: mg_camera, N, sorted_ids, tile_ranges, means2d, conic_opacity, rgb, masks, final_T, n_contrib,
                  dL_dimage, dL_dmeans2d, dL_dconic, dL_dopacity, dL_drgb, dL_dmask, tile_order=None):
    _check(lib().mg_render_bwd(C.byref(cam), C.c_int64(N), _ptr(sorted_ids, I32), _ptr(tile_ranges, I32),
                               _ptr(tile_order, I32), _ptr(means2d, F32), _ptr(conic_opacity, F32), _ptr(rgb, F32), _ptr(masks, F32),
                               _ptr(final_T, F32), _ptr(n_contrib, I32), _ptr(dL_dimage, F32), _ptr(dL_dmeans2d, F32),
                               _ptr(dL_dconic, F32), _ptr(dL_dopacity, F32), _ptr(dL_drgb, F32), _ptr(dL_dmask, F32),
                               _stream()))


def mg_preprocess_bwd(cam: mg_camera, means, log_scales, quats, opacity_logits, sh, radii, clamped, dL_dmeans2d,
                      dL_dconic, dL_dopacity, dL_drgb, dL_dmeans, dL_dlog_scales, dL_dquats, dL_dopacity_logits,
                      dL_dsh):
    N = means.shape[0]
    _check(lib().mg_preprocess_bwd(C.byref(cam), C.c_int64(N), _ptr(means, F32), _ptr(log_scales, F32),
                                   _ptr(quats, F32), _ptr(opacity_logits, F32), _ptr(sh, F32), _ptr(radii, I32),
                                   _ptr(clamped, U8), _ptr(dL_dmeans2d, F32), _ptr(dL_dconic, F32),
                                   _ptr(dL_dopacity, F32), _ptr(dL_drgb, F32), _ptr(dL_dmeans, F32),
                                   _ptr(dL_dlog_scales, F32), _ptr(dL_dquats, F32), _ptr(dL_dopacity_logits, F32),
                                   _ptr(dL_dsh, F32), _stream()))


def mg_mask_sample(scores, uniforms, tau, masks, soft=None):
    N = scores.shape[0]
    _check(lib().mg_mask_sample(C.c_int64(N), _ptr(scores, F32), _ptr(uniforms, F32), C.c_float(tau), _ptr(masks, F32),
                                _ptr(soft, F32), _stream()))


def mg_mask_sample_bwd(soft, dL_dmask, tau, dL_dscores):
    N = soft.shape[0]
    _check(lib().mg_mask_sample_bwd(C.c_int64(N), _ptr(soft, F32), _ptr(dL_dmask, F32), C.c_float(tau),
                                    _ptr(dL_dscores, F32), _stream()))


def mg_mask_loss(masks, lambda_m, dL_dmask, stats):
    N = masks.shape[0]
    _check(lib().mg_mask_loss(C.c_int64(N), _ptr(masks, F32), C.c_float(lambda_m), _ptr(dL_dmask, F32),
                              _ptr(stats, torch.float64), _stream()))


def mg_mask_prune_keep(scores, uniforms, keep):
    N, S = scores.shape[0], uniforms.shape[0]
    _check(lib().mg_mask_prune_keep(C.c_int64(N), C.c_int32(S), _ptr(scores, F32), _ptr(uniforms, F32), _ptr(keep, U8),
                                    _stream()))


def mg_compact_workspace_bytes(N) -> int:
    return int(lib().mg_compact_workspace_bytes(int(N)))


def mg_compact(keep, src, dst, workspace, N_out_host=None):
    """src / dst: lists of contiguous fp32 tensors with N rows each (row size = numel / N)."""
    N = keep.shape[0]
    n = len(src)
    srcp = (C.c_void_p * n)(*[t.data_ptr() for t in src])
    dstp = (C.c_void_p * n)(*[t.data_ptr() for t in dst])
    rows = (C.c_int32 * n)(*[(t.numel() // N if N else 1) for t in src])
    for t in list(src) + list(dst):
        assert t.is_contiguous() and t.dtype == F32 and t.device.type == "cuda"
    _check(lib().mg_compact(C.c_int64(N), _ptr(keep, U8), C.c_int32(n), srcp, dstp, rows, _ptr(workspace, U8),
                            C.c_size_t(workspace.numel()), _ptr(N_out_host, torch.int64, "cpu"), _stream()))


def mg_render_loss_workspace_bytes(width, height) -> int:
    return int(lib().mg_render_loss_workspace_bytes(int(width), int(height)))


def mg_render_loss(image, target, lambda_dssim, dL_dimage, stats, workspace):
    _, H, W = image.shape
    _check(lib().mg_render_loss(C.c_int32(W), C.c_int32(H), _ptr(image, F32), _ptr(target, F32), C.c_float(lambda_dssim),
                                _ptr(dL_dimage, F32), _ptr(stats, torch.float64), _ptr(workspace, U8),
                                C.c_size_t(workspace.numel()), _stream()))


RENDER_LOSS_STATIC_MAX_PIXELS = 1 << 21  # MG_RENDER_LOSS_STATIC_MAX_PIXELS of include/mg.h


def mg_render_loss_static(image, target, lambda_dssim, dL_dimage, stats):
    """mg_render_loss without a workspace argument, for callers that cannot allocate device memory: the scratch is an
    array inside libmg.so (72 MiB per GPU), shared by all calls on a device -- calls that overlap on the GPU race.
    Images of more than RENDER_LOSS_STATIC_MAX_PIXELS pixels raise MgError(MG_ERR_CAPACITY).  See include/mg.h."""
    _, H, W = image.shape
    _check(lib().mg_render_loss_static(C.c_int32(W), C.c_int32(H), _ptr(image, F32), _ptr(target, F32),
                                       C.c_float(lambda_dssim), _ptr(dL_dimage, F32), _ptr(stats, torch.float64), _stream()))


def mg_density_stats(dL_dmeans2d, radii, scale, grad_accum, denom, max_radii):
    N = radii.shape[0]
    _check(lib().mg_density_stats(C.c_int64(N), _ptr(dL_dmeans2d, F32), _ptr(radii, I32), C.c_float(scale[0]),
                                  C.c_float(scale[1]), _ptr(grad_accum, F32), _ptr(denom, F32), _ptr(max_radii, F32),
                                  _stream()))


class mg_adam_group(C.Structure):
    _fields_ = [("param", C.c_void_p), ("grad", C.c_void_p), ("m", C.c_void_p), ("v", C.c_void_p),
                ("n_rows", C.c_int64), ("row_floats", C.c_int32), ("lr", C.c_float)]


def mg_adam_step(groups, beta1, beta2, eps, step, radii=None):
    """groups: list of (param, grad, m, v, lr) with contiguous fp32 device tensors of one shape [n_rows, ...] each."""
    arr = (mg_adam_group * max(len(groups), 1))()
    for k, (p, g, m, v, lr) in enumerate(groups):
        for t in (p, g, m, v):
            assert t.is_contiguous() and t.dtype == F32 and t.device.type == "cuda" and t.shape == p.shape
        n_rows = p.shape[0]
        arr[k].param, arr[k].grad, arr[k].m, arr[k].v = p.data_ptr(), g.data_ptr(), m.data_ptr(), v.data_ptr()
        arr[k].n_rows, arr[k].row_floats, arr[k].lr = n_rows, (p.numel() // n_rows if n_rows else 1), float(lr)
    _check(lib().mg_adam_step(C.c_int32(len(groups)), arr, C.c_float(beta1), C.c_float(beta2), C.c_float(eps),
                              C.c_int64(step), _ptr(radii, I32), _stream()))


def mg_measure_fp32_peak(min_seconds=0.05):
    """-> dict of TFLOP/s: scalar FFMA and packed f32x2, sustained and best round (synchronous)."""
    out = (C.c_double * 4)()
    scratch = torch.zeros(1, dtype=F32, device="cuda")
    _check(lib().mg_measure_fp32_peak(C.c_double(min_seconds), out, _ptr(scratch, F32), _stream()))
    return {"ffma_sustained": out[0], "ffma_best": out[1], "ffma2_sustained": out[2], "ffma2_best": out[3]}


class Frame:
    """Device buffers of one camera view + the five calls in order.  Allocation and marshalling only.

    uint32 arrays of the C-ABI (tiles_touched, sorted_ids, tile_ranges, n_contrib) are held as torch.int32
    tensors (same bits; torch has no arithmetic on uint32).
    """

    def __init__(self, cam_like, N, device="cuda"):
        self.cam_like = cam_like
        self.cam = camera(cam_like)
        self.N = N
        K = (cam_like.sh_degree + 1) ** 2
        H, W = cam_like.height, cam_like.width
        gw, gh = grid(cam_like)
        e = lambda *s, dt=F32: torch.empty(*s, dtype=dt, device=device)
        self.means2d, self.depths, self.conic_opacity, self.rgb = e(N, 2), e(N), e(N, 4), e(N, 3)
        self.radii, self.rects, self.tiles_touched = e(N, dt=I32), e(N, 4, dt=I32), e(N, dt=I32)
        self.clamped = e(N, dt=U8)
        self.tile_ranges = e(gw * gh, 2, dt=I32)
        self.tile_order = e(gw * gh, dt=I32)  # scheduling hint: longest tile lists first
        self.image, self.final_T, self.n_contrib = e(3, H, W), e(H, W), e(H, W, dt=I32)
        self.dL_dmeans2d, self.dL_dconic, self.dL_dopacity = e(N, 2), e(N, 3), e(N)
        self.dL_drgb, self.dL_dmask = e(N, 3), e(N)
        self.dL_dmeans, self.dL_dlog_scales, self.dL_dquats = e(N, 3), e(N, 3), e(N, 4)
        self.dL_dopacity_logits, self.dL_dsh = e(N), e(N, K, 3)
        self.R_dev = torch.zeros(1, dtype=torch.int64, device=device)  # mg_preprocess's counter (caller-owned)
        self.R_host = torch.zeros(2, dtype=torch.int64).pin_memory()
        self.R_capacity = 0
        self.R = 0
        self.sorted_ids = None
        self.workspace = None

    def set_camera(self, cam_like):
        """Point the frame at another camera of the same image size (buffers are reused)."""
        assert (cam_like.width, cam_like.height, cam_like.sh_degree) == (self.cam_like.width, self.cam_like.height,
                                                                         self.cam_like.sh_degree)
        self.cam_like = cam_like
        self.cam = camera(cam_like)

    def reserve(self, R_capacity):
        """(Re)allocate sorted_ids and the sort workspace for at most R_capacity duplicated keys."""
        if R_capacity > self.R_capacity or self.sorted_ids is None:
            self.R_capacity = int(R_capacity)
            self.sorted_ids = torch.empty(max(self.R_capacity, 1), dtype=I32, device=self.means2d.device)
            nbytes = mg_workspace_bytes(self.N, self.cam.width, self.cam.height, self.R_capacity)
            self.workspace = torch.empty(nbytes, dtype=U8, device=self.means2d.device)

    def preprocess(self, g):
        mg_preprocess(self.cam, g["means"], g["log_scales"], g["quats"], g["opacity_logits"], g["sh"], self.means2d,
                      self.depths, self.conic_opacity, self.rgb, self.radii, self.rects, self.tiles_touched,
                      self.clamped, self.R_dev, self.R_host[0:1])

    def bin_sort(self):
        mg_bin_sort(self.cam, self.depths, self.rects, self.tiles_touched, self.R_capacity, self.workspace,
                    self.sorted_ids, self.tile_ranges, self.R_host[1:2], self.tile_order)

    def render_fwd(self, masks):
        mg_render_fwd(self.cam, self.sorted_ids, self.tile_ranges, self.means2d, self.conic_opacity, self.rgb, masks,
                      self.image, self.final_T, self.n_contrib, self.tile_order)

    def render_bwd(self, masks, dL_dimage):
        mg_render_bwd(self.cam, self.N, self.sorted_ids, self.tile_ranges, self.means2d, self.conic_opacity, self.rgb,
                      masks, self.final_T, self.n_contrib, dL_dimage, self.dL_dmeans2d, self.dL_dconic,
                      self.dL_dopacity, self.dL_drgb, self.dL_dmask, self.tile_order)

    def preprocess_bwd(self, g):
        mg_preprocess_bwd(self.cam, g["means"], g["log_scales"], g["quats"], g["opacity_logits"], g["sh"], self.radii,
                          self.clamped, self.dL_dmeans2d, self.dL_dconic, self.dL_dopacity, self.dL_drgb,
                          self.dL_dmeans, self.dL_dlog_scales, self.dL_dquats, self.dL_dopacity_logits, self.dL_dsh)

    def forward(self, g, masks):
        """Calls 1-3.  Sizes the sort buffers from the exact R (one stream sync) unless they already fit."""
        self.preprocess(g)
        torch.cuda.current_stream().synchronize()
        self.R = int(self.R_host[0])
        self.reserve(self.R)
        self.bin_sort()
        self.render_fwd(masks)

    def backward(self, g, masks, dL_dimage):
        self.render_bwd(masks, dL_dimage)
        self.preprocess_bwd(g)

    def step(self, g, masks, dL_dimage):
        """One pass of the whole hot path with pre-reserved buffers and no host sync (bench inner loop)."""
        self.preprocess(g)
        self.bin_sort()
        self.render_fwd(masks)
        self.render_bwd(masks, dL_dimage)
        self.preprocess_bwd(g)


def upload(scene, device="cuda"):
    """Scene arrays (numpy fp32) -> dict of device tensors + masks."""
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(device)
    g = dict(means=t(scene.means), log_scales=t(scene.log_scales), quats=t(scene.quats),
             opacity_logits=t(scene.opacity_logits), sh=t(scene.sh))
    return g, t(scene.masks)
