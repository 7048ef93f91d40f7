"""CPU oracle for the masked-rasterization hot path (TEST INFRASTRUCTURE, not the product).

ctypes binding of oracle/mg_oracle.cpp (fp64, brute force; see that file's header for the
paper citations).  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this package; paper_2412_20522_b200 never does.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

_lib = None


class _Cam(C.Structure):
    _fields_ = [("width", C.c_int32), ("height", C.c_int32), ("fx", C.c_double), ("fy", C.c_double),
                ("cx", C.c_double), ("cy", C.c_double), ("R", C.c_double * 9), ("t", C.c_double * 3),
                ("bg", C.c_double * 3), ("sh_degree", C.c_int32)]


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
    return _lib


def set_threads(n: int) -> None:
    os.environ["OMP_NUM_THREADS"] = str(n)


def _cam(cam) -> _Cam:
    """The camera the GPU sees is fp32; the oracle takes those same values, upcast."""
    f = lambda v: float(np.float32(v))
    c = _Cam()
    c.width, c.height = int(cam.width), int(cam.height)
    c.fx, c.fy, c.cx, c.cy = f(cam.fx), f(cam.fy), f(cam.cx), f(cam.cy)
    for i, v in enumerate(np.asarray(cam.R, np.float64).reshape(-1)):
        c.R[i] = f(v)
    for i, v in enumerate(np.asarray(cam.t, np.float64).reshape(-1)):
        c.t[i] = f(v)
    for i, v in enumerate(cam.bg):
        c.bg[i] = f(v)
    c.sh_degree = int(cam.sh_degree)
    return c


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _in(a, dtype):
    return np.ascontiguousarray(a, dtype=dtype)


def grid(cam):
    return (cam.width + 15) // 16, (cam.height + 15) // 16


def preprocess(cam, means, log_scales, quats, opacity_logits, sh):
    """O1-O8.  Inputs: the fp32 arrays the GPU gets (upcast exactly) or fp64 (FD pin).  Returns fp64/int arrays."""
    N = means.shape[0]
    means, log_scales, quats = _in(means, np.float64), _in(log_scales, np.float64), _in(quats, np.float64)
    opacity_logits, sh = _in(opacity_logits, np.float64), _in(sh, np.float64)
    assert sh.shape == (N, (cam.sh_degree + 1) ** 2, 3)
    out = dict(means2d=np.zeros((N, 2)), depths=np.zeros(N), conic_opacity=np.zeros((N, 4)), rgb=np.zeros((N, 3)),
               radii=np.zeros(N, np.int32), rects=np.zeros((N, 4), np.int32), tiles_touched=np.zeros(N, np.uint32),
               clamped=np.zeros(N, np.uint8), margin=np.zeros(N))
    c = _cam(cam)
    rc = lib().orc_preprocess(C.byref(c), C.c_int64(N), _p(means), _p(log_scales), _p(quats), _p(opacity_logits), _p(sh),
                              _p(out["means2d"]), _p(out["depths"]), _p(out["conic_opacity"]), _p(out["rgb"]),
                              _p(out["radii"]), _p(out["rects"]), _p(out["tiles_touched"]), _p(out["clamped"]),
                              _p(out["margin"]))
    assert rc == 0
    return out


def bin_sort(cam, depths, rects, tiles_touched, tile_select=None):
    """O9.  depths are taken as fp32 (their bit pattern is the sort key).  tile_select: optional uint8 per tile."""
    N = depths.shape[0]
    depths, rects, tiles_touched = _in(depths, np.float32), _in(rects, np.int32), _in(tiles_touched, np.uint32)
    R = int(tiles_touched.astype(np.uint64).sum())
    gw, gh = grid(cam)
    sorted_ids = np.zeros(max(R, 1), np.uint32)
    tile_ranges = np.zeros((gw * gh, 2), np.uint32)
    R_out = C.c_uint64(0)
    c = _cam(cam)
    sel = None if tile_select is None else _in(tile_select, np.uint8)
    assert sel is None or sel.shape == (gw * gh,)
    rc = lib().orc_bin_sort(C.byref(c), C.c_int64(N), _p(depths), _p(rects), _p(tiles_touched), _p(sorted_ids),
                            _p(tile_ranges), C.byref(R_out), None if sel is None else _p(sel))
    assert rc == 0 and (R_out.value == R if sel is None else R_out.value <= R)
    return sorted_ids[:R_out.value], tile_ranges


def _counts(out, counts):
    c = [int(v) for v in counts]
    out["pair_evals"], out["pair_evals_masked"] = c[0] + c[1], c[1]
    out["blends"], out["blends_masked"] = c[2] + c[3], c[3]


def render_fwd(cam, sorted_ids, tile_ranges, means2d, conic_opacity, rgb, masks):
    """O10.  Returns dict(image [3,H,W], final_T, n_contrib, margin, hash) + the work counters of SURVEY.md 8(d):
    pair_evals / blends (totals) and pair_evals_masked / blends_masked (the part on entries with M == 0)."""
    H, W = cam.height, cam.width
    sorted_ids, tile_ranges = _in(sorted_ids, np.uint32), _in(tile_ranges, np.uint32)
    means2d, conic_opacity, rgb = _in(means2d, np.float64), _in(conic_opacity, np.float64), _in(rgb, np.float64)
    masks = _in(masks, np.float32)
    out = dict(image=np.zeros((3, H, W)), final_T=np.zeros((H, W)), n_contrib=np.zeros((H, W), np.uint32),
               margin=np.zeros((H, W)), hash=np.zeros((H, W), np.uint64))
    counts = np.zeros(4, np.uint64)
    c = _cam(cam)
    rc = lib().orc_render_fwd(C.byref(c), _p(sorted_ids), _p(tile_ranges), _p(means2d), _p(conic_opacity), _p(rgb),
                              _p(masks), _p(out["image"]), _p(out["final_T"]), _p(out["n_contrib"]), _p(out["margin"]),
                              _p(out["hash"]), _p(counts))
    assert rc == 0
    _counts(out, counts)
    return out


def render_bwd(cam, N, sorted_ids, tile_ranges, means2d, conic_opacity, rgb, masks, dL_dimage, cutoff=0.0):
    """O11.  Returns dict of fp64 gradients (+ sens flags when cutoff > 0, + revisit counts)."""
    sorted_ids, tile_ranges = _in(sorted_ids, np.uint32), _in(tile_ranges, np.uint32)
    means2d, conic_opacity, rgb = _in(means2d, np.float64), _in(conic_opacity, np.float64), _in(rgb, np.float64)
    masks, dL_dimage = _in(masks, np.float32), _in(dL_dimage, np.float64)
    assert dL_dimage.shape == (3, cam.height, cam.width)
    out = dict(dL_dmeans2d=np.zeros((N, 2)), dL_dconic=np.zeros((N, 3)), dL_dopacity=np.zeros(N),
               dL_drgb=np.zeros((N, 3)), dL_dmask=np.zeros(N), sens=np.zeros(N, np.uint32))
    counts = np.zeros(4, np.uint64)
    c = _cam(cam)
    rc = lib().orc_render_bwd(C.byref(c), C.c_int64(N), _p(sorted_ids), _p(tile_ranges), _p(means2d), _p(conic_opacity),
                              _p(rgb), _p(masks), _p(dL_dimage), _p(out["dL_dmeans2d"]), _p(out["dL_dconic"]),
                              _p(out["dL_dopacity"]), _p(out["dL_drgb"]), _p(out["dL_dmask"]),
                              _p(out["sens"]) if cutoff > 0 else None, C.c_double(cutoff), _p(counts))
    assert rc == 0
    _counts(out, counts)
    return out


def preprocess_bwd(cam, means, log_scales, quats, opacity_logits, sh, dL_dmeans2d, dL_dconic, dL_dopacity, dL_drgb):
    """O12.  Returns dict of fp64 gradients w.r.t. the five raw input arrays."""
    N = means.shape[0]
    K = (cam.sh_degree + 1) ** 2
    means, log_scales, quats = _in(means, np.float64), _in(log_scales, np.float64), _in(quats, np.float64)
    opacity_logits, sh = _in(opacity_logits, np.float64), _in(sh, np.float64)
    g2, gc, go, gr = (_in(dL_dmeans2d, np.float64), _in(dL_dconic, np.float64), _in(dL_dopacity, np.float64),
                      _in(dL_drgb, np.float64))
    out = dict(dL_dmeans=np.zeros((N, 3)), dL_dlog_scales=np.zeros((N, 3)), dL_dquats=np.zeros((N, 4)),
               dL_dopacity_logits=np.zeros(N), dL_dsh=np.zeros((N, K, 3)))
    c = _cam(cam)
    rc = lib().orc_preprocess_bwd(C.byref(c), C.c_int64(N), _p(means), _p(log_scales), _p(quats), _p(opacity_logits),
                                  _p(sh), _p(g2), _p(gc), _p(go), _p(gr), _p(out["dL_dmeans"]),
                                  _p(out["dL_dlog_scales"]), _p(out["dL_dquats"]), _p(out["dL_dopacity_logits"]),
                                  _p(out["dL_dsh"]))
    assert rc == 0
    return out


def full_forward(cam, scene_arrays, masks):
    """Whole forward path in the oracle (fp64 between stages; depth key = fp32 rounding of fp64 depth)."""
    pre = preprocess(cam, *scene_arrays)
    ids, ranges = bin_sort(cam, pre["depths"].astype(np.float32), pre["rects"], pre["tiles_touched"])
    fwd = render_fwd(cam, ids, ranges, pre["means2d"], pre["conic_opacity"], pre["rgb"], masks)
    return pre, ids, ranges, fwd


def full_backward(cam, scene_arrays, masks, pre, ids, ranges, dL_dimage, cutoff=0.0):
    N = scene_arrays[0].shape[0]
    rb = render_bwd(cam, N, ids, ranges, pre["means2d"], pre["conic_opacity"], pre["rgb"], masks, dL_dimage, cutoff)
    pb = preprocess_bwd(cam, *scene_arrays, rb["dL_dmeans2d"], rb["dL_dconic"], rb["dL_dopacity"], rb["dL_drgb"])
    return rb, pb
