"""mg_render_loss_static: the render loss for callers that cannot allocate device memory.

Who needs it: code that runs inside a host application which reserved the whole GPU for its own memory manager and
passes in nothing but input and output buffers; plug-ins and callbacks under a "no allocation after initialisation"
rule; frame loops that cannot afford the device-wide stall of cudaMalloc / cudaFree.  mg_render_loss wants a workspace
from such a caller (9 floats per pixel) that it has nowhere to take from; mg_render_loss_static keeps that scratch in a
fixed array inside libmg.so instead (at most 2^21 pixels, 72 MiB per GPU) and takes inputs and outputs only.

What is checked: on two calls in a row -- the second on a smaller image, so that it runs over what the first one left in
the shared array -- the loss statistics and dL/dimage agree with mg_render_loss given a caller workspace, within the
tolerances tests/test_gpu_render_loss.py holds that path to against the oracle.  (The kernels are the same, so the
gradient is in fact expected to be identical; the three sums are accumulated with atomics in both paths and may differ
in the last bits.)  An image beyond the limit must be refused with MG_ERR_CAPACITY and a message that states the limit,
before anything touches the GPU -- that part runs without one.

This file is named to be collected last: with `pytest -x` a failure here cannot hide another test.  It depends on no
state of the tests before it and passes alone in a fresh process as well (the first call on a device does its own set-up).
"""
import ctypes as C

import numpy as np
import pytest


def _images(h, w, seed):
    rng = np.random.default_rng(seed)
    yy, xx = np.mgrid[0:h, 0:w]
    base = 0.5 + 0.4 * np.sin(xx / 17.0)[None] * np.cos(yy / 23.0)[None] * np.array([1.0, 0.7, 0.4])[:, None, None]
    target = base.astype(np.float32)
    image = np.clip(target + rng.normal(0, 0.05, target.shape), 0, 1).astype(np.float32)
    return image, target


@pytest.mark.gpu
def test_static_scratch_matches_the_workspace_path_on_two_calls_in_a_row():
    import torch

    from paper_2412_20522_b200 import binding as mg

    lam = 0.2
    # first the bench image size (ragged 32x32 tiles on both edges), then a smaller one over the first call's leftovers
    cases = [(840, 1297, 11), (211, 333, 12)]
    dev = []
    for h, w, seed in cases:  # every buffer exists before the first call: the calls under test get inputs and outputs only
        x, y = _images(h, w, seed)
        img, tgt = torch.from_numpy(x).cuda(), torch.from_numpy(y).cuda()
        dev.append(dict(img=img, tgt=tgt, grad_static=torch.full_like(img, float("nan")), grad_ws=torch.full_like(img, float("nan")),
                        stats_static=torch.full((3,), float("nan"), dtype=torch.float64, device="cuda"),
                        stats_ws=torch.full((3,), float("nan"), dtype=torch.float64, device="cuda"),
                        ws=torch.empty(mg.mg_render_loss_workspace_bytes(w, h), dtype=torch.uint8, device="cuda")))
    for d in dev:  # the two calls of the new entry point, back to back on one stream
        mg.mg_render_loss_static(d["img"], d["tgt"], lam, d["grad_static"], d["stats_static"])
    for d in dev:  # the existing path, each call with a workspace of its own
        mg.mg_render_loss(d["img"], d["tgt"], lam, d["grad_ws"], d["stats_ws"], d["ws"])
    torch.cuda.synchronize()
    for d, (h, w, _) in zip(dev, cases):
        st, ref_st = d["stats_static"].cpu().numpy(), d["stats_ws"].cpu().numpy()
        assert np.isfinite(st).all() and np.isfinite(ref_st).all(), (h, w, st, ref_st)
        assert st[0] == pytest.approx(ref_st[0], rel=1e-6, abs=1e-12)  # mean |I - G|
        assert st[1] == pytest.approx(ref_st[1], rel=2e-5, abs=1e-7)   # mean SSIM
        assert st[2] == pytest.approx(ref_st[2], rel=2e-5, abs=1e-7)   # L_render
        g, ref = d["grad_static"].cpu().numpy().astype(np.float64), d["grad_ws"].cpu().numpy().astype(np.float64)
        assert np.isfinite(g).all() and np.abs(ref).max() > 0
        tol = 1e-3 * np.abs(ref) + 2e-5 * np.abs(ref).max()
        bad = np.abs(g - ref) > tol
        assert not bad.any(), (h, w, int(bad.sum()), float(np.abs(g - ref).max()))
        assert np.linalg.norm(g - ref) <= 1e-4 * np.linalg.norm(ref)


def test_static_scratch_rejects_an_image_beyond_its_limit():
    """Needs no GPU: the size is checked before any CUDA call, so the null pointers are never looked at."""
    from paper_2412_20522_b200 import binding as mg
    from paper_2412_20522_b200 import build

    build.build()
    L = mg.lib()
    null = C.c_void_p(0)
    limit = mg.RENDER_LOSS_STATIC_MAX_PIXELS
    assert limit == 1 << 21 and 1920 * 1080 <= limit
    for w, h in ((2048, 1025), (1 << 20, 3), (46341, 46341)):  # the last one would overflow a 32-bit product
        rc = L.mg_render_loss_static(C.c_int32(w), C.c_int32(h), null, null, C.c_float(0.2), null, null, null)
        msg = L.mg_last_error_string().decode()
        assert rc == mg.MG_ERR_CAPACITY, (w, h, rc, msg)
        assert str(limit) in msg and "mg_render_loss " in msg, msg
    rc = L.mg_render_loss_static(C.c_int32(0), C.c_int32(5), null, null, C.c_float(0.2), null, null, null)
    assert rc == mg.MG_ERR_INVALID_ARG
