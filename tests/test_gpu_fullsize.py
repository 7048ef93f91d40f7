"""Parity at BASELINE.json's full sizes -- configs[2] (3 M Gaussians, 1297x840: the bench workload), configs[3]
(2.8 M, 1264x832, indoor) and configs[4] (6 M, 1920x1080, keep-probability 0.9: the largest size and the
longest tile lists), camera 0, SH degree 3 -- in the launch configuration bench.py times.  Projection, sort and projection-backward are compared in full; the two
blend kernels on a seeded sample of tiles the oracle can walk in seconds (the other tiles' ranges are
emptied for both sides, which leaves the sampled tiles' arithmetic untouched)."""
import numpy as np
import pytest
import torch

import parity_util as pu
from paper_2412_20522_b200 import binding as mg
from paper_2412_20522_b200 import scenes

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", params=[3, 4, 5])
def full(request, oracle):
    sc = scenes.make(request.param)
    fr, g, m, gimg = pu.run_gpu(sc)
    yield sc, fr, g, m, gimg
    del fr, g, m, gimg
    torch.cuda.empty_cache()


def test_full_size_projection_and_sort(full, oracle):
    sc, fr, *_ = full
    cam = sc.camera
    s1 = pu.check_preprocess(fr, sc, cam, max_flag_frac=0.02)
    ids, ranges = pu.check_bin_sort(fr, cam)
    assert fr.R > 10_000_000
    print("PARITY", sc.name, "full size", dict(R=fr.R, preprocess=s1))


def test_full_size_blend_on_sampled_tiles(full, oracle):
    sc, fr, g, m, gimg = full
    cam = sc.camera
    gw, gh = mg.grid(cam)
    rng = np.random.default_rng(12)
    lens = (pu.u32(fr.tile_ranges)[:, 1] - pu.u32(fr.tile_ranges)[:, 0]).astype(np.int64)
    tiles = set(rng.choice(gw * gh, 40, replace=False).tolist())
    tiles |= {int(np.argmax(lens)), gw - 1, gw * gh - 1, gw * (gh - 1)}  # longest list + ragged corners
    tiles = sorted(tiles)
    ranges_full = pu.u32(fr.tile_ranges).copy()
    ranges_s = np.zeros_like(ranges_full)
    ranges_s[tiles] = ranges_full[tiles]
    ids = pu.u32(fr.sorted_ids)[: fr.R]
    ref, s3 = pu.check_render_fwd(fr, cam, sc.masks, ids, ranges_s, tiles=tiles, max_flag_frac=4e-3)
    print("PARITY", sc.name, "full size fwd sampled tiles", dict(tiles=len(tiles), render_fwd=s3))
    # backward restricted to the same tiles on both sides
    keep_ranges = fr.tile_ranges.clone()
    fr.tile_ranges.copy_(torch.from_numpy(ranges_s.view(np.int32)).cuda())
    fr.render_bwd(m, gimg)
    torch.cuda.synchronize()
    try:
        _, s4 = pu.check_render_bwd(fr, cam, sc.N, sc.masks, ids, ranges_s, sc.dL_dimage(), max_flag_frac=2e-3)
        print("PARITY", sc.name, "full size bwd sampled tiles", dict(render_bwd=s4))
    finally:
        fr.tile_ranges.copy_(keep_ranges)
        fr.render_bwd(m, gimg)
        torch.cuda.synchronize()


@pytest.mark.parametrize("cam_index", [5, 10, 15])
def test_config5_other_cameras_on_the_circle(oracle, cam_index):
    """BASELINE.json configs[4]: "timed over 20 cameras on a circle of radius 8".  Camera 0 is the `full` fixture; the
    same full-size checks for three more of the 20 views (the scene looks different from every side: other Gaussians
    are culled, other depth order, other R): projection on all 6 M Gaussians, the sort on all keys bit-exactly, both
    blend kernels on sampled tiles, projection backward in the 2-norm."""
    sc = scenes.make(5)
    cam = sc.cameras[cam_index]
    fr, g, m, gimg = pu.run_gpu(sc, cam_index=cam_index)
    s1 = pu.check_preprocess(fr, sc, cam, max_flag_frac=0.02)
    ids, ranges = pu.check_bin_sort(fr, cam)
    assert fr.R > 40_000_000
    gw, gh = mg.grid(cam)
    lens = (ranges[:, 1].astype(np.int64) - ranges[:, 0])
    tiles = sorted(set(np.random.default_rng(cam_index).choice(gw * gh, 20, replace=False).tolist()) | {int(np.argmax(lens)), gw * gh - 1})
    ranges_s = np.zeros_like(ranges)
    ranges_s[tiles] = ranges[tiles]
    _, s3 = pu.check_render_fwd(fr, cam, sc.masks, ids, ranges_s, tiles=tiles, max_flag_frac=5e-3)
    fr.tile_ranges.copy_(torch.from_numpy(ranges_s.view(np.int32)).cuda())
    fr.render_bwd(m, gimg)
    torch.cuda.synchronize()
    _, s4 = pu.check_render_bwd(fr, cam, sc.N, sc.masks, ids, ranges_s, sc.dL_dimage(cam_index), max_flag_frac=2e-3)
    fr.tile_ranges.copy_(torch.from_numpy(ranges.view(np.int32)).cuda())
    fr.render_bwd(m, gimg)
    fr.preprocess_bwd(g)
    torch.cuda.synchronize()
    _, s5 = pu.check_preprocess_bwd(fr, sc, cam)
    for k, v in s5.items():
        assert v <= 2e-4, f"{k}: relative 2-norm error {v:.2e}"
    print("PARITY", f"cfg5 camera {cam_index}", dict(R=fr.R, preprocess=s1, render_fwd=s3, render_bwd=s4, preprocess_bwd=s5))
    del fr, g, m, gimg
    torch.cuda.empty_cache()


def test_full_size_projection_backward(full, oracle):
    sc, fr, *_ = full
    cam = sc.camera
    ref5, s5 = pu.check_preprocess_bwd(fr, sc, cam)
    for k, v in s5.items():
        assert v <= 2e-4, f"{k}: relative 2-norm error {v:.2e}"
    print("PARITY", sc.name, "full size", dict(preprocess_bwd=s5))


def test_full_size_invariants(full):
    """Properties that hold at any size: partition of unity (Eq. 16 telescoped) and range bookkeeping."""
    sc, fr, g, m, gimg = full
    ranges = pu.u32(fr.tile_ranges).astype(np.int64)
    assert (ranges[:, 1] >= ranges[:, 0]).all() and ranges[-1, 1] == fr.R and ranges[0, 0] == 0
    assert (ranges[1:, 0] == ranges[:-1, 1]).all()
    assert int(pu.u32(fr.tiles_touched).astype(np.int64).sum()) == fr.R
    # white splats, black background: image + final_T == 1 at every pixel
    rgb_keep = fr.rgb.clone()
    fr.rgb.fill_(1.0)
    fr.render_fwd(m)
    torch.cuda.synchronize()
    s = fr.image[0] + fr.final_T
    assert float((s - 1).abs().max()) < 2e-5
    fr.rgb.copy_(rgb_keep)
    fr.render_fwd(m)
    torch.cuda.synchronize()
