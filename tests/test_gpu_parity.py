"""GPU parity tests: the CUDA path through the C-ABI against the CPU oracle, on the same seeded inputs.

Staged mode: the oracle's stage k runs on the GPU's fp32
outputs of stage k-1, so integers (sorted ids, tile ranges, last-contributor indices) compare bit for bit
and floats within north_star's tolerances.  End-to-end mode compares against the oracle run from the raw
inputs in fp64.  Pixels / Gaussians whose decisions sit within fp32 reach of a threshold are excluded,
counted, and the count is bounded.
"""
import numpy as np
import pytest
import torch

import parity_util as pu
from paper_2412_20522_b200 import binding as mg
from paper_2412_20522_b200 import scenes

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _need_gpu():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    mg.lib()  # fails loudly if libmg.so is missing: there is no fallback


# Largest fraction of Gaussians the end-to-end gradient comparison may exempt as threshold-sensitive (at most twice the
# count observed on the B200, profiles/r03_parity_counts.md; cfg2: 0.375 observed).
# End to end the fp32 chain (projection -> blend -> two backward stages) is held against the fp64 chain from the raw
# inputs at north_star's 1e-3 relative, elementwise, with the absolute floor of the staged projection-backward comparison
# (1e-4 of the array's largest element: an element that is the sum of cancelling per-pixel terms has no relative accuracy
# of its own).  Measured on the B200 at this tolerance: worst error / tolerance 0.24 (cfg4_small dL_dmeans2d), 0.235 (cfg2
# dL_dquats), <= 0.16 everywhere else.  (With a floor of 1e-5 every array of every scene still passes except ONE element
# each of cfg2 dL_dquats, at 1.09 x, and cfg4_small dL_dmeans2d, at 1.03 x.)
E2E_GRAD_RTOL = 1e-3
E2E_GRAD_FLOOR = 1e-4
E2E_GRAD_BUDGET = {"tiny": 0.0, "cfg1": 0.136, "cfg2": 0.40, "cfg3_small": 0.072, "cfg4_small": 0.064}
# Scenes whose END-TO-END comparison is ill-posed in fp32 and is therefore held in the 2-norm only.  "needles": the conic
# that mg_preprocess stores is fp32 (relative rounding 6e-8 per component); at a pixel thousands of pixels from the
# centre of a long thin splat the terms A dx^2, B dx dy, C dy^2 reach 1e4..1e6 and cancel, so that rounding alone moves
# the exponent by 1e-3..1e-1 whatever the blend kernel does.  The kernel's own arithmetic on those splats is checked by
# the STAGED test (the oracle runs on the fp32 conics), elementwise, with no allowance.
E2E_L2_ONLY = {"needles": 5e-3}  # observed 2.2e-3


def small_scenes():
    return {
        "tiny": lambda: scenes.tiny_fd_scene(),
        "cfg1": lambda: scenes.config1(),
        "cfg2": lambda: scenes.config2(),
        # ragged image (partial tiles on both edges), outdoor generator with huge background splats
        "cfg3_small": lambda: scenes.config3(n=60_000, width=333, height=211),
        "cfg4_small": lambda: scenes.config4(n=50_000, width=320, height=208),
        # long thin splats far from their centres: the terms of the exponent reach 1e4..1e6 and cancel
        "needles": lambda: scenes.needles(),
    }


@pytest.fixture(scope="module", params=list(small_scenes()))
def run(request, oracle):
    sc = small_scenes()[request.param]()
    fr, g, m, gimg = pu.run_gpu(sc)
    return request.param, sc, fr


def test_staged_parity_all_five_calls(run, oracle):
    name, sc, fr = run
    cam = sc.camera
    s1 = pu.check_preprocess(fr, sc, cam, max_flag_frac=0.02)
    ids, ranges = pu.check_bin_sort(fr, cam)
    _, s3 = pu.check_render_fwd(fr, cam, sc.masks, ids, ranges)
    _, s4 = pu.check_render_bwd(fr, cam, sc.N, sc.masks, ids, ranges, sc.dL_dimage())
    ref5, s5 = pu.check_preprocess_bwd(fr, sc, cam)
    vis = fr.radii.cpu().numpy() > 0
    for k, v in s5.items():
        assert v <= 1e-4, f"{k}: relative 2-norm error {v:.2e}"
    for k in ref5:
        pu.grad_close(pu.f64(getattr(fr, k))[vis], ref5[k][vis], k, rtol=1e-3, floor_frac=1e-4)
    print("PARITY", name, "staged", dict(preprocess=s1, render_fwd=s3, render_bwd=s4, preprocess_bwd=s5))


def test_end_to_end_image_parity(run, oracle):
    """fp64 oracle from the raw inputs vs the GPU image; threshold-sensitive pixels excluded and counted."""
    name, sc, fr = run
    cam = sc.camera
    pre, ids, ranges, fwd = oracle.full_forward(cam, pu.arrays(sc), sc.masks)
    img = pu.f64(fr.image)
    if name in E2E_L2_ONLY:
        rel = np.linalg.norm(img - fwd["image"]) / np.linalg.norm(fwd["image"])
        print(name, "e2e image (2-norm only): l2", rel)
        assert rel < E2E_L2_ONLY[name]
        return
    # sensitive: a blend decision within CUT_E2E of its threshold, or a Gaussian of the pixel's tile whose
    # integer decisions (radius, rect) or depth order are within fp32 reach of flipping
    flag = fwd["margin"] < pu.CUT_E2E
    gpu = pu.gpu_pre(fr)
    unstable = np.nonzero((pre["radii"] != gpu["radii"]) | (pre["rects"] != gpu["rects"]).any(1))[0]
    order_differs = not np.array_equal(pu.u32(fr.sorted_ids)[: fr.R], ids) if fr.R == len(ids) else True
    tol = pu.IMG_ATOL + pu.IMG_RTOL * np.abs(fwd["image"])
    err = np.abs(img - fwd["image"])
    bad = (err > tol).any(0) & ~flag
    # a pixel may also differ because a Gaussian's rect/order differs between fp32 and fp64: bound their number
    frac_bad = bad.mean()
    limit = 0.0 if (len(unstable) == 0 and not order_differs) else 5e-3
    assert frac_bad <= limit, f"{name}: {bad.sum()} non-flagged pixels outside tolerance (unstable={len(unstable)})"
    assert flag.mean() < 0.1
    rel = np.linalg.norm(img - fwd["image"]) / np.linalg.norm(fwd["image"])
    assert rel < 1e-3
    print(name, "e2e image: flagged", int(flag.sum()), "bad", int(bad.sum()), "unstable", len(unstable), "l2", rel)


def test_end_to_end_gradient_parity(run, oracle):
    """fp64 oracle from the raw inputs vs the GPU's gradients w.r.t. the raw inputs and the masks: ELEMENTWISE (1e-3
    relative) on every Gaussian the oracle does not flag as threshold-sensitive at CUT_E2E and whose integer decisions
    (radius, rect) agree between fp32 and fp64, plus the 2-norm over all of them."""
    name, sc, fr = run
    cam = sc.camera
    g = sc.dL_dimage().astype(np.float64)
    pre, ids, ranges, fwd = oracle.full_forward(cam, pu.arrays(sc), sc.masks)
    rb, pb = oracle.full_backward(cam, pu.arrays(sc), sc.masks, pre, ids, ranges, g, cutoff=pu.CUT_E2E)
    gpu = pu.gpu_pre(fr)
    unstable = (pre["radii"] != gpu["radii"]) | (pre["rects"] != gpu["rects"]).any(1)
    # a Gaussian whose rect differs changes the lists of the tiles at its border: the pixels there (and the Gaussians
    # blended behind it at those pixels) see one entry more or less.  Scenes with such Gaussians are compared in the
    # 2-norm only; the others elementwise on the non-flagged Gaussians.
    order_same = fr.R == len(ids) and np.array_equal(pu.u32(fr.sorted_ids)[: fr.R], ids)
    # On every scene of this module the fp32 and the fp64 chain produce the same lists (observed on the B200); were that
    # to change, the elementwise branch below would silently stop running -- so it is asserted, not assumed.
    assert order_same and not unstable.any(), f"{name}: fp32 and fp64 lists differ (unstable={int(unstable.sum())})"
    clean = (rb["sens"] == 0) & ~unstable
    ref = {k: v for k, v in list(rb.items()) + list(pb.items()) if k.startswith("dL_")}
    if order_same and name not in E2E_L2_ONLY:
        out = pu.grads_vs_ref(fr, ref, list(ref), clean, max_flag_frac=E2E_GRAD_BUDGET[name], l2_clean=2e-4,
                              rtol=E2E_GRAD_RTOL, floor_frac=E2E_GRAD_FLOOR)
    else:
        out = {}
        for k, r in ref.items():
            out[k + "_l2"] = float(np.linalg.norm(pu.f64(getattr(fr, k)) - r) / max(np.linalg.norm(r), 1e-300))
            lim = E2E_L2_ONLY.get(name, pu.L2_ALL)
            assert out[k + "_l2"] < lim, f"{name} {k}: relative 2-norm error {out[k + '_l2']:.2e}"
    print("PARITY", name, "e2e gradients", dict(order_same=bool(order_same), unstable=int(unstable.sum()), **out))


def test_masked_gaussians_get_only_mask_gradient(run):
    """PAPER.md:50 (Fig. 1): a masked splat gets a mask gradient but no alpha/colour gradient."""
    name, sc, fr = run
    masked = (sc.masks == 0) & (fr.radii.cpu().numpy() > 0)
    for k in ("dL_dmeans2d", "dL_dconic", "dL_dopacity", "dL_drgb", "dL_dmeans", "dL_dlog_scales", "dL_dquats",
              "dL_dopacity_logits", "dL_dsh"):
        assert not getattr(fr, k).cpu().numpy()[masked].any(), k
    dm = fr.dL_dmask.cpu().numpy()
    if name != "tiny":
        assert np.count_nonzero(dm[masked]) > 0.5 * masked.sum()
    culled = fr.radii.cpu().numpy() == 0
    assert not dm[culled].any()


def test_delete_equivalence_on_gpu(oracle):
    """rendering with masks == rendering only the kept Gaussians (images to fp32 rounding)."""
    sc = scenes.config2(n=30_000, width=256, height=256)
    fr, *_ = pu.run_gpu(sc)
    keep = sc.masks > 0
    sub = scenes.Scene("sub", sc.means[keep], sc.log_scales[keep], sc.quats[keep], sc.opacity_logits[keep],
                       sc.sh[keep], np.ones(int(keep.sum()), np.float32), sc.cameras, sc.seed)
    fr2, *_ = pu.run_gpu(sub)
    assert torch.equal(fr.image, fr2.image) and torch.equal(fr.final_T, fr2.final_T)


def test_unmasked_equals_all_ones(oracle):
    sc = scenes.config1()
    ones = np.ones(sc.N, np.float32)
    fr, *_ = pu.run_gpu(sc, masks=ones)
    cam = sc.camera
    ids, ranges = pu.check_bin_sort(fr, cam)
    _, s3 = pu.check_render_fwd(fr, cam, ones, ids, ranges)
    _, s4 = pu.check_render_bwd(fr, cam, sc.N, ones, ids, ranges, sc.dL_dimage())
    print("PARITY", "cfg1 all-ones masks", dict(render_fwd=s3, render_bwd=s4))


def test_fractional_masks(oracle):
    """Eq. 4 is affine in M: any real mask value is legal (reading 7)."""
    sc = scenes.config2(n=20_000, width=192, height=160)
    m = np.random.default_rng(0).random(sc.N).astype(np.float32)
    fr, *_ = pu.run_gpu(sc, masks=m)
    cam = sc.camera
    ids, ranges = pu.check_bin_sort(fr, cam)
    _, s3 = pu.check_render_fwd(fr, cam, m, ids, ranges)
    _, s4 = pu.check_render_bwd(fr, cam, sc.N, m, ids, ranges, sc.dL_dimage())
    print("PARITY", "cfg2 20k fractional masks", dict(render_fwd=s3, render_bwd=s4))


def test_background_colour(oracle):
    sc = scenes.config1()
    sc.cameras[0].bg = (0.9, 0.3, 0.5)
    fr, *_ = pu.run_gpu(sc)
    cam = sc.camera
    ids, ranges = pu.check_bin_sort(fr, cam)
    _, s3 = pu.check_render_fwd(fr, cam, sc.masks, ids, ranges)
    _, s4 = pu.check_render_bwd(fr, cam, sc.N, sc.masks, ids, ranges, sc.dL_dimage())
    print("PARITY", "cfg1 background colour", dict(render_fwd=s3, render_bwd=s4))


@pytest.mark.parametrize("degree", [1, 2])
def test_sh_degrees_1_and_2(oracle, degree):
    """The configs use SH degree 0 and 3 only; mg_preprocess / mg_preprocess_bwd have one kernel instance per degree, and
    degree 1 (48-byte rows: float4 loads) and degree 2 (108-byte rows: not a multiple of 16, scalar loads by flat position)
    take different staging paths.  config 2's geometry, N ragged against a warp and a block, higher bands strong enough to
    clamp channels; the whole path is run, projection and projection backward are compared (staged)."""
    import dataclasses

    base = scenes.config2()
    n = 20_011
    sh = scenes._sh(np.random.default_rng(70 + degree), n, degree, 0.5, 0.3)
    sc = dataclasses.replace(base, name=f"cfg2_sh{degree}", means=base.means[:n], log_scales=base.log_scales[:n],
                             quats=base.quats[:n], opacity_logits=base.opacity_logits[:n], sh=sh, masks=base.masks[:n],
                             cameras=[dataclasses.replace(base.camera, sh_degree=degree)])
    fr, g, m, gimg = pu.run_gpu(sc)
    cam = sc.camera
    s1 = pu.check_preprocess(fr, sc, cam, max_flag_frac=0.02)
    assert s1["n_clamped"] > 0, "the scene should clamp some channels"
    ref5, s5 = pu.check_preprocess_bwd(fr, sc, cam)
    vis = fr.radii.cpu().numpy() > 0
    for k, v in s5.items():
        assert v <= 1e-4, f"{k}: relative 2-norm error {v:.2e}"
    for k in ref5:
        pu.grad_close(pu.f64(getattr(fr, k))[vis], ref5[k][vis], k, rtol=1e-3, floor_frac=1e-4)
    print("PARITY", sc.name, "staged", dict(preprocess=s1, preprocess_bwd=s5))


def test_projection_backward_with_dense_upstream_gradients(oracle):
    """mg_preprocess_bwd alone at N = 1.2 M with EVERY visible Gaussian carrying a gradient (a view early in training:
    little saturation).  The geometry kernel queues the Gaussians that need the chain; at this density a block's
    queue fills several times per sweep.  Compared with the oracle's VJP of the same upstream gradients."""
    sc = scenes.config3(n=1_200_000, width=640, height=416)
    cam = sc.camera
    g, m = mg.upload(sc)
    fr = mg.Frame(cam, sc.N)
    fr.preprocess(g)
    torch.cuda.synchronize()
    rng = np.random.default_rng(5)
    up = dict(dL_dmeans2d=rng.standard_normal((sc.N, 2)), dL_dconic=rng.standard_normal((sc.N, 3)),
              dL_dopacity=rng.standard_normal(sc.N), dL_drgb=rng.standard_normal((sc.N, 3)))
    for k, v in up.items():
        getattr(fr, k).copy_(torch.from_numpy(v.astype(np.float32)))
    fr.preprocess_bwd(g)
    torch.cuda.synchronize()
    vis = fr.radii.cpu().numpy() > 0
    assert vis.mean() > 0.5
    ref5, s5 = pu.check_preprocess_bwd(fr, sc, cam)
    for k, v in s5.items():
        assert v <= 2e-4, f"{k}: relative 2-norm error {v:.2e}"
    # elementwise on a well-conditioned subset: conic -> covariance amplifies the fp32 rounding of the upstream
    # gradient by the splat's anisotropy squared; random (not rendered) dL/dconic does not cancel the way a real one does
    for k in ("dL_dopacity_logits", "dL_dsh"):
        pu.grad_close(pu.f64(getattr(fr, k))[vis], ref5[k][vis], k, rtol=1e-3, floor_frac=1e-4)
    print("dense upstream", s5)


def test_lookback_failure_is_reported_not_returned_as_an_order(monkeypatch):
    """include/mg.h, mg_bin_sort "Internal failure": a look-back that gives up must not yield a wrong order.  Injected
    through the hook of the TEST build of the library (libmg_testing.so, -DMG_TESTING; the shipped libmg.so has no such
    hook): every look-back gives up at once.  The first radix tile of a pass has no predecessor and never looks back, so
    the scene must span several tiles for the injection to reach anything."""
    import ctypes as C
    import os

    from paper_2412_20522_b200 import build

    sc = scenes.config2()
    assert sc.N > 8 * 4096  # a radix tile is 4096 keys (RS_THREADS * RS_ITEMS of binsort.cu): at least 8 look-backs per pass
    g, m = mg.upload(sc)
    fr = mg.Frame(sc.camera, sc.N)
    fr.forward(g, m)
    torch.cuda.synchronize()
    R = fr.R
    good, good_ids = fr.tile_ranges.clone(), fr.sorted_ids.clone()
    assert os.path.exists(build.LIB_TESTING), "libmg_testing.so not built (python -m paper_2412_20522_b200.build)"
    tl = mg.load_library(build.LIB_TESTING)
    tl.mg_debug_set_lookback_spin_limit.restype = None
    tl.mg_debug_set_lookback_spin_limit.argtypes = [C.c_int]
    assert not hasattr(mg.lib(), "mg_debug_set_lookback_spin_limit")
    monkeypatch.setattr(mg, "_lib", tl)  # from here on the binding's calls go through the test build
    try:
        tl.mg_debug_set_lookback_spin_limit(0)
        fr.sorted_ids.fill_(-1)
        fr.bin_sort()
        torch.cuda.synchronize()
        assert int(fr.R_host[1]) == -1  # UINT64_MAX read as int64
        assert not fr.tile_ranges.any() and (fr.sorted_ids == -1).all()
        fr.render_fwd(m)  # harmless: every range is empty
        torch.cuda.synchronize()
        assert (fr.n_contrib == 0).all()
    finally:
        tl.mg_debug_set_lookback_spin_limit(-1)
    fr.bin_sort()  # the test build without the injection: the same result as the shipped library
    torch.cuda.synchronize()
    assert int(fr.R_host[1]) == R and torch.equal(fr.tile_ranges, good) and torch.equal(fr.sorted_ids[:R], good_ids[:R])


# ------------------------------------------------------------------ edge cases
def test_empty_scene():
    sc = scenes.config1(n=1)
    sc2 = scenes.Scene("empty", sc.means[:0], sc.log_scales[:0], sc.quats[:0], sc.opacity_logits[:0], sc.sh[:0],
                       sc.masks[:0], sc.cameras, 0)
    sc2.cameras[0].bg = (0.1, 0.2, 0.3)
    fr, *_ = pu.run_gpu(sc2)
    assert fr.R == 0
    img = fr.image.cpu().numpy()
    np.testing.assert_allclose(img[0], 0.1, rtol=1e-6)
    np.testing.assert_allclose(img[2], 0.3, rtol=1e-6)
    assert (fr.final_T == 1).all() and (fr.n_contrib == 0).all()
    assert (fr.tile_ranges[:, 0] == fr.tile_ranges[:, 1]).all()


def test_everything_culled_and_all_masked():
    sc = scenes.config1()
    behind = sc.means.copy()
    behind[:, 2] = -behind[:, 2]
    sc_b = scenes.Scene("behind", behind, sc.log_scales, sc.quats, sc.opacity_logits, sc.sh, sc.masks, sc.cameras, 0)
    fr, *_ = pu.run_gpu(sc_b)
    assert fr.R == 0 and (fr.radii == 0).all() and not fr.image.any()
    for k in ("dL_dmeans", "dL_dlog_scales", "dL_dquats", "dL_dopacity_logits", "dL_dsh", "dL_dmask"):
        assert not getattr(fr, k).any()
    fr0, *_ = pu.run_gpu(sc, masks=np.zeros(sc.N, np.float32))
    assert not fr0.image.any() and (fr0.final_T == 1).all()
    assert (fr0.n_contrib > 0).any()  # masked Gaussians still "engage in the forward pass"
    assert fr0.dL_dmask.abs().sum() > 0 and not fr0.dL_dopacity.any()


def test_capacity_overflow_is_reported_not_written():
    sc = scenes.config1()
    g, m = mg.upload(sc)
    fr = mg.Frame(sc.camera, sc.N)
    fr.preprocess(g)
    torch.cuda.synchronize()
    R = int(fr.R_host[0])
    fr.reserve(R // 2)
    fr.sorted_ids.fill_(-1)
    fr.bin_sort()
    torch.cuda.synchronize()
    assert int(fr.R_host[1]) == R > fr.R_capacity
    assert (fr.sorted_ids == -1).all() and not fr.tile_ranges.any()
    fr.render_fwd(m)  # harmless: every range is empty
    torch.cuda.synchronize()
    assert (fr.n_contrib == 0).all()
    with pytest.raises(mg.MgError) as e:
        mg.mg_bin_sort(fr.cam, fr.depths, fr.rects, fr.tiles_touched, R, fr.workspace[:1024], fr.sorted_ids, fr.tile_ranges)
    assert e.value.code == mg.MG_ERR_CAPACITY


def test_huge_splat_covers_every_tile(oracle):
    """A Gaussian touching all tiles (key duplication by the whole warp) + ties in depth (order by index)."""
    sc = scenes.config1(n=300)
    sc.log_scales[:3] = 1.0
    sc.means[:3] = [0.0, 0.0, 3.0]  # three identical huge Gaussians: equal depth bits
    sc.opacity_logits[:3] = -2.0
    fr, *_ = pu.run_gpu(sc)
    gw, gh = mg.grid(sc.camera)
    assert (pu.u32(fr.tiles_touched)[:3] == gw * gh).all()
    ids, ranges = pu.check_bin_sort(fr, sc.camera)
    _, s3 = pu.check_render_fwd(fr, sc.camera, sc.masks, ids, ranges)
    print("PARITY", "cfg1 huge splats", dict(render_fwd=s3))


def test_many_tiles_three_sort_passes(oracle):
    """More than 65536 tiles -> three passes over the tile bits (4112 x 272 image = 257 x 17... use 4352x4112)."""
    cam0 = scenes.config1().camera
    W, H = 4400, 4000  # 275 x 250 = 68750 tiles > 2^16
    cam = scenes.Camera(W, H, 120.0 * W / 128, 120.0 * W / 128, W / 2, H / 2, cam0.R, cam0.t, sh_degree=0)
    sc = scenes.config1(n=2000)
    sc.cameras = [cam]
    sc.log_scales -= 2.5
    g, m = mg.upload(sc)
    fr = mg.Frame(cam, sc.N)
    fr.forward(g, m)
    torch.cuda.synchronize()
    pu.check_bin_sort(fr, cam)


def _length_class(n):
    """include/mg.h: class(0) = 0, class(n) = 1 + 8 floor(log2 n) + the next 3 bits of n."""
    n = np.asarray(n, np.int64)
    msb = np.zeros_like(n)
    nz = n > 0
    msb[nz] = np.floor(np.log2(n[nz])).astype(np.int64)
    msb[nz] -= (1 << msb[nz]) > n[nz]  # guard log2 rounding
    msb[nz] += (1 << (msb[nz] + 1)) <= n[nz]
    frac = np.where(msb >= 3, (n >> np.maximum(msb - 3, 0)) & 7, (n << np.maximum(3 - msb, 0)) & 7)
    return np.where(nz, 1 + 8 * msb + frac, 0)


def test_tile_order_is_a_permutation_with_longest_lists_first(run):
    """mg_bin_sort's scheduling hint: a permutation of the tiles, list-length class never increasing."""
    name, sc, fr = run
    order = fr.tile_order.cpu().numpy().astype(np.int64)
    ranges = fr.tile_ranges.cpu().numpy().astype(np.int64)
    ntiles = ranges.shape[0]
    assert sorted(order.tolist()) == list(range(ntiles))
    cls = _length_class(ranges[order, 1] - ranges[order, 0])
    assert (np.diff(cls) <= 0).all()


def test_tile_order_does_not_change_the_image(run):
    """The render calls give bit-identical per-pixel outputs with the hint and without it (row-major)."""
    name, sc, fr = run
    g, m = mg.upload(sc)
    fr.render_fwd(m)
    img, fT, nc = fr.image.clone(), fr.final_T.clone(), fr.n_contrib.clone()
    mg.mg_render_fwd(fr.cam, fr.sorted_ids, fr.tile_ranges, fr.means2d, fr.conic_opacity, fr.rgb, m, fr.image,
                     fr.final_T, fr.n_contrib, tile_order=None)
    torch.cuda.synchronize()
    assert torch.equal(img, fr.image) and torch.equal(fT, fr.final_T) and torch.equal(nc, fr.n_contrib)


@pytest.mark.parametrize("seed,W,H,n,big_frac,tie_levels", [
    (0, 16, 16, 500, 0.5, 3),          # a single tile, heavy depth ties
    (1, 530, 40, 3000, 0.1, 0),        # 34 x 3 tiles: two 32-bin words in x, one in y
    (2, 40, 1100, 3000, 0.1, 50),      # 3 x 69 tiles: three words in y
    (3, 2100, 2100, 40_000, 0.02, 0),  # 132 x 132 tiles: five words both ways
    (4, 1297, 840, 200_000, 0.05, 1000),
    (5, 333, 211, 70_000, 1.0, 7),     # every rect is large: long runs per record
])
def test_bin_sort_random_rects_through_the_c_abi(oracle, seed, W, H, n, big_frac, tie_levels):
    """mg_bin_sort alone on synthetic (depth, rect) inputs that the projection would not produce together: depth
    ties (order by index), rects of every shape incl. whole-image ones, culled entries, odd grid shapes -- compared
    bit for bit with the oracle's list builder."""
    rng = np.random.default_rng(seed)
    cam0 = scenes.config1().camera
    cam = scenes.Camera(W, H, 100.0, 100.0, W / 2, H / 2, cam0.R, cam0.t, sh_degree=0)
    gw, gh = mg.grid(cam)
    x0 = rng.integers(0, gw, n)
    y0 = rng.integers(0, gh, n)
    big = rng.uniform(size=n) < big_frac
    wx = np.where(big, rng.integers(1, gw + 1, n), rng.integers(1, 4, n))
    wy = np.where(big, rng.integers(1, gh + 1, n), rng.integers(1, 4, n))
    x1, y1 = np.minimum(x0 + wx, gw), np.minimum(y0 + wy, gh)
    culled = rng.uniform(size=n) < 0.2
    rects = np.stack([x0, y0, x1, y1], 1).astype(np.int32)
    rects[culled] = 0
    tt = ((rects[:, 2] - rects[:, 0]) * (rects[:, 3] - rects[:, 1])).astype(np.uint32)
    depths = rng.uniform(0.3, 50.0, n).astype(np.float32)
    if tie_levels:
        depths = (np.round(depths * tie_levels / 50.0) * (50.0 / tie_levels) + 0.25).astype(np.float32)
    R = int(tt.astype(np.int64).sum())
    ids_ref, ranges_ref = orc_bin_sort(oracle, cam, depths, rects, tt)
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    ws = torch.empty(mg.mg_workspace_bytes(n, W, H, R), dtype=torch.uint8, device="cuda")
    sorted_ids = torch.empty(max(R, 1), dtype=torch.int32, device="cuda")
    ranges = torch.empty(gw * gh, 2, dtype=torch.int32, device="cuda")
    order = torch.empty(gw * gh, dtype=torch.int32, device="cuda")
    R_host = torch.zeros(1, dtype=torch.int64).pin_memory()
    mg.mg_bin_sort(mg.camera(cam), d(depths), d(rects), d(tt.view(np.int32)), R, ws, sorted_ids, ranges, R_host, order)
    torch.cuda.synchronize()
    assert int(R_host[0]) == R
    assert np.array_equal(pu.u32(ranges), ranges_ref)
    assert np.array_equal(pu.u32(sorted_ids)[:R], ids_ref)
    assert sorted(order.cpu().numpy().tolist()) == list(range(gw * gh))


def orc_bin_sort(oracle, cam, depths, rects, tt):
    return oracle.bin_sort(cam, depths, rects, tt)


def test_degenerate_gaussians(oracle):
    """The degenerate inputs the method has, mixed into config 1: a zero quaternion (its normalisation is 0/0: the
    covariance is not a number and the Gaussian is culled, `det > 0` being false), vanishing scales (the covariance is
    the 0.3 dilation alone), a very large scale (its rect covers the image), opacity logits of +-30 (opacity 1 -> the
    0.99 clamp is active and cuts the gradient to the logit; opacity 1e-13 -> never passes the alpha filter), a centre
    exactly on the near plane (z = 0.2: culled, the test is z > 0.2) and one behind the camera.  Staged parity of all
    five calls, and no output of any call is non-finite."""
    sc = scenes.config1()
    n = sc.N
    sc.quats[0] = 0.0
    sc.log_scales[1] = -60.0
    sc.log_scales[2] = [2.0, -60.0, 1.0]
    sc.log_scales[3] = 3.0
    sc.means[3] = [0.1, -0.1, 4.0]
    sc.opacity_logits[3] = -2.0
    sc.opacity_logits[4] = 30.0
    sc.opacity_logits[5] = -30.0
    sc.means[6] = [0.3, 0.2, 0.2]
    sc.means[7] = [0.0, 0.0, -3.0]
    sc.quats[8] = [0.0, 0.0, 0.0, 1e-15]  # tiny but inside the domain of include/mg.h (|q|^2 a normal fp32 number)
    fr, g, m, gimg = pu.run_gpu(sc)
    cam = sc.camera
    radii = fr.radii.cpu().numpy()
    assert radii[0] == 0 and radii[6] == 0 and radii[7] == 0, "zero quaternion, near plane and behind the camera are culled"
    assert radii[1] > 0 and radii[3] > 0 and radii[8] > 0
    gw, gh = mg.grid(cam)
    assert pu.u32(fr.tiles_touched)[3] == gw * gh
    for k in ("means2d", "depths", "conic_opacity", "rgb", "image", "final_T", "dL_dmeans2d", "dL_dconic", "dL_dopacity",
              "dL_drgb", "dL_dmask", "dL_dmeans", "dL_dlog_scales", "dL_dquats", "dL_dopacity_logits", "dL_dsh"):
        assert torch.isfinite(getattr(fr, k)).all(), k
    s1 = pu.check_preprocess(fr, sc, cam, max_flag_frac=0.02)
    ids, ranges = pu.check_bin_sort(fr, cam)
    _, s3 = pu.check_render_fwd(fr, cam, sc.masks, ids, ranges)
    _, s4 = pu.check_render_bwd(fr, cam, n, sc.masks, ids, ranges, sc.dL_dimage())
    ref5, s5 = pu.check_preprocess_bwd(fr, sc, cam)
    vis = radii > 0
    for k, v in s5.items():
        assert v <= 1e-4, f"{k}: relative 2-norm error {v:.2e}"
    for k in ref5:
        pu.grad_close(pu.f64(getattr(fr, k))[vis], ref5[k][vis], k, rtol=1e-3, floor_frac=1e-4)
    assert float(fr.dL_dopacity_logits[4]) == 0.0 or abs(float(fr.dL_dopacity_logits[4])) < 1e-12, "sigmoid'(30) ~ 1e-13"
    print("PARITY", "cfg1 degenerate Gaussians", dict(preprocess=s1, render_fwd=s3, render_bwd=s4, preprocess_bwd=s5))
