"""Helpers for the GPU-vs-oracle parity tests (tolerances are derived in DESIGN.md "Parity procedure")."""
import numpy as np
import torch

import oracle as orc
from paper_2412_20522_b200 import binding as mg

# image: north_star's tolerance
IMG_ATOL, IMG_RTOL = 1e-5, 1e-4
# gradients: north_star's 1e-3 relative, plus an absolute floor relative to the array's scale
GRAD_RTOL = 1e-3
# decision-margin cut-offs (relative distance of a decision from its flip point)
CUT_STAGED = 2e-5
CUT_E2E = 2e-4


def arrays(sc):
    return (sc.means, sc.log_scales, sc.quats, sc.opacity_logits, sc.sh)


def u32(t):
    """torch int32 tensor holding uint32 bits -> numpy uint32."""
    return t.detach().cpu().numpy().view(np.uint32)


def f64(t):
    return t.detach().cpu().numpy().astype(np.float64)


def run_gpu(sc, cam_index=0, dL_dimage=None, masks=None):
    cam = sc.cameras[cam_index]
    g, m = mg.upload(sc)
    if masks is not None:
        m = torch.from_numpy(np.ascontiguousarray(masks, np.float32)).cuda()
    fr = mg.Frame(cam, sc.N)
    fr.forward(g, m)
    if dL_dimage is None:
        dL_dimage = sc.dL_dimage(cam_index)
    gimg = torch.from_numpy(dL_dimage).cuda()
    fr.backward(g, m, gimg)
    torch.cuda.synchronize()
    assert int(fr.R_host[1]) == fr.R
    return fr, g, m, gimg


def gpu_pre(fr):
    return dict(means2d=f64(fr.means2d), depths=fr.depths.cpu().numpy(), conic_opacity=f64(fr.conic_opacity),
                rgb=f64(fr.rgb), radii=fr.radii.cpu().numpy(), rects=fr.rects.cpu().numpy(),
                tiles_touched=u32(fr.tiles_touched), clamped=fr.clamped.cpu().numpy())


def check_preprocess(fr, sc, cam, max_flag_frac=0.01):
    """Stage 1 against the oracle run on the same fp32 inputs."""
    ref = orc.preprocess(cam, *arrays(sc))
    got = gpu_pre(fr)
    # integer decisions: exact unless the fp64 value sits within fp32 reach of a flip point
    radius = np.maximum(ref["radii"], got["radii"]).astype(np.float64)
    flag = ref["margin"] < 2e-3 + 2e-5 * radius
    same_int = (ref["radii"] == got["radii"]) & (ref["rects"] == got["rects"]).all(1) & \
               (ref["tiles_touched"] == got["tiles_touched"])
    bad = ~same_int & ~flag
    assert not bad.any(), f"{bad.sum()} Gaussians differ in radius/rect outside the margin, e.g. {np.nonzero(bad)[0][:5]}"
    n_flag_diff = int((~same_int).sum())
    assert flag.mean() <= max_flag_frac, f"{flag.mean():.4f} of Gaussians are margin-flagged"
    vis = (ref["radii"] > 0) & (got["radii"] > 0)
    # clamp flags (they gate dL/dsh in mg_preprocess_bwd): bit k set <=> channel k clamped at 0.  A flag may differ from
    # the fp64 decision only where the colour itself is within the colour tolerance of 0 on both sides.
    n_clamp_diff = 0
    for k in range(3):
        rb, gb = (ref["clamped"] >> k) & 1, (got["clamped"] >> k) & 1
        assert not (got["rgb"][vis, k][gb[vis] == 1]).any(), "a channel flagged as clamped must be exactly 0"
        diff = vis & (rb != gb)
        n_clamp_diff += int(diff.sum())
        near0 = np.maximum(np.abs(ref["rgb"][:, k]), np.abs(got["rgb"][:, k])) <= 1e-5
        assert not (diff & ~near0).any(), f"channel {k}: {(diff & ~near0).sum()} clamp flags differ away from 0"
    assert not got["clamped"][got["radii"] == 0].any()
    np.testing.assert_allclose(got["depths"], ref["depths"], rtol=2e-6, atol=1e-6)
    np.testing.assert_allclose(got["means2d"][vis], ref["means2d"][vis], rtol=2e-6, atol=5e-4)
    A, B, Cc, o = ref["conic_opacity"][vis].T
    cond = A * Cc / np.maximum(A * Cc - B * B, 1e-300)
    tol = (2e-6 * cond + 1e-5) * np.maximum(A, Cc)
    err = np.abs(got["conic_opacity"][vis][:, :3] - ref["conic_opacity"][vis][:, :3]).max(1)
    assert (err <= tol).all(), f"conic error {np.max(err / tol):.2f}x tolerance"
    np.testing.assert_allclose(got["conic_opacity"][vis][:, 3], o, rtol=5e-6, atol=1e-7)
    # colour: clamp decisions can flip only where the unclamped value is ~0
    np.testing.assert_allclose(got["rgb"][vis], ref["rgb"][vis], rtol=2e-5, atol=5e-6)
    culled = ref["radii"] == 0
    both = culled & (got["radii"] == 0)
    for k in ("means2d", "conic_opacity", "rgb"):
        assert not got[k][both].any()
    return dict(n_flagged=int(flag.sum()), flag_frac=float(flag.mean()), n_int_diff=n_flag_diff, n_visible=int(vis.sum()), n_clamp_diff=n_clamp_diff,
                n_clamped=int(((got["clamped"] > 0) & vis).sum()))


def check_bin_sort(fr, cam):
    """Stage 2, staged: the oracle's lists from the GPU's own fp32 depths and rects -- bit exact."""
    got = gpu_pre(fr)
    ids_ref, ranges_ref = orc.bin_sort(cam, got["depths"], got["rects"], got["tiles_touched"])
    R = len(ids_ref)
    assert fr.R == R
    ranges = u32(fr.tile_ranges)
    assert np.array_equal(ranges, ranges_ref), "tile_ranges differ"
    assert np.array_equal(u32(fr.sorted_ids)[:R], ids_ref), "sorted_ids differ"
    return ids_ref, ranges_ref


def check_render_fwd(fr, cam, masks, ids, ranges, cut=CUT_STAGED, max_flag_frac=1e-3, tiles=None):
    """Stage 3, staged: oracle blend on the GPU's fp32 splats and lists."""
    got = gpu_pre(fr)
    ref = orc.render_fwd(cam, ids, ranges, got["means2d"], got["conic_opacity"], got["rgb"], masks)
    img, Tf, nc = f64(fr.image), f64(fr.final_T), u32(fr.n_contrib)
    sel = np.ones((cam.height, cam.width), bool) if tiles is None else tile_pixel_mask(cam, tiles)
    flag = (ref["margin"] < cut) & sel
    ok = sel & ~flag
    err = np.abs(img - ref["image"])
    tol = IMG_ATOL + IMG_RTOL * np.abs(ref["image"])
    assert (err <= tol)[:, ok].all(), f"image error {np.max((err / tol)[:, ok]):.2f}x tolerance at non-flagged pixels"
    assert (np.abs(Tf - ref["final_T"]) <= IMG_ATOL + IMG_RTOL * ref["final_T"])[ok].all()
    assert np.array_equal(nc[ok], ref["n_contrib"][ok]), f"{(nc != ref['n_contrib'])[ok].sum()} n_contrib differ"
    # flagged pixels: one flipped alpha decision changes a pixel by at most ~1/255; a flipped stop by ~0.01
    assert (err[:, flag] <= 2e-2).all() if flag.any() else True
    assert flag.sum() <= max_flag_frac * sel.sum(), f"{flag.sum()} pixels margin-flagged"
    return ref, dict(n_flagged=int(flag.sum()), flag_frac=float(flag.sum() / max(sel.sum(), 1)),
                     n_contrib_diff=int((nc != ref["n_contrib"])[sel].sum()), max_err=float(err[:, ok].max()))


def tile_pixel_mask(cam, tiles):
    gw = (cam.width + 15) // 16
    m = np.zeros((cam.height, cam.width), bool)
    for t in tiles:
        ty, tx = divmod(int(t), gw)
        m[ty * 16:(ty + 1) * 16, tx * 16:(tx + 1) * 16] = True
    return m


def grad_close(got, ref, name, rtol=GRAD_RTOL, floor_frac=1e-5, mask=None):
    """|d| <= rtol |ref| + floor_frac * max|ref|  elementwise (optionally on rows where mask is True)."""
    scale = np.abs(ref).max() if ref.size else 0.0
    err = np.abs(got - ref)
    tol = rtol * np.abs(ref) + floor_frac * scale + 1e-30
    if mask is not None:
        err, tol = err[mask], tol[mask]
    worst = float((err / tol).max()) if err.size else 0.0
    assert worst <= 1.0, f"{name}: error {worst:.2f}x tolerance"
    return worst


L2_CLEAN = 1e-4  # relative 2-norm error of a gradient array over its non-flagged elements
L2_ALL = 2e-3    # ... over every element: a flagged Gaussian may differ by whole alpha >= 1/255 contributions


def grads_vs_ref(fr, ref, names, clean, max_flag_frac, l2_clean=L2_CLEAN, l2_all=L2_ALL, rtol=GRAD_RTOL, floor_frac=1e-5):
    """Elementwise on the non-flagged Gaussians (north_star: 1e-3 relative) + the two 2-norm bounds."""
    out = {}
    for k in names:
        g = f64(getattr(fr, k))
        out[k] = round(grad_close(g, ref[k], k, rtol=rtol, floor_frac=floor_frac, mask=clean), 4)
        nrm_c, nrm = np.linalg.norm(ref[k][clean]), np.linalg.norm(ref[k])
        if nrm_c > 0:
            out[k + "_l2clean"] = float(np.linalg.norm((g - ref[k])[clean]) / nrm_c)
            assert out[k + "_l2clean"] <= l2_clean, f"{k}: relative 2-norm error {out[k + '_l2clean']:.2e} on non-flagged Gaussians"
        if nrm > 0:
            out[k + "_l2"] = float(np.linalg.norm(g - ref[k]) / nrm)
            assert out[k + "_l2"] <= l2_all, f"{k}: relative 2-norm error {out[k + '_l2']:.2e}"
    out["n_flagged"] = int((~clean).sum())
    out["flag_frac"] = float((~clean).mean())
    assert out["flag_frac"] <= max_flag_frac, f"{out['n_flagged']} Gaussians flagged ({out['flag_frac']:.4f} > {max_flag_frac})"
    return out


def check_render_bwd(fr, cam, N, masks, ids, ranges, dL_dimage, cut=CUT_STAGED, max_flag_frac=0.15):
    """Stage 4, staged."""
    got = gpu_pre(fr)
    ref = orc.render_bwd(cam, N, ids, ranges, got["means2d"], got["conic_opacity"], got["rgb"], masks,
                         dL_dimage.astype(np.float64), cutoff=cut)
    clean = ref["sens"] == 0
    names = ["dL_dmeans2d", "dL_dconic", "dL_dopacity", "dL_drgb", "dL_dmask"]
    return ref, grads_vs_ref(fr, ref, names, clean, max_flag_frac)


def check_preprocess_bwd(fr, sc, cam):
    """Stage 5, staged: oracle VJP with the GPU's own upstream gradients."""
    ref = orc.preprocess_bwd(cam, *arrays(sc), f64(fr.dL_dmeans2d), f64(fr.dL_dconic), f64(fr.dL_dopacity),
                             f64(fr.dL_drgb))
    # the oracle re-derives the cull decision in fp64; compare where both agree a Gaussian is visible
    vis = fr.radii.cpu().numpy() > 0
    out = {}
    for k in ("dL_dmeans", "dL_dlog_scales", "dL_dquats", "dL_dopacity_logits", "dL_dsh"):
        g = f64(getattr(fr, k))
        assert not g[~vis].any(), f"{k}: culled Gaussians must get exact zeros"
        nrm = np.linalg.norm(ref[k][vis])
        rel = np.linalg.norm((g - ref[k])[vis]) / max(nrm, 1e-300)
        out[k + "_l2"] = float(rel)
    return ref, out


def check_adam_step(got, ref, p_before, g, lr, beta1, beta2, eps, step, name=""):
    """(p', m', v') of mg_adam_step against the oracle's, tolerances derived from the kernel's fp32 arithmetic
    (e = 2^-24; every operation of csrc/optimizer.cu adam_one is one correctly rounded IEEE operation):

    m' = fma(beta1, m, fl(fl(1 - beta1) g)): the constant, the product and the fma are rounded once each, so
        |dm'| <= e (2 |(1 - beta1) g| + |m'|).
      The bound is relative to the TERMS, not to the result: beta1 m and (1 - beta1) g have either sign and can cancel; a
      bound relative to m' alone fails there (0.26 % of the elements of the test distribution, on the GPU and in an fp32
      numpy emulation alike) although nothing is wrong.
    v' = fma(beta2, v, fl(fl(fl(1 - beta2) g) g)): both terms are >= 0, nothing cancels: |dv'| <= 4.5 e v' < 4e-7 v'.
    p' = fl(p - u), u = fl(fl(step_size m') / denom), denom = fma(fl(sqrt v'), c, eps):
        |dp'| <= |du/dm'| |dm'| + 9.3 e |u| + e |p'|,   du/dm' = step_size / denom.
      The first term matters where m' cancelled while v' is small (the tests draw m and v independently of g); without it
      4 elements in 5.4 M of the emulation exceed the bound.  Used as 1e-6 |u| + 1.2e-7 |p'| + 1.1 x the first term.
    """
    e = 2.0 ** -24
    (p_got, m_got, v_got), (p_ref, m_ref, v_ref) = got, ref
    g = np.asarray(g, np.float64)
    bc1, bc2 = 1.0 - beta1 ** step, 1.0 - beta2 ** step
    dm = 1.1 * e * (2.0 * np.abs((1.0 - beta1) * g) + np.abs(m_ref))
    bad = np.abs(np.asarray(m_got, np.float64) - m_ref) > dm + 1e-37
    assert not bad.any(), (name, "first moment", int(bad.sum()), "of", bad.size)
    np.testing.assert_allclose(v_got, v_ref, rtol=4e-7, atol=1e-37, err_msg=name)
    u = np.abs(p_ref - np.asarray(p_before, np.float64))
    du_dm = (lr / bc1) / (np.sqrt(v_ref / bc2) + eps)
    bad = np.abs(np.asarray(p_got, np.float64) - p_ref) > 1e-6 * u + 1.2e-7 * np.abs(p_ref) + du_dm * dm + 1e-30
    assert not bad.any(), (name, "parameter", int(bad.sum()), "of", bad.size)
