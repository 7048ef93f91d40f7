"""Pins of the CPU oracle against what the paper and the mathematics fix.

Nothing here touches the CUDA path.  Every check is written independently of oracle/mg_oracle.cpp
(numpy re-derivations, closed forms, scipy's spherical harmonics, finite differences, invariants).
Citations: PAPER.md line + equation.
"""
import numpy as np
import pytest

from paper_2412_20522_b200 import scenes

ALPHA_MIN, ALPHA_MAX, T_MIN = 1.0 / 255.0, 0.99, 1e-4


def arrays(sc):
    return (sc.means, sc.log_scales, sc.quats, sc.opacity_logits, sc.sh)


# ---------------------------------------------------------------- independent numpy blend
def np_tile_lists(cam, depths_f32, rects, tiles_touched):
    """(tile, depth_bits, index) lexsort -- the library routine of pin P11."""
    gw, gh = (cam.width + 15) // 16, (cam.height + 15) // 16
    keys_t, keys_d, keys_i = [], [], []
    bits = depths_f32.astype(np.float32).view(np.uint32)
    for i in np.nonzero(tiles_touched)[0]:
        x0, y0, x1, y1 = rects[i]
        for ty in range(y0, y1):
            for tx in range(x0, x1):
                keys_t.append(ty * gw + tx)
                keys_d.append(bits[i])
                keys_i.append(i)
    keys_t, keys_d, keys_i = np.array(keys_t, np.int64), np.array(keys_d, np.int64), np.array(keys_i, np.int64)
    o = np.lexsort((keys_i, keys_d, keys_t))
    ids = keys_i[o].astype(np.uint32)
    t_sorted = keys_t[o]
    ranges = np.zeros((gw * gh, 2), np.uint32)
    for t in range(gw * gh):
        ranges[t, 0] = np.searchsorted(t_sorted, t, "left")
        ranges[t, 1] = np.searchsorted(t_sorted, t, "right")
    return ids, ranges


def np_pixel(px, py, ids, m2, co, rgb, m, bg, masked=True):
    """One pixel, written from Eq. 1-2 (masked=False) or Eq. 3-4 (masked=True) + the thresholds."""
    if len(ids) == 0:
        return np.array(bg, float), 1.0, 0, np.zeros(0), np.zeros(0), np.zeros(0, bool)
    d = m2[ids] - np.array([px, py], float)
    A, B, C, o = co[ids].T
    power = -0.5 * (A * d[:, 0] ** 2 + 2 * B * d[:, 0] * d[:, 1] + C * d[:, 1] ** 2)
    alpha = np.minimum(ALPHA_MAX, o * np.exp(power))
    ok = (power <= 0) & (alpha >= ALPHA_MIN)
    a = np.where(ok, (m[ids] if masked else 1.0) * alpha, 0.0)
    Tn = np.cumprod(1 - a)
    stop = np.nonzero(ok & (Tn < T_MIN))[0]
    n = stop[0] if len(stop) else len(ids)
    Ti = np.concatenate([[1.0], Tn[:-1]])
    w = (a * Ti)[:n]
    col = (w[:, None] * rgb[ids[:n]]).sum(0)
    Tfin = Tn[n - 1] if n > 0 else 1.0
    last = n  # entries consumed: those in front of the stopping entry, or the whole list (reading 5)
    return col + Tfin * np.array(bg, float), Tfin, last, alpha[:n], Ti[:n], ok[:n]


@pytest.fixture(scope="module")
def cfg1(oracle):
    sc = scenes.config1()
    pre, ids, ranges, fwd = oracle.full_forward(sc.camera, arrays(sc), sc.masks)
    return sc, pre, ids, ranges, fwd


# ---------------------------------------------------------------- P11 / P12: lists
def test_P11_bin_sort_equals_library_lexsort(oracle, cfg1):
    sc, pre, ids, ranges, _ = cfg1
    ids_np, ranges_np = np_tile_lists(sc.camera, pre["depths"].astype(np.float32), pre["rects"], pre["tiles_touched"])
    assert np.array_equal(ids, ids_np)
    assert np.array_equal(ranges, ranges_np)


def test_P12_list_invariants(oracle, cfg1):
    sc, pre, ids, ranges, _ = cfg1
    gw = (sc.camera.width + 15) // 16
    assert int((ranges[:, 1] - ranges[:, 0]).sum()) == int(pre["tiles_touched"].sum()) == len(ids)
    bits = pre["depths"].astype(np.float32).view(np.uint32)
    for t, (s, e) in enumerate(ranges):
        tx, ty = t % gw, t // gw
        r = pre["rects"][ids[s:e]]
        assert np.all((r[:, 0] <= tx) & (tx < r[:, 2]) & (r[:, 1] <= ty) & (ty < r[:, 3]))
        assert np.all(np.diff(bits[ids[s:e]].astype(np.int64)) >= 0)


def test_bin_sort_ties_by_index_and_empty(oracle):
    cam = scenes.Camera(64, 32, 50, 50, 32, 16, np.eye(3), np.zeros(3))
    depths = np.array([2.0, 1.0, 2.0, 1.0, 5.0], np.float32)
    rects = np.array([[0, 0, 2, 1], [0, 0, 4, 2], [1, 0, 2, 2], [0, 0, 1, 1], [0, 0, 0, 0]], np.int32)
    tt = np.array([2, 8, 2, 1, 0], np.uint32)
    ids, ranges = oracle.bin_sort(cam, depths, rects, tt)
    assert ids[ranges[0, 0]:ranges[0, 1]].tolist() == [1, 3, 0]
    assert ids[ranges[1, 0]:ranges[1, 1]].tolist() == [1, 0, 2]
    assert ids[ranges[5, 0]:ranges[5, 1]].tolist() == [1, 2]
    ids0, ranges0 = oracle.bin_sort(cam, depths, rects * 0, tt * 0)
    assert len(ids0) == 0 and np.all(ranges0[:, 0] == ranges0[:, 1])


# ---------------------------------------------------------------- P1: m == 1 is the unmasked blend of Eq. 1-2
def test_P1_all_ones_mask_is_unmasked_blend(oracle, cfg1):
    sc, pre, ids, ranges, _ = cfg1
    cam = sc.camera
    ones = np.ones(sc.N, np.float32)
    fwd = oracle.render_fwd(cam, ids, ranges, pre["means2d"], pre["conic_opacity"], pre["rgb"], ones)
    gw = (cam.width + 15) // 16
    rng = np.random.default_rng(5)
    for _ in range(600):
        px, py = int(rng.integers(cam.width)), int(rng.integers(cam.height))
        s, e = ranges[(py // 16) * gw + px // 16]
        col, Tfin, last, *_ = np_pixel(px, py, ids[s:e], pre["means2d"], pre["conic_opacity"], pre["rgb"], ones, cam.bg,
                                       masked=False)
        np.testing.assert_allclose(fwd["image"][:, py, px], col, rtol=1e-12, atol=1e-14)
        np.testing.assert_allclose(fwd["final_T"][py, px], Tfin, rtol=1e-12)
        assert fwd["n_contrib"][py, px] == last


def test_masked_blend_matches_eq3_eq4_numpy(oracle, cfg1):
    sc, pre, ids, ranges, fwd = cfg1
    cam = sc.camera
    gw = (cam.width + 15) // 16
    rng = np.random.default_rng(6)
    for _ in range(600):
        px, py = int(rng.integers(cam.width)), int(rng.integers(cam.height))
        s, e = ranges[(py // 16) * gw + px // 16]
        col, Tfin, last, *_ = np_pixel(px, py, ids[s:e], pre["means2d"], pre["conic_opacity"], pre["rgb"], sc.masks, cam.bg)
        np.testing.assert_allclose(fwd["image"][:, py, px], col, rtol=1e-12, atol=1e-14)
        np.testing.assert_allclose(fwd["final_T"][py, px], Tfin, rtol=1e-12)
        assert fwd["n_contrib"][py, px] == last


# ---------------------------------------------------------------- P2: delete-equivalence
@pytest.mark.parametrize("cfg", [1, 2])
def test_P2_delete_equivalence(oracle, cfg):
    sc = scenes.config1() if cfg == 1 else scenes.config2(n=20000, width=256, height=256)
    cam = sc.camera
    _, _, _, fwd = oracle.full_forward(cam, arrays(sc), sc.masks)
    keep = sc.masks > 0
    sub = tuple(a[keep] for a in arrays(sc))
    _, _, _, fwd_sub = oracle.full_forward(cam, sub, np.ones(int(keep.sum()), np.float32))
    assert np.array_equal(fwd["image"], fwd_sub["image"])  # bit-identical: a masked entry multiplies T by exactly 1
    assert np.array_equal(fwd["final_T"], fwd_sub["final_T"])
    # and the image does differ from the unmasked render (the masks are doing something)
    _, _, _, fwd_all = oracle.full_forward(cam, arrays(sc), np.ones(sc.N, np.float32))
    assert np.abs(fwd_all["image"] - fwd["image"]).max() > 1e-2


def test_stop_uses_post_mask_T(oracle):
    """A masked opaque Gaussian must not stop the pixel (reading 3)."""
    cam = scenes.Camera(16, 16, 10, 10, 8, 8, np.eye(3), np.zeros(3), bg=(0.0, 0.0, 0.0))
    n = 6
    m2 = np.full((n, 2), 7.0)
    co = np.tile(np.array([0.01, 0.0, 0.01, 0.999]), (n, 1))
    rgb = np.tile(np.array([0.2, 0.4, 0.6]), (n, 1))
    rgb[5] = [1.0, 0.0, 0.0]
    ids = np.arange(n, dtype=np.uint32)
    ranges = np.array([[0, n]], np.uint32)
    m = np.array([0, 0, 0, 0, 0, 1], np.float32)
    f = oracle.render_fwd(cam, ids, ranges, m2, co, rgb, m)
    assert f["n_contrib"][7, 7] == 6 and abs(f["image"][0, 7, 7] - 0.99) < 1e-12
    f1 = oracle.render_fwd(cam, ids, ranges, m2, co, rgb, np.ones(n, np.float32))
    # unmasked: T = 0.01 after the first, 1e-4(1+eps) after the second, the third would give 1e-6 -> stop;
    # the stopping entry is neither blended nor counted (reading 4)
    assert f1["n_contrib"][7, 7] == 2 and abs(f1["final_T"][7, 7] - 1e-4) < 1e-12


# ---------------------------------------------------------------- P4: Eq. 16 and the telescoping sum
def test_P4_final_T_product_and_partition_of_unity(oracle, cfg1):
    sc, pre, ids, ranges, fwd = cfg1
    cam = sc.camera
    white = np.ones_like(pre["rgb"])
    f1 = oracle.render_fwd(cam, ids, ranges, pre["means2d"], pre["conic_opacity"], white, sc.masks)
    np.testing.assert_allclose(f1["image"][0] + f1["final_T"], 1.0, rtol=0, atol=1e-13)
    gw = (cam.width + 15) // 16
    rng = np.random.default_rng(7)
    for _ in range(300):
        px, py = int(rng.integers(cam.width)), int(rng.integers(cam.height))
        s, e = ranges[(py // 16) * gw + px // 16]
        _, _, _, alpha, _, ok = np_pixel(px, py, ids[s:e], pre["means2d"], pre["conic_opacity"], pre["rgb"], sc.masks, cam.bg)
        prod = np.prod(1 - alpha[ok] * sc.masks[ids[s:e]][: len(ok)][ok])  # Eq. 16
        np.testing.assert_allclose(fwd["final_T"][py, px], prod, rtol=1e-12)


# ---------------------------------------------------------------- P5: single splat closed form (Eq. 18, N = 1)
@pytest.mark.parametrize("m", [0.0, 1.0, 0.3])
def test_P5_single_splat_closed_form(oracle, m):
    bg = (0.3, 0.6, 0.1)
    cam = scenes.Camera(16, 16, 10, 10, 8, 8, np.eye(3), np.zeros(3), bg=bg)
    m2 = np.array([[6.3, 9.1]])
    co = np.array([[0.08, 0.02, 0.05, 0.8]])
    c = np.array([[0.9, 0.2, 0.5]])
    ids, ranges = np.array([0], np.uint32), np.array([[0, 1]], np.uint32)
    masks = np.array([m], np.float32)
    mm = float(masks[0])
    f = oracle.render_fwd(cam, ids, ranges, m2, co, c, masks)
    g = np.random.default_rng(1).standard_normal((3, 16, 16))
    b = oracle.render_bwd(cam, 1, ids, ranges, m2, co, c, masks, g)
    yy, xx = np.mgrid[0:16, 0:16]
    dx, dy = m2[0, 0] - xx, m2[0, 1] - yy
    alpha = co[0, 3] * np.exp(-0.5 * (co[0, 0] * dx * dx + 2 * co[0, 1] * dx * dy + co[0, 2] * dy * dy))
    alpha = np.where(alpha >= ALPHA_MIN, alpha, 0.0)
    bgv = np.float32(bg).astype(np.float64)[:, None, None]  # the camera is fp32 on both sides
    img = mm * alpha * c[0][:, None, None] + (1 - mm * alpha) * bgv
    np.testing.assert_allclose(f["image"], img, rtol=1e-13, atol=1e-15)
    dm = (alpha * (g * (c[0][:, None, None] - bgv)).sum(0)).sum()
    np.testing.assert_allclose(b["dL_dmask"][0], dm, rtol=1e-12)
    np.testing.assert_allclose(b["dL_drgb"][0], (mm * alpha * g).sum((1, 2)), rtol=1e-12, atol=1e-15)
    do = (mm * (g * (c[0][:, None, None] - bgv)).sum(0) * np.where(alpha > 0, alpha / co[0, 3], 0)).sum()
    np.testing.assert_allclose(b["dL_dopacity"][0], do, rtol=1e-12, atol=1e-15)


# ---------------------------------------------------------------- P6: Fig. 1 shaped case + Eq. 18 evaluated directly
def test_P6_fig1_five_splats_masked_get_only_mask_gradient(oracle):
    """Five Gaussians on a ray, G2 and G5 masked (Fig. 1).  b_{i+1} by its direct definition."""
    bg = (0.25, 0.1, 0.4)
    cam = scenes.Camera(16, 16, 10, 10, 8, 8, np.eye(3), np.zeros(3), bg=bg)
    rng = np.random.default_rng(3)
    n = 5
    m2 = 7.5 + rng.uniform(-2, 2, (n, 2))
    co = np.column_stack([rng.uniform(0.02, 0.06, n), rng.uniform(-0.01, 0.01, n), rng.uniform(0.02, 0.06, n),
                          rng.uniform(0.3, 0.9, n)])
    c = rng.uniform(0, 1, (n, 3))
    masks = np.array([1, 0, 1, 1, 0], np.float32)
    ids, ranges = np.arange(n, dtype=np.uint32), np.array([[0, n]], np.uint32)
    g = rng.standard_normal((3, 16, 16))
    f = oracle.render_fwd(cam, ids, ranges, m2, co, c, masks)
    b = oracle.render_bwd(cam, n, ids, ranges, m2, co, c, masks, g)
    for i in (1, 4):
        assert np.all(b["dL_dmeans2d"][i] == 0) and np.all(b["dL_dconic"][i] == 0)
        assert b["dL_dopacity"][i] == 0 and np.all(b["dL_drgb"][i] == 0)
        assert abs(b["dL_dmask"][i]) > 1e-3
    # Eq. 18 with T_i, b_{i+1}, T_{N+1} from their definitions (no recursion)
    yy, xx = np.mgrid[0:16, 0:16]
    alpha = np.zeros((n, 16, 16))
    for i in range(n):
        dx, dy = m2[i, 0] - xx, m2[i, 1] - yy
        a_ = co[i, 3] * np.exp(-0.5 * (co[i, 0] * dx * dx + 2 * co[i, 1] * dx * dy + co[i, 2] * dy * dy))
        alpha[i] = np.where(a_ >= ALPHA_MIN, a_, 0)
    assert alpha.max() < ALPHA_MAX
    fac = 1 - masks[:, None, None] * alpha
    Tfin = np.prod(fac, 0)
    assert Tfin.min() > 0.01  # no stop in this case
    bgv = np.float32(bg).astype(np.float64)[:, None, None]  # the camera is fp32 on both sides
    for i in range(n):
        Ti = np.prod(fac[:i], 0)
        bnext = np.zeros((3, 16, 16))
        for j in range(i + 1, n):
            bnext += masks[j] * alpha[j] * np.prod(fac[i + 1:j], 0) * c[j][:, None, None]
        dm = alpha[i] * Ti * (g * (c[i][:, None, None] - bnext)).sum(0) - alpha[i] * Tfin / fac[i] * (g * bgv).sum(0)
        np.testing.assert_allclose(b["dL_dmask"][i], dm.sum(), rtol=1e-11)
    np.testing.assert_allclose(f["final_T"], Tfin, rtol=1e-13)


# ---------------------------------------------------------------- P3: exact mask flip differences
def test_P3_mask_gradient_equals_exact_flip_difference(oracle, cfg1):
    """C is affine in each M_i (Eq. 3-4, Eq. 14), so dL/dM_i = L(M_i=1) - L(M_i=0) exactly."""
    sc, pre, ids, ranges, fwd = cfg1
    cam = sc.camera
    g = sc.dL_dimage().astype(np.float64)
    rb = oracle.render_bwd(cam, sc.N, ids, ranges, pre["means2d"], pre["conic_opacity"], pre["rgb"], sc.masks, g)
    visible = np.nonzero(pre["radii"] > 0)[0]
    rng = np.random.default_rng(11)
    checked = 0
    for i in rng.choice(visible, 150, replace=False):
        L = []
        same = True
        for v in (1.0, 0.0):
            m = sc.masks.copy()
            m[i] = v
            f = oracle.render_fwd(cam, ids, ranges, pre["means2d"], pre["conic_opacity"], pre["rgb"], m)
            same &= np.array_equal(f["hash"], fwd["hash"])
            L.append((g * f["image"]).sum())
        if not same:
            continue
        checked += 1
        np.testing.assert_allclose(rb["dL_dmask"][i], L[0] - L[1], rtol=1e-9, atol=1e-11)
    assert checked > 100
    # pin 2 of north_star: masked Gaussians that pass the alpha filter somewhere get a nonzero mask gradient
    masked_vis = visible[sc.masks[visible] == 0]
    assert np.count_nonzero(rb["dL_dmask"][masked_vis]) > 0.9 * len(masked_vis)
    assert np.all(rb["dL_dopacity"][masked_vis] == 0) and np.all(rb["dL_drgb"][masked_vis] == 0)
    assert np.all(rb["dL_dmeans2d"][masked_vis] == 0) and np.all(rb["dL_dconic"][masked_vis] == 0)


# ---------------------------------------------------------------- P7: permutation of the input order
def test_P7_input_permutation(oracle):
    sc = scenes.config1()
    cam = sc.camera
    g = sc.dL_dimage().astype(np.float64)
    pre, ids, ranges, fwd = oracle.full_forward(cam, arrays(sc), sc.masks)
    assert len(np.unique(pre["depths"].astype(np.float32))) == sc.N
    rb, pb = oracle.full_backward(cam, arrays(sc), sc.masks, pre, ids, ranges, g)
    perm = np.random.default_rng(2).permutation(sc.N)
    arr_p = tuple(a[perm] for a in arrays(sc))
    pre2, ids2, ranges2, fwd2 = oracle.full_forward(cam, arr_p, sc.masks[perm])
    rb2, pb2 = oracle.full_backward(cam, arr_p, sc.masks[perm], pre2, ids2, ranges2, g)
    assert np.array_equal(fwd["image"], fwd2["image"])
    np.testing.assert_allclose(rb2["dL_dmask"], rb["dL_dmask"][perm], rtol=1e-10, atol=1e-14)
    for k in pb:
        np.testing.assert_allclose(pb2[k], pb[k][perm], rtol=1e-9, atol=1e-13)


# ---------------------------------------------------------------- P8: isotropic on-axis closed form (EWA)
def test_P8_isotropic_on_axis_closed_form(oracle):
    f, z, sigma, logit = 200.0, 4.0, 0.05, 0.4
    cam = scenes.Camera(64, 64, f, f, 32, 32, np.eye(3), np.zeros(3))
    means = np.array([[0.0, 0.0, z]])
    ls = np.full((1, 3), np.log(sigma))
    q = np.array([[0.3, -0.5, 0.2, 0.7]])
    sh = np.zeros((1, 1, 3))
    pre = oracle.preprocess(cam, means, ls, q, np.array([logit]), sh)
    var = (f * sigma / z) ** 2 + 0.3
    np.testing.assert_allclose(pre["conic_opacity"][0], [1 / var, 0, 1 / var, 1 / (1 + np.exp(-logit))], rtol=1e-12, atol=1e-15)
    np.testing.assert_allclose(pre["means2d"][0], [31.5, 31.5], rtol=1e-13)
    assert pre["radii"][0] == int(np.ceil(3 * np.sqrt(var + np.sqrt(0.1))))  # floor 0.1 under the sqrt (reading 14)
    np.testing.assert_allclose(pre["rgb"][0], 0.5)
    ids, ranges = oracle.bin_sort(cam, pre["depths"], pre["rects"], pre["tiles_touched"])
    fw = oracle.render_fwd(cam, ids, ranges, pre["means2d"], pre["conic_opacity"], pre["rgb"], np.ones(1, np.float32))
    o = 1 / (1 + np.exp(-logit))
    for r in (0, 1, 3, 5):
        a = o * np.exp(-(r + 0.5) ** 2 * 2 / (2 * var))  # pixel (31+r+1, 31+r+1)... offset (r+.5, r+.5)
        if a >= ALPHA_MIN:
            np.testing.assert_allclose(fw["image"][0, 32 + r, 32 + r], a * 0.5, rtol=1e-12)
    g = np.random.default_rng(0).standard_normal((3, 64, 64))
    rb, pb = oracle.full_backward(cam, (means, ls, q, np.array([logit]), sh), np.ones(1, np.float32), pre, ids, ranges, g)
    np.testing.assert_allclose(pb["dL_dquats"], 0, atol=1e-12 * np.abs(pb["dL_dlog_scales"]).max())


# ---------------------------------------------------------------- P9: spherical harmonics vs scipy
def _sh_probe(oracle, dirs, degree):
    """Y_j(dir) read back through orc_preprocess: colour_k - 0.5 = 0.25 * Y_j with sh = 0.25 e_j."""
    K = (degree + 1) ** 2
    Y = np.zeros((len(dirs), K))
    # six cameras at the origin looking along +-x, +-y, +-z; each sees one cube face with margin
    faces = [((0, 0, 1)), ((0, 0, -1)), ((1, 0, 0)), ((-1, 0, 0)), ((0, 1, 0)), ((0, -1, 0))]
    axis = np.argmax(np.abs(dirs), axis=1)
    sign = np.sign(dirs[np.arange(len(dirs)), axis])
    face_of = {(2, 1): 0, (2, -1): 1, (0, 1): 2, (0, -1): 3, (1, 1): 4, (1, -1): 5}
    fidx = np.array([face_of[(int(a), int(s))] for a, s in zip(axis, sign)])
    for fi, look in enumerate(faces):
        sel = np.nonzero(fidx == fi)[0]
        if not len(sel):
            continue
        down = (0.0, 1.0, 0.0) if look[1] == 0 else (0.0, 0.0, 1.0)
        R, t = scenes.look_at((0, 0, 0), look, down)
        cam = scenes.Camera(256, 256, 100.0, 100.0, 128, 128, R, t, sh_degree=degree)
        means = dirs[sel] * 3.0
        n = len(sel)
        ls = np.full((n, 3), -4.0)
        q = np.tile([1.0, 0, 0, 0], (n, 1))
        for j0 in range(0, K, 3):
            sh = np.zeros((n, K, 3))
            for k in range(3):
                if j0 + k < K:
                    sh[:, j0 + k, k] = 0.25
            pre = oracle.preprocess(cam, means, ls, q, np.zeros(n), sh)
            assert np.all(pre["radii"] > 0) and np.all(pre["clamped"] == 0)
            for k in range(3):
                if j0 + k < K:
                    Y[sel, j0 + k] = (pre["rgb"][:, k] - 0.5) / 0.25
    return Y


def test_P9_sh_basis_matches_scipy_and_is_orthonormal(oracle):
    from scipy.special import sph_harm_y

    rng = np.random.default_rng(0)
    d = rng.standard_normal((400, 3))
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    Y = _sh_probe(oracle, d, 3)
    theta, phi = np.arccos(d[:, 2]), np.arctan2(d[:, 1], d[:, 0])
    j = 0
    for l in range(4):
        for m in range(-l, l + 1):
            c = sph_harm_y(l, abs(m), theta, phi)  # complex, Condon-Shortley phase included
            ref = c.real if m == 0 else np.sqrt(2) * (c.real if m > 0 else c.imag)
            np.testing.assert_allclose(Y[:, j], ref, rtol=0, atol=1e-12, err_msg=f"l={l} m={m}")
            j += 1
    # addition theorem: sum_m Y_lm^2 = (2l+1)/(4 pi)
    for l in range(4):
        np.testing.assert_allclose((Y[:, l * l:(l + 1) ** 2] ** 2).sum(1), (2 * l + 1) / (4 * np.pi), rtol=1e-12)
    # orthonormality by Gauss-Legendre quadrature on the cube-face parametrisation of the sphere
    x, w = np.polynomial.legendre.leggauss(24)
    u, v = np.meshgrid(x, x)
    wt = np.outer(w, w) / (1 + u * u + v * v) ** 1.5
    pts, wts = [], []
    for ax in range(3):
        for s in (1, -1):
            p = np.zeros(u.shape + (3,))
            p[..., ax] = s
            p[..., (ax + 1) % 3] = u
            p[..., (ax + 2) % 3] = v
            pts.append((p / np.linalg.norm(p, axis=-1, keepdims=True)).reshape(-1, 3))
            wts.append(wt.reshape(-1))
    pts, wts = np.concatenate(pts), np.concatenate(wts)
    np.testing.assert_allclose(wts.sum(), 4 * np.pi, rtol=1e-9)
    Yq = _sh_probe(oracle, pts, 3)
    gram = (Yq * wts[:, None]).T @ Yq
    np.testing.assert_allclose(gram, np.eye(16), atol=1e-8)


def test_sh_degree0_colour_is_direction_independent(oracle, cfg1):
    sc, pre, *_ = cfg1
    vis = pre["radii"] > 0
    ref = np.maximum(0.5 + 0.5 * np.sqrt(1 / np.pi) * sc.sh[:, 0, :].astype(np.float64), 0)
    np.testing.assert_allclose(pre["rgb"][vis], ref[vis], rtol=1e-14)
    assert np.array_equal(pre["clamped"][vis], ((0.5 + 0.5 * np.sqrt(1 / np.pi) * sc.sh[:, 0, :].astype(np.float64)) < 0)[vis] @ np.array([1, 2, 4]))


# ---------------------------------------------------------------- projection: independent numpy EWA
def test_projection_matches_numpy_ewa(oracle):
    """O1-O7 re-derived with numpy matrices (J W Sigma W^T J^T + 0.3 I)."""
    sc = scenes.config2(n=3000, width=256, height=256)
    cam = sc.camera
    pre = oracle.preprocess(cam, *arrays(sc))
    gw, gh = 16, 16
    R, t = np.asarray(cam.R, np.float32).astype(np.float64), np.asarray(cam.t, np.float32).astype(np.float64)
    fx, fy, cx, cy = (float(np.float32(v)) for v in (cam.fx, cam.fy, cam.cx, cam.cy))
    nvis, margins = 0, []
    for i in range(0, sc.N, 7):
        p = sc.means[i].astype(np.float64)
        tc = R @ p + t
        if tc[2] <= 0.2:
            assert pre["radii"][i] == 0
            continue
        s = np.exp(sc.log_scales[i].astype(np.float64))
        w, x, y, z = sc.quats[i].astype(np.float64) / np.linalg.norm(sc.quats[i].astype(np.float64))
        Rot = np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - w * z), 2 * (x * z + w * y)],
                        [2 * (x * y + w * z), 1 - 2 * (x * x + z * z), 2 * (y * z - w * x)],
                        [2 * (x * z - w * y), 2 * (y * z + w * x), 1 - 2 * (x * x + y * y)]])
        np.testing.assert_allclose(Rot @ Rot.T, np.eye(3), atol=1e-12)
        Sig = Rot @ np.diag(s * s) @ Rot.T
        lx, ly = 1.3 * cam.width / (2 * fx), 1.3 * cam.height / (2 * fy)
        xt, yt = np.clip(tc[0] / tc[2], -lx, lx) * tc[2], np.clip(tc[1] / tc[2], -ly, ly) * tc[2]
        J = np.array([[fx / tc[2], 0, -fx * xt / tc[2] ** 2], [0, fy / tc[2], -fy * yt / tc[2] ** 2]])
        cov = J @ R @ Sig @ R.T @ J.T + 0.3 * np.eye(2)
        lam = np.linalg.eigvalsh(cov)[-1]
        m2 = np.array([fx * tc[0] / tc[2] + cx - 0.5, fy * tc[1] / tc[2] + cy - 0.5])
        mid, det = 0.5 * (cov[0, 0] + cov[1, 1]), np.linalg.det(cov)
        lam_f = mid + np.sqrt(max(mid * mid - det, 0.1))
        assert lam_f >= lam - 1e-9
        rad = int(np.ceil(3 * np.sqrt(lam_f)))
        x0, x1 = np.clip(np.floor((m2[0] - rad) / 16), 0, gw), np.clip(np.floor((m2[0] + rad + 15) / 16), 0, gw)
        y0, y1 = np.clip(np.floor((m2[1] - rad) / 16), 0, gh), np.clip(np.floor((m2[1] + rad + 15) / 16), 0, gh)
        if (x1 - x0) * (y1 - y0) == 0:
            assert pre["radii"][i] == 0 and pre["tiles_touched"][i] == 0
            continue
        nvis += 1
        conic = np.linalg.inv(cov)
        np.testing.assert_allclose(pre["conic_opacity"][i, :3], [conic[0, 0], conic[0, 1], conic[1, 1]], rtol=1e-9)
        np.testing.assert_allclose(pre["conic_opacity"][i, 3], 1 / (1 + np.exp(-float(sc.opacity_logits[i]))), rtol=1e-13)
        np.testing.assert_allclose(pre["means2d"][i], m2, rtol=1e-12)
        np.testing.assert_allclose(pre["depths"][i], tc[2], rtol=1e-14)
        assert pre["radii"][i] == rad
        assert pre["rects"][i].tolist() == [x0, y0, x1, y1] and pre["tiles_touched"][i] == (x1 - x0) * (y1 - y0)
        # `margin` (gates which Gaussians the GPU comparison may exempt from bit-exact integers): how far, in pixels /
        # depth units, the nearest of this Gaussian's integer decisions is from flipping -- the near-plane test, the
        # ceil of the radius, the four floors of the tile rectangle (a quotient in tiles is 16 pixels per unit).
        to_int = lambda v: abs(v - np.rint(v))
        quot = [(m2[0] - rad) / 16, (m2[0] + rad + 15) / 16, (m2[1] - rad) / 16, (m2[1] + rad + 15) / 16]
        want = min(abs(tc[2] - 0.2), to_int(3 * np.sqrt(lam_f)), 16 * min(to_int(q) for q in quot))
        np.testing.assert_allclose(pre["margin"][i], want, rtol=1e-6, atol=1e-9)
        margins.append(want)
    assert nvis > 200
    # the pin bites: margins spread over the whole range a distance to the nearest integer can take, and moving an input
    # by less than a Gaussian's margin leaves its integers alone while the smallest margins sit near a flip
    margins = np.array(margins)
    assert margins.min() < 0.02 and margins.max() > 0.3 and (margins <= 0.5 + 1e-12).all()


# ---------------------------------------------------------------- tile shift (pixel-centre convention, reading 15)
def test_shift_principal_point_by_one_tile(oracle):
    sc = scenes.config1()
    cam = sc.camera
    _, _, _, f0 = oracle.full_forward(cam, arrays(sc), sc.masks)
    cam2 = scenes.Camera(cam.width, cam.height, cam.fx, cam.fy, cam.cx + 16, cam.cy, cam.R, cam.t, cam.bg, cam.sh_degree)
    _, _, _, f1 = oracle.full_forward(cam2, arrays(sc), sc.masks)
    np.testing.assert_allclose(f1["image"][:, :, 16:], f0["image"][:, :, :-16], rtol=0, atol=1e-13)


# ---------------------------------------------------------------- P10: finite differences through the whole path
def _loss(oracle, cam, arrs, masks, g):
    pre, ids, ranges, fwd = oracle.full_forward(cam, arrs, masks)
    sig = (pre["radii"].copy(), pre["rects"].copy(), fwd["hash"].copy(), ids.copy())
    return float((g * fwd["image"]).sum()), sig, (pre, ids, ranges, fwd)


@pytest.mark.parametrize("seed,degree", [(100, 3), (101, 1), (102, 0)])
def test_P10_finite_differences_all_inputs(oracle, seed, degree):
    sc = scenes.tiny_fd_scene(seed=seed, sh_degree=degree)
    cam = sc.camera
    arrs = [a.astype(np.float64) for a in arrays(sc)]
    g = sc.dL_dimage().astype(np.float64)
    L0, sig0, (pre, ids, ranges, fwd) = _loss(oracle, cam, arrs, sc.masks, g)
    assert fwd["blends"] > 500
    rb, pb = oracle.full_backward(cam, arrs, sc.masks, pre, ids, ranges, g)
    # the clamp row of the readings: Gaussian 0 has opacity ~0.999, so some pixels are clamped
    assert 1 / (1 + np.exp(-arrs[3][0])) > 0.99
    names = ["dL_dmeans", "dL_dlog_scales", "dL_dquats", "dL_dopacity_logits", "dL_dsh"]
    h = 1e-6
    rng = np.random.default_rng(seed)
    n_ok = n_rej = 0
    for ai, name in enumerate(names):
        flat_n = arrs[ai].size
        probes = range(flat_n) if ai < 4 else rng.choice(flat_n, min(flat_n, 40), replace=False)
        for k in probes:
            Ls, same = [], True
            for sgn in (1, -1):
                a2 = [a.copy() for a in arrs]
                a2[ai].reshape(-1)[k] += sgn * h
                L, sig, _ = _loss(oracle, cam, a2, sc.masks, g)
                same &= all(np.array_equal(x, y) for x, y in zip(sig, sig0))
                Ls.append(L)
            if not same:
                n_rej += 1
                continue
            n_ok += 1
            fd = (Ls[0] - Ls[1]) / (2 * h)
            an = pb[name].reshape(-1)[k]
            assert abs(fd - an) <= 2e-6 * max(1.0, abs(an)) + 1e-7, (name, k, fd, an)
    assert n_ok > 5 * max(n_rej, 1), (n_ok, n_rej)
    # quaternion gradient is w.r.t. the raw quaternion through the normalisation: q . dL/dq = 0 (reading 20)
    dots = (pb["dL_dquats"] * arrs[2]).sum(1)
    np.testing.assert_allclose(dots, 0, atol=1e-10 * max(1.0, np.abs(pb["dL_dquats"]).max()))


def test_fd_render_stage_gradients(oracle):
    """FD of L w.r.t. the render-stage inputs (mean2d, conic, opacity, colour) incl. a clamped pixel."""
    sc = scenes.tiny_fd_scene(seed=103)
    cam = sc.camera
    pre, ids, ranges, fwd = oracle.full_forward(cam, arrays(sc), sc.masks)
    g = sc.dL_dimage().astype(np.float64)
    rb = oracle.render_bwd(cam, sc.N, ids, ranges, pre["means2d"], pre["conic_opacity"], pre["rgb"], sc.masks, g)
    h = 1e-6
    ins = {"means2d": pre["means2d"], "conic_opacity": pre["conic_opacity"], "rgb": pre["rgb"]}
    n_ok = 0
    for key, gname in (("means2d", "dL_dmeans2d"), ("conic_opacity", None), ("rgb", "dL_drgb")):
        for k in range(ins[key].size):
            Ls, same = [], True
            for sgn in (1, -1):
                mod = {kk: v.copy() for kk, v in ins.items()}
                mod[key].reshape(-1)[k] += sgn * h
                f = oracle.render_fwd(cam, ids, ranges, mod["means2d"], mod["conic_opacity"], mod["rgb"], sc.masks)
                same &= np.array_equal(f["hash"], fwd["hash"])
                Ls.append((g * f["image"]).sum())
            if not same:
                continue
            n_ok += 1
            fd = (Ls[0] - Ls[1]) / (2 * h)
            if key == "conic_opacity":
                i, j = divmod(k, 4)
                an = rb["dL_dopacity"][i] if j == 3 else rb["dL_dconic"][i, j]
            else:
                an = rb[gname].reshape(-1)[k]
            assert abs(fd - an) <= 2e-6 * max(1.0, abs(an)) + 1e-7, (key, k, fd, an)
    assert n_ok > 50


# ---------------------------------------------------------------- work counters (numerators of bench.py's throughput)
def np_pixel_margins(px, py, ids, m2, co, m):
    """Decision margins of one pixel, from DESIGN.md section 5's definition ("the smallest relative distance of any
    decision the walk took from its flip point"), written with numpy array operations on the whole list."""
    if len(ids) == 0:
        return np.inf, np.inf, 0, np.zeros(0)
    d = m2[ids] - np.array([px, py], float)
    A, B, C, o = co[ids].T
    power = -0.5 * (A * d[:, 0] ** 2 + 2 * B * d[:, 0] * d[:, 1] + C * d[:, 1] ** 2)
    oG = o * np.exp(np.minimum(power, 0.0))
    alpha = np.minimum(ALPHA_MAX, oG)
    ok = (power <= 0) & (alpha >= ALPHA_MIN)
    a = np.where(ok, m[ids] * alpha, 0.0)
    Tn = np.cumprod(1 - a)
    stop = np.nonzero(ok & (Tn < T_MIN))[0]
    nvis = stop[0] + 1 if len(stop) else len(ids)  # entries visited, the stopping one included
    v = slice(0, nvis)
    inside = power[v] <= 0
    mg_alpha = (np.abs(alpha[v] - ALPHA_MIN) / ALPHA_MIN)[inside]
    mg_T = (np.abs(Tn[v] - T_MIN) / T_MIN)[ok[v]]
    mg_clamp = (np.abs(oG[v] - ALPHA_MAX) / ALPHA_MAX)[ok[v]]
    mg = min(mg_alpha.min() if mg_alpha.size else np.inf, mg_T.min() if mg_T.size else np.inf)
    return mg, (mg_clamp.min() if mg_clamp.size else np.inf), nvis, alpha[v]


@pytest.mark.parametrize("cfg", [1, 2])
def test_work_counters_match_an_independent_count(oracle, cfg):
    """"a pair evaluation = one (list entry, pixel) visited before the pixel stops; a blend = a pair
    evaluation that passes the alpha filter (masked or not)".  The oracle's counters (numerators of every throughput
    and roofline number of bench.py) against a count taken from the numpy Eq. 3-4 loop, masked and unmasked entries
    separately, forward (the stopping entry is visited and passes the filter) and backward (positions n_contrib..1)."""
    sc = scenes.config1() if cfg == 1 else scenes.config2(n=60000, width=128, height=96)  # cfg 2: ~800 pixels stop
    cam = sc.camera
    pre, ids, ranges, fwd = oracle.full_forward(cam, arrays(sc), sc.masks)
    g = sc.dL_dimage().astype(np.float64)
    rb = oracle.render_bwd(cam, sc.N, ids, ranges, pre["means2d"], pre["conic_opacity"], pre["rgb"], sc.masks, g)
    gw = (cam.width + 15) // 16
    f_ev = [0, 0]; f_bl = [0, 0]; b_ev = [0, 0]; b_bl = [0, 0]  # [unmasked, masked]
    n_stopped = 0
    for py in range(cam.height):
        for px in range(cam.width):
            s, e = ranges[(py // 16) * gw + px // 16]
            lst = ids[s:e]
            _, _, n, _, _, ok = np_pixel(px, py, lst, pre["means2d"], pre["conic_opacity"], pre["rgb"], sc.masks, cam.bg)
            stopped = n < len(lst)
            n_stopped += stopped
            mk = sc.masks[lst[:n]] == 0
            for j, sel in enumerate((~mk, mk)):
                b_ev[j] += int(sel.sum()); b_bl[j] += int((ok & sel).sum())
                f_ev[j] += int(sel.sum()); f_bl[j] += int((ok & sel).sum())
            if stopped:  # the entry that stops the pixel: visited, passes the filter, never masked (reading 3)
                assert sc.masks[lst[n]] != 0
                f_ev[0] += 1; f_bl[0] += 1
    assert (fwd["pair_evals"] - fwd["pair_evals_masked"], fwd["pair_evals_masked"]) == tuple(f_ev)
    assert (fwd["blends"] - fwd["blends_masked"], fwd["blends_masked"]) == tuple(f_bl)
    assert (rb["pair_evals"] - rb["pair_evals_masked"], rb["pair_evals_masked"]) == tuple(b_ev)
    assert (rb["blends"] - rb["blends_masked"], rb["blends_masked"]) == tuple(b_bl)
    assert fwd["pair_evals"] - rb["pair_evals"] == n_stopped == fwd["blends"] - rb["blends"]
    assert f_ev[1] > 0 and f_bl[1] > 0 and (cfg == 1 or n_stopped > 0)
    # the committed table the bench reads was written from these counters
    import json, os
    wc = json.load(open(os.path.join(os.path.dirname(__file__), "..", "oracle", "work_counts.json")))
    if cfg == 1:
        assert wc["1"]["fwd_pair_evals"] == fwd["pair_evals"] and wc["1"]["bwd_blends_masked"] == rb["blends_masked"]


def test_bin_sort_tile_select_is_the_full_result_restricted_to_the_selected_tiles(oracle):
    """orc_bin_sort's tile_select branch (bench.py's bounded cpu_baseline sample): selected tiles keep exactly the
    list of the unselected run, the others are empty, R = the sum of the kept lists."""
    sc = scenes.config2(n=20000, width=256, height=256)
    cam = sc.camera
    pre = oracle.preprocess(cam, *arrays(sc))
    d32 = pre["depths"].astype(np.float32)
    ids, ranges = oracle.bin_sort(cam, d32, pre["rects"], pre["tiles_touched"])
    ntiles = ranges.shape[0]
    sel = np.zeros(ntiles, np.uint8)
    sel[1::3] = 1
    ids_s, ranges_s = oracle.bin_sort(cam, d32, pre["rects"], pre["tiles_touched"], sel)
    kept = 0
    for t in range(ntiles):
        s, e = ranges_s[t]
        if sel[t]:
            assert np.array_equal(ids_s[s:e], ids[ranges[t, 0]:ranges[t, 1]])
            kept += int(e - s)
        else:
            assert s == e
    assert kept == len(ids_s) and 0 < kept < len(ids)
    assert (np.diff(ranges_s.reshape(-1).astype(np.int64)) >= 0).all()  # ranges tile the array in tile order


def test_margins_and_sens_flags_follow_their_definition(oracle, cfg1):
    """The per-pixel decision margin and the per-Gaussian `sens` count decide which elements a GPU parity test may
    exempt.  (a) Both against a numpy evaluation of DESIGN.md section 5's definition.  (b) The property they exist
    for: perturbing the render-stage inputs by fp32-sized relative amounts changes decisions only at pixels whose
    margin is below the cut-off, and moves the gradient only of Gaussians with sens > 0 beyond the tolerance."""
    sc, pre, ids, ranges, fwd = cfg1
    cam = sc.camera
    gw = (cam.width + 15) // 16
    cut = 2e-4
    g = sc.dL_dimage().astype(np.float64)
    rb = oracle.render_bwd(cam, sc.N, ids, ranges, pre["means2d"], pre["conic_opacity"], pre["rgb"], sc.masks, g, cutoff=cut)
    sens = np.zeros(sc.N, np.int64)
    for py in range(cam.height):
        for px in range(cam.width):
            s, e = ranges[(py // 16) * gw + px // 16]
            lst = ids[s:e]
            mg, mgc, nvis, alpha = np_pixel_margins(px, py, lst, pre["means2d"], pre["conic_opacity"], sc.masks)
            if np.isfinite(mg):
                np.testing.assert_allclose(fwd["margin"][py, px], mg, rtol=1e-9)
            else:
                assert fwd["margin"][py, px] > 1e29
            if min(mg, mgc) < cut:
                np.add.at(sens, lst[:nvis][alpha >= (1 - cut) * ALPHA_MIN], 1)
    assert np.array_equal(sens, rb["sens"].astype(np.int64)) and sens.sum() > 0
    # (b) relative perturbation of 2e-7 (a few fp32 ulps) of centres, conics and opacities
    rng = np.random.default_rng(9)
    m2p = pre["means2d"] * (1 + 2e-7 * rng.uniform(-1, 1, pre["means2d"].shape))
    cop = pre["conic_opacity"] * (1 + 2e-7 * rng.uniform(-1, 1, pre["conic_opacity"].shape))
    fwd_p = oracle.render_fwd(cam, ids, ranges, m2p, cop, pre["rgb"], sc.masks)
    changed = fwd_p["hash"] != fwd["hash"]
    assert not (changed & (fwd["margin"] >= cut)).any()
    rb_p = oracle.render_bwd(cam, sc.N, ids, ranges, m2p, cop, pre["rgb"], sc.masks, g)
    for k in ("dL_dmask", "dL_dopacity", "dL_drgb"):
        ref = rb[k]
        err = np.abs(rb_p[k] - ref)
        tol = 1e-3 * np.abs(ref) + 1e-5 * np.abs(ref).max()
        bad = (err > tol).reshape(sc.N, -1).any(1)
        assert not (bad & (rb["sens"] == 0)).any(), k
