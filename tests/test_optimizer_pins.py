"""Pins of the f4 oracle (oracle/optimizer.py; readings 27-28) against things
other than itself: torch.optim.Adam (a library routine), closed forms of Adam's recursion, a scalar hand loop;
the density statistics against a per-Gaussian Python loop and their invariants.  Runs with -m "not gpu"."""
import math

import numpy as np
import torch

from oracle import optimizer as opt


def test_adam_equals_library_adam_over_several_steps_and_groups():
    """Kingma & Ba Algorithm 1 as the library implements it (fp64, eps outside the bias-corrected root): any slip in
    the moment recursions, the bias correction or the place of eps shows within a few steps."""
    rng = np.random.default_rng(0)
    shapes = [(50, 3), (50, 4), (50,), (50, 16, 3), (50, 2)]
    lrs = [1.6e-4, 1e-3, 5e-2, 2.5e-3, 1e-2]
    b1, b2, eps = 0.9, 0.999, 1e-15
    ps = [rng.normal(0, 1, s) for s in shapes]
    tp = [torch.tensor(p.copy(), dtype=torch.float64, requires_grad=True) for p in ps]
    lib = torch.optim.Adam([dict(params=[t], lr=lr) for t, lr in zip(tp, lrs)], betas=(b1, b2), eps=eps)
    ms = [np.zeros(s) for s in shapes]
    vs = [np.zeros(s) for s in shapes]
    for t in range(1, 8):
        gs = [rng.normal(0, 10.0 ** rng.uniform(-6, 1), s) for s in shapes]
        for k in range(len(shapes)):
            tp[k].grad = torch.tensor(gs[k])
            ps[k], ms[k], vs[k] = opt.adam_step(ps[k], gs[k], ms[k], vs[k], lrs[k], b1, b2, eps, t)
        lib.step()
        for k in range(len(shapes)):
            np.testing.assert_allclose(ps[k], tp[k].detach().numpy(), rtol=1e-12, atol=1e-15)
            st = lib.state[tp[k]]
            np.testing.assert_allclose(ms[k], st["exp_avg"].numpy(), rtol=1e-12, atol=1e-300)
            np.testing.assert_allclose(vs[k], st["exp_avg_sq"].numpy(), rtol=1e-12, atol=1e-300)


def test_first_step_from_zero_moments_is_a_sign_step():
    """t = 1, m = v = 0: m_hat = g, v_hat = g^2, so p moves by lr g / (|g| + eps): -lr sign(g) up to eps."""
    g = np.array([3.0, -2e-5, 1e-9, -7.0, 0.0])
    p = np.array([1.0, 2.0, 3.0, 4.0, 5.0])
    lr, eps = 0.01, 1e-15
    pn, mn, vn = opt.adam_step(p, g, np.zeros(5), np.zeros(5), lr, 0.9, 0.999, eps, 1)
    np.testing.assert_allclose(pn, p - lr * g / (np.abs(g) + eps), rtol=1e-14)
    np.testing.assert_allclose(pn[:4], p[:4] - lr * np.sign(g[:4]), atol=lr * 2e-6)
    assert pn[4] == p[4]  # zero gradient, zero moments: no move
    np.testing.assert_allclose(mn, 0.1 * g, rtol=1e-14)
    np.testing.assert_allclose(vn, 0.001 * g * g, rtol=1e-12)


def test_constant_gradient_closed_form_at_step_t():
    """Constant g from zero moments: m_t = (1 - b1^t) g and v_t = (1 - b2^t) g^2 (geometric sums), so every step is the
    sign step and p_t = p_0 - t lr g / (|g| + eps)."""
    g = np.array([0.5, -4.0])
    p = np.array([0.0, 0.0])
    m = np.zeros(2)
    v = np.zeros(2)
    b1, b2, lr, eps = 0.8, 0.95, 0.1, 1e-12
    for t in range(1, 12):
        p, m, v = opt.adam_step(p, g, m, v, lr, b1, b2, eps, t)
        np.testing.assert_allclose(m, (1 - b1 ** t) * g, rtol=1e-12)
        np.testing.assert_allclose(v, (1 - b2 ** t) * g * g, rtol=1e-12)
        np.testing.assert_allclose(p, -t * lr * g / (np.abs(g) + eps), rtol=1e-10)


def test_scalar_hand_loop():
    """One parameter, three steps, every quantity typed out with math.* on Python floats."""
    b1, b2, lr, eps = 0.9, 0.999, 0.02, 1e-8
    p, m, v = 0.7, 0.0, 0.0
    pa, ma, va = np.array([0.7]), np.zeros(1), np.zeros(1)
    for t, g in enumerate([0.3, -1.1, 0.05], start=1):
        m = b1 * m + (1 - b1) * g
        v = b2 * v + (1 - b2) * g * g
        p = p - lr * (m / (1 - math.pow(b1, t))) / (math.sqrt(v / (1 - math.pow(b2, t))) + eps)
        pa, ma, va = opt.adam_step(pa, np.array([g]), ma, va, lr, b1, b2, eps, t)
        assert abs(pa[0] - p) < 1e-15 and abs(ma[0] - m) < 1e-16 and abs(va[0] - v) < 1e-16


def test_row_restriction_leaves_invisible_rows_untouched():
    rng = np.random.default_rng(3)
    p, g, m, v = (rng.normal(0, 1, (20, 3)) for _ in range(4))
    v = np.abs(v)
    vis = rng.random(20) < 0.5
    pn, mn, vn = opt.adam_step(p, g, m, v, 0.01, 0.9, 0.999, 1e-15, 5, row_visible=vis)
    pf, mf, vf = opt.adam_step(p, g, m, v, 0.01, 0.9, 0.999, 1e-15, 5)
    assert np.array_equal(pn[~vis], p[~vis]) and np.array_equal(mn[~vis], m[~vis]) and np.array_equal(vn[~vis], v[~vis])
    assert np.array_equal(pn[vis], pf[vis]) and np.array_equal(mn[vis], mf[vis]) and np.array_equal(vn[vis], vf[vis])


def test_density_stats_equal_a_per_gaussian_loop():
    rng = np.random.default_rng(5)
    n = 300
    g = rng.normal(0, 1e-3, (n, 2))
    radii = rng.integers(0, 40, n) * (rng.random(n) < 0.7)
    acc0, den0, mx0 = rng.random(n), rng.integers(0, 5, n).astype(float), rng.integers(0, 30, n).astype(float)
    sx, sy = 648.5, 420.0
    acc, den, mx = opt.density_stats(g, radii, acc0, den0, mx0, scale=(sx, sy))
    for i in range(n):
        if radii[i] > 0:
            assert abs(acc[i] - (acc0[i] + math.hypot(sx * g[i, 0], sy * g[i, 1]))) < 1e-15
            assert den[i] == den0[i] + 1
            assert mx[i] == max(mx0[i], float(radii[i]))
        else:
            assert acc[i] == acc0[i] and den[i] == den0[i] and mx[i] == mx0[i]


def test_density_stats_invariants():
    """Accumulating k views: denom counts the views a Gaussian was visible in; grad_accum / denom lies between the
    smallest and the largest per-view norm; the norm of the summed gradient never exceeds grad_accum (triangle
    inequality); max_radii is the running maximum."""
    rng = np.random.default_rng(6)
    n, views = 200, 6
    acc, den, mx = np.zeros(n), np.zeros(n), np.zeros(n)
    gsum = np.zeros((n, 2))
    seen = np.zeros(n)
    lo, hi, rmax = np.full(n, np.inf), np.zeros(n), np.zeros(n)
    for _ in range(views):
        g = rng.normal(0, 1, (n, 2))
        radii = rng.integers(1, 50, n) * (rng.random(n) < 0.6)
        acc, den, mx = opt.density_stats(g, radii, acc, den, mx)
        vis = radii > 0
        nrm = np.linalg.norm(g, axis=1)
        gsum[vis] += g[vis]
        seen[vis] += 1
        lo[vis] = np.minimum(lo[vis], nrm[vis])
        hi[vis] = np.maximum(hi[vis], nrm[vis])
        rmax = np.maximum(rmax, radii)
    assert np.array_equal(den, seen) and np.array_equal(mx, rmax)
    s = seen > 0
    avg = acc[s] / den[s]
    assert (avg >= lo[s] - 1e-12).all() and (avg <= hi[s] + 1e-12).all()
    assert (np.linalg.norm(gsum, axis=1) <= acc + 1e-12).all()
    assert not acc[~s].any()
