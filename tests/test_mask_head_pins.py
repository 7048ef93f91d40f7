"""Pins of the mask-head oracle (oracle/mask_head.py) against what the paper and the
mathematics fix: the Gumbel-max property, library softmax / argmax, finite differences, closed forms of Eq. 7.
Runs with -m "not gpu"."""
import numpy as np
import pytest
from scipy.special import softmax

from oracle import mask_head as mh


def draws(n, seed, shape=(2,)):
    rng = np.random.default_rng(seed)
    return rng.uniform(1e-12, 1.0 - 1e-12, size=(n,) + shape)


def test_gumbel_max_property_fixes_noise_formula_and_category():
    """the sample is one category out of 2 scores; by the Gumbel-max theorem P(M = 1) =
    softmax(s)_1 = sigmoid(s_1 - s_0), whatever tau.  A sign error in g, swapped categories or u instead of
    -log u all move the frequency far outside the band."""
    n = 400_000
    for s0, s1 in [(0.0, 0.0), (0.3, -1.2), (-2.0, 1.0), (1.5, 1.6)]:
        scores = np.tile([s0, s1], (n, 1))
        for tau in (0.5, 1.0, 3.0):
            m = mh.sample(scores, draws(n, 7), tau)["mask"]
            p = 1.0 / (1.0 + np.exp(-(s1 - s0)))
            assert abs(m.mean() - p) < 5.0 * np.sqrt(p * (1 - p) / n), (s0, s1, tau, m.mean(), p)


def test_soft_and_hard_sample_equal_library_softmax_and_argmax():
    rng = np.random.default_rng(1)
    n = 5000
    scores = rng.normal(0, 2, (n, 2))
    u = draws(n, 2)
    for tau in (0.25, 1.0, 2.0):
        r = mh.sample(scores, u, tau)
        pert = scores - np.log(-np.log(u))
        np.testing.assert_allclose(r["soft"], softmax(pert / tau, axis=1)[:, 1], rtol=1e-12, atol=1e-300)
        assert np.array_equal(r["mask"], np.argmax(pert, axis=1).astype(float))
        assert ((r["mask"] == 1) == (r["soft"] > 0.5)).all()


def test_straight_through_gradient_is_the_derivative_of_the_soft_sample():
    """Finite differences of y_1(s) in fp64 (central, h = 1e-6) against sample_bwd."""
    rng = np.random.default_rng(3)
    n = 200
    scores = rng.normal(0, 1.5, (n, 2))
    u = draws(n, 4)
    w = rng.normal(0, 1, n)
    for tau in (0.5, 1.0):
        soft = mh.sample(scores, u, tau)["soft"]
        got = mh.sample_bwd(soft, w, tau)
        h = 1e-6
        for k in range(2):
            sp, sm = scores.copy(), scores.copy()
            sp[:, k] += h
            sm[:, k] -= h
            fd = w * (mh.sample(sp, u, tau)["soft"] - mh.sample(sm, u, tau)["soft"]) / (2 * h)
            np.testing.assert_allclose(got[:, k], fd, rtol=1e-6, atol=1e-9)
        np.testing.assert_allclose(got.sum(axis=1), 0.0, atol=1e-15)  # softmax of 2: the two derivatives cancel


def test_mask_loss_closed_forms_and_gradient():
    """Eq. 7-8: L_m = (mean M)^2; all ones -> 1, all zeros -> 0, half -> 1/4."""
    n = 1000
    assert mh.mask_loss(np.ones(n), 0.7)[0] == pytest.approx(0.7)
    assert mh.mask_loss(np.zeros(n), 0.7)[0] == 0.0
    m = np.zeros(n)
    m[::2] = 1
    loss, grad = mh.mask_loss(m, 2.0)
    assert loss == pytest.approx(2.0 * 0.25)
    # gradient with respect to a continuous relaxation of M, by finite differences
    rng = np.random.default_rng(5)
    mc = rng.uniform(0, 1, 50)
    _, g = mh.mask_loss(mc, 1.3)
    for i in (0, 17, 49):
        e = np.zeros(50)
        e[i] = 1e-6
        fd = (mh.mask_loss(mc + e, 1.3)[0] - mh.mask_loss(mc - e, 1.3)[0]) / 2e-6
        assert g[i] == pytest.approx(fd, rel=1e-8)


def test_prune_rule_keeps_exactly_the_gaussians_sampled_at_least_once():
    """10 samples, remove those never sampled.  P(removed) = (1 - p)^10."""
    n = 200_000
    scores = np.tile([0.0, -1.0], (n, 1))  # p = sigmoid(-1) = 0.2689
    u10 = draws(10, 11, shape=(n, 2))
    keep, _ = mh.prune_keep(scores, u10)
    p_removed = (1 - 1 / (1 + np.e)) ** 10
    assert abs((~keep).mean() - p_removed) < 5 * np.sqrt(p_removed * (1 - p_removed) / n)
    # equals the OR of ten library argmaxes
    ref = np.zeros(n, bool)
    for k in range(10):
        ref |= np.argmax(scores - np.log(-np.log(u10[k])), axis=1) == 1
    assert np.array_equal(keep, ref)
    assert not mh.prune_keep(np.tile([0.0, -80.0], (100, 1)), u10[:, :100])[0].any()
    assert mh.prune_keep(np.tile([0.0, 80.0], (100, 1)), u10[:, :100])[0].all()


def test_compaction_is_stable_and_complete():
    rng = np.random.default_rng(9)
    n = 1000
    keep = rng.uniform(size=n) < 0.3
    arrays = [rng.normal(size=(n, 3)), rng.normal(size=(n, 16, 3)), np.arange(n, dtype=np.float64)]
    out, cnt = mh.compact(keep, arrays)
    assert cnt == keep.sum() and all(o.shape[0] == cnt for o in out)
    j = 0
    for i in range(n):  # written out: row i of the input is row j of the output iff kept
        if keep[i]:
            assert out[2][j] == i and np.array_equal(out[0][j], arrays[0][i]) and np.array_equal(out[1][j], arrays[1][i])
            j += 1
    assert j == cnt


def test_uniforms_at_and_beyond_the_endpoints():
    """Reading 29: a uniform outside (0,1) is taken as the nearest fp32 value inside it, [2^-126, 1 - 2^-24].  Held against
    the closed forms of the noise at those two values (not against the oracle's own clamp), and against what the
    definition implies: values beyond the interval behave like its end, every output is finite, the noise is
    non-decreasing in u, and a pair (0, 0) -- whose unclamped noise would be inf - inf -- gives the noise-free sample."""
    g_lo = -np.log(126.0 * np.log(2.0))            # -ln(-ln 2^-126)
    g_hi = -np.log(-np.log1p(-(2.0 ** -24)))       # -ln(-ln(1 - 2^-24))
    assert mh.gumbel(0.0) == pytest.approx(g_lo, rel=1e-14) and mh.gumbel(1.0) == pytest.approx(g_hi, rel=1e-14)
    assert -4.48 < g_lo < -4.46 and 16.63 < g_hi < 16.64
    for beyond, end in ((-0.5, 0.0), (1e-45, 0.0), (-np.inf, 0.0), (1.5, 1.0), (np.inf, 1.0)):
        assert mh.gumbel(beyond) == mh.gumbel(end)
    u = np.array([0.0, 1e-45, np.finfo(np.float32).tiny, 1e-20, 0.25, 0.5, 0.75, 1.0 - 2.0 ** -24, 1.0])
    g = mh.gumbel(u)
    assert np.isfinite(g).all() and (np.diff(g) >= 0).all()
    s = np.array([[0.3, -0.2], [1.0, 2.5]])
    for pair in ((0.0, 0.0), (1.0, 1.0)):
        r = mh.sample(s, np.tile(np.array(pair), (2, 1)), tau=0.7)
        np.testing.assert_allclose(r["soft"], 1.0 / (1.0 + np.exp(-(s[:, 1] - s[:, 0]) / 0.7)), rtol=1e-14)
        assert np.array_equal(r["mask"], (s[:, 1] > s[:, 0]).astype(np.float64))
    # the extreme pairs decide the sample whatever the scores (|g_hi - g_lo| = 21.1 against scores of a few units)
    assert mh.sample(s, np.tile(np.array((0.0, 1.0)), (2, 1)))["mask"].tolist() == [1.0, 1.0]
    assert mh.sample(s, np.tile(np.array((1.0, 0.0)), (2, 1)))["mask"].tolist() == [0.0, 0.0]
