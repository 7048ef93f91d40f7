"""Pins of the render-loss oracle (oracle/render_loss.py): closed forms, a brute-force
window sum, finite differences.  Runs with -m "not gpu"."""
import numpy as np
import pytest

from oracle import render_loss as rl


def images(h=23, w=37, seed=0):
    rng = np.random.default_rng(seed)
    return rng.uniform(0, 1, (3, h, w)), rng.uniform(0, 1, (3, h, w))


def test_window_is_normalised_gaussian():
    w = rl.window()
    assert len(w) == 11 and abs(w.sum() - 1) < 1e-15 and np.allclose(w, w[::-1])
    assert w[5] / w[4] == pytest.approx(np.exp(1 / (2 * 1.5 ** 2)), rel=1e-12)  # exp(-0)/exp(-1/(2 sigma^2))


def test_blur_equals_brute_force_window_sum_with_zero_padding():
    x, _ = images(9, 13, 1)
    w = rl.window()
    got = rl.blur(x)
    for c, i, j in [(0, 0, 0), (1, 4, 6), (2, 8, 12), (0, 2, 11)]:
        s = 0.0
        for di in range(-5, 6):
            for dj in range(-5, 6):
                ii, jj = i + di, j + dj
                if 0 <= ii < 9 and 0 <= jj < 13:
                    s += w[di + 5] * w[dj + 5] * x[c, ii, jj]
        assert got[c, i, j] == pytest.approx(s, rel=1e-13)


def test_identical_images_give_zero_loss_and_ssim_one():
    x, _ = images()
    r = rl.render_loss(x, x.copy(), 0.2)
    assert r["l1"] == 0 and r["ssim"] == pytest.approx(1.0, abs=1e-14) and r["loss"] == pytest.approx(0.0, abs=1e-14)


def test_lambda_zero_is_l1_and_its_gradient_is_the_sign():
    x, y = images(seed=2)
    r = rl.render_loss(x, y, 0.0)
    assert r["loss"] == pytest.approx(np.abs(x - y).mean(), rel=1e-14)
    assert np.array_equal(r["dL_dimage"] * x.size, np.sign(x - y))


def test_constant_images_closed_form():
    """Far from the border, constant images a and b: sigma's vanish, SSIM = (2ab + C1)/(a^2 + b^2 + C1)."""
    a, b = 0.3, 0.7
    x, y = np.full((3, 31, 31), a), np.full((3, 31, 31), b)
    sm, _ = rl.ssim_map(x, y)
    assert sm[1, 15, 15] == pytest.approx((2 * a * b + rl.C1) / (a * a + b * b + rl.C1), rel=1e-12)


def test_gradient_matches_central_finite_differences():
    x, y = images(17, 19, 3)
    for lam in (0.2, 1.0):
        r = rl.render_loss(x, y, lam)
        rng = np.random.default_rng(4)
        for _ in range(25):
            c, i, j = rng.integers(3), rng.integers(17), rng.integers(19)
            h = 1e-6
            xp, xm = x.copy(), x.copy()
            xp[c, i, j] += h
            xm[c, i, j] -= h
            fd = (rl.render_loss(xp, y, lam)["loss"] - rl.render_loss(xm, y, lam)["loss"]) / (2 * h)
            assert r["dL_dimage"][c, i, j] == pytest.approx(fd, rel=2e-6, abs=1e-11)
