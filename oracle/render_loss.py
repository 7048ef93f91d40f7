"""CPU oracle of the render loss -- TEST INFRASTRUCTURE, not the product.

Plain numpy / scipy, fp64.  Only tests/ may import this.

What the paper fixes: Eq. 8: L = L_render + lambda_m L_m, where L_render is "the original
rendering loss" -- the paper does not define it.  Reading 26: the loss of the
3DGS method the paper builds on (its reference [14]; "We modify the CUDA rasterization code of 3DGS",
PAPER.md:156):

    L_render = (1 - lambda) * mean |I - G|  +  lambda * (1 - mean SSIM(I, G)),      lambda = 0.2 by default,

SSIM per channel with an 11 x 11 Gaussian window (sigma = 1.5, normalised, separable), zero padding,
C1 = 0.01^2, C2 = 0.03^2, means over all 3 H W elements:

    mu1 = w * I, mu2 = w * G, s1 = w * I^2 - mu1^2, s2 = w * G^2 - mu2^2, s12 = w * (I G) - mu1 mu2
    SSIM = (2 mu1 mu2 + C1)(2 s12 + C2) / ((mu1^2 + mu2^2 + C1)(s1 + s2 + C2))

The window filter is scipy.ndimage.correlate1d applied along y then x (a library routine; mode="constant").
The gradient with respect to I is the chain rule through the five filtered maps, written out; it is pinned by
central finite differences in tests/test_render_loss_pins.py.
"""
from __future__ import annotations

import numpy as np
from scipy.ndimage import correlate1d

C1 = 0.01 ** 2
C2 = 0.03 ** 2
WINDOW = 11
SIGMA = 1.5


def window():
    x = np.arange(WINDOW, dtype=np.float64) - WINDOW // 2
    g = np.exp(-(x * x) / (2.0 * SIGMA * SIGMA))
    return g / g.sum()


def blur(a):
    """w * a per channel: separable 11-tap correlation, zero padding.  a [3,H,W]."""
    w = window()
    out = correlate1d(np.asarray(a, np.float64), w, axis=1, mode="constant", cval=0.0)
    return correlate1d(out, w, axis=2, mode="constant", cval=0.0)


def ssim_map(img, tgt):
    x, y = np.asarray(img, np.float64), np.asarray(tgt, np.float64)
    mu1, mu2 = blur(x), blur(y)
    e1, e2, e12 = blur(x * x), blur(y * y), blur(x * y)
    s1, s2, s12 = e1 - mu1 * mu1, e2 - mu2 * mu2, e12 - mu1 * mu2
    A, B = 2 * mu1 * mu2 + C1, 2 * s12 + C2
    C, D = mu1 * mu1 + mu2 * mu2 + C1, s1 + s2 + C2
    return A * B / (C * D), (mu1, mu2, A, B, C, D)


def render_loss(img, tgt, lam=0.2):
    """Returns dict(loss, l1, ssim, dL_dimage [3,H,W])."""
    x, y = np.asarray(img, np.float64), np.asarray(tgt, np.float64)
    n = x.size
    l1 = np.abs(x - y).sum() / n
    sm, (mu1, mu2, A, B, C, D) = ssim_map(x, y)
    ssim = sm.sum() / n
    loss = (1.0 - lam) * l1 + lam * (1.0 - ssim)
    # d SSIM(q) / d(mu1, E[x^2], E[xy])(q), the filtered maps held as independent variables
    # (s1 = e1 - mu1^2 and s12 = e12 - mu1 mu2 depend on mu1: dB/dmu1 = -2 mu2, dD/dmu1 = -2 mu1)
    CD = C * D
    d_mu1 = (2 * mu2 * B - 2 * mu2 * A) / CD - A * B / (CD * CD) * (2 * mu1 * D - 2 * mu1 * C)
    d_e1 = -A * B / (C * D * D)
    d_e12 = 2 * A / CD
    # back through the (symmetric) window: each filtered map is w * (.), so the adjoint is the same filter
    d_ssim = blur(d_mu1) + 2 * x * blur(d_e1) + y * blur(d_e12)
    grad = (1.0 - lam) * np.sign(x - y) / n - lam * d_ssim / n
    return dict(loss=loss, l1=l1, ssim=ssim, dL_dimage=grad)
