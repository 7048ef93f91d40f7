"""CPU oracle of density-control statistics and the optimiser step -- TEST INFRASTRUCTURE,
not the product.

Plain numpy, fp64, one statement per step; no blocking, no fusion.  Only tests/ and bench.py's cpu_baseline leg may
import this.

What the paper fixes: nothing beyond the words.  PAPER.md:124 (sec. 3.5): "This pruning procedure is applied at every
densification step, and every 1000 iterations after densification"; "without altering the 3DGS pipeline
such as ... the densification scheme"; "All models are trained for 30,000 iterations"; PAPER.md:205
"mask learning rate".  So the method keeps the density control and the optimiser of the 3DGS method it modifies and
prints neither.  Readings taken (readings 27-28):

 27 density-control statistics, accumulated after every backward pass over the Gaussians VISIBLE in that view
    (radius > 0, i.e. not culled by mg_preprocess):
        grad_accum[i] += || (sx dL/dmean2d_x, sy dL/dmean2d_y) ||_2        screen-space positional gradient norm
        denom[i]      += 1                                                  number of views the Gaussian was seen in
        max_radii[i]   = max(max_radii[i], radius_i)                        largest screen radius seen, pixels
    (sx, sy) converts the gradient from this library's pixel units (reading 19) to whatever unit the caller's threshold
    is in (the 3DGS lineage uses normalised device coordinates: sx = W/2, sy = H/2); (1, 1) keeps pixels.
    A densification step then looks at grad_accum / denom; that decision and the cloning/splitting itself need the
    paper's training data to validate and are out of scope.
 28 optimiser: Adam (Kingma & Ba 2015, Algorithm 1) with bias correction, one learning rate per attribute group
    (means, log-scales, quaternions, opacity logits, SH, the 2 mask scores):
        m <- b1 m + (1 - b1) g ;  v <- b2 v + (1 - b2) g^2
        p <- p - lr (m / (1 - b1^t)) / (sqrt(v / (1 - b2^t)) + eps),   t = 1, 2, ... the step number
    Optionally restricted to the Gaussians visible in the view (rows with radius 0 are left untouched: parameter AND
    moments), the "sparse" variant that skips the rows which received no gradient at all.

Parity pinned (tests/test_optimizer_pins.py): Adam against torch.optim.Adam (a library routine, fp64, several steps,
several groups), the closed form of the first step (u = lr g / (|g| + eps)), a constant-gradient closed form at step t,
a scalar hand loop; the statistics against a per-Gaussian Python loop and the triangle-inequality invariant.
"""
from __future__ import annotations

import numpy as np


def density_stats(dL_dmeans2d, radii, grad_accum, denom, max_radii, scale=(1.0, 1.0)):
    """Reading 27.  dL_dmeans2d [N,2], radii [N] int; grad_accum, denom, max_radii [N] float64 are UPDATED copies
    (returned); Gaussians with radii == 0 are left unchanged."""
    g = np.asarray(dL_dmeans2d, np.float64)
    r = np.asarray(radii)
    acc = np.array(grad_accum, np.float64, copy=True)
    den = np.array(denom, np.float64, copy=True)
    mx = np.array(max_radii, np.float64, copy=True)
    vis = r > 0
    gx = scale[0] * g[:, 0]
    gy = scale[1] * g[:, 1]
    norm = np.sqrt(gx * gx + gy * gy)
    acc[vis] = acc[vis] + norm[vis]
    den[vis] = den[vis] + 1.0
    mx[vis] = np.maximum(mx[vis], r[vis].astype(np.float64))
    return acc, den, mx


def adam_step(p, g, m, v, lr, beta1, beta2, eps, t, row_visible=None):
    """Reading 28.  p, g, m, v: arrays of one attribute group, shape [N, ...]; t >= 1 the step number.  Returns the
    updated (p, m, v) as new fp64 arrays.  row_visible [N] bool (optional): rows where it is False are returned
    unchanged (parameter and both moments)."""
    p = np.asarray(p, np.float64)
    g = np.asarray(g, np.float64)
    m = np.asarray(m, np.float64)
    v = np.asarray(v, np.float64)
    m_new = beta1 * m + (1.0 - beta1) * g
    v_new = beta2 * v + (1.0 - beta2) * g * g
    m_hat = m_new / (1.0 - beta1 ** t)
    v_hat = v_new / (1.0 - beta2 ** t)
    p_new = p - lr * m_hat / (np.sqrt(v_hat) + eps)
    if row_visible is not None:
        keep = np.asarray(row_visible, bool)
        sel = keep.reshape((-1,) + (1,) * (p.ndim - 1))
        p_new = np.where(sel, p_new, p)
        m_new = np.where(sel, m_new, m)
        v_new = np.where(sel, v_new, v)
    return p_new, m_new, v_new
