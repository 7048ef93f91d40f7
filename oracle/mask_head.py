"""CPU oracle of the mask head -- TEST INFRASTRUCTURE, not the product.

Plain numpy, fp64, one statement per step of the paper's text; no blocking, no fusion.  Only tests/ and
bench.py's cpu_baseline leg may import this.  Random numbers are INPUTS (uniforms in (0,1)), never drawn here.

What the paper fixes (sec. 3.3): "we assign 2 learnable mask scores for each Gaussian, and
apply Gumbel-Softmax to sample one differentiable category out of the 2 scores, denoted M_i in {0,1}";
(sec. 3.5, Eq. 7-8): L_m = (1/N sum M_i)^2, L = L_render + lambda_m L_m;
"we sample each Gaussian 10 times and remove those that are never sampled".

Readings (readings 22-25): the Gumbel-Softmax estimator is the standard one of the paper's
reference [13] with a hard (one-hot) forward sample and the soft sample's derivative in the backward pass
(straight-through); category 1 = "present"; the temperature tau is not stated in the paper -> a parameter;
a tie (equal perturbed scores) gives M = 0.

  g_k   = -log(-log(u_k)),  u_k in (0,1)                       Gumbel(0,1) noise, k = 0, 1
          (reading 29: a uniform outside the open interval -- fp32 generators on [0,1) return exactly 0 with probability
          2^-24 per draw, and rounding to fp32 can give exactly 1 -- is taken as the nearest fp32 value inside it:
          u is clamped to [2^-126, 1 - 2^-24], so g lies in [-4.47, 16.64] and d is always finite)
  d     = (s_1 + g_1) - (s_0 + g_0)
  y_1   = softmax((s + g)/tau)_1 = 1 / (1 + exp(-d / tau))      soft sample
  M     = 1 if d > 0 else 0                                     hard sample = argmax of the perturbed scores
  dM/ds_1 := dy_1/ds_1 = y_1 (1 - y_1) / tau,   dM/ds_0 := -dM/ds_1      (straight-through)

The hard decision d > 0 is a floating-point decision of an integer: `sample` returns the margin |d| so that
a comparison can exclude elements whose decision sits within rounding reach of the tie.
Parity pinned: closed forms, finite differences, sampling frequencies (tests/test_mask_head_pins.py).
"""
from __future__ import annotations

import numpy as np


U_MIN = float(np.finfo(np.float32).tiny)                 # 2^-126, the smallest normal fp32
U_MAX = float(np.float32(1.0) - np.float32(2.0 ** -24))  # 1 - 2^-24, the largest fp32 below 1


def gumbel(u):
    u = np.clip(np.asarray(u, np.float64), U_MIN, U_MAX)  # reading 29
    return -np.log(-np.log(u))


def sample(scores, u, tau=1.0):
    """scores [N,2], u [N,2] uniforms in (0,1).  Returns dict(mask [N] in {0,1}, soft [N] = y_1, margin [N] = |d|)."""
    s = np.asarray(scores, np.float64)
    g = gumbel(u)
    d = (s[:, 1] + g[:, 1]) - (s[:, 0] + g[:, 0])
    soft = 1.0 / (1.0 + np.exp(-d / tau))
    mask = (d > 0.0).astype(np.float64)
    return dict(mask=mask, soft=soft, margin=np.abs(d))


def sample_bwd(soft, dL_dmask, tau=1.0):
    """Straight-through: dL/ds_1 = dL/dM * y_1 (1 - y_1) / tau, dL/ds_0 = -dL/ds_1.  Returns [N,2]."""
    y = np.asarray(soft, np.float64)
    t = np.asarray(dL_dmask, np.float64) * y * (1.0 - y) / tau
    return np.stack([-t, t], axis=1)


def mask_loss(mask, lambda_m):
    """Eq. 7-8: lambda_m * L_m = lambda_m * (mean M)^2 and its gradient lambda_m * 2 * mean(M) / N per element."""
    m = np.asarray(mask, np.float64)
    n = m.shape[0]
    mean = m.sum() / n if n else 0.0
    loss = lambda_m * mean * mean
    grad = np.full(n, lambda_m * 2.0 * mean / n if n else 0.0)
    return loss, grad


def prune_keep(scores, u10, tau=1.0):
    """keep a Gaussian iff it is sampled (M = 1) in at least one of the draws u10 [S,N,2]."""
    keep = np.zeros(np.asarray(scores).shape[0], bool)
    margin = np.full(keep.shape, np.inf)
    for k in range(np.asarray(u10).shape[0]):
        r = sample(scores, u10[k], tau)
        keep |= r["mask"] > 0
        margin = np.minimum(margin, r["margin"])
    return keep, margin


def compact(keep, arrays):
    """Stable compaction of every attribute array (rows of kept Gaussians, in order)."""
    keep = np.asarray(keep, bool)
    return [np.ascontiguousarray(a[keep]) for a in arrays], int(keep.sum())
