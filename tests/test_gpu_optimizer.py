"""GPU parity of f4: mg_density_stats and mg_adam_step through the C-ABI against oracle/optimizer.py.

Tolerances of the Adam step: derived from the kernel's arithmetic in parity_util.check_adam_step (same fp32 inputs on both
sides, scalars included: they cross the C-ABI as float).  The statistics: one sqrt + 3 roundings, 4e-7 relative.
"""
import numpy as np
import pytest
import torch

from paper_2412_20522_b200 import binding as mg

import parity_util as pu

pytestmark = pytest.mark.gpu

GROUP_ROWS = [("means", 3, 1.6e-4), ("log_scales", 3, 5e-3), ("quats", 4, 1e-3), ("opacity_logits", 1, 5e-2),
              ("sh", 48, 2.5e-3), ("mask_scores", 2, 1e-2)]


@pytest.fixture(scope="module", autouse=True)
def _need_gpu():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    mg.lib()


def _groups(rng, n, rows=GROUP_ROWS):
    out = []
    for name, rf, lr in rows:
        shape = (n, rf) if rf > 1 else (n,)
        p = rng.normal(0, 1, shape).astype(np.float32)
        g = (rng.normal(0, 1, shape) * 10.0 ** rng.uniform(-7, 1, shape)).astype(np.float32)
        g[rng.random(shape) < 0.1] = 0.0
        m = (rng.normal(0, 1, shape) * 1e-2).astype(np.float32)
        v = (rng.random(shape) * 1e-3).astype(np.float32)
        out.append([name, p, g, m, v, lr])
    return out


def _run(groups, b1, b2, eps, step, radii=None):
    dev = [[torch.from_numpy(a.copy()).cuda() for a in (p, g, m, v)] + [lr] for _, p, g, m, v, lr in groups]
    mg.mg_adam_step([tuple(d) for d in dev], b1, b2, eps, step, None if radii is None else torch.from_numpy(radii).cuda())
    torch.cuda.synchronize()
    return [(d[0].cpu().numpy(), d[2].cpu().numpy(), d[3].cpu().numpy()) for d in dev]


def _check(groups, got, b1, b2, eps, step, vis=None):
    from oracle import optimizer as opt

    # Same inputs on both sides: beta1, beta2, eps and lr cross the C-ABI as `float` (include/mg.h), so the oracle gets
    # the fp32-rounded values the kernel receives, upcast -- 1 - 0.999f differs from 1 - 0.999 by 1.3e-5 relative,
    # which is an input difference, not arithmetic error.
    f32 = lambda x: float(np.float32(x))
    b1, b2, eps = f32(b1), f32(b2), f32(eps)
    for (name, p, g, m, v, lr), (pg, mgot, vgot) in zip(groups, got):
        pr, mr, vr = opt.adam_step(p, g, m, v, f32(lr), b1, b2, eps, step, row_visible=vis)
        pu.check_adam_step((pg, mgot, vgot), (pr, mr, vr), p, g, f32(lr), b1, b2, eps, step, name)
        if vis is not None:  # untouched rows: bit-identical
            assert np.array_equal(pg[~vis], p[~vis]) and np.array_equal(mgot[~vis], m[~vis]) and np.array_equal(vgot[~vis], v[~vis])


@pytest.mark.parametrize("n", [1, 5, 1023, 4097, 200_000])
@pytest.mark.parametrize("step", [1, 7, 30000])
def test_adam_step_parity_all_groups_one_launch(n, step):
    """Sizes span several blocks, group boundaries inside a launch and ragged tails (n * row_floats not a multiple of 4)."""
    rng = np.random.default_rng(n + step)
    groups = _groups(rng, n)
    got = _run(groups, 0.9, 0.999, 1e-15, step)
    _check(groups, got, 0.9, 0.999, 1e-15, step)


def test_adam_step_parity_at_the_bench_size():
    """The size bench.py times (next_rows.optimizer): 3 M Gaussians, all attribute groups in one launch, 59 floats per
    Gaussian = 177 M parameters -- block indices past 2^16 per group, element offsets past 2^27."""
    n = 3_000_000
    rng = np.random.default_rng(33)
    groups = _groups(rng, n)
    got = _run(groups, 0.9, 0.999, 1e-15, 7)
    _check(groups, got, 0.9, 0.999, 1e-15, 7)


def test_adam_first_step_from_zero_moments_is_a_sign_step():
    rng = np.random.default_rng(0)
    g = rng.normal(0, 1, (1000, 3)).astype(np.float32)
    p = rng.normal(0, 1, (1000, 3)).astype(np.float32)
    z = np.zeros_like(p)
    (pn, mn, vn), = _run([["x", p, g, z, z, 0.01]], 0.9, 0.999, 1e-15, 1)
    np.testing.assert_allclose(pn, p - 0.01 * np.sign(g), atol=2e-7 * (np.abs(p).max() + 1))


def test_adam_visible_rows_only():
    rng = np.random.default_rng(9)
    n = 50_001
    radii = (rng.integers(1, 30, n) * (rng.random(n) < 0.4)).astype(np.int32)
    groups = _groups(rng, n)
    got = _run(groups, 0.9, 0.999, 1e-15, 12, radii=radii)
    _check(groups, got, 0.9, 0.999, 1e-15, 12, vis=radii > 0)


def test_adam_empty_and_argument_checks():
    mg.mg_adam_step([], 0.9, 0.999, 1e-15, 1)
    z = torch.zeros(0, 3, device="cuda")
    mg.mg_adam_step([(z, z.clone(), z.clone(), z.clone(), 0.1)], 0.9, 0.999, 1e-15, 1)
    t = torch.zeros(8, 3, device="cuda")
    with pytest.raises(mg.MgError):
        mg.mg_adam_step([(t, t.clone(), t.clone(), t.clone(), 0.1)], 0.9, 0.999, 1e-15, 0)  # step counts from 1
    with pytest.raises(mg.MgError):
        mg.mg_adam_step([(t, t.clone(), t.clone(), t.clone(), 0.1)] * 9, 0.9, 0.999, 1e-15, 1)
    with pytest.raises(mg.MgError):  # with radii, every group has one row per Gaussian
        t2 = torch.zeros(4, 3, device="cuda")
        mg.mg_adam_step([(t, t.clone(), t.clone(), t.clone(), 0.1), (t2, t2.clone(), t2.clone(), t2.clone(), 0.1)],
                        0.9, 0.999, 1e-15, 1, radii=torch.ones(8, dtype=torch.int32, device="cuda"))


@pytest.mark.parametrize("n", [0, 1, 777, 300_000, 3_000_000])
def test_density_stats_parity(n):
    from oracle import optimizer as opt

    rng = np.random.default_rng(n)
    g = (rng.normal(0, 1, (n, 2)) * 10.0 ** rng.uniform(-8, -2, (n, 1))).astype(np.float32)
    radii = (rng.integers(1, 400, n) * (rng.random(n) < 0.7)).astype(np.int32)
    acc0 = (rng.random(n) * 1e-3).astype(np.float32)
    den0 = rng.integers(0, 100, n).astype(np.float32)
    mx0 = rng.integers(0, 300, n).astype(np.float32)
    scale = (648.5, 420.0)
    d = [torch.from_numpy(a.copy()).cuda() for a in (g, radii, acc0, den0, mx0)]
    mg.mg_density_stats(d[0], d[1], scale, d[2], d[3], d[4])
    torch.cuda.synchronize()
    acc, den, mx = opt.density_stats(g, radii, acc0, den0, mx0, scale)
    np.testing.assert_allclose(d[2].cpu().numpy(), acc, rtol=4e-7, atol=1e-37)
    assert np.array_equal(d[3].cpu().numpy(), den) and np.array_equal(d[4].cpu().numpy(), mx)
    inv = radii == 0
    assert np.array_equal(d[2].cpu().numpy()[inv], acc0[inv])
