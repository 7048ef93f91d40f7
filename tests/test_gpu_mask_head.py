"""GPU parity of the mask head against oracle/mask_head.py on the same seeded inputs.
Hard decisions (d > 0) are integers decided by floating point: elements whose fp64 margin |d| is within fp32
reach of the tie are excluded, counted, and the count is bounded; every other element must match exactly."""
import numpy as np
import pytest
import torch

from oracle import mask_head as mh
from paper_2412_20522_b200 import binding as mg
from paper_2412_20522_b200 import scenes

pytestmark = pytest.mark.gpu

CUT = 2e-5  # |d| below this (d is O(1..10)) counts as threshold-sensitive


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


@pytest.mark.parametrize("n", [1, 33, 100_037, 3_000_000])
@pytest.mark.parametrize("tau", [1.0, 0.5])
def test_sample_loss_and_backward(n, tau):
    scores, u, _, g = scenes.mask_head_inputs(n)
    ref = mh.sample(scores, u, tau)
    masks, soft = torch.empty(n, device="cuda"), torch.empty(n, device="cuda")
    mg.mg_mask_sample(dev(scores), dev(u), tau, masks, soft)
    got_m, got_s = masks.cpu().numpy().astype(np.float64), soft.cpu().numpy().astype(np.float64)
    ok = ref["margin"] > CUT
    assert (~ok).sum() <= max(2, 2e-4 * n)
    assert np.array_equal(got_m[ok], ref["mask"][ok])
    np.testing.assert_allclose(got_s, ref["soft"], rtol=2e-5, atol=1e-6)
    # loss on the GPU's masks (staged): exact sum, fp64 loss, gradient added in place
    lam = float(np.float32(0.37))  # the C-ABI takes lambda_m as a float
    dmask = dev(g.copy())
    stats = torch.zeros(3, dtype=torch.float64, device="cuda")
    mg.mg_mask_loss(masks, lam, dmask, stats)
    loss, grad = mh.mask_loss(got_m, lam)
    st = stats.cpu().numpy()
    assert st[0] == got_m.sum() and st[2] == pytest.approx(got_m.mean(), rel=1e-15)
    assert st[1] == pytest.approx(loss, rel=1e-13)
    np.testing.assert_allclose(dmask.cpu().numpy(), (g.astype(np.float64) + grad), rtol=2e-7, atol=1e-12)
    # straight-through backward on the GPU's soft sample (staged)
    dscores = torch.empty(n, 2, device="cuda")
    mg.mg_mask_sample_bwd(soft, dmask, tau, dscores)
    want = mh.sample_bwd(got_s, dmask.cpu().numpy(), tau)
    np.testing.assert_allclose(dscores.cpu().numpy(), want, rtol=1e-5, atol=1e-12)


@pytest.mark.parametrize("n", [1, 2049, 100_037])
def test_prune_rule_and_compaction(n):
    scores, _, u10, _ = scenes.mask_head_inputs(n, seed=11)
    keep_ref, margin = mh.prune_keep(scores, u10)
    keep = torch.empty(n, dtype=torch.uint8, device="cuda")
    mg.mg_mask_prune_keep(dev(scores), dev(u10), keep)
    got = keep.cpu().numpy().astype(bool)
    ok = margin > CUT
    assert (~ok).sum() <= max(2, 2e-3 * n)
    assert np.array_equal(got[ok], keep_ref[ok])
    # compaction by the GPU's own flags (staged): bit-exact rows, in order
    rng = np.random.default_rng(3)
    arrays = [rng.normal(size=(n, 3)).astype(np.float32), rng.normal(size=(n, 4)).astype(np.float32),
              rng.normal(size=(n,)).astype(np.float32), rng.normal(size=(n, 16, 3)).astype(np.float32), scores]
    src = [dev(a) for a in arrays]
    dst = [torch.full_like(t, float("nan")) for t in src]
    ws = torch.empty(mg.mg_compact_workspace_bytes(n), dtype=torch.uint8, device="cuda")
    n_out = torch.zeros(1, dtype=torch.int64).pin_memory()
    mg.mg_compact(keep, src, dst, ws, n_out)
    torch.cuda.synchronize()
    want, cnt = mh.compact(got, arrays)
    assert int(n_out[0]) == cnt
    for d, w in zip(dst, want):
        assert np.array_equal(d.cpu().numpy()[:cnt], w)


def test_compaction_edge_cases():
    n = 5000
    a = np.arange(n * 3, dtype=np.float32).reshape(n, 3)
    ws = torch.empty(mg.mg_compact_workspace_bytes(n), dtype=torch.uint8, device="cuda")
    n_out = torch.zeros(1, dtype=torch.int64).pin_memory()
    for flags in (np.zeros(n, np.uint8), np.ones(n, np.uint8)):
        dst = [torch.zeros(n, 3, device="cuda")]
        mg.mg_compact(dev(flags), [dev(a)], dst, ws, n_out)
        torch.cuda.synchronize()
        assert int(n_out[0]) == int(flags.sum())
        if flags.all():
            assert np.array_equal(dst[0].cpu().numpy(), a)
    # nothing to do
    mg.mg_compact(torch.empty(0, dtype=torch.uint8, device="cuda"), [], [], ws, n_out)
    torch.cuda.synchronize()
    assert int(n_out[0]) == 0


def test_uniforms_at_and_beyond_the_endpoints():
    """include/mg.h / DESIGN.md reading 29: a uniform outside (0,1) is taken as the nearest fp32 value inside it.  Every
    pair of {0, 1, a denormal, 2^-126, 1 - 2^-24, a negative value, a value above 1} with ordinary ones, through
    mg_mask_sample and mg_mask_prune_keep: finite outputs, and the oracle's hard and soft samples."""
    special = np.array([0.0, 1.0, 1e-45, np.finfo(np.float32).tiny, 1.0 - 2.0 ** -24, -3.0, 7.0, 0.5, 0.013], np.float32)
    a, b = np.meshgrid(special, special, indexing="ij")
    u = np.stack([a.ravel(), b.ravel()], axis=1).astype(np.float32)
    n = u.shape[0]
    scores = np.random.default_rng(3).normal(0.0, 2.0, (n, 2)).astype(np.float32)
    for tau in (1.0, 0.5):
        ref = mh.sample(scores, u, tau)
        masks, soft = torch.empty(n, device="cuda"), torch.empty(n, device="cuda")
        mg.mg_mask_sample(dev(scores), dev(u), tau, masks, soft)
        got_m, got_s = masks.cpu().numpy().astype(np.float64), soft.cpu().numpy().astype(np.float64)
        assert np.isfinite(got_s).all() and np.isfinite(ref["soft"]).all()
        ok = ref["margin"] > CUT
        assert ok.sum() >= n - 2
        assert np.array_equal(got_m[ok], ref["mask"][ok])
        np.testing.assert_allclose(got_s, ref["soft"], atol=2e-5, rtol=0)
    u10 = np.stack([np.roll(u, k, axis=0) for k in range(10)]).astype(np.float32)
    keep_ref, margin = mh.prune_keep(scores, u10)
    keep = torch.empty(n, dtype=torch.uint8, device="cuda")
    mg.mg_mask_prune_keep(dev(scores), dev(u10), keep)
    ok = margin > CUT
    assert np.array_equal(keep.cpu().numpy().astype(bool)[ok], keep_ref[ok])
