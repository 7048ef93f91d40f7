"""GPU parity of mg_render_loss against oracle/render_loss.py on the same seeded images:
sizes that span several 16x16 tiles with ragged edges, the bench image size, identical images, lambda 0 / 1."""
import numpy as np
import pytest
import torch

from oracle import render_loss as rl
from paper_2412_20522_b200 import binding as mg

pytestmark = pytest.mark.gpu


def run(x, y, lam):
    _, H, W = x.shape
    img, tgt = torch.from_numpy(x).cuda(), torch.from_numpy(y).cuda()
    grad = torch.empty_like(img)
    stats = torch.zeros(3, dtype=torch.float64, device="cuda")
    ws = torch.empty(mg.mg_render_loss_workspace_bytes(W, H), dtype=torch.uint8, device="cuda")
    mg.mg_render_loss(img, tgt, lam, grad, stats, ws)
    torch.cuda.synchronize()
    return stats.cpu().numpy(), grad.cpu().numpy().astype(np.float64)


def images(h, w, seed, smooth=False):
    rng = np.random.default_rng(seed)
    x = rng.uniform(0, 1, (3, h, w)).astype(np.float32)
    if smooth:  # a rendered-image-like pair: smooth target, noisy estimate of it
        yy, xx = np.mgrid[0:h, 0:w]
        base = 0.5 + 0.4 * np.sin(xx / 17.0)[None] * np.cos(yy / 23.0)[None] * np.array([1.0, 0.7, 0.4])[:, None, None]
        y = base.astype(np.float32)
        x = np.clip(y + rng.normal(0, 0.05, y.shape), 0, 1).astype(np.float32)
    else:
        y = rng.uniform(0, 1, (3, h, w)).astype(np.float32)
    return x, y


@pytest.mark.parametrize("h,w,smooth", [(1, 1, False), (16, 16, False), (37, 53, False), (211, 333, True), (840, 1297, True)])
@pytest.mark.parametrize("lam", [0.2, 1.0, 0.0])
def test_render_loss_parity(h, w, smooth, lam):
    x, y = images(h, w, 5, smooth)
    st, grad = run(x, y, lam)
    ref = rl.render_loss(x, y, lam)
    assert st[0] == pytest.approx(ref["l1"], rel=1e-6, abs=1e-12)
    assert st[1] == pytest.approx(ref["ssim"], rel=2e-5, abs=1e-7)
    assert st[2] == pytest.approx(ref["loss"], rel=2e-5, abs=1e-7)
    g = ref["dL_dimage"]
    tol = 1e-3 * np.abs(g) + 2e-5 * np.abs(g).max()
    bad = np.abs(grad - g) > tol
    assert not bad.any(), (int(bad.sum()), float(np.abs(grad - g).max()), float(np.abs(g).max()))
    assert np.linalg.norm(grad - g) <= 1e-4 * np.linalg.norm(g) + 1e-30


def test_identical_images():
    x, _ = images(64, 80, 9)
    st, grad = run(x, x.copy(), 0.2)
    assert st[0] == 0 and abs(st[1] - 1) < 1e-6 and abs(st[2]) < 1e-6
    assert np.abs(grad).max() < 1e-9
