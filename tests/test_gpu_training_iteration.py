"""One whole training iteration of the paper's method through the C-ABI (every call except the optimiser):
mask sample -> preprocess -> bin_sort -> render_fwd -> render_loss -> render_bwd -> mask_loss -> mask_sample_bwd ->
preprocess_bwd, against the same chain of the CPU oracles in fp64 run from the same raw inputs (the hard mask
sample is staged: the oracle chain uses the GPU's masks, whose own parity is tested in test_gpu_mask_head.py).
End-to-end mode: decisions that sit on a threshold may differ between fp32 and fp64, so gradients are compared in
relative 2-norm."""
import numpy as np
import pytest
import torch

import oracle as orc
from oracle import mask_head as mh
from oracle import render_loss as rl
from paper_2412_20522_b200 import binding as mg
from paper_2412_20522_b200 import scenes

pytestmark = pytest.mark.gpu

TAU, LAMBDA_M, LAMBDA_DSSIM = 1.0, float(np.float32(0.05)), float(np.float32(0.2))


@pytest.mark.parametrize("name", ["cfg1", "cfg2"])
def test_training_iteration_chain(name):
    sc = scenes.config1() if name == "cfg1" else scenes.config2()
    cam, n = sc.camera, sc.N
    scores, u, _, _ = scenes.mask_head_inputs(n, seed=21, score_sigma=1.0)
    g, _ = mg.upload(sc)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    # target image: the scene rendered with every mask = 1 plus seeded noise (only an input of the loss; the noise
    # keeps I - G away from 0, where the L1 term's sign is decided by rounding on either side)
    fr = mg.Frame(cam, n)
    fr.forward(g, torch.ones(n, device="cuda"))
    noise = np.random.default_rng(5).normal(0.0, 0.05, (3, cam.height, cam.width)).astype(np.float32)
    target = (fr.image + torch.from_numpy(noise).cuda()).contiguous()
    # ---- GPU chain
    masks, soft = torch.empty(n, device="cuda"), torch.empty(n, device="cuda")
    mg.mg_mask_sample(dev(scores), dev(u), TAU, masks, soft)
    fr.forward(g, masks)
    dL_dimage = torch.empty_like(fr.image)
    lstats = torch.zeros(3, dtype=torch.float64, device="cuda")
    ws = torch.empty(mg.mg_render_loss_workspace_bytes(cam.width, cam.height), dtype=torch.uint8, device="cuda")
    mg.mg_render_loss(fr.image, target, LAMBDA_DSSIM, dL_dimage, lstats, ws)
    fr.backward(g, masks, dL_dimage)
    mstats = torch.zeros(3, dtype=torch.float64, device="cuda")
    mg.mg_mask_loss(masks, LAMBDA_M, fr.dL_dmask, mstats)
    dL_dscores = torch.empty(n, 2, device="cuda")
    mg.mg_mask_sample_bwd(soft, fr.dL_dmask, TAU, dL_dscores)
    torch.cuda.synchronize()
    # ---- oracle chain (fp64) on the same raw inputs and the GPU's hard masks
    m_np = masks.cpu().numpy()
    arrs = (sc.means, sc.log_scales, sc.quats, sc.opacity_logits, sc.sh)
    pre, ids, ranges, fwd = orc.full_forward(cam, arrs, m_np)
    loss = rl.render_loss(fwd["image"], target.cpu().numpy().astype(np.float64), LAMBDA_DSSIM)
    rb, pb = orc.full_backward(cam, arrs, m_np, pre, ids, ranges, loss["dL_dimage"])
    lm, gm = mh.mask_loss(m_np, LAMBDA_M)
    soft_ref = mh.sample(scores, u, TAU)["soft"]
    dsc = mh.sample_bwd(soft_ref, rb["dL_dmask"] + gm, TAU)
    # ---- compare
    ls = lstats.cpu().numpy()
    assert ls[2] == pytest.approx(loss["loss"], rel=1e-3, abs=1e-7)
    assert mstats.cpu().numpy()[1] == pytest.approx(lm, rel=1e-12)
    rel = lambda a, b: np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)
    errs = {"dL_dscores": rel(dL_dscores.cpu().numpy().astype(np.float64), dsc)}
    for k, ref in pb.items():
        if k.startswith("dL_"):
            errs[k] = rel(getattr(fr, k).cpu().numpy().astype(np.float64), ref)
    print(name, "L_render", ls[2], {k: f"{v:.1e}" for k, v in errs.items()})
    for k, v in errs.items():
        assert v < 1e-3, (k, v)
    assert np.abs(dsc).sum() > 0
