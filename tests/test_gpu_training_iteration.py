"""Two whole training iterations of the paper's method through the C-ABI:
mask sample -> preprocess -> bin_sort -> render_fwd -> render_loss -> render_bwd -> mask_loss -> mask_sample_bwd ->
preprocess_bwd -> density statistics -> Adam step, against the same chain of the CPU oracles in fp64 run from the same
raw inputs (staged where a decision or a state crosses: the oracle chain uses the GPU's hard masks, whose own parity is
tested in test_gpu_mask_head.py, and starts each iteration from the GPU's current fp32 parameters and moments).
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

import parity_util as pu

pytestmark = pytest.mark.gpu

TAU, LAMBDA_M, LAMBDA_DSSIM = 1.0, float(np.float32(0.05)), float(np.float32(0.2))


# scalars that cross the C-ABI as `float` are fp32 values here too, so that oracle and kernel get the same inputs
_f32 = lambda x: float(np.float32(x))
LRS = {k: _f32(v) for k, v in dict(means=1.6e-4, log_scales=5e-3, quats=1e-3, opacity_logits=5e-2, sh=2.5e-3, scores=1e-2).items()}
B1, B2, EPS = _f32(0.9), _f32(0.999), _f32(1e-15)


@pytest.mark.parametrize("name", ["cfg1", "cfg2"])
def test_training_iteration_chain(name):
    from oracle import optimizer as opt

    sc = scenes.config1() if name == "cfg1" else scenes.config2()
    cam, n = sc.camera, sc.N
    scores_np, _, _, _ = scenes.mask_head_inputs(n, seed=21, score_sigma=1.0)
    g, _ = mg.upload(sc)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    f64 = lambda t: t.cpu().numpy().astype(np.float64)
    # target image: the scene rendered with every mask = 1 plus seeded noise (only an input of the loss; the noise
    # keeps I - G away from 0, where the L1 term's sign is decided by rounding on either side)
    fr = mg.Frame(cam, n)
    fr.forward(g, torch.ones(n, device="cuda"))
    noise = np.random.default_rng(5).normal(0.0, 0.05, (3, cam.height, cam.width)).astype(np.float32)
    target = (fr.image + torch.from_numpy(noise).cuda()).contiguous()
    # trainable state on the device: the five attribute arrays of `g` + the mask scores, with Adam moments
    names = ["means", "log_scales", "quats", "opacity_logits", "sh", "scores"]
    params = dict(g)
    params["scores"] = dev(scores_np.astype(np.float32))
    mom = {k: (torch.zeros_like(v), torch.zeros_like(v)) for k, v in params.items()}
    acc, den, mxr = (torch.zeros(n, device="cuda") for _ in range(3))
    rel = lambda a, b: np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)
    for it in (1, 2):
        _, u, _, _ = scenes.mask_head_inputs(n, seed=21 + it, score_sigma=1.0)
        g_it = {k: params[k] for k in names[:5]}
        before = {k: f64(v) for k, v in params.items()}
        mom_before = {k: (f64(a), f64(b)) for k, (a, b) in mom.items()}
        stats_before = (f64(acc), f64(den), f64(mxr))
        # ---- GPU chain
        masks, soft = torch.empty(n, device="cuda"), torch.empty(n, device="cuda")
        mg.mg_mask_sample(params["scores"], dev(u), TAU, masks, soft)
        fr.forward(g_it, masks)
        dL_dimage = torch.empty_like(fr.image)
        lstats = torch.zeros(3, dtype=torch.float64, device="cuda")
        ws = torch.empty(mg.mg_render_loss_workspace_bytes(cam.width, cam.height), dtype=torch.uint8, device="cuda")
        mg.mg_render_loss(fr.image, target, LAMBDA_DSSIM, dL_dimage, lstats, ws)
        fr.backward(g_it, masks, dL_dimage)
        mstats = torch.zeros(3, dtype=torch.float64, device="cuda")
        mg.mg_mask_loss(masks, LAMBDA_M, fr.dL_dmask, mstats)
        dL_dscores = torch.empty(n, 2, device="cuda")
        mg.mg_mask_sample_bwd(soft, fr.dL_dmask, TAU, dL_dscores)
        mg.mg_density_stats(fr.dL_dmeans2d, fr.radii, (cam.width / 2, cam.height / 2), acc, den, mxr)
        grads = dict(means=fr.dL_dmeans, log_scales=fr.dL_dlog_scales, quats=fr.dL_dquats,
                     opacity_logits=fr.dL_dopacity_logits, sh=fr.dL_dsh, scores=dL_dscores)
        grads_np = {k: f64(v) for k, v in grads.items()}
        mg.mg_adam_step([(params[k], grads[k], mom[k][0], mom[k][1], LRS[k]) for k in names], B1, B2, EPS, it)
        torch.cuda.synchronize()
        # ---- oracle chain (fp64) from the parameters this iteration started with and the GPU's hard masks
        m_np = masks.cpu().numpy()
        arrs = tuple(before[k] for k in names[:5])
        pre, ids, ranges, fwd = orc.full_forward(cam, arrs, m_np)
        loss = rl.render_loss(fwd["image"], f64(target), LAMBDA_DSSIM)
        rb, pb = orc.full_backward(cam, arrs, m_np, pre, ids, ranges, loss["dL_dimage"])
        lm, gm = mh.mask_loss(m_np, LAMBDA_M)
        soft_ref = mh.sample(before["scores"], u, TAU)["soft"]
        dsc = mh.sample_bwd(soft_ref, rb["dL_dmask"] + gm, TAU)
        # ---- compare the gradients
        ls = lstats.cpu().numpy()
        assert ls[2] == pytest.approx(loss["loss"], rel=1e-3, abs=1e-7)
        assert mstats.cpu().numpy()[1] == pytest.approx(lm, rel=1e-12)
        errs = {"dL_dscores": rel(grads_np["scores"], dsc)}
        for k, ref in pb.items():
            if k.startswith("dL_"):
                errs[k] = rel(f64(getattr(fr, k)), ref)
        print(name, "iteration", it, "L_render", ls[2], {k: f"{v:.1e}" for k, v in errs.items()})
        for k, v in errs.items():
            assert v < 1e-3, (k, v)
        assert np.abs(dsc).sum() > 0
        # ---- the statistics and the step (staged on the GPU's own gradients): elementwise
        a_ref, d_ref, r_ref = opt.density_stats(f64(fr.dL_dmeans2d), fr.radii.cpu().numpy(), *stats_before,
                                                scale=(cam.width / 2, cam.height / 2))
        np.testing.assert_allclose(f64(acc), a_ref, rtol=1e-6, atol=1e-30)
        assert np.array_equal(f64(den), d_ref) and np.array_equal(f64(mxr), r_ref)
        for k in names:
            p_ref, m_ref, v_ref = opt.adam_step(before[k], grads_np[k], *mom_before[k], LRS[k], B1, B2, EPS, it)
            pu.check_adam_step((f64(params[k]), f64(mom[k][0]), f64(mom[k][1])), (p_ref, m_ref, v_ref), before[k],
                               grads_np[k], LRS[k], B1, B2, EPS, it, k)
        assert (f64(params["means"]) != before["means"]).any()
