"""The inference path: compact away the Gaussians with M = 0, then project, sort and
render forward-only with every mask = 1.  The paper's claim behind masked rasterization (masked
Gaussians "will not affect the rendered result and act as pruned") is checked on the GPU path itself:
the masked render of ALL Gaussians equals, bit for bit, the unmasked render of the compacted survivors -- and the
composition compact -> preprocess -> bin_sort -> render_fwd(M = 1) is compared with the ORACLE run on the survivors:
staged (lists bit-exact, blend within north_star's image tolerance) and end to end from the raw compacted inputs."""
import numpy as np
import pytest
import torch

import parity_util as pu
from paper_2412_20522_b200 import binding as mg
from paper_2412_20522_b200 import scenes

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("name", ["cfg1", "cfg2", "cfg3_small", "cfg3_full"])
def test_masked_render_equals_render_of_the_compacted_survivors(name, oracle):
    sc = {"cfg1": scenes.config1, "cfg2": scenes.config2, "cfg3_small": lambda: scenes.config3(n=60_000, width=333, height=211),
          "cfg3_full": scenes.config3}[name]()
    cam = sc.camera
    g, m = mg.upload(sc)
    fr = mg.Frame(cam, sc.N)
    fr.forward(g, m)  # masked render of all Gaussians
    torch.cuda.synchronize()
    # compaction by the masks (keep = M != 0), stable
    keep = (m != 0).to(torch.uint8)
    names = ["means", "log_scales", "quats", "opacity_logits", "sh"]
    src = [g[k] for k in names]
    dst = [torch.empty_like(t) for t in src]
    ws = torch.empty(mg.mg_compact_workspace_bytes(sc.N), dtype=torch.uint8, device="cuda")
    n_out = torch.zeros(1, dtype=torch.int64).pin_memory()
    mg.mg_compact(keep, src, dst, ws, n_out)
    torch.cuda.synchronize()
    n_kept = int(n_out[0])
    assert n_kept == int((sc.masks != 0).sum())
    g2 = {k: t[:n_kept].contiguous() for k, t in zip(names, dst)}
    for k in names:  # the compacted arrays are the kept rows, in order
        assert torch.equal(g2[k], g[k][keep.bool()])
    fr2 = mg.Frame(cam, n_kept)
    fr2.forward(g2, torch.ones(n_kept, device="cuda"))
    torch.cuda.synchronize()
    assert fr2.R <= fr.R
    assert torch.equal(fr.image, fr2.image), float((fr.image - fr2.image).abs().max())
    assert torch.equal(fr.final_T, fr2.final_T)
    print(name, "N", sc.N, "kept", n_kept, "R", fr.R, "->", fr2.R)
    # ---- against the oracle: the survivors as a scene of their own, every mask = 1
    kb = sc.masks != 0
    sub = scenes.Scene("survivors", sc.means[kb], sc.log_scales[kb], sc.quats[kb], sc.opacity_logits[kb], sc.sh[kb],
                       np.ones(n_kept, np.float32), sc.cameras, sc.seed)
    ones = sub.masks
    s1 = pu.check_preprocess(fr2, sub, cam, max_flag_frac=0.02)
    ids2, ranges2 = pu.check_bin_sort(fr2, cam)  # the oracle's lists from the GPU's depths and rects: bit-exact
    if name != "cfg3_full":
        _, s3 = pu.check_render_fwd(fr2, cam, ones, ids2, ranges2, max_flag_frac=2e-3)
        pre, ids, ranges, fwd = oracle.full_forward(cam, pu.arrays(sub), ones)  # end to end, fp64 from the raw inputs
        img = pu.f64(fr2.image)
        flag = fwd["margin"] < pu.CUT_E2E
        err = np.abs(img - fwd["image"])
        bad = (err > pu.IMG_ATOL + pu.IMG_RTOL * np.abs(fwd["image"])).any(0) & ~flag
        same_lists = fr2.R == len(ids) and np.array_equal(pu.u32(fr2.sorted_ids)[: fr2.R], ids)
        assert bad.mean() <= (0.0 if same_lists else 5e-3), f"{bad.sum()} non-flagged pixels outside tolerance"
        assert flag.mean() < 0.02
        print("PARITY", name, "inference vs oracle", dict(preprocess=s1, render_fwd=s3, e2e_flagged=int(flag.sum()),
                                                           e2e_bad=int(bad.sum()), same_lists=bool(same_lists)))
    else:  # full size: the blend on sampled tiles the oracle can walk in seconds
        gw, gh = mg.grid(cam)
        lens = (ranges2[:, 1].astype(np.int64) - ranges2[:, 0])
        tiles = sorted(set(np.random.default_rng(3).choice(gw * gh, 24, replace=False).tolist()) | {int(np.argmax(lens)), gw - 1, gw * gh - 1})
        ranges_s = np.zeros_like(ranges2)
        ranges_s[tiles] = ranges2[tiles]
        _, s3 = pu.check_render_fwd(fr2, cam, ones, ids2, ranges_s, tiles=tiles, max_flag_frac=2e-3)
        print("PARITY", name, "inference vs oracle (sampled tiles)", dict(preprocess=s1, render_fwd=s3))
