"""The inference path: compact away the Gaussians with M = 0, then project, sort and
render forward-only with every mask = 1.  The paper's claim behind masked rasterization (masked
Gaussians "will not affect the rendered result and act as pruned") is checked on the GPU path itself:
the masked render of ALL Gaussians equals, bit for bit, the unmasked render of the compacted survivors."""
import numpy as np
import pytest
import torch

import parity_util as pu
from paper_2412_20522_b200 import binding as mg
from paper_2412_20522_b200 import scenes

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("name", ["cfg1", "cfg2", "cfg3_small", "cfg3_full"])
def test_masked_render_equals_render_of_the_compacted_survivors(name):
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
