"""include/mg.h: "Calls may overlap on different streams, and be issued from different host threads, as long as they share
no output or scratch buffer: the library keeps no device-side state of its own".  Two host threads, each with its own
stream, frame buffers and scene, run the whole hot path repeatedly at the same time; every result must be what the same
frame gives when it runs alone -- bit for bit for the integers, the image and final_T (deterministic), and within the
reordering of float atomics for the gradients."""
import threading

import numpy as np
import pytest
import torch

from paper_2412_20522_b200 import binding as mg
from paper_2412_20522_b200 import scenes

pytestmark = pytest.mark.gpu

EXACT = ["radii", "rects", "tiles_touched", "clamped", "tile_ranges", "n_contrib", "image", "final_T", "means2d", "depths",
         "conic_opacity", "rgb"]
GRADS = ["dL_dmeans2d", "dL_dconic", "dL_dopacity", "dL_drgb", "dL_dmask", "dL_dmeans", "dL_dlog_scales", "dL_dquats",
         "dL_dopacity_logits", "dL_dsh"]


def _snapshot(fr):
    out = {k: getattr(fr, k).clone() for k in EXACT + GRADS}
    out["sorted_ids"] = fr.sorted_ids[: fr.R].clone()
    out["R"] = fr.R
    return out


def _run_alone(sc):
    g, m = mg.upload(sc)
    gimg = torch.from_numpy(sc.dL_dimage()).cuda()
    fr = mg.Frame(sc.camera, sc.N)
    fr.forward(g, m)
    fr.backward(g, m, gimg)
    torch.cuda.synchronize()
    return _snapshot(fr)


def test_two_frames_on_two_streams_from_two_threads():
    mg.lib()
    specs = [lambda: scenes.config2(), lambda: scenes.config3(n=60_000, width=333, height=211)]
    scs = [f() for f in specs]
    alone = [_run_alone(sc) for sc in scs]
    results, errors = [None, None], []
    start = threading.Barrier(2)

    def worker(k):
        try:
            torch.cuda.set_device(0)
            st = torch.cuda.Stream()
            with torch.cuda.stream(st):
                sc = scs[k]
                g, m = mg.upload(sc)
                gimg = torch.from_numpy(sc.dL_dimage()).cuda()
                fr = mg.Frame(sc.camera, sc.N)
                fr.forward(g, m)  # sizes the sort buffers (one stream sync)
                st.synchronize()
                start.wait()
                for _ in range(40):  # no host sync inside: the two streams' kernels interleave on the device
                    fr.step(g, m, gimg)
                st.synchronize()
                assert int(fr.R_host[1]) == fr.R, "the sort saw another R than the projection reported"
                results[k] = _snapshot(fr)
        except Exception as e:  # noqa: BLE001 -- reported in the main thread
            errors.append((k, repr(e)))

    threads = [threading.Thread(target=worker, args=(k,)) for k in range(2)]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    assert not errors, errors
    for k in range(2):
        ref, got = alone[k], results[k]
        assert got["R"] == ref["R"]
        for name in EXACT + ["sorted_ids"]:
            assert torch.equal(got[name], ref[name]), (k, name)
        for name in GRADS:
            a, b = got[name].double(), ref[name].double()
            scale = float(b.abs().max())
            assert float((a - b).abs().max()) <= 2e-5 * scale + 1e-30, (k, name)
