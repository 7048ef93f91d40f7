"""Exact work counts of the workloads, from the oracle only (numerators of bench.py's throughput).

    python -m oracle.count_work 1 2 3     ->  oracle/work_counts.json

A pair evaluation = one (list entry, pixel) visited before the pixel stops; a blend = a pair evaluation
that passes the alpha filter, masked or not.  Backward counts are the pairs the reverse
traversal revisits (positions n_contrib..1) and the blends among them.  Every count also comes split by the
entry's mask (`*_masked` = the part on entries with M == 0): under DESIGN.md reading 5 the forward pass never
has to look at a masked entry and the backward pass owes it dL/dM only, so the algorithmic flop counts of
bench.py charge the two kinds differently.  Camera 0 of each config.  The counters are pinned by
tests/test_oracle_pins.py::test_work_counters_match_an_independent_count.
"""
import json
import os
import sys
import time

import numpy as np

import oracle as orc
from paper_2412_20522_b200 import scenes

OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "work_counts.json")


def count(cfg: int) -> dict:
    sc = scenes.make(cfg)
    cam = sc.camera
    arrs = (sc.means, sc.log_scales, sc.quats, sc.opacity_logits, sc.sh)
    t = time.time()
    pre, ids, ranges, fwd = orc.full_forward(cam, arrs, sc.masks)
    rb = orc.render_bwd(cam, sc.N, ids, ranges, pre["means2d"], pre["conic_opacity"], pre["rgb"], sc.masks,
                        sc.dL_dimage().astype(np.float64))
    lens = (ranges[:, 1] - ranges[:, 0]).astype(np.int64)
    return dict(config=cfg, N=sc.N, width=cam.width, height=cam.height, visible=int((pre["radii"] > 0).sum()),
                R=int(len(ids)), fwd_pair_evals=fwd["pair_evals"], fwd_blends=fwd["blends"],
                fwd_pair_evals_masked=fwd["pair_evals_masked"], fwd_blends_masked=fwd["blends_masked"],
                bwd_pair_evals=rb["pair_evals"], bwd_blends=rb["blends"],
                bwd_pair_evals_masked=rb["pair_evals_masked"], bwd_blends_masked=rb["blends_masked"],
                stopped_pixels=int((fwd["final_T"] < 1e-3).sum()), list_len_max=int(lens.max()),
                list_len_median=int(np.median(lens)), oracle_seconds=round(time.time() - t, 1))


if __name__ == "__main__":
    data = json.load(open(OUT)) if os.path.exists(OUT) else {}
    for c in [int(a) for a in sys.argv[1:]] or [1, 2]:
        data[str(c)] = count(c)
        print(data[str(c)], flush=True)
        json.dump(data, open(OUT, "w"), indent=1, sort_keys=True)
