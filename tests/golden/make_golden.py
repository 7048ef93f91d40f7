"""Writes tests/golden/tiny_scene.txt: a regression net for the ORACLE itself.

    python tests/golden/make_golden.py

Calls only oracle/ and the seeded input generator (paper_2412_20522_b200/scenes.py, which holds none of the
method's arithmetic).  No value comes from the CUDA path.  The paper (arXiv 2412.20522) prints no worked
numeric example for the masked blend (Fig. 1, is qualitative), so these are not the paper's
numbers: they freeze the oracle's output on the 8-Gaussian finite-difference scene, so that a later edit of
the oracle that changes its arithmetic shows up as a diff here and must be justified (DESIGN.md readings).
The pins that tie the oracle to the paper are in tests/test_oracle_pins.py.
"""
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)

import oracle as orc  # noqa: E402
from paper_2412_20522_b200 import scenes  # noqa: E402

OUT = os.path.join(HERE, "tiny_scene.txt")
PIXELS = [(5, 7), (16, 16), (20, 11), (31, 31), (0, 0), (13, 22)]  # (x, y)


def compute():
    sc = scenes.tiny_fd_scene()
    cam = sc.camera
    arrs = (sc.means, sc.log_scales, sc.quats, sc.opacity_logits, sc.sh)
    pre, ids, ranges, fwd = orc.full_forward(cam, arrs, sc.masks)
    g = sc.dL_dimage().astype(np.float64)
    rb, pb = orc.full_backward(cam, arrs, sc.masks, pre, ids, ranges, g)
    rows = [("R", float(len(ids))), ("image_sum", float(fwd["image"].sum())), ("final_T_sum", float(fwd["final_T"].sum())),
            ("n_contrib_sum", float(fwd["n_contrib"].sum()))]
    for x, y in PIXELS:
        for c in range(3):
            rows.append((f"image[{c}][{y}][{x}]", float(fwd["image"][c, y, x])))
        rows.append((f"final_T[{y}][{x}]", float(fwd["final_T"][y, x])))
        rows.append((f"n_contrib[{y}][{x}]", float(fwd["n_contrib"][y, x])))
    for k in sorted(rb):
        if k.startswith("dL_"):
            rows.append((f"{k}_sum", float(np.sum(rb[k]))))
            rows.append((f"{k}_abs_sum", float(np.abs(rb[k]).sum())))
    for k in sorted(pb):
        if k.startswith("dL_"):
            rows.append((f"{k}_sum", float(np.sum(pb[k]))))
            rows.append((f"{k}_abs_sum", float(np.abs(pb[k]).sum())))
    return rows


if __name__ == "__main__":
    with open(OUT, "w") as f:
        f.write("# oracle output on scenes.tiny_fd_scene() (8 Gaussians, 32x32, SH degree 3, bg = (0.2, 0.5, 0.7));\n"
                "# written by tests/golden/make_golden.py from oracle/ only -- not the paper's numbers (it prints none)\n")
        for k, v in compute():
            f.write(f"{k} {v!r}\n")
    print("wrote", OUT)
