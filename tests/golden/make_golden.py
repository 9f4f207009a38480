"""Writes tests/golden/tiny_oracle.txt: values of the CPU oracle on BASELINE.json config 1 ("tiny", seeded).

    python tests/golden/make_golden.py

Calls only oracle/ and the seeded scene generator (no CUDA path).  The paper prints no worked
numerical example of the rasterizer -- its numbers are dataset metrics -- so this fixture is not a paper value:
it freezes the oracle's own output so that a later change to the oracle's arithmetic (which must cite the
passage that justifies it) shows up as a diff of this file.  What the oracle computes is pinned to the paper
and to closed forms in tests/test_oracle_*.py.
"""
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

PIXELS = [(0, 0), (127, 0), (0, 127), (127, 127), (64, 64), (31, 97), (100, 45), (77, 77)]
PRIMS = [0, 1, 17, 255, 512, 1023]


def golden_lines():
    from oracle import gabsplat_oracle as orc
    from paper_2508_05343_b200 import scenes
    scene = scenes.make_scene("tiny")
    cam = scenes.make_cameras("tiny")[0]
    dL = scenes.make_image_grad("tiny", 0, cam)
    b = orc.bin_sort(scene, cam)
    f = orc.render_forward(scene, cam)
    g = orc.render_backward(scene, cam, dL)
    out = ["# oracle on config 1 (tiny): Eq.2, 9-13 of PAPER.md as read in DESIGN.md 3; written by make_golden.py",
           "num_instances %d" % b["num_instances"],
           "keys_head " + " ".join("%016x" % int(k) for k in b["keys"][:8]),
           "ids_head " + " ".join("%d" % int(i) for i in b["ids"][:8])]
    for x, y in PIXELS:
        out.append("pixel %d %d  rgb %.12e %.12e %.12e  T %.12e  n_contrib %d" % (
            x, y, f["image"][0, y, x], f["image"][1, y, x], f["image"][2, y, x], f["final_T"][y, x], f["n_contrib"][y, x]))
    for i in PRIMS:
        out.append("grad %d  d_means %s  d_opacity %.12e  d_freqs0 %s  d_weights %s" % (
            i, " ".join("%.12e" % v for v in g["d_means"][i]), g["d_opacities"][i],
            " ".join("%.12e" % v for v in g["d_freqs"][i, 0]), " ".join("%.12e" % v for v in g["d_weights"][i])))
    return out


if __name__ == "__main__":
    path = os.path.join(HERE, "tiny_oracle.txt")
    with open(path, "w") as fh:
        fh.write("\n".join(golden_lines()) + "\n")
    print("wrote", path)
