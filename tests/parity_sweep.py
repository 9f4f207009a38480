"""Parity of the CUDA path against the CPU oracle on every view of a config, as a table (not a pytest module):

    python tests/parity_sweep.py [config] [K]        # default: unbounded (BASELINE.json config 3), its own K

Per view: instance count; sorted keys, ids and tile ranges bit-exact or not; undecidable pixels (reading C18); image
max error on decidable pixels; last contributor exact or not there; the worst gradient tensor (max-norm relative
error, dL/dimage zeroed on the undecidable pixels for both sides).  The oracle runs on the host cores (~10 s per
view at 1M primitives).  Output committed as profiles/r01_parity_sweep.md.
"""
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(HERE))
sys.path.insert(0, HERE)


def main():
    from gpu_helpers import rel_inf, run_gpu
    from oracle import gabsplat_oracle as orc
    from paper_2508_05343_b200 import scenes
    name = sys.argv[1] if len(sys.argv) > 1 else "unbounded"
    K = int(sys.argv[2]) if len(sys.argv) > 2 else None
    scene = scenes.make_scene(name, K=K)
    cams = scenes.make_cameras(name)
    print("| view | D | lists bit-exact | undecidable px | image max err (decidable) | last contributor exact | worst gradient |")
    print("|---|---|---|---|---|---|---|")
    for view, cam in enumerate(cams):
        dL = scenes.make_image_grad(name, view, cam)
        f = orc.render_forward(scene, cam)
        dec = np.minimum(f["margin"][..., 0], f["margin"][..., 1]) > 1e-4
        dLm = (dL * dec[None]).astype(np.float32)
        g = run_gpu(scene, cam, dLm)[0]
        o = orc.render_backward(scene, cam, dLm)
        b = orc.bin_sort(scene, cam)
        lists = (np.array_equal(g["keys"], b["keys"]) and np.array_equal(g["ids"], b["ids"])
                 and np.array_equal(g["tile_ranges"], b["tile_ranges"]))
        err = np.abs(g["image"].astype(np.float64) - f["image"]).max(axis=0)
        w = {n: rel_inf(g[n], o[n]) for n in ("d_means", "d_scales", "d_rotations", "d_opacities", "d_sh", "d_freqs",
                                              "d_weights", "d_mean2d")}
        worst = max(w, key=w.get)
        print("| %d | %d | %s | %d | %.1e | %s | %.1e (%s) |" % (
            view, g["D"], "yes" if lists else "NO", int((~dec).sum()), err[dec].max(),
            "yes" if np.array_equal(g["n_contrib"][dec], f["n_contrib"][dec]) else "NO", w[worst], worst), flush=True)


if __name__ == "__main__":
    main()
