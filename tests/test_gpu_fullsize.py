"""-m gpu parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times: every view of configs 3
(unbounded, 1M primitives, 1297x840) and 2 (object, 300k, 800x800), four views of config 4 (large, 3M, 1957x1266),
config 5 (K in {1, 2, 8} and the all-omega-zero case at 1M / 1297x840, two views each) and the primitive variants (f4) at
config 3's size -- the whole image, final T, last
contributor and EVERY gradient tensor against the oracle, UNMASKED, at north_star's tolerances.

The image (and so its gradient) is discontinuous where a skip / stop / clamp decision crosses its threshold; within
fp32 evaluation error of a threshold both outcomes are correct renderings (reading C18).  At exactly the
pixels where the oracle's own margin is below DELTA, the CUDA path's decisions (gabsplat_trace_pixels, verified here
to reproduce the forward image bit for bit) are handed to the oracle's decision-injected mode, which REJECTS any
injected outcome that is farther than DELTA from its threshold (`violations` must be 0).  What is compared is then
unique: no pixel is masked, no tolerance is loosened.
"""
import json
import os

import numpy as np
import pytest

from paper_2508_05343_b200 import scenes

pytestmark = pytest.mark.gpu

IMG_TOL = 1e-4        # north_star: rendered images max abs error <= 1e-4
GRAD_TOL = 1e-3       # north_star: gradients relative error <= 1e-3 (per tensor, inf-norm; reading C19)
DELTA = 1e-4          # reading C18 (why not 1e-5: DESIGN.md "Tolerances" -- the MUFU phase error at |phase| ~ 300 rad)
GRADS = ("d_means", "d_scales", "d_rotations", "d_opacities", "d_sh", "d_freqs", "d_weights", "d_mean2d", "d_mean2d_abs")
REPORT = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "gpurun_out", "parity_fullsize.jsonl")


def _report(rec):
    try:
        os.makedirs(os.path.dirname(REPORT), exist_ok=True)
        with open(REPORT, "a") as f:
            f.write(json.dumps(rec) + "\n")
    except OSError:
        pass


def gpu_decisions(gb, ctx, dev, cam, pixels):
    """The CUDA forward's decisions at `pixels` in the oracle's `inject` format, checked against the forward image."""
    import torch
    ds, proj, bins, fwd = dev["scene"], dev["proj"], dev["bins"], dev["fwd"]
    cnt = gb.gabsplat_count_pairs(ctx, ds, cam, proj, bins)
    px = torch.from_numpy(np.ascontiguousarray(pixels, np.int32)).cuda()
    nb = cnt[px[:, 1].long(), px[:, 0].long(), 2].to(torch.int64)
    offsets = torch.zeros(px.shape[0] + 1, dtype=torch.int64, device="cuda")
    offsets[1:] = torch.cumsum(nb, 0)
    entries, colour_T, info = gb.gabsplat_trace_pixels(ctx, ds, cam, proj, bins, px, offsets.to(torch.int32))
    torch.cuda.synchronize()
    info = info.cpu().numpy().view(np.uint32)
    assert np.array_equal(info[:, 1], nb.cpu().numpy().astype(np.uint32))          # nothing dropped
    # the trace IS the forward: colour, final T and last contributor bit for bit
    img = fwd.image[:, px[:, 1].long(), px[:, 0].long()].T.contiguous()
    assert torch.equal(img.view(torch.int32), colour_T[:, :3].contiguous().view(torch.int32))
    assert torch.equal(fwd.final_T[px[:, 1].long(), px[:, 0].long()].view(torch.int32), colour_T[:, 3].contiguous().view(torch.int32))
    assert np.array_equal(fwd.n_contrib[px[:, 1].long(), px[:, 0].long()].cpu().numpy().view(np.uint32), info[:, 0])
    return dict(pixels=np.ascontiguousarray(pixels, np.int32), offsets=offsets.cpu().numpy().astype(np.uint32),
                entries=entries.cpu().numpy().view(np.uint32), stop_pos=info[:, 2].copy(), delta=DELTA)


def full_compare(tag, scene, cam, dL, grad_tol=GRAD_TOL):
    import torch
    from oracle import gabsplat_oracle as orc
    from paper_2508_05343_b200 import binding as gb
    from gpu_helpers import ctx, run_gpu, rel_inf
    o_fwd = orc.render_forward(scene, cam)
    margin = np.minimum(o_fwd["margin"][..., 0], o_fwd["margin"][..., 1])
    und = margin <= DELTA
    ys, xs = np.nonzero(und)
    pixels = np.stack([xs, ys], axis=1).astype(np.int32)
    g, dev = run_gpu(scene, cam, dL)
    # integer stages, bit-exact in full
    o_bin = orc.bin_sort(scene, cam)
    assert g["D"] == o_bin["num_instances"]
    assert np.array_equal(g["keys"], o_bin["keys"]) and np.array_equal(g["ids"], o_bin["ids"])
    assert np.array_equal(g["tile_ranges"], o_bin["tile_ranges"])
    inject = gpu_decisions(gb, ctx(), dev, cam, pixels) if len(pixels) else None
    o = orc.render_backward(scene, cam, dL, inject=inject)
    assert o["violations"] == 0, o["violations"]
    # the whole image, final T and last contributor, every pixel
    err = np.abs(g["image"].astype(np.float64) - o["image"]).max(axis=0)
    errT = np.abs(g["final_T"].astype(np.float64) - o["final_T"])
    assert err.max() <= IMG_TOL, err.max()
    assert errT.max() <= IMG_TOL, errT.max()
    assert np.array_equal(g["n_contrib"], o["n_contrib"])
    # decidable pixels need no injection: the un-injected oracle agrees there too
    assert np.array_equal(g["n_contrib"][~und], o_fwd["n_contrib"][~und])
    rec = dict(case=tag, N=scene.N, K=scene.K, D=int(g["D"]), pixels=int(und.size), undecidable=int(und.sum()),
               undecidable_at_1e5=int((margin <= 1e-5).sum()), image_max_err=float(err.max()), final_T_max_err=float(errT.max()))
    worst, elem = {}, {}
    for n in GRADS:
        ref = o["d_absmean2d"] if n == "d_mean2d_abs" else o[n]
        worst[n] = rel_inf(g[n], ref)
        # reading C19, second figure: per-element relative error over the elements above 1e-3 of the tensor's max
        big = np.abs(ref) > 1e-3 * np.abs(ref).max() if ref.size else np.zeros(ref.shape, bool)
        elem[n] = float((np.abs(g[n].astype(np.float64) - ref)[big] / np.abs(ref)[big]).max()) if big.any() else 0.0
    rec["grad_rel_inf"] = worst
    rec["grad_rel_elementwise"] = elem
    _report(rec)
    bad = {k: v for k, v in worst.items() if not v <= grad_tol}
    assert not bad, (bad, worst)
    assert max(elem.values()) <= 5e-2, elem
    culled = g["tiles_touched"] == 0
    for n in GRADS:
        assert not np.any(g[n][culled])
    return rec


@pytest.mark.parametrize("view", range(8))
def test_unbounded_every_view(view):
    """BASELINE.json config 3, the headline workload, all 8 seeded views, forward + backward."""
    scene = scenes.make_scene("unbounded")
    cam = scenes.make_cameras("unbounded")[view]
    full_compare("unbounded/view%d" % view, scene, cam, scenes.make_image_grad("unbounded", view, cam))


@pytest.mark.parametrize("K,zero,view", [(1, False, 1), (2, False, 2), (8, False, 3), (4, True, 4),
                                         (1, False, 5), (2, False, 6), (8, False, 7), (4, True, 0)])
def test_filter_bank_sweep_full_size(K, zero, view):
    """BASELINE.json config 5: the K sweep and the all-omega-zero case at 1M primitives / 1297x840 (the synthetic
    stand-in for the paper's F ablation, Table 3)."""
    scene = scenes.make_scene("unbounded", K=K, zero_weights=zero)
    cam = scenes.make_cameras("unbounded")[view]
    full_compare("unbounded/K%d%s/view%d" % (K, "/zero_weights" if zero else "", view), scene, cam,
                 scenes.make_image_grad("unbounded", view, cam))


def test_zero_weights_equals_k0_full_size():
    """PAPER.md:131 at full size: K=4 with all weights zero renders the K=0 (plain Gaussian) image bit for bit."""
    from gpu_helpers import run_gpu
    cam = scenes.make_cameras("unbounded")[4]
    g4, _ = run_gpu(scenes.make_scene("unbounded", zero_weights=True), cam)
    g0, _ = run_gpu(scenes.make_scene("unbounded", K=0), cam)
    assert np.array_equal(g4["image"], g0["image"])
    assert np.array_equal(g4["n_contrib"], g0["n_contrib"])


@pytest.mark.parametrize("variant,view", [(1, 1), (2, 2), (3, 5)])
def test_variants_full_size(variant, view):
    """SURVEY 8(f) f4 at the headline size: the line-integral amplitude, the Mip 2D filter (:224) and
    both, on 1M primitives / 1297x840 -- whole-screen rectangles, |phase| up to ~300 rad, the fp64 value track and the
    variant chain rule of the projection backward on every visible primitive; same unmasked comparison as the plain
    primitive (the injected decisions are taken on the folded records the blend kernels see)."""
    scene = scenes.make_scene("unbounded")
    scene.variant = variant
    cam = scenes.make_cameras("unbounded")[view]
    full_compare("unbounded/variant%d/view%d" % (variant, view), scene, cam, scenes.make_image_grad("unbounded", view, cam))


@pytest.mark.parametrize("view", [0, 3, 5, 6])
def test_large_views(view):
    """BASELINE.json config 4: 3M primitives, 1957x1266, ~50 M instances, forward + backward."""
    scene = scenes.make_scene("large")
    cam = scenes.make_cameras("large")[view]
    full_compare("large/view%d" % view, scene, cam, scenes.make_image_grad("large", view, cam))


@pytest.mark.parametrize("view", range(8))
def test_object_views(view):
    """BASELINE.json config 2 (300k primitives in the unit ball, 800x800, white background).  The config is forward
    only; the backward is compared as well since it costs nothing extra here."""
    scene = scenes.make_scene("object")
    cam = scenes.make_cameras("object")[view]
    full_compare("object/view%d" % view, scene, cam, scenes.make_image_grad("object", view, cam))


def test_buffers_reused_across_views():
    """The timed configuration of bench.py: ONE Projected / Binning / FwdOut / Grads set cycled through different
    views by the fused gabsplat_preprocess_bin_sort (no keys, no count read-back).  Rows of culled primitives keep
    whatever an earlier view left there (gabsplat.h: unspecified) -- nothing may depend on them: every view must give
    what a run on fresh buffers gives."""
    import torch
    from paper_2508_05343_b200 import binding as gb
    from gpu_helpers import ctx, run_gpu
    c = ctx()
    scene = scenes.make_scene("unbounded", N=250000)
    cams = scenes.make_cameras("unbounded")
    ds = gb.upload_scene(scene)
    views = [0, 5, 2, 7, 0]
    fresh = {}
    for v in set(views):
        dL = scenes.make_image_grad("unbounded", v, cams[v])
        fresh[v] = run_gpu(scene, cams[v], dL)[0]
    cap = max(f["D"] for f in fresh.values()) + 17
    proj = gb.Projected(ds.N, ds.K, ds.means.device)
    bins = gb.Binning(ds.N, cams[0], cap, ds.means.device, with_keys=False)
    fwd = gb.FwdOut(cams[0], ds.means.device, cap)
    grads = gb.Grads(ds.N, ds.K, ds.means.device)
    for v in views:
        dL = torch.from_numpy(scenes.make_image_grad("unbounded", v, cams[v])).cuda()
        gb.gabsplat_preprocess_bin_sort(c, ds, cams[v], proj, bins, read_count=False)
        gb.gabsplat_render_forward(c, ds, cams[v], proj, bins, fwd)
        gb.gabsplat_render_backward(c, ds, cams[v], proj, bins, fwd, dL, grads)
        torch.cuda.synchronize()
        f = fresh[v]
        D = f["D"]
        assert int(bins.num_instances[0].item()) == D
        assert np.array_equal(bins.ids.cpu().numpy().view(np.uint32)[:D], f["ids"])
        assert np.array_equal(bins.tile_ranges.cpu().numpy().view(np.uint32), f["tile_ranges"])
        assert np.array_equal(fwd.image.cpu().numpy(), f["image"])
        assert np.array_equal(fwd.n_contrib.cpu().numpy().view(np.uint32), f["n_contrib"])
        for n in GRADS:
            a, b = getattr(grads, n).cpu().numpy(), f[n]
            # equal up to the order of the fp32 atomic accumulation
            assert np.allclose(a, b, rtol=1e-4, atol=2e-6 * max(np.abs(b).max(), 1e-30)), n
            assert not np.any(a[f["tiles_touched"] == 0]), n
