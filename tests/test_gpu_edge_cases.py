"""-m gpu edge cases of the C ABI: empty and fully culled scenes, capacity overflow, status codes, and the
host-buffer convenience call."""
import numpy as np
import pytest

from paper_2508_05343_b200 import scenes

pytestmark = pytest.mark.gpu


def _mods():
    import torch
    from paper_2508_05343_b200 import binding as gb
    from gpu_helpers import ctx, run_gpu
    return torch, gb, ctx(), run_gpu


def test_empty_scene():
    torch, gb, ctx, run_gpu = _mods()
    scene = scenes.make_scene("tiny", N=0)
    cam = scenes.make_cameras("tiny")[0]
    cam.bg = (0.25, 0.5, 0.75)
    dL = np.ones((3, cam.height, cam.width), np.float32)
    g, _ = run_gpu(scene, cam, dL)
    assert g["D"] == 0
    assert np.all(g["tile_ranges"] == 0)
    assert np.all(g["n_contrib"] == 0) and np.all(g["final_T"] == 1.0)
    for ch, v in enumerate(cam.bg):
        assert np.all(g["image"][ch] == np.float32(v))


def test_all_culled():
    """Everything behind the camera: no instances, background image, zero gradients."""
    torch, gb, ctx, run_gpu = _mods()
    scene = scenes.make_scene("tiny")
    scene.means[:, 2] -= 10.0
    cam = scenes.make_cameras("tiny")[0]
    dL = scenes.make_image_grad("tiny", 0, cam)
    g, _ = run_gpu(scene, cam, dL)
    assert g["D"] == 0 and np.all(g["tiles_touched"] == 0)
    assert np.all(g["image"] == 0)
    for n in ("d_means", "d_scales", "d_rotations", "d_opacities", "d_sh", "d_freqs", "d_weights"):
        assert np.all(g[n] == 0)


def test_capacity_overflow_reports_required_count():
    torch, gb, ctx, run_gpu = _mods()
    scene = scenes.make_scene("tiny")
    cam = scenes.make_cameras("tiny")[0]
    ds = gb.upload_scene(scene)
    proj = gb.gabsplat_preprocess(ctx, ds, cam)
    full = gb.gabsplat_bin_sort(ctx, ds.N, proj, cam)
    D = full.D
    assert D > 16
    small = gb.Binning(ds.N, cam, D - 1, ds.means.device)
    with pytest.raises(gb.GabsplatError) as e:
        gb.gabsplat_bin_sort(ctx, ds.N, proj, cam, bin=small)
    assert e.value.code == gb.CAPACITY
    torch.cuda.synchronize()
    assert int(small.num_instances[0].item()) == D          # the required count is left on the device
    exact = gb.gabsplat_bin_sort(ctx, ds.N, proj, cam, bin=gb.Binning(ds.N, cam, D, ds.means.device))
    assert torch.equal(exact.keys[:D], full.keys[:D]) and torch.equal(exact.ids[:D], full.ids[:D])
    # slack capacity gives the same list
    slack = gb.gabsplat_bin_sort(ctx, ds.N, proj, cam, bin=gb.Binning(ds.N, cam, 3 * D + 5, ds.means.device))
    assert torch.equal(slack.keys[:D], full.keys[:D]) and torch.equal(slack.ids[:D], full.ids[:D])
    assert torch.equal(slack.tile_ranges, full.tile_ranges)


def test_invalid_arguments():
    torch, gb, ctx, run_gpu = _mods()
    scene = scenes.make_scene("tiny", N=8)
    cam = scenes.make_cameras("tiny")[0]
    ds = gb.upload_scene(scene)
    bad = scenes.make_camera(0, 16, 10.0, cam.world_to_cam)
    with pytest.raises(gb.GabsplatError) as e:
        gb.gabsplat_preprocess(ctx, ds, bad, out=gb.Projected(8, 4, ds.means.device))
    assert e.value.code == gb.INVALID_ARG
    ds.sh_degree = 4
    with pytest.raises(gb.GabsplatError) as e:
        gb.gabsplat_preprocess(ctx, ds, cam)
    assert e.value.code == gb.INVALID_ARG


def test_async_path_without_readback_matches():
    """read_count=False (no host sync inside the call) gives the same result as the synchronising call."""
    torch, gb, ctx, run_gpu = _mods()
    scene = scenes.make_scene("tiny")
    cam = scenes.make_cameras("tiny")[0]
    ds = gb.upload_scene(scene)
    proj = gb.gabsplat_preprocess(ctx, ds, cam)
    a = gb.gabsplat_bin_sort(ctx, ds.N, proj, cam)
    b = gb.gabsplat_bin_sort(ctx, ds.N, proj, cam, bin=gb.Binning(ds.N, cam, a.D + 100, ds.means.device),
                             read_count=False)
    torch.cuda.synchronize()
    assert b.D is None
    assert torch.equal(a.keys[:a.D], b.keys[:a.D]) and torch.equal(a.tile_ranges, b.tile_ranges)


def test_side_stream():
    torch, gb, ctx, run_gpu = _mods()
    scene = scenes.make_scene("tiny")
    cam = scenes.make_cameras("tiny")[0]
    ref, _ = run_gpu(scene, cam)
    st = torch.cuda.Stream()
    ds = gb.upload_scene(scene)
    torch.cuda.synchronize()
    with torch.cuda.stream(st):
        proj = gb.gabsplat_preprocess(ctx, ds, cam, stream=st)
        bins = gb.gabsplat_bin_sort(ctx, ds.N, proj, cam, stream=st)
        fwd = gb.gabsplat_render_forward(ctx, ds, cam, proj, bins, stream=st)
    st.synchronize()
    assert np.array_equal(fwd.image.cpu().numpy(), ref["image"])


def test_render_host_matches_device_path():
    torch, gb, ctx, run_gpu = _mods()
    scene = scenes.make_scene("tiny")
    cam = scenes.make_cameras("tiny")[0]
    dL = scenes.make_image_grad("tiny", 0, cam)
    ref, _ = run_gpu(scene, cam, dL)

    class H:
        pass
    h = H()
    for n in ("means", "scales", "rotations", "opacities", "sh", "freqs", "weights"):
        setattr(h, n, torch.from_numpy(getattr(scene, n)).pin_memory())
    h.sh_degree = 3
    cap = ref["D"] + 10
    arena = torch.zeros(gb.host_arena_bytes(scene.N, scene.K, cam, cap), dtype=torch.uint8, device="cuda")
    img = torch.zeros((3, cam.height, cam.width), dtype=torch.float32).pin_memory()
    names = ("d_means", "d_scales", "d_rotations", "d_opacities", "d_sh", "d_freqs", "d_weights")
    grads = {n: torch.zeros(ref[n].shape, dtype=torch.float32).pin_memory() for n in names}
    gb.gabsplat_render_host(ctx, h, cam, cap, img, torch.from_numpy(dL).pin_memory(), grads, arena)
    assert np.array_equal(img.numpy(), ref["image"])
    for n in names:
        assert np.allclose(grads[n].numpy(), ref[n], rtol=1e-4, atol=1e-6 * np.abs(ref[n]).max())


def test_render_host_refuses_bad_arguments_before_copying():
    """A scene or camera the device calls would refuse (z_near <= 0, unknown variant) is refused by gabsplat_render_host
    itself, before any copy is queued on its internal streams: INVALID_ARG, the host image untouched, and the same
    buffers render correctly in the next call."""
    import copy
    torch, gb, ctx, run_gpu = _mods()
    scene = scenes.make_scene("tiny")
    cam = scenes.make_cameras("tiny")[0]
    ref, _ = run_gpu(scene, cam)

    class H:
        pass
    h = H()
    for n in ("means", "scales", "rotations", "opacities", "sh", "freqs", "weights"):
        setattr(h, n, torch.from_numpy(getattr(scene, n)).pin_memory())
    h.sh_degree = 3
    cap = ref["D"] + 10
    arena = torch.zeros(gb.host_arena_bytes(scene.N, scene.K, cam, cap), dtype=torch.uint8, device="cuda")
    img = torch.full((3, cam.height, cam.width), -1.0, dtype=torch.float32).pin_memory()
    bad_cam = copy.copy(cam)
    bad_cam.z_near = 0.0
    with pytest.raises(gb.GabsplatError) as err:
        gb.gabsplat_render_host(ctx, h, bad_cam, cap, img, None, None, arena)
    assert err.value.code == gb.INVALID_ARG and "camera" in str(err.value)
    h.variant = 7
    with pytest.raises(gb.GabsplatError) as err:
        gb.gabsplat_render_host(ctx, h, cam, cap, img, None, None, arena)
    assert err.value.code == gb.INVALID_ARG and "scene" in str(err.value)
    torch.cuda.synchronize()
    assert float(img.min()) == -1.0 and float(img.max()) == -1.0
    h.variant = 0
    gb.gabsplat_render_host(ctx, h, cam, cap, img, None, None, arena)
    assert np.array_equal(img.numpy(), ref["image"])


def test_inference_forward_has_no_blend_state():
    """A forward run without blend_state (inference) gives the same image bit for bit, and the backward refuses
    it with INVALID_ARG instead of silently re-deciding anything."""
    torch, gb, ctx, run_gpu = _mods()
    scene = scenes.make_scene("tiny")
    cam = scenes.make_cameras("tiny")[0]
    dL = torch.from_numpy(scenes.make_image_grad("tiny", 0, cam)).cuda()
    ds = gb.upload_scene(scene)
    proj = gb.gabsplat_preprocess(ctx, ds, cam)
    bins = gb.gabsplat_bin_sort(ctx, ds.N, proj, cam)
    train = gb.gabsplat_render_forward(ctx, ds, cam, proj, bins)
    infer = gb.gabsplat_render_forward(ctx, ds, cam, proj, bins, save_state=False)
    torch.cuda.synchronize()
    assert torch.equal(train.image, infer.image) and torch.equal(train.n_contrib, infer.n_contrib)
    with pytest.raises(gb.GabsplatError) as e:
        gb.gabsplat_render_backward(ctx, ds, cam, proj, bins, infer, dL)
    assert e.value.code == gb.INVALID_ARG
    # the saved lists: per half tile at most the tile's list length, ids inside the tile's list
    tiles = cam.tiles_x * cam.tiles_y
    counts = train.blend_state[:].view(torch.int32)[:2 * tiles].cpu().numpy().reshape(tiles, 2)
    ranges = bins.tile_ranges.cpu().numpy().view(np.uint32).reshape(tiles, 2)
    assert np.all(counts <= (ranges[:, 1] - ranges[:, 0])[:, None])
    assert counts.sum() > 0


def test_backward_leaves_its_workspace_zero():
    """gabsplat_render_backward needs an all-zero gradient scratch and returns it all zero: two backward calls
    through the same Grads object give the same gradients (up to the order of the fp32 atomics)."""
    torch, gb, ctx, run_gpu = _mods()
    scene = scenes.make_scene("tiny")
    cam = scenes.make_cameras("tiny")[0]
    dL = torch.from_numpy(scenes.make_image_grad("tiny", 0, cam)).cuda()
    ds = gb.upload_scene(scene)
    proj = gb.gabsplat_preprocess(ctx, ds, cam)
    bins = gb.gabsplat_bin_sort(ctx, ds.N, proj, cam)
    fwd = gb.gabsplat_render_forward(ctx, ds, cam, proj, bins)
    g = gb.gabsplat_render_backward(ctx, ds, cam, proj, bins, fwd, dL)
    torch.cuda.synchronize()
    assert int(g.workspace.count_nonzero().item()) == 0
    first = {n: getattr(g, n).clone() for n in ("d_means", "d_sh", "d_freqs", "d_weights", "d_opacities")}
    g.d_means.fill_(123.0)                      # outputs are fully overwritten
    gb.gabsplat_render_backward(ctx, ds, cam, proj, bins, fwd, dL, g)
    torch.cuda.synchronize()
    assert int(g.workspace.count_nonzero().item()) == 0
    for n, ref in first.items():
        assert torch.allclose(getattr(g, n), ref, rtol=1e-4, atol=2e-6 * float(ref.abs().max()))


def test_fused_preprocess_bin_sort_equals_the_two_calls():
    """gabsplat_preprocess_bin_sort (value track on the side stream beside the binning) gives bit-identical
    projected arrays, lists and image."""
    torch, gb, ctx, run_gpu = _mods()
    scene = scenes.make_scene("unbounded", N=60000)
    base = scenes.make_cameras("unbounded")[2]
    cam = scenes.make_camera(331, 213, 290.0, base.world_to_cam, base.bg)
    ds = gb.upload_scene(scene)
    p1 = gb.gabsplat_preprocess(ctx, ds, cam)
    b1 = gb.gabsplat_bin_sort(ctx, ds.N, p1, cam)
    f1 = gb.gabsplat_render_forward(ctx, ds, cam, p1, b1, save_state=False)
    p2 = gb.Projected(ds.N, ds.K, ds.means.device)
    b2 = gb.Binning(ds.N, cam, b1.capacity, ds.means.device)
    for _ in range(3):       # repeated: the side stream must be ordered against the next call too
        gb.gabsplat_preprocess_bin_sort(ctx, ds, cam, p2, b2)
        f2 = gb.gabsplat_render_forward(ctx, ds, cam, p2, b2, save_state=False)
    torch.cuda.synchronize()
    assert b2.D == b1.D
    for n in ("mean2d", "depth", "radius", "conic_opacity", "rgb", "rgb_clamped", "freq2d", "tiles_touched", "rect", "packed"):
        assert torch.equal(getattr(p1, n), getattr(p2, n)), n
    assert torch.equal(b1.ids[:b1.D], b2.ids[:b1.D]) and torch.equal(b1.tile_ranges, b2.tile_ranges)
    assert torch.equal(b1.keys[:b1.D], b2.keys[:b1.D])
    assert torch.equal(f1.image, f2.image)


@pytest.mark.parametrize("levels", [1, 3, 60, 6000])
def test_depth_sort_paths(levels):
    """The depth order of the visible primitives comes from the bucketed sort when the depths spread and from the
    stable radix passes when a bucket overflows (thousands of primitives at one depth): 6000 primitives on `levels`
    planes facing the camera -- one plane: every key equal, the order is the index order and the radix passes run;
    three planes: three huge buckets (radix passes); 60 planes: the bucketed path with 100-way ties inside a bucket;
    6000 levels: the bucketed path.  Lists bit-exact either way."""
    from oracle import gabsplat_oracle as orc
    from gpu_helpers import run_gpu
    scene = scenes.make_scene("tiny", N=6000)
    z = -0.9 + 1.8 * (np.arange(6000) % levels) / max(levels, 1)
    scene.means[:, 2] = z.astype(np.float32)          # the tiny camera looks down +z: depth = z + 4 exactly
    cam = scenes.make_cameras("tiny")[0]
    g, _ = run_gpu(scene, cam)
    o = orc.bin_sort(scene, cam)
    if levels == 1:
        assert len(np.unique(g["depth_bits"][g["tiles_touched"] != 0])) == 1
    assert g["D"] == o["num_instances"]
    assert np.array_equal(g["keys"], o["keys"]) and np.array_equal(g["ids"], o["ids"])
    assert np.array_equal(g["tile_ranges"], o["tile_ranges"])


def test_launch_order_hint_changes_nothing_but_the_order():
    """gabsplat_fwd_out.tile_work (list entries every tile consumed) fed back as gabsplat_binning.tile_work_hint: the
    tile order becomes the order of min(hint, list length), still a permutation; image, final T, last contributor,
    lists and gradients are bit-identical (only the forward's launch order changed)."""
    import torch
    from paper_2508_05343_b200 import binding as gb
    from gpu_helpers import ctx
    from test_gpu_parity import _ragged_case
    scene, cam = _ragged_case("unbounded", 40000, 403, 251, 360.0)
    dL = torch.from_numpy(np.random.default_rng(5).standard_normal((3, cam.height, cam.width)).astype(np.float32)).cuda()
    c = ctx()
    ds = gb.upload_scene(scene)
    proj = gb.gabsplat_preprocess(c, ds, cam)
    bins = gb.gabsplat_bin_sort(c, ds.N, proj, cam)
    fwd = gb.FwdOut(cam, ds.means.device, bins.capacity)
    fwd.tile_work = torch.full((bins.n_tiles,), -1, dtype=torch.int32, device="cuda")
    gb.gabsplat_render_forward(c, ds, cam, proj, bins, fwd)
    g0 = gb.gabsplat_render_backward(c, ds, cam, proj, bins, fwd, dL)
    torch.cuda.synchronize()
    n = (bins.tile_ranges[:, 1] - bins.tile_ranges[:, 0]).cpu().numpy()
    work = fwd.tile_work.cpu().numpy()
    assert np.all(work >= 0) and np.all(work <= n)                     # every tile wrote it
    assert np.all((work % 128 == 0) | (work == n))                     # whole staging batches, or the whole list
    last = fwd.n_contrib.cpu().numpy().reshape(-1)
    assert work.max() >= 1 and last.max() <= n.max()
    ref = dict(image=fwd.image.clone(), T=fwd.final_T.clone(), nc=fwd.n_contrib.clone(), ids=bins.ids.clone(),
               ranges=bins.tile_ranges.clone(), order=bins.tile_order.clone())
    # second render of the view, with the hint
    bins.tile_work_hint = fwd.tile_work.clone()
    gb.gabsplat_bin_sort(c, ds.N, proj, cam, bins)
    gb.gabsplat_render_forward(c, ds, cam, proj, bins, fwd)
    g1 = gb.gabsplat_render_backward(c, ds, cam, proj, bins, fwd, dL)
    torch.cuda.synchronize()
    order = bins.tile_order.cpu().numpy()
    assert np.array_equal(np.sort(order), np.arange(bins.n_tiles))     # a permutation
    key = np.minimum(work, n)[order]
    # descending up to the 256 buckets of the counting sort behind it
    assert key[0] == key.max() and np.all(np.diff(key.astype(np.int64)) <= max(1, int(key.max()) // 255 + 1))
    assert not np.array_equal(order, ref["order"].cpu().numpy())
    assert torch.equal(fwd.image, ref["image"]) and torch.equal(fwd.final_T, ref["T"]) and torch.equal(fwd.n_contrib, ref["nc"])
    assert torch.equal(bins.ids, ref["ids"]) and torch.equal(bins.tile_ranges, ref["ranges"])
    for name in ("d_means", "d_scales", "d_rotations", "d_opacities", "d_sh", "d_freqs", "d_weights"):
        a, b = getattr(g0, name), getattr(g1, name)
        assert torch.allclose(a, b, rtol=1e-4, atol=2e-6 * float(a.abs().max()))   # equal up to the order of the fp32 atomics
