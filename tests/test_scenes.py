"""Seeded input generators: determinism and the stated distributions."""
import numpy as np

from paper_2508_05343_b200 import scenes


def test_splitmix64_reference_vector():
    # SplitMix64 (Steele, Lea, Flood 2014) published test vector for seed 1234567.
    with np.errstate(over="ignore"):
        idx = np.arange(1, 4, dtype=np.uint64)
        out = scenes._mix(np.uint64(1234567) + idx * scenes._GAMMA)
    assert [int(v) for v in out] == [6457827717110365317, 3203168211198807973, 9817491932198370423]


def test_stream_is_counter_based():
    a = scenes.Stream(7, 3)
    x = a.uniform(10)
    b = scenes.Stream(7, 3)
    y = np.concatenate([b.uniform(4), b.uniform(6)])
    assert np.array_equal(x, y)
    assert not np.array_equal(x, scenes.Stream(7, 4).uniform(10))


def test_tiny_scene_recipe():
    s = scenes.make_scene("tiny")
    s2 = scenes.make_scene("tiny")
    for a, b in zip((s.means, s.scales, s.rotations, s.opacities, s.sh, s.freqs, s.weights),
                    (s2.means, s2.scales, s2.rotations, s2.opacities, s2.sh, s2.freqs, s2.weights)):
        assert a.dtype == np.float32 and a.flags.c_contiguous and np.array_equal(a, b)
    assert s.N == 1024 and s.K == 4 and s.sh.shape == (1024, 16, 3)
    assert np.all(np.abs(s.means) <= 1) and np.all(s.scales > 0)
    assert np.allclose(np.linalg.norm(s.rotations, axis=1), 1, atol=1e-6)
    assert np.all((s.opacities > 0) & (s.opacities < 1)) and np.all((s.weights >= 0) & (s.weights < 1))
    assert np.all(np.linalg.norm(s.freqs, axis=2) <= 8 + 1e-5)
    assert abs(np.log(s.scales).mean() + 3.0) < 0.05 and abs(np.log(s.scales).std() - 0.5) < 0.05
    cam = scenes.make_cameras("tiny")[0]
    assert np.array_equal(cam.world_to_cam, np.array([[1, 0, 0, 0], [0, 1, 0, 0], [0, 0, 1, 4]], np.float32))
    assert (cam.tiles_x, cam.tiles_y) == (8, 8) and cam.cx == 63.5


def test_unbounded_recipe_small_N():
    s = scenes.make_scene("unbounded", N=20000, K=2)
    r = np.linalg.norm(s.means[14000:], axis=1)
    assert s.K == 2 and r.min() >= 20 - 1e-3 and r.max() <= 50 + 1e-3
    assert abs(s.means[:14000, 1].std() - 1.0) < 0.05 and abs(s.means[:14000, 0].std() - 3.0) < 0.1
    cams = scenes.make_cameras("unbounded")
    assert len(cams) == 8 and cams[0].width == 1297 and cams[0].height == 840
    for c in cams:
        W = c.world_to_cam[:, :3].astype(np.float64)
        assert np.allclose(W @ W.T, np.eye(3), atol=1e-6)
    z = scenes.make_scene("unbounded", N=1000, zero_weights=True)
    assert not z.weights.any()
    g = scenes.make_image_grad("tiny", 0, scenes.make_cameras("tiny")[0])
    assert g.shape == (3, 128, 128) and abs(g.std() - 1) < 0.02
