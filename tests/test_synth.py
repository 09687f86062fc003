"""The seeded input generator: determinism, shapes and the structure BASELINE.json's configs ask for."""
import numpy as np

import synth


def test_render_is_deterministic_and_typed():
    cfg = synth.make_config(1)
    a, b = synth.render_frame(cfg), synth.render_frame(cfg)
    assert all(np.array_equal(x, y) for x, y in zip(a, b))
    assert a[0].shape == (48, 64) and a[0].dtype == np.uint8 and len(a) == 2
    cfg2 = synth.make_config(2)
    imgs = synth.render_frame(cfg2)
    assert len(imgs) == 3 and imgs[0].dtype == np.float32 and imgs[0].shape == (256, 320)
    assert 0.0 <= imgs[0].min() and imgs[0].max() <= 1.0
    # per-image Gaussian noise: the same scene rendered for camera 0 twice with different noise seeds differs slightly
    n0 = synth.render_camera(cfg2["cams"][0], cfg2["scene"], noise_seed=1)
    n1 = synth.render_camera(cfg2["cams"][0], cfg2["scene"], noise_seed=2)
    d = (n0 - n1)[(n0 > 0.05) & (n0 < 0.95) & (n1 > 0.05) & (n1 < 0.95)]
    assert 0.012 < d.std() < 0.016          # sqrt(2) * 0.01


def test_config_shapes_match_baseline_json():
    c3 = synth.make_config(3)
    assert [f["n_planes"] for f in c3["families"]] == [96, 32] and c3["params"]["window"] == 9
    assert c3["cams"][0]["width"] == 1280 and c3["cams"][0]["k1"] == -0.05 and len(c3["cams"]) == 3
    c4 = synth.make_config(4)
    assert c4["crop"] == (384, 256, 512, 512) and c4["families_crop"][0]["n_planes"] == 192
    assert c4["families_crop"][0]["d_last"] == 80.0 and c4["params_low"]["window"] == 7
    c5 = synth.make_config(5)
    assert [f["n_planes"] for f in c5["families"]] == [192, 64] and c5["n_frames"] == 32 and c5["step_m"] == 0.5
    assert len(c3["scene"]["boxes"]) >= 1 + 40 + 10


def test_mask_and_hash():
    m = synth.make_mask(1280, 1024, seed=4)
    assert m.shape == (1024, 1280) and m.dtype == np.uint8 and set(np.unique(m)) <= {0, 1}
    assert 8 * 40 * 40 * 0.5 < m.sum() <= 8 * 300 * 200
    assert np.array_equal(m, synth.make_mask(1280, 1024, seed=4)) and not np.array_equal(m, synth.make_mask(1280, 1024, seed=5))
    u = np.array([synth.uniform(7, 1, i) for i in range(4000)])
    assert abs(u.mean() - 0.5) < 0.02 and abs(u.std() - 12 ** -0.5) < 0.02 and 0 < u.min() and u.max() < 1


def test_moving_rig_changes_the_frame():
    c5 = synth.make_config(5)
    cam = dict(c5["cams"][0])
    cam.update(width=160, height=128, fx=43.75, fy=43.75, cx=79.625, cy=63.625)   # 1/8 resolution for speed
    a = synth.render_camera(cam, c5["scene"], (0, 0, 0.0))
    b = synth.render_camera(cam, c5["scene"], (0, 0, 0.5))
    assert a.shape == (128, 160) and np.abs(a - b).mean() > 1e-3
