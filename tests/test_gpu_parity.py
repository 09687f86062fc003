"""-m gpu: the CUDA path, called through the C ABI, against the oracle on the same seeded inputs.

Gates (BASELINE.json north_star; derivations in DESIGN.md "Tolerances"):
  index   >= 99.9 % of oracle-valid pixels, a differing index only as a tie in the oracle's own cost vector (2e-4)
  cost    |c1 - c1_oracle| <= 1e-4 wherever the indices agree
  depth   within 1e-3 relative on >= 99.9 % of the pixels whose indices agree, and on ALL of them within
          1e-3 + 3e-4 * (|ds|/s) / pden  (the parabola's conditioning at the 1e-4 cost tolerance)
  valid   bit-exact on pixels the oracle does not mark fragile
  N_eval  the kernel's counter of finite (pixel, plane, view) costs equals the oracle's within 0.1 %
"""
import numpy as np
import pytest

import oracle
import synth
from parity_helpers import assert_gates, gpu_objects, run_multires, run_single

pytestmark = pytest.mark.gpu


def _small_rig(W=70, H=45, n_views=1, xi=0.9, rot=False, dist=None, dtype="u8", seed=7, fov=200.0):
    """A small seeded rig + plane scene whose sizes are not multiples of the 32x32 tile (ragged tails)."""
    kw = dict(width=W, height=H, fx=0.45 * W, fy=0.45 * W, cx=W / 2.0 - 0.3, cy=H / 2.0 + 0.2, xi=xi, fov_max_deg=fov)
    if dist:
        kw.update(dist)
    centres = [(0.3, 0, 0), (-0.25, 0.05, 0), (0.0, -0.3, 0.02), (0.2, 0.2, 0)][:n_views]
    yaws = [8.0, -6.0, 3.0, -2.0] if rot else [0.0] * 4
    cams = [synth.camera(**kw)] + [synth.camera(centre=c, yaw_deg=yaws[i], **kw) for i, c in enumerate(centres)]
    cfg = dict(name="small", dtype=dtype, ref_index=0, cams=cams,
               families=[synth.family((0, 0, 1), 24, 0.8, 30.0, "inverse")],
               params=synth.params(5, synth.VAR_FLOOR_U8 if dtype == "u8" else synth.VAR_FLOOR_F32, 60.0),
               scene=synth.scene_plane(3.0, (0.5, 2.0), seed=seed))
    return cfg


# ---- the five BASELINE.json configs ---------------------------------------------------------------------------------
@pytest.mark.parametrize("idx", [1, 2, 3])
def test_config_single_resolution(idx):
    cfg = synth.make_config(idx)
    images = synth.render_frame(cfg, 0)
    _, _, stats, counters = run_single(cfg, images)
    assert_gates(stats)
    assert counters["n_launches"] >= 1


def test_paper_workload_shape_four_rotated_views():
    """the paper's own workload shape (5 cameras = 4 rotated matching views, 1024x544, 64 + 30 planes,
    9x9): the run-time view loop of the generic kernel variant at full size."""
    cfg = synth.make_config(6)
    images = synth.render_frame(cfg, 3)
    _, _, stats, counters = run_single(cfg, images)
    assert_gates(stats)
    assert stats["n_oracle_valid"] > 50000 and counters["n_eval"] > 10_000_000


def test_paper_multiscale_shape_and_its_batch():
    """the paper's multi-scale estimator at its own shape -- 512 x 272 full field of view
    (7 x 7) + the 572 x 332 centre crop at full resolution (9 x 9), four rotated matching views, 64 + 30 planes -- through
    fsw_compute_depth_multires against the oracle, and two frame sets through fsw_compute_depth_multires_batch,
    bit-identical to their single calls."""
    import torch
    import paper_1809_06132_b200 as fsw
    cfg = synth.make_config(7)
    _, _, ctx = gpu_objects(cfg)
    images = synth.render_frame(cfg, 2)
    ref, test, stats, counters = run_multires(cfg, images, None, ctx=ctx)
    assert_gates(stats, fragile_frac=0.12)
    assert stats["n_oracle_valid"] > 50000
    k = ref["kbest"]
    assert ((k >= 0) & (k >> 14 == 1)).sum() > 50000 and ((k >= 0) & (k >> 14 == 0)).sum() > 50000
    pl, pc = fsw.PlaneSet(cfg["families_low"]), fsw.PlaneSet(cfg["families_crop"])
    sets = [[torch.from_numpy(im).cuda() for im in fr] for fr in (images, synth.render_frame(cfg, 9))]
    masks = [torch.from_numpy(synth.make_mask(1024, 544, 21)).cuda(), None]
    singles, n_eval = [], 0
    for st, m in zip(sets, masks):
        singles.append(oracle.compare.to_numpy(ctx.compute_depth_multires(pl, pc, cfg["params_low"], cfg["params_crop"], cfg["crop"], st, m)))
        n_eval += ctx.last_counters()["n_eval"]
    outs = ctx.compute_depth_multires_batch(pl, pc, cfg["params_low"], cfg["params_crop"], cfg["crop"], sets, masks)
    torch.cuda.synchronize()
    c = ctx.last_counters()
    # downsample, pack + low sweep, pack + crop sweep; a sweep is two launches where the plane split keeps tiles whole
    assert c["n_eval"] == n_eval and 5 <= c["n_launches"] <= 7, c
    for s in range(2):
        got = oracle.compare.to_numpy(outs[s])
        for key in ("depth", "best_cost", "second_cost", "plane_index", "valid_reason"):
            assert np.array_equal(singles[s][key], got[key], equal_nan=True), (s, key)
    assert (oracle.compare.to_numpy(outs[0])["depth"][masks[0].cpu().numpy() != 0] == 0).all()


def test_paper_half_resolution_shape():
    """PAPER.md:249 "half resolution": 512 x 272, 7 x 7, the same planes and views (synth.make_config(8))."""
    cfg = synth.make_config(8)
    images = synth.render_frame(cfg, 1)
    _, _, stats, counters = run_single(cfg, images)
    assert_gates(stats, fragile_frac=0.12)
    assert stats["n_oracle_valid"] > 15000


def test_camera_subset_three_of_five_cameras():
    """the three-camera configuration.  fsw_rig_subset gives the rig of the listed cameras: its
    maps equal those of a rig created from those cameras directly, and match the oracle."""
    import torch
    import paper_1809_06132_b200 as fsw
    full = synth.make_config(6)
    cfg = synth.make_config(6, cameras=(0, 1, 2))
    images = synth.render_frame(cfg, 5)
    assert all(np.array_equal(a, b) for a, b in zip(images, synth.render_frame(full, 5)[:3]))
    sub = fsw.Rig(full["cams"], 0).subset([0, 1, 2])
    ctx_sub = fsw.Context(sub, 0)
    ref, test, stats, counters = run_single(cfg, images)            # rig created from the three cameras
    assert_gates(stats, fragile_frac=0.12)
    planes = fsw.PlaneSet(cfg["families"])
    dev = [torch.from_numpy(im).cuda() for im in images]
    got = oracle.compare.to_numpy(ctx_sub.compute_depth(planes, cfg["params"], dev))
    for key in ("depth", "best_cost", "second_cost", "plane_index", "valid_reason"):
        assert np.array_equal(test[key], got[key], equal_nan=True), key
    assert ctx_sub.last_counters()["n_eval"] == counters["n_eval"]


def test_multires_batch_host_small():
    """fsw_compute_depth_multires_batch_host on a small rig: three frame sets, masks on some, equal to the single
    host calls bit for bit."""
    import paper_1809_06132_b200 as fsw
    cfg = _small_rig(W=128, H=96, n_views=3, rot=True, fov=170.0)
    _, _, ctx = gpu_objects(cfg)
    pl = fsw.PlaneSet([synth.family((0, 0, 1), 16, 0.8, 30.0, "inverse")])
    pc = fsw.PlaneSet([synth.family((0, 0, 1), 24, 0.8, 40.0, "inverse"), synth.family((0, 1, 0), 5, 0.5, 1.5, "linear")])
    p_lo = synth.params(5, synth.VAR_FLOOR_U8, 60.0)
    p_hi = synth.params(7, synth.VAR_FLOOR_U8, 80.0, 0.2, 0.3, 48, 1.1, filters=3)
    crop = (35, 27, 61, 40)
    sets = [synth.render_frame(dict(cfg, scene=synth.scene_plane(2.0 + 0.6 * s, (0.5, 2.0), seed=70 + s)), 0) for s in range(3)]
    masks = [synth.make_mask(128, 96, 80, n_rects=2), None, synth.make_mask(128, 96, 81, n_rects=1)]
    singles = [oracle.compare.to_numpy(ctx.compute_depth_multires(pl, pc, p_lo, p_hi, crop, st, m, host=True)) for st, m in zip(sets, masks)]
    outs = ctx.compute_depth_multires_batch(pl, pc, p_lo, p_hi, crop, sets, masks, host=True)
    for s in range(3):
        got = oracle.compare.to_numpy(outs[s])
        for key in ("depth", "best_cost", "second_cost", "plane_index", "valid_reason"):
            assert np.array_equal(singles[s][key], got[key], equal_nan=True), (s, key)
    assert (singles[0]["plane_index"] >= 0).sum() > 1000
    with pytest.raises(fsw.FswError):
        ctx.compute_depth_multires_batch(pl, pc, p_lo, p_hi, (100, 27, 61, 40), sets, masks, host=True)   # crop leaves the image


@pytest.mark.parametrize("n_views,best_k", [(2, 1), (4, 1), (4, 2), (3, 2), (2, 2)])
def test_best_k_view_aggregation(n_views, best_k):
    """SURVEY 8(f) 4 / reading Q26: the mean of the best_k lowest per-view costs.  One view is corrupted
    in a band so that the aggregation rule matters; best_k >= views is the plain mean bit for bit."""
    import torch
    import paper_1809_06132_b200 as fsw
    cfg = _small_rig(W=150, H=101, n_views=n_views, rot=True, fov=170.0)
    images = synth.render_frame(dict(cfg, scene=synth.scene_boxes(seed=5)), 0)
    images[1] = images[1].copy()
    images[1][:, 40:90] = np.random.default_rng(3).integers(0, 255, (101, 50), dtype=np.uint8)
    p = dict(cfg["params"], best_k=best_k, filters=3, alpha_upper=0.4, alpha_lower=0.4, beta=1.05, horizon_row=50)
    fams = [synth.family((0, 0, 1), 24, 0.8, 30.0, "inverse"), synth.family((0, 1, 0), 5, 0.6, 1.6, "linear")]
    _, _, ctx = gpu_objects(cfg)
    ref, test, stats, _ = run_single(cfg, images, params=p, families=fams, ctx=ctx)
    assert_gates(stats, depth_frac_over_tol=0.01)
    plain, _, _, _ = run_single(cfg, images, params=dict(p, best_k=0), families=fams, ctx=ctx)
    if best_k >= n_views:
        assert np.array_equal(ref["kbest"], plain["kbest"])
        planes = fsw.PlaneSet(fams)
        dev = [torch.from_numpy(im).cuda() for im in images]
        a = oracle.compare.to_numpy(ctx.compute_depth(planes, p, dev))
        b = oracle.compare.to_numpy(ctx.compute_depth(planes, dict(p, best_k=0), dev))
        for key in ("depth", "best_cost", "second_cost", "plane_index", "valid_reason"):
            assert np.array_equal(a[key], b[key], equal_nan=True), key
    else:
        assert (ref["kbest"] != plain["kbest"]).sum() > 50      # the rule matters on this input
        ctx.set_split("on")                                      # and the plane split carries it as well
        _, split, stats2, _ = run_single(cfg, images, params=p, families=fams, ctx=ctx)
        for key in ("depth", "best_cost", "second_cost", "plane_index", "valid_reason"):
            assert np.array_equal(test[key], split[key], equal_nan=True), key
    with pytest.raises(fsw.FswError) as ei:
        ctx.compute_depth(fsw.PlaneSet(fams), dict(p, best_k=3), [torch.from_numpy(im).cuda() for im in images])
    assert ei.value.code == fsw.binding.E_UNSUPPORTED


def test_filter_before_merge_order():
    """SURVEY 8(f) 4 / reading Q27: each scale filtered on its own, then merged -- against the oracle, with strict
    thresholds for the crop pass so that half-resolution estimates fill in, single call and batch."""
    import torch
    import paper_1809_06132_b200 as fsw
    cfg = _small_rig(W=128, H=96, n_views=2, fov=170.0)
    images = synth.render_frame(dict(cfg, scene=synth.scene_boxes(seed=12, n_boxes=8)), 0)
    cfg.update(families_low=[synth.family((0, 0, 1), 16, 0.8, 30.0, "inverse")],
               families_crop=[synth.family((0, 0, 1), 32, 0.8, 40.0, "inverse")],
               params_low=synth.params(5, synth.VAR_FLOOR_U8, 60.0, 0.25, 0.35, 24, 1.1, filters=3),
               params_crop=dict(synth.params(7, synth.VAR_FLOOR_U8, 80.0, 0.03, 0.05, 48, 1.15, filters=3), filter_before_merge=1),
               crop=(35, 27, 61, 40))
    mask = np.zeros((96, 128), np.uint8)
    mask[10:30, 50:90] = 1
    _, _, ctx = gpu_objects(cfg)
    ref, test, stats, _ = run_multires(cfg, images, mask, ctx=ctx)
    assert_gates(stats, depth_frac_over_tol=0.01)
    k = ref["kbest"]
    x0, y0, w, h = cfg["crop"]
    inside = np.zeros(mask.shape, bool)
    inside[y0:y0 + h, x0:x0 + w] = True
    filled = inside & (ref["reason"] == 0) & (k >= 0) & ((k >> 14) == 0)
    assert filled.sum() > 20 and (inside & (ref["reason"] == 0) & ((k >> 14) == 1)).sum() > 20
    other = dict(cfg, params_crop=dict(cfg["params_crop"], filter_before_merge=0))
    ref2, _, stats2, _ = run_multires(other, images, mask, ctx=ctx)
    assert_gates(stats2, depth_frac_over_tol=0.01)
    assert (ref["reason"] == 0).sum() > (ref2["reason"] == 0).sum()      # filtering first keeps more
    pl, pc = fsw.PlaneSet(cfg["families_low"]), fsw.PlaneSet(cfg["families_crop"])
    dev = [torch.from_numpy(im).cuda() for im in images]
    outs = ctx.compute_depth_multires_batch(pl, pc, cfg["params_low"], cfg["params_crop"], cfg["crop"], [dev, dev],
                                            [torch.from_numpy(mask).cuda(), None])
    torch.cuda.synchronize()
    got = oracle.compare.to_numpy(outs[0])
    for key in ("depth", "best_cost", "second_cost", "plane_index", "valid_reason"):
        assert np.array_equal(test[key], got[key], equal_nan=True), key


@pytest.mark.parametrize("depth_kind,filter_first", [(0, 0), (1, 1)])
def test_plane_consistent_upsampling(depth_kind, filter_first):
    """SURVEY 8(f) 4 / reading Q28: pixels that take the half-resolution estimate intersect their own ray with the
    refined plane of the half-resolution pixel (range and z-depth, both merge orders), against the oracle."""
    cfg = _small_rig(W=128, H=96, n_views=2, fov=170.0)
    images = synth.render_frame(dict(cfg, scene=synth.scene_boxes(seed=12, n_boxes=8)), 0)
    cfg.update(families_low=[synth.family((0, 0, 1), 16, 0.8, 30.0, "inverse"), synth.family((0, 1, 0), 4, 0.8, 1.6, "linear")],
               families_crop=[synth.family((0, 0, 1), 32, 0.8, 40.0, "inverse")],
               params_low=synth.params(5, synth.VAR_FLOOR_U8, 60.0, 0.3, 0.4, 24, 1.05, filters=3),
               params_crop=dict(synth.params(7, synth.VAR_FLOOR_U8, 80.0, 0.2, 0.3, 48, 1.1, filters=3, depth_kind=depth_kind),
                                upsample_plane=1, filter_before_merge=filter_first),
               crop=(35, 27, 61, 40))
    mask = np.zeros((96, 128), np.uint8)
    mask[60:80, 20:60] = 1
    ref, test, stats, _ = run_multires(cfg, images, mask)
    assert_gates(stats, depth_frac_over_tol=0.01)
    k = ref["kbest"]
    from_lo = (k >= 0) & ((k >> 14) == 0) & (ref["reason"] == 0)
    assert from_lo.sum() > 500
    plain = dict(cfg, params_crop=dict(cfg["params_crop"], upsample_plane=0))
    ref0, _, _, _ = run_multires(plain, images, mask)
    assert (np.abs(ref0["depth"][from_lo] - ref["depth"][from_lo]) > 1e-6 * ref["depth"][from_lo]).mean() > 0.5


@pytest.mark.parametrize("idx", [1, 2])
def test_config_with_filters(idx):
    """C1 / C2 name no filters; SURVEY 8(d) asks for both the raw-valid set and alpha = 0.3/0.3, beta = 1.2."""
    cfg = synth.make_config(idx)
    images = synth.render_frame(cfg, 0)
    p = dict(cfg["params"], alpha_upper=0.3, alpha_lower=0.3, beta=1.2, filters=3, horizon_row=cfg["cams"][0]["height"] // 2)
    ref, test, stats, _ = run_single(cfg, images, params=p)
    assert_gates(stats)
    assert 0 < stats["n_oracle_valid"] < stats["n_oracle_raw_valid"]


def test_config4_multires_merge_and_mask():
    cfg = synth.make_config(4)
    images = synth.render_frame(cfg, 0)
    mask = synth.make_mask(1280, 1024, cfg["mask_seed"])
    ref, test, stats, counters = run_multires(cfg, images, mask)
    assert_gates(stats)
    # outside the crop every value is the nearest-neighbour upsampled half-resolution one (no crop flag)
    x0, y0, w, h = cfg["crop"]
    outside = np.ones(mask.shape, bool)
    outside[y0:y0 + h, x0:x0 + w] = False
    k = test["plane_index"].astype(np.int32)
    assert not ((k[outside] >= 0) & ((k[outside] >> 14) & 1).astype(bool)).any()
    assert (test["depth"][mask != 0] == 0).all() and (test["valid_reason"][mask != 0] != 0).all()
    # downsample, footprint pack + low sweep, footprint pack + crop sweep (two launches each where tiles stay whole)
    assert 5 <= counters["n_launches"] <= 7


@pytest.mark.parametrize("frame", [0, 31])
def test_config5_stream_frames(frame):
    cfg = synth.make_config(5)
    images = synth.render_frame(cfg, frame)
    mask = synth.make_mask(1280, 1024, cfg["mask_seed"] + frame)
    _, test, stats, _ = run_single(cfg, images, mask)
    assert_gates(stats)
    assert (test["depth"][mask != 0] == 0).all()


def test_config5_batch_of_8_as_benchmarked():
    """The launch configuration bench.py times: 8 consecutive C5 frame sets (with their masks) in ONE sweep launch
    (fsw_compute_depth_batch) at full size.  One frame set of the launch is gated against the oracle, and every set
    must be bit-identical to its own single-set call."""
    import torch
    import paper_1809_06132_b200 as fsw
    cfg = synth.make_config(5)
    _, _, ctx = gpu_objects(cfg)
    planes = fsw.PlaneSet(cfg["families"])
    frames = list(range(8, 16))
    sets = [synth.render_frame(cfg, f) for f in frames]
    masks = [synth.make_mask(1280, 1024, cfg["mask_seed"] + f) for f in frames]
    dev_sets = [[torch.from_numpy(im).cuda() for im in st] for st in sets]
    dev_masks = [torch.from_numpy(m).cuda() for m in masks]
    outs = ctx.compute_depth_batch(planes, cfg["params"], dev_sets, dev_masks)
    torch.cuda.synchronize()
    counters = ctx.last_counters()
    assert 2 <= counters["n_launches"] <= 3  # one footprint pack, one sweep (two with whole + halved tiles)
    batch = [oracle.compare.to_numpy(o) for o in outs]
    n_eval, n_eval_set = 0, []
    for s in range(8):
        single = oracle.compare.to_numpy(ctx.compute_depth(planes, cfg["params"], dev_sets[s], dev_masks[s]))
        n_eval_set.append(ctx.last_counters()["n_eval"])
        n_eval += n_eval_set[-1]
        for key in ("depth", "best_cost", "second_cost", "plane_index", "valid_reason"):
            assert np.array_equal(single[key], batch[s][key], equal_nan=True), (s, key)
    assert counters["n_eval"] == n_eval
    s = 5
    ref = oracle.compute_depth(cfg["cams"], cfg["ref_index"], cfg["families"], cfg["params"], sets[s], masks[s], keep_cost=True)
    cond = oracle.compare.depth_conditioning(ref, oracle.plane_table(cfg["families"])[0])
    stats = oracle.compare.compare_maps(ref, batch[s], ref["cost"], depth_cond=cond)
    # the batch counter is the sum of the single-set counters (above); this set's share is held to the oracle
    stats["n_eval_oracle"], stats["n_eval_test"] = ref["n_eval"], n_eval_set[s]
    assert_gates(stats)
    assert (batch[s]["depth"][masks[s] != 0] == 0).all()


# ---- cost volume, element by element --------------------------------------------------------------------------------
def test_debug_cost_volume_matches_oracle():
    cfg = synth.make_config(2)
    images = synth.render_frame(cfg, 0)
    ref, test, stats, _ = run_single(cfg, images, debug_cost=True)
    vol, ovol = test["cost_volume"].astype(np.float64), ref["cost"]
    fin_o, fin_t = np.isfinite(ovol), np.isfinite(vol)
    frag = ref["fragile_geom"] != 0
    assert not ((fin_o != fin_t) & ~frag[None]).any()
    both = fin_o & fin_t
    assert np.abs(vol[both] - ovol[both]).max() <= 1e-4
    assert_gates(stats)


# ---- edge cases ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("window", [3, 5, 7, 9, 11, 13, 15])
def test_every_window_size_ragged_image(window):
    cfg = _small_rig(W=70, H=45)
    cfg["params"] = dict(cfg["params"], window=window)
    images = synth.render_frame(cfg, 0)
    _, _, stats, _ = run_single(cfg, images)
    assert_gates(stats, depth_frac_over_tol=0.001 if window >= 5 else 0.01)
    assert stats["n_oracle_valid"] > 0


@pytest.mark.parametrize("n_views,rot,dist,dtype", [
    (1, False, None, "f32"),
    (3, True, None, "u8"),
    (2, True, dict(k1=-0.03, k2=0.004, p1=0.0008, p2=-0.0006), "u8"),
    (4, True, dict(k1=-0.04), "f32"),
])
def test_views_rotation_distortion_dtype(n_views, rot, dist, dtype):
    cfg = _small_rig(W=96, H=64, n_views=n_views, rot=rot, dist=dist, dtype=dtype, fov=170.0)
    images = synth.render_frame(cfg, 0)
    _, _, stats, _ = run_single(cfg, images)
    assert_gates(stats)
    assert stats["n_oracle_valid"] > 500


def test_two_families_linear_ground_roi_z_depth_no_subpixel():
    cfg = synth.make_config(2)
    images = synth.render_frame(cfg, 0)
    fams = [synth.family((0, 0, 1), 20, 1.0, 40.0, "inverse"), synth.family((0, 1, 0), 9, 1.2, 2.0, "linear"),
            synth.family((0, 0, 1), 1, 2.5, 2.5, "linear")]
    for sub, kind in ((1, 1), (0, 0)):
        p = dict(cfg["params"], roi=(37, 21, 201, 150), depth_kind=kind, subpixel=sub, filters=3, alpha_upper=0.2,
                 alpha_lower=0.35, beta=1.1, horizon_row=100)
        ref, test, stats, _ = run_single(cfg, images, params=p, families=fams)
        assert_gates(stats)
        outside = np.ones(ref["depth"].shape, bool)
        outside[21:21 + 150, 37:37 + 201] = False
        assert (test["depth"][outside] == 0).all() and (test["plane_index"][outside] == -1).all()
        assert (ref["kbest"] >= 20).any()  # the ground family wins somewhere


def test_degenerate_inputs():
    import torch
    import paper_1809_06132_b200 as fsw
    cfg = _small_rig(W=64, H=48)
    fsw_mod, rig, ctx = gpu_objects(cfg)
    images = synth.render_frame(cfg, 0)
    # (a) everything masked -> all invalid, reasons say why
    mask = np.ones((48, 64), np.uint8)
    ref, test, stats, _ = run_single(cfg, images, mask, ctx=ctx)
    assert (test["depth"] == 0).all() and stats["valid_mismatch_total"] == 0
    assert set(np.unique(test["valid_reason"])) <= {fsw.REASON_NO_PLANE, fsw.REASON_MASKED}
    # (b) constant images: cost = 0.5 on every plane, lowest index wins, the cost filter rejects everything
    flat = [np.full((48, 64), 90, np.uint8)] * 2
    p = dict(cfg["params"], filters=1, alpha_upper=0.3, alpha_lower=0.3)
    ref, test, stats, _ = run_single(cfg, flat, params=p, ctx=ctx)
    assert (test["depth"] == 0).all() and stats["valid_mismatch_total"] == 0
    k = test["plane_index"]
    assert np.array_equal(k[k >= 0], ref["kbest"][ref["kbest"] >= 0])
    assert np.abs(test["best_cost"][k >= 0] - 0.5).max() < 1e-6
    # (c) ROI entirely outside the field of view / clipped away -> no plane anywhere, nothing evaluated
    p = dict(cfg["params"], roi=(0, 0, 3, 3))
    ref, test, stats, counters = run_single(cfg, images, params=p, ctx=ctx)
    assert (test["plane_index"] == -1).all() and counters["n_eval"] == 0 and ref["n_eval"] == 0
    # (d) the largest plane set the ABI accepts
    fams = [synth.family((0, 0, 1), 1024, 0.8, 30.0, "inverse")]
    ref, test, stats, _ = run_single(cfg, images, families=fams, ctx=ctx)
    assert_gates(stats, depth_frac_over_tol=0.05)  # 1024 planes over 64x48 pixels: every cost curve is flat
    # (e) bad arguments are errors, not crashes
    planes = fsw.PlaneSet(cfg["families"])
    dev = [torch.from_numpy(im).cuda() for im in images]
    for bad in (dict(window=4), dict(window=17), dict(range_max=0.0), dict(filters=8)):
        with pytest.raises(fsw.FswError) as ei:
            ctx.compute_depth(planes, dict(cfg["params"], **bad), dev)
        assert ei.value.code == fsw.binding.E_INVALID_ARG


def test_host_call_equals_device_call_and_is_deterministic():
    cfg = synth.make_config(2)
    images = synth.render_frame(cfg, 0)
    _, _, ctx = gpu_objects(cfg)
    p = dict(cfg["params"], filters=3, alpha_upper=0.3, alpha_lower=0.3, beta=1.2, horizon_row=128)
    _, a, _, _ = run_single(cfg, images, params=p, ctx=ctx)
    _, b, _, _ = run_single(cfg, images, params=p, ctx=ctx, host=True)
    _, c, _, _ = run_single(cfg, images, params=p, ctx=ctx)
    for key in ("depth", "best_cost", "second_cost", "plane_index", "valid_reason"):
        assert np.array_equal(a[key], b[key], equal_nan=True), key
        assert np.array_equal(a[key], c[key], equal_nan=True), key


def test_async_host_calls_on_two_streams():
    """fsw_context_set_host_async: host calls that do not synchronize, issued alternately on two streams through two
    contexts (bench.py's end-to-end arrangement), give the maps of the synchronous host call."""
    import torch
    import paper_1809_06132_b200 as fsw
    cfg = _small_rig(W=150, H=77, n_views=2, fov=170.0)
    rig = fsw.Rig(cfg["cams"], cfg["ref_index"])
    planes = fsw.PlaneSet(cfg["families"])
    ctxs = [fsw.Context(rig, 0), fsw.Context(rig, 0)]
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    sets = [[torch.from_numpy(im).pin_memory() for im in synth.render_frame(dict(cfg, scene=synth.scene_plane(2.0 + 0.5 * s, (0.5, 2.0), seed=40 + s)), 0)]
            for s in range(6)]
    masks = [torch.from_numpy(synth.make_mask(150, 77, 60 + s, n_rects=2)).pin_memory() for s in range(6)]
    sync = [oracle.compare.to_numpy(ctxs[0].compute_depth(planes, cfg["params"], sets[s], masks[s], host=True)) for s in range(6)]
    for c in ctxs:
        c.set_host_async(True)
    pinned = [{k: torch.empty((77, 150), dtype=t).pin_memory() for k, t in
               (("depth", torch.float32), ("best_cost", torch.float32), ("second_cost", torch.float32),
                ("plane_index", torch.int16), ("valid_reason", torch.uint8))} for _ in range(6)]
    for b in range(3):  # batches of two frame sets, alternating contexts / streams
        with torch.cuda.stream(streams[b % 2]):
            ctxs[b % 2].compute_depth_batch(planes, cfg["params"], sets[2 * b:2 * b + 2], masks[2 * b:2 * b + 2], host=True,
                                            outs=pinned[2 * b:2 * b + 2])
    torch.cuda.synchronize()
    for s in range(6):
        for key in ("depth", "best_cost", "second_cost", "plane_index", "valid_reason"):
            assert np.array_equal(sync[s][key], pinned[s][key].numpy(), equal_nan=True), (s, key)
    for c in ctxs:
        c.close()


def test_multires_host_call_small():
    """S10 on a small rig: host-buffer call, crop not aligned to the tile grid, odd crop origin."""
    cfg = _small_rig(W=128, H=96, n_views=2, fov=170.0)
    images = synth.render_frame(cfg, 0)
    cfg.update(families_low=[synth.family((0, 0, 1), 16, 0.8, 30.0, "inverse")],
               families_crop=[synth.family((0, 0, 1), 32, 0.8, 40.0, "inverse")],
               params_low=synth.params(5, synth.VAR_FLOOR_U8, 60.0),
               params_crop=synth.params(7, synth.VAR_FLOOR_U8, 80.0, 0.2, 0.3, 48, 1.1, filters=3),
               crop=(35, 27, 61, 40))
    mask = synth.make_mask(128, 96, 11, n_rects=2)
    mask[:, :] = 0
    mask[10:30, 50:90] = 1
    for host in (False, True):
        ref, test, stats, _ = run_multires(cfg, images, mask, host=host)
        assert_gates(stats)
        assert (ref["kbest"] >> 14 == 1).any() and ((ref["kbest"] >= 0) & (ref["kbest"] >> 14 == 0)).any()


def test_batch_equals_single_calls():
    """fsw_compute_depth_batch: n frame sets in one sweep launch give exactly the maps of n separate calls
    (device and host variants; masks may be missing for some sets), and the counters are the totals."""
    import torch
    import paper_1809_06132_b200 as fsw
    cfg = _small_rig(W=150, H=77, n_views=2, fov=170.0)
    _, _, ctx = gpu_objects(cfg)
    planes = fsw.PlaneSet(cfg["families"])
    p = dict(cfg["params"], filters=3, alpha_upper=0.3, alpha_lower=0.3, beta=1.1, horizon_row=40)
    sets, masks = [], []
    for s in range(5):
        c = dict(cfg, scene=synth.scene_plane(2.0 + 0.7 * s, (0.5, 2.0), seed=20 + s))
        sets.append(synth.render_frame(c, 0))
        masks.append(synth.make_mask(150, 77, 30 + s, n_rects=2) if s % 2 == 0 else None)
    singles, n_eval = [], 0
    for s in range(5):
        dev = [torch.from_numpy(im).cuda() for im in sets[s]]
        dm = None if masks[s] is None else torch.from_numpy(masks[s]).cuda()
        singles.append(oracle.compare.to_numpy(ctx.compute_depth(planes, p, dev, dm)))
        n_eval += ctx.last_counters()["n_eval"]
    dev_sets = [[torch.from_numpy(im).cuda() for im in st] for st in sets]
    dev_masks = [None if m is None else torch.from_numpy(m).cuda() for m in masks]
    outs = ctx.compute_depth_batch(planes, p, dev_sets, dev_masks)
    torch.cuda.synchronize()
    c = ctx.last_counters()
    assert c["n_eval"] == n_eval and 2 <= c["n_launches"] <= 3
    houts = ctx.compute_depth_batch(planes, p, sets, masks, host=True)
    for s in range(5):
        a, b = oracle.compare.to_numpy(outs[s]), oracle.compare.to_numpy(houts[s])
        for key in ("depth", "best_cost", "second_cost", "plane_index", "valid_reason"):
            assert np.array_equal(singles[s][key], a[key], equal_nan=True), (s, key)
            assert np.array_equal(singles[s][key], b[key], equal_nan=True), (s, key)
        if masks[s] is not None:
            assert (a["depth"][masks[s] != 0] == 0).all()
    # one set against the oracle, so that the batch path is pinned to more than itself
    ref = oracle.compute_depth(cfg["cams"], cfg["ref_index"], cfg["families"], p, sets[3], masks[3], keep_cost=True)
    st = oracle.compare.compare_maps(ref, oracle.compare.to_numpy(outs[3]), ref["cost"])
    assert st["index_match_frac"] >= 0.999 and st["max_dc1"] <= 1e-4 and st["valid_mismatch_nonfragile"] == 0, st
    with pytest.raises(fsw.FswError):
        ctx.compute_depth_batch(planes, p, [], None)


def test_plane_split_is_bit_identical_to_the_unsplit_sweep():
    """fsw_context_set_split: tiles swept as two half plane ranges (ascending below the cut, descending above it) and
    merged must give exactly the maps, the cost volume and the counters of the unsplit sweep -- cut inside a family
    (with the neighbour across the cut), cut at a family boundary, two planes only, the multi-resolution call and a
    batch; and the automatic mode must split a single full-size frame set but not a batch of eight."""
    import torch
    import paper_1809_06132_b200 as fsw
    keys = ("depth", "best_cost", "second_cost", "plane_index", "valid_reason")

    def both(ctx, run):
        res = []
        for mode in ("off", "on"):
            ctx.set_split(mode)
            out = run()
            torch.cuda.synchronize()
            res.append((oracle.compare.to_numpy(out), ctx.last_counters()))
        (a, ca), (b, cb) = res
        assert ca["n_split_launches"] == 0 and cb["n_split_launches"] >= 1
        for key in keys + (("cost_volume",) if "cost_volume" in a else ()):
            assert np.array_equal(a[key], b[key], equal_nan=True), key
        for key in ("n_eval", "n_raw_valid", "n_valid"):
            assert ca[key] == cb[key], key
        return a

    fam_sets = [
        [synth.family((0, 0, 1), 24, 0.8, 30.0, "inverse")],                                       # cut inside the family
        [synth.family((0, 0, 1), 12, 0.8, 30.0, "inverse"), synth.family((0, 1, 0), 24, 0.4, 1.6, "linear")],  # at the boundary
        [synth.family((0, 0, 1), 9, 0.8, 30.0, "inverse"), synth.family((0, 1, 0), 4, 0.4, 1.6, "linear"),
         synth.family((0.1, 0.2, 1), 7, 1.0, 20.0, "linear")],                                     # three families
        [synth.family((0, 0, 1), 2, 2.0, 4.0, "inverse")],                                         # two planes: 1 + 1
        [synth.family((0, 0, 1), 1, 3.0, 3.0, "inverse"), synth.family((0, 1, 0), 1, 1.0, 1.0, "linear")],
    ]
    cfg = _small_rig(W=150, H=101, n_views=2, fov=170.0)
    _, _, ctx = gpu_objects(cfg)
    images = synth.render_frame(dict(cfg, scene=synth.scene_boxes(seed=5)), 0)
    dev = [torch.from_numpy(im).cuda() for im in images]
    p = dict(cfg["params"], filters=3, alpha_upper=0.4, alpha_lower=0.4, beta=1.05, horizon_row=50)
    for fams in fam_sets:
        planes = fsw.PlaneSet(fams)
        a = both(ctx, lambda: ctx.compute_depth(planes, p, dev, None, debug_cost=True))
        assert (a["plane_index"] >= 0).any()
    # the split path against the oracle on its own (second family mostly wins below the horizon)
    ctx.set_split("on")
    ref, test, stats, _ = run_single(cfg, images, params=p, families=fam_sets[1], ctx=ctx)
    assert_gates(stats, depth_frac_over_tol=0.01)
    # batch and multi-resolution calls
    planes = fsw.PlaneSet(fam_sets[0])
    sets = [dev, [torch.from_numpy(im).cuda() for im in synth.render_frame(cfg, 0)]]
    for s in range(2):
        ctx.set_split("off")
        single = oracle.compare.to_numpy(ctx.compute_depth(planes, p, sets[s], None))
        ctx.set_split("on")
        outs = ctx.compute_depth_batch(planes, p, sets, None)
        torch.cuda.synchronize()
        for key in keys:
            assert np.array_equal(single[key], oracle.compare.to_numpy(outs[s])[key], equal_nan=True), (s, key)
    pl, pc = fsw.PlaneSet(fam_sets[0]), fsw.PlaneSet(fam_sets[1])
    pp = dict(p, window=3)
    both(ctx, lambda: ctx.compute_depth_multires(pl, pc, pp, p, (40, 30, 70, 50), dev, None))
    ctx.close()
    # automatic mode at full size
    cfg = synth.make_config(3)
    _, _, ctx = gpu_objects(cfg)
    planes = fsw.PlaneSet(cfg["families"])
    dev = [torch.from_numpy(im).cuda() for im in synth.render_frame(cfg, 0)]
    res = {}
    # auto: the heavy tiles whole in the unsplit kernel + the light ones in halves as its programmatic dependent launch
    # (both on the caller's stream); on: every tile in halves, one launch
    for mode in ("off", "auto", "on"):
        ctx.set_split(mode)
        res[mode] = oracle.compare.to_numpy(ctx.compute_depth(planes, cfg["params"], dev, None))
        c = ctx.last_counters()
        assert c["n_split_launches"] == (0 if mode == "off" else 1)
        assert c["n_launches"] == (3 if mode == "auto" else 2), (mode, c)   # pack + sweep(s)
    for mode in ("auto", "on"):
        for key in keys:
            assert np.array_equal(res["off"][key], res[mode][key], equal_nan=True), (mode, key)
    ctx.set_split("auto")
    ctx.compute_depth_batch(planes, cfg["params"], [dev] * 8, None)
    assert ctx.last_counters()["n_split_launches"] == 0
    ctx.close()


@pytest.mark.parametrize("window", [7, 11])
def test_plane_split_two_launches_other_windows(window):
    """An image with more live tiles than SMs and a window other than 9 x 9 (other tile geometry): the automatic mode
    sweeps the heavy tiles whole and the rest in halves (two launches on the caller's stream, the second a programmatic
    dependent of the first) and gives the unsplit maps bit for bit; so does a back-to-back series of such calls."""
    import torch
    import paper_1809_06132_b200 as fsw
    cfg = _small_rig(W=1216, H=808, n_views=2, fov=170.0)
    _, _, ctx = gpu_objects(cfg)
    planes = fsw.PlaneSet([synth.family((0, 0, 1), 9, 0.8, 30.0, "inverse"), synth.family((0, 1, 0), 4, 0.4, 1.6, "linear")])
    dev = [torch.from_numpy(im).cuda() for im in synth.render_frame(cfg, 0)]
    p = dict(cfg["params"], window=window, filters=3, alpha_upper=0.4, alpha_lower=0.4, beta=1.05, horizon_row=400)
    res = {}
    for mode in ("off", "auto", "on"):
        ctx.set_split(mode)
        res[mode] = oracle.compare.to_numpy(ctx.compute_depth(planes, p, dev, None))
        c = ctx.last_counters()
        assert (c["n_split_launches"], c["n_launches"]) == {"off": (0, 2), "auto": (1, 3), "on": (1, 2)}[mode], c
        res[mode + "_n_eval"] = c["n_eval"]
    assert res["off_n_eval"] == res["auto_n_eval"] == res["on_n_eval"] > 0
    for mode in ("auto", "on"):
        for key in ("depth", "best_cost", "second_cost", "plane_index", "valid_reason"):
            assert np.array_equal(res["off"][key], res[mode][key], equal_nan=True), (mode, key)
    assert (res["off"]["plane_index"] >= 0).sum() > 100000
    # calls issued back to back without a host synchronisation: the pack kernel of a call must not start before both
    # sweep launches of the call before it are through (the dependent launch completes after the first one)
    ctx.set_split("auto")
    outs = [ctx.compute_depth(planes, p, dev, None) for _ in range(6)]
    torch.cuda.synchronize()
    for o in outs:
        o = oracle.compare.to_numpy(o)
        for key in ("depth", "best_cost", "second_cost", "plane_index", "valid_reason"):
            assert np.array_equal(res["off"][key], o[key], equal_nan=True), key
    ctx.close()


def test_split_call_captured_into_a_cuda_graph():
    """include/fsw.h: the whole / halved launches of FSW_SPLIT_AUTO are two launches on the caller's stream, the second a
    programmatic dependent of the first; captured into a CUDA graph and replayed they give the maps of the eager call."""
    import torch
    import paper_1809_06132_b200 as fsw
    cfg = synth.make_config(3)
    _, _, ctx = gpu_objects(cfg)
    planes = fsw.PlaneSet(cfg["families"])
    dev = [torch.from_numpy(im).cuda() for im in synth.render_frame(cfg, 0)]
    keys = ("depth", "best_cost", "second_cost", "plane_index", "valid_reason")
    eager = ctx.compute_depth(planes, cfg["params"], dev, None)
    c = ctx.last_counters()
    assert (c["n_split_launches"], c["n_launches"]) == (1, 3), c
    eager = {k: eager[k].clone() for k in keys}
    side = torch.cuda.Stream()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.stream(side):
        ctx.compute_depth(planes, cfg["params"], dev, None)     # scratch of the context is allocated outside the capture
        torch.cuda.synchronize()
        with torch.cuda.graph(graph, stream=side):
            out = ctx.compute_depth(planes, cfg["params"], dev, None)
    for _ in range(3):
        for k in keys:
            out[k].zero_()
        graph.replay()
        torch.cuda.synchronize()
        for k in keys:
            assert np.array_equal(eager[k].cpu().numpy(), out[k].cpu().numpy(), equal_nan=True), k
    ctx.close()


def test_bfloat16_and_float_footprints_agree_bitwise():
    """8-bit views are staged as bfloat16 footprints (exact for integers up to 256), float views as float footprints:
    the same integer-valued views given as uint8 and as float32 must produce bit-identical maps, and a call that
    mixes both types (falls back to float footprints) as well."""
    import torch
    import paper_1809_06132_b200 as fsw
    cfg = _small_rig(W=131, H=83, n_views=2, fov=170.0)
    images = synth.render_frame(cfg, 0)
    assert images[0].dtype == np.uint8
    _, _, ctx = gpu_objects(cfg)
    planes = fsw.PlaneSet(cfg["families"])
    outs = []
    # the reference image stays 8-bit (its type decides how the centring constant is rounded); only the views change
    for kinds in (("u8", "u8", "u8"), ("u8", "f32", "f32"), ("u8", "f32", "u8")):
        dev = [torch.from_numpy(im if k == "u8" else im.astype(np.float32)).cuda() for im, k in zip(images, kinds)]
        outs.append(oracle.compare.to_numpy(ctx.compute_depth(planes, cfg["params"], dev)))
    for o in outs[1:]:
        for key in ("depth", "best_cost", "second_cost", "plane_index", "valid_reason"):
            assert np.array_equal(outs[0][key], o[key], equal_nan=True), key
    assert (outs[0]["plane_index"] >= 0).sum() > 1000


@pytest.mark.parametrize("idx,window,gamma,delta", [(2, 5, 0.5, 0.3), (3, 5, 0.5, 0.3), (2, 9, 0.2, 0.5), (1, 3, 2.0, 0.25)])
def test_continuity_filter_bit_exact_against_oracle(idx, window, gamma, delta):
    """fsw_filter_continuity (third filter + mask) on the depth map the sweep produced: validity, reasons
    and surviving depths must equal the oracle's filter on the same float32 map bit for bit (integer / comparison
    work: both sides compare in double precision)."""
    import torch
    import paper_1809_06132_b200 as fsw
    cfg = synth.make_config(idx)
    images = synth.render_frame(cfg, 0)
    W, H = cfg["cams"][0]["width"], cfg["cams"][0]["height"]
    _, _, ctx = gpu_objects(cfg)
    planes = fsw.PlaneSet(cfg["families"])
    p = dict(cfg["params"], filters=3 if idx > 1 else 0, alpha_upper=0.3, alpha_lower=0.3, beta=1.1, horizon_row=H // 2)
    dev = [torch.from_numpy(np.ascontiguousarray(im)).cuda() for im in images]
    swept = ctx.compute_depth(planes, p, dev)          # no mask here: the mask comes after the filters
    mask = synth.make_mask(W, H, 77, n_rects=3)
    if idx == 1:  # the generator's rectangles are larger than this 64 x 48 image
        mask = np.zeros((H, W), np.uint8)
        mask[10:20, 30:50] = 1
    out = ctx.filter_continuity(swept["depth"], window, gamma, delta, torch.from_numpy(mask).cuda())
    torch.cuda.synchronize()
    d_in = swept["depth"].cpu().numpy()
    ref_d, ref_r = oracle.filter_continuity(d_in, window, gamma, delta, mask)
    assert np.array_equal(out["valid_reason"].cpu().numpy(), ref_r)
    assert np.array_equal(out["depth"].cpu().numpy().astype(np.float64), ref_d)
    n_in, n_out = int((d_in > 0).sum()), int((ref_d > 0).sum())
    assert 0 < n_out <= n_in
    if idx > 1:  # the scenes with depth edges: every verdict occurs
        assert n_out < n_in and (ref_r == 5).sum() > 0 and (ref_r == 4).sum() > 0
    # without mask and reason map; pitched input view
    out2 = ctx.filter_continuity(swept["depth"], window, gamma, delta, None, want_reason=False)
    ref2, _ = oracle.filter_continuity(d_in, window, gamma, delta)
    assert np.array_equal(out2["depth"].cpu().numpy().astype(np.float64), ref2)


def test_continuity_filter_delta_boundary_is_decided_in_double():
    """Reading Q25: a centre whose consistent share equals delta exactly is kept.  With a 9 x 9 window and delta = 0.3
    that is 24 consistent neighbours of 80 (and 36 of 120 with 11 x 11): 24/80 == 0.3 in double, whereas a float
    0.3f = 0.300000012 would reject the pixel.  gamma and delta cross the ABI as doubles."""
    import torch
    cfg = _small_rig(W=64, H=48)
    _, _, ctx = gpu_objects(cfg)
    for window, n_keep in ((9, 24), (11, 36)):
        d = np.zeros((48, 64), np.float32)
        cy, cx, hw = 24, 30, window // 2
        d[cy, cx] = 5.0
        cells = [(cy + dy, cx + dx) for dy in range(-hw, hw + 1) for dx in range(-hw, hw + 1) if (dy, dx) != (0, 0)]
        for (y, x) in cells[:n_keep]:
            d[y, x] = 5.2                      # consistent: |5.2 - 5.0| < 0.5
        for (y, x) in cells[n_keep:n_keep + 10]:
            d[y, x] = 9.0                      # valid but not consistent
        for n_cons, kept in ((n_keep, True), (n_keep - 1, False)):
            dd = d.copy()
            if n_cons < n_keep:
                dd[cells[0]] = 9.0
            out = ctx.filter_continuity(torch.from_numpy(dd).cuda(), window, 0.5, 0.3)
            torch.cuda.synchronize()
            ref_d, ref_r = oracle.filter_continuity(dd, window, 0.5, 0.3)
            got_d, got_r = out["depth"].cpu().numpy(), out["valid_reason"].cpu().numpy()
            assert (ref_d[cy, cx] > 0) == kept and (got_d[cy, cx] > 0) == kept, (window, n_cons)
            assert np.array_equal(got_r, ref_r) and np.array_equal(got_d.astype(np.float64), ref_d)


def test_continuity_filter_argument_errors():
    import torch
    import paper_1809_06132_b200 as fsw
    cfg = _small_rig(W=64, H=48)
    _, _, ctx = gpu_objects(cfg)
    d = torch.ones((48, 64), dtype=torch.float32, device="cuda")
    for kw in (dict(window=4), dict(window=17), dict(gamma=0.0), dict(delta=1.5)):
        with pytest.raises(fsw.FswError):
            ctx.filter_continuity(d, **kw)
    out = ctx.filter_continuity(d)   # constant map: unchanged
    assert torch.equal(out["depth"], d) and int(out["valid_reason"].sum()) == 0
    # the binding refuses tensors the kernel would write out of bounds: wrong type, wrong shape, wrong device
    with pytest.raises(AssertionError):
        ctx.filter_continuity(d.double())
    with pytest.raises(AssertionError):
        ctx.filter_continuity(d[:40])
    planes = fsw.PlaneSet(cfg["families"])
    dev = [torch.from_numpy(im).cuda() for im in synth.render_frame(cfg, 0)]
    for bad in (dict(plane_index=torch.empty((48, 64), dtype=torch.float32, device="cuda")),
                dict(depth=torch.empty((40, 64), dtype=torch.float32, device="cuda")),
                dict(depth=torch.empty((48, 64), dtype=torch.float32))):
        out = dict(depth=torch.empty((48, 64), dtype=torch.float32, device="cuda"))
        out.update(bad)
        with pytest.raises(AssertionError):
            ctx.compute_depth(planes, cfg["params"], dev, out=out)
