"""Pins of the oracle's variants (run with -m "not gpu").

Reading Q26 -- occlusion-robust best-k view aggregation (SPEC.md:233 names it as a configuration option; the paper is
silent beyond "more than two cameras"): the cost of a plane is the mean of the k lowest per-view costs
among the valid views.  Pinned by what fixes it without the oracle's own aggregation code: k >= number of views is the
plain mean; k = 1 is the element-wise minimum of the cost volumes of the two-camera sub-rigs; a view corrupted by
construction is dropped and the exact plane index of the integer-disparity construction comes back.

Reading Q27 -- filter each scale, then merge (the alternative order of Q20: SPEC.md:301 fixes merge-then-filter, the
paper's multi-scale experiment is unfiltered).  Pinned by its limiting cases: with thresholds that reject
every full-resolution estimate the result is the filtered half-resolution map upsampled (fill-in), with thresholds
that reject nothing both orders agree, and outside the crop the full-resolution pass never shows.

Reading Q28 -- plane-consistent upsampling (the alternative SURVEY Q18 notes): a pixel that takes the half-resolution
estimate intersects its own ray with the refined plane of the half-resolution pixel.  Pinned by geometry: the upsampled
points of one half-resolution pixel lie ON that plane (n.X = d*), which the copied ranges do not; a fronto-parallel
scene plane that coincides with a sweep plane comes back with the exact z at every upsampled pixel.
"""
import numpy as np

import oracle
import synth
from test_oracle_sweep import _pinhole_pair

INF = float("inf")


def _three_pinhole_cameras(W=64, H=40, fx=40.0, b=0.5):
    ref, right = _pinhole_pair(W, H, fx, b)
    left = dict(ref)
    left["t"] = np.array([b, 0.0, 0.0])     # centre at x = -b: the scene shifts the other way
    return ref, left, right


def _shifted_images(W, H, disparity, seed=5):
    rng = np.random.default_rng(seed)
    big = rng.uniform(0, 255, (H, W + 32))
    ref = big[:, 16:16 + W].copy()
    right = big[:, 16 + disparity:16 + disparity + W].copy()   # camera at +b: view(u) = ref(u + disparity)
    left = big[:, 16 - disparity:16 - disparity + W].copy()
    return ref, left, right


def test_best_k_limits_mean_and_single_view_minimum():
    W, H = 64, 40
    cams = _three_pinhole_cameras(W, H)
    fams = [synth.family((0, 0, 1), 8, 20.0, 2.5, "inverse")]          # disparities 1..8 px
    imgs = _shifted_images(W, H, 5)
    prm = synth.params(5, 1e-6, 1e3)
    mean = oracle.compute_depth(cams, 0, fams, prm, imgs, keep_cost=True)
    for k in (2, 3, 7):       # k >= number of valid views: the plain mean, bit for bit
        same = oracle.compute_depth(cams, 0, fams, dict(prm, best_k=k), imgs, keep_cost=True)
        assert np.array_equal(same["cost"], mean["cost"]) and same["n_eval"] == mean["n_eval"]
    best1 = oracle.compute_depth(cams, 0, fams, dict(prm, best_k=1), imgs, keep_cost=True)
    single = [oracle.compute_depth([cams[0], cams[v]], 0, fams, prm, [imgs[0], imgs[v]], keep_cost=True)["cost"] for v in (1, 2)]
    assert np.array_equal(best1["cost"], np.minimum(single[0], single[1]))      # +inf where a view is invalid
    assert best1["n_eval"] == mean["n_eval"]        # the counter counts finite per-view costs, not the ones kept
    # the mean of the two lies between the single-view costs; the best one is never above it
    both = np.isfinite(single[0]) & np.isfinite(single[1])
    assert np.allclose(mean["cost"][both], 0.5 * (single[0][both] + single[1][both]), atol=1e-15)
    assert (best1["cost"][both] <= mean["cost"][both] + 1e-15).all()
    # brute force for single pixels goes through the same aggregation rule
    for (px, py) in [(30, 20), (12, 9), (50, 31)]:
        got = oracle.pixel_costs(cams, 0, fams, dict(prm, best_k=1), imgs, px, py)
        fin = np.isfinite(got)
        assert np.array_equal(fin, np.isfinite(best1["cost"][:, py, px]))
        assert np.allclose(got[fin], best1["cost"][:, py, px][fin], atol=1e-12)


def test_best_k_drops_a_view_that_is_wrong_by_construction():
    """Integer-disparity construction with two views; the right view is replaced by unrelated texture in a band (an
    "occluder").  The mean over both views no longer recovers the plane there; the best single view does, exactly."""
    W, H, true_k = 64, 40, 4
    cams = _three_pinhole_cameras(W, H)
    fams = [synth.family((0, 0, 1), 8, 20.0, 2.5, "inverse")]
    ref, left, right = _shifted_images(W, H, true_k + 1)
    rng = np.random.default_rng(99)
    right[:, 20:44] = rng.uniform(0, 255, (H, 24))
    prm = synth.params(5, 1e-6, 1e3)
    mean = oracle.compute_depth(cams, 0, fams, prm, [ref, left, right], keep_cost=True)
    best1 = oracle.compute_depth(cams, 0, fams, dict(prm, best_k=1), [ref, left, right], keep_cost=True)
    left_only = oracle.compute_depth(cams[:2], 0, fams, prm, [ref, left], keep_cost=True)
    seen_left = np.isfinite(left_only["cost"][true_k])              # pixels whose window the left view covers
    assert seen_left.sum() > 0.5 * W * H
    assert (best1["kbest"][seen_left] == true_k).all()
    assert best1["cost"][true_k][seen_left].max() < 1e-12           # the intact view matches exactly: cost 0
    band = seen_left.copy()
    band[:, :22] = False
    band[:, 42:] = False
    assert (mean["cost"][true_k][band] > 0.05).mean() > 0.5         # the mean carries the wrong view's cost
    assert (mean["kbest"][band] != true_k).any()                    # and loses the plane on some of those pixels


def _multires_setup():
    kw = dict(width=96, height=64, fx=40.0, fy=40.0, cx=47.7, cy=31.8, xi=0.9, fov_max_deg=170.0)
    cams = [synth.camera(**kw), synth.camera(centre=(0.3, 0, 0), yaw_deg=5.0, **kw), synth.camera(centre=(-0.3, 0.02, 0), **kw)]
    scene = synth.scene_boxes(seed=12, n_boxes=8)
    imgs = [synth.quantize(synth.render_camera(c, scene), "u8") for c in cams]
    fl = [synth.family((0, 0, 1), 12, 0.8, 30.0, "inverse")]
    fc = [synth.family((0, 0, 1), 20, 0.8, 40.0, "inverse")]
    p_lo = synth.params(5, synth.VAR_FLOOR_U8, 60.0, 0.25, 0.35, 16, 1.1, filters=3)   # horizon in half-resolution rows
    p_hi = synth.params(7, synth.VAR_FLOOR_U8, 80.0, 0.02, 0.02, 32, 1.15, filters=3)     # strict: leaves room for fill-in
    return cams, imgs, fl, fc, p_lo, p_hi, (30, 20, 40, 28)


def test_filter_before_merge_limiting_cases():
    cams, imgs, fl, fc, p_lo, p_hi, crop = _multires_setup()
    H, W = imgs[0].shape
    x0, y0, cw, ch = crop
    up = lambda a: np.repeat(np.repeat(a, 2, axis=0), 2, axis=1)[:H, :W]
    mask = np.zeros((H, W), np.uint8)
    mask[10:30, 60:80] = 1
    first = oracle.compute_depth_multires(cams, 0, fl, fc, p_lo, dict(p_hi, filter_before_merge=1), crop, imgs, mask)
    after = oracle.compute_depth_multires(cams, 0, fl, fc, p_lo, p_hi, crop, imgs, mask)
    # the half-resolution pass on its own, filtered with its own thresholds
    lo = oracle.compute_depth([oracle.camera_half(c) for c in cams], 0, fl, p_lo, [oracle.downsample2(im) for im in imgs])
    outside = np.ones((H, W), bool)
    outside[y0:y0 + ch, x0:x0 + cw] = False
    free = mask == 0
    # outside the crop: the filtered half-resolution map, upsampled (then the mask)
    assert np.array_equal(first["depth"][outside & free], up(lo["depth"])[outside & free])
    assert not ((first["kbest"][outside] >= 0) & ((first["kbest"][outside] >> 14) == 1)).any()
    assert (first["depth"][mask != 0] == 0).all() and (first["reason"][mask != 0] != 0).all()
    # inside: a surviving full-resolution estimate wins; where it was filtered a surviving half-resolution one fills in
    hi_valid = (first["hi"]["valid"] != 0)
    inside = ~outside & free
    assert np.array_equal(first["depth"][inside & hi_valid], first["hi"]["depth"][inside & hi_valid])
    fill = inside & ~hi_valid & (up(lo["depth"]) > 0)
    assert fill.any() and np.array_equal(first["depth"][fill], up(lo["depth"])[fill])
    assert ((first["kbest"][fill] >> 14) == 0).all()
    # filtering first can only keep more: every pixel valid under merge-then-filter with the SAME thresholds for both
    # passes stays valid when each pass is filtered with those thresholds first
    p_same_lo = dict(p_lo, alpha_upper=p_hi["alpha_upper"], alpha_lower=p_hi["alpha_lower"], beta=p_hi["beta"], horizon_row=p_hi["horizon_row"] // 2)
    a = oracle.compute_depth_multires(cams, 0, fl, fc, p_same_lo, p_hi, crop, imgs)
    f = oracle.compute_depth_multires(cams, 0, fl, fc, p_same_lo, dict(p_hi, filter_before_merge=1), crop, imgs)
    assert not ((a["valid"] != 0) & (f["valid"] == 0)).any() and (f["valid"] != 0).sum() >= (a["valid"] != 0).sum()
    # limiting cases: (i) thresholds that reject every full-resolution estimate -> the filtered half-resolution map
    none_hi = dict(p_hi, alpha_upper=-1.0, alpha_lower=-1.0, filter_before_merge=1)
    r = oracle.compute_depth_multires(cams, 0, fl, fc, p_lo, none_hi, crop, imgs)
    assert np.array_equal(r["depth"], up(lo["depth"]))
    # (ii) no filters at all: both orders are the plain merge
    off_lo, off_hi = dict(p_lo, filters=0), dict(p_hi, filters=0)
    r1 = oracle.compute_depth_multires(cams, 0, fl, fc, off_lo, off_hi, crop, imgs)
    r2 = oracle.compute_depth_multires(cams, 0, fl, fc, off_lo, dict(off_hi, filter_before_merge=1), crop, imgs)
    for key in ("depth", "c1", "c2", "kbest", "reason"):
        assert np.array_equal(r1[key], r2[key]), key
    assert after["n_eval"] == first["n_eval"]


def test_plane_consistent_upsampling_puts_the_points_on_the_chosen_plane():
    cams, imgs, fl, fc, p_lo, p_hi, crop = _multires_setup()
    H, W = imgs[0].shape
    off = dict(filters=0)
    copy = oracle.compute_depth_multires(cams, 0, fl, fc, dict(p_lo, **off), dict(p_hi, **off), crop, imgs)
    plane = oracle.compute_depth_multires(cams, 0, fl, fc, dict(p_lo, **off), dict(p_hi, upsample_plane=1, **off), crop, imgs)
    lo = plane["lo"]
    s_lo, d_lo, f_lo, n_fam = oracle.plane_table(fl)
    from_lo = (plane["kbest"] >= 0) & ((plane["kbest"] >> 14) == 0)
    assert from_lo.sum() > 500
    # costs, index and the pixels supplied by the crop pass are untouched
    for key in ("c1", "c2", "kbest"):
        assert np.array_equal(copy[key], plane[key]), key
    hi_px = (plane["kbest"] >> 14) == 1
    assert np.array_equal(copy["depth"][hi_px], plane["depth"][hi_px])
    n_checked, off_plane_copy = 0, 0
    for y, x in list(zip(*np.nonzero(from_lo & (plane["reason"] == 0))))[::7]:
        yl, xl = y >> 1, x >> 1
        k = lo["kbest"][yl, xl]
        sk = s_lo[k] + lo["delta"][yl, xl] * ((s_lo[k + 1] - s_lo[k]) if lo["delta"][yl, xl] != 0 else 0.0)
        d_star = 1.0 / sk
        r = oracle.back_project(cams[0], x, y)
        X = plane["depth"][y, x] * r                               # the reconstructed point (range along the unit ray)
        assert abs(n_fam[f_lo[k]] @ X - d_star) < 1e-9 * d_star    # lies on the refined plane of the half-res pixel
        Xc = copy["depth"][y, x] * r
        off_plane_copy += abs(n_fam[f_lo[k]] @ Xc - d_star) > 1e-6 * d_star
        n_checked += 1
    assert n_checked > 50 and off_plane_copy > 0.5 * n_checked     # the copied ranges do not have that property
    # the four children of a half-resolution pixel share one plane: their z-depths agree (fronto-parallel family)
    zmap = oracle.compute_depth_multires(cams, 0, fl, fc, dict(p_lo, **off), dict(p_hi, upsample_plane=1, depth_kind=1, **off), crop, imgs)
    blocks = 0
    for yl in range(2, H // 2 - 2, 3):
        for xl in range(2, W // 2 - 2, 5):
            blk = (slice(2 * yl, 2 * yl + 2), slice(2 * xl, 2 * xl + 2))
            if from_lo[blk].all() and (zmap["reason"][blk] == 0).all():
                assert np.ptp(zmap["depth"][blk]) < 1e-9 * zmap["depth"][blk].max()
                blocks += 1
    assert blocks > 20
