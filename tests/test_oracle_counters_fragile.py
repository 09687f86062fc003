"""Pins of the oracle's by-products (run with -m "not gpu"): the N_eval counter and the fragile maps.

N_eval is the unit the roofline credits ((pixel, plane, view) triples with a finite per-view
cost) and the gate the kernel's own counter is held to; the fragile maps decide which pixels the
validity gate excuses.  Neither is compared with itself here: the counter is held to a numpy brute force, to the
finite entries of the cost volume, to additivity over views and to the surveyor's printed C1 counts
(tests/golden/survey_spot_values.txt); the flags are held to what they promise -- a threshold or a geometric limit
moved by less than its epsilon may change the verdict of flagged pixels only -- and to an upper bound on how many pixels
they may excuse.
"""
import math
import os

import numpy as np

import oracle
import oracle.compare
import synth
from conftest import read_golden
from test_oracle_sweep import _np_project, _np_ray

GOLD = os.path.join(os.path.dirname(__file__), "golden")


# ----------------------------------------------------------------------------------------------------------------------
# N_eval
# ----------------------------------------------------------------------------------------------------------------------
def _np_valid_views(cams, fams_nd, shapes, w, range_max, px, py):
    """Number of views whose whole w x w window around (px, py) maps into the view, per plane; numpy only, written
    independently of oracle/ (bisection undistortion from test_oracle_sweep)."""
    ref = cams[0]
    H, W = shapes[0]
    h = w // 2
    out = []
    for (n, d) in fams_nd:
        n = np.asarray(n, dtype=float)
        cnt = 0
        for vi in range(1, len(cams)):
            view = cams[vi]
            R = view["R"] @ ref["R"].T
            T = view["t"] - R @ ref["t"]
            ok = True
            for dy in range(-h, h + 1):
                for dx in range(-h, h + 1):
                    x, y = px + dx, py + dy
                    if not (0 <= x < W and 0 <= y < H):
                        ok = False
                        break
                    r = _np_ray(ref, x, y)
                    if r is None or n @ r <= 1e-9 or d / (n @ r) > range_max:
                        ok = False
                        break
                    uv = _np_project(view, R @ (r * d / (n @ r)) + T)
                    Hv, Wv = shapes[vi]
                    if uv is None or not (0 <= uv[0] < Wv - 1 and 0 <= uv[1] < Hv - 1):
                        ok = False
                        break
                if not ok:
                    break
            cnt += 1 if ok else 0
        out.append(cnt)
    return np.array(out)


def _tiny_three_camera_rig():
    kw = dict(width=26, height=20, fx=12.0, fy=12.0, cx=13.0, cy=10.0, xi=1.0, k1=-0.05, fov_max_deg=185.0)
    cams = [synth.camera(**kw), synth.camera(centre=(-0.4, 0, 0), yaw_deg=-10, **kw),
            synth.camera(centre=(0.4, 0.02, 0.05), yaw_deg=10, **kw)]
    fams = [synth.family((0, 0, 1), 4, 1.0, 20.0, "inverse"), synth.family((0, 1, 0), 2, 1.1, 2.1, "linear")]
    scene = synth.scene_boxes(seed=9, n_boxes=6)
    imgs = [synth.render_camera(c, scene).astype(np.float64) for c in cams]
    return cams, fams, imgs, synth.params(3, synth.VAR_FLOOR_F32, 40.0)


def test_n_eval_equals_numpy_brute_force_count_on_a_tiny_rig():
    cams, fams, imgs, prm = _tiny_three_camera_rig()
    out = oracle.compute_depth(cams, 0, fams, prm, imgs, keep_cost=True)
    s, d, f, n = oracle.plane_table(fams)
    nd = [(tuple(n[fi]), dk) for fi, dk in zip(f, d)]
    shapes = [im.shape for im in imgs]
    total = 0
    H, W = shapes[0]
    for py in range(H):
        for px in range(W):
            cnt = _np_valid_views(cams, nd, shapes, 3, 40.0, px, py)
            total += int(cnt.sum())
            # a plane has a finite averaged cost exactly when at least one view counted
            assert np.array_equal(cnt > 0, np.isfinite(out["cost"][:, py, px])), (px, py)
    assert total > 500
    assert out["n_eval"] == total


def test_n_eval_is_the_finite_entries_with_one_view_and_additive_over_views():
    # one matching view: every finite entry of the cost volume is exactly one evaluation
    cfg = synth.make_config(1)
    imgs = synth.render_frame(cfg)
    out = oracle.compute_depth(cfg["cams"], 0, cfg["families"], cfg["params"], imgs, keep_cost=True)
    assert out["n_eval"] == int(np.isfinite(out["cost"]).sum())
    # several views: the count of the rig is the sum of the counts of its two-camera sub-rigs (a finite per-view cost
    # does not depend on the other views), and lies between the finite entries and views x finite entries
    cams, fams, imgs, prm = _tiny_three_camera_rig()
    both = oracle.compute_depth(cams, 0, fams, prm, imgs, keep_cost=True)
    parts = [oracle.compute_depth([cams[0], cams[v]], 0, fams, prm, [imgs[0], imgs[v]], keep_cost=True) for v in (1, 2)]
    assert both["n_eval"] == parts[0]["n_eval"] + parts[1]["n_eval"]
    fin = int(np.isfinite(both["cost"]).sum())
    assert fin <= both["n_eval"] <= 2 * fin
    assert fin == int((np.isfinite(parts[0]["cost"]) | np.isfinite(parts[1]["cost"])).sum())
    # the region of interest restricts the outputs that are counted, not the windows
    roi = dict(prm, roi=(5, 4, 9, 7))
    sub = oracle.compute_depth(cams, 0, fams, roi, imgs, keep_cost=True)
    views = np.isfinite(parts[0]["cost"]).astype(int) + np.isfinite(parts[1]["cost"]).astype(int)
    assert sub["n_eval"] == int(views[:, 4:11, 5:14].sum())


def test_c1_counts_printed_by_the_surveyor():
    """tests/golden/survey_spot_values.txt (SURVEY.md 8(c) row "planes", 8(d) row C1): 2867 of the 3072 pixels of C1
    have r_z > 0, and 2361 are raw-valid with the 5 x 5 window (geometry only: independent of the texture)."""
    g = read_golden(os.path.join(GOLD, "survey_spot_values.txt"))
    cfg = synth.make_config(1)
    ref = cfg["cams"][0]
    rz_pos = 0
    for y in range(ref["height"]):
        for x in range(ref["width"]):
            r = oracle.back_project(ref, x, y)
            rz_pos += 1 if (r is not None and r[2] > 0) else 0
    assert rz_pos == int(g["c1_rz_positive"][0])
    out = oracle.compute_depth(cfg["cams"], 0, cfg["families"], cfg["params"], synth.render_frame(cfg), keep_cost=True)
    assert int(out["raw_valid"].sum()) == int(g["c1_raw_valid"][0])
    # every raw-valid pixel has r_z > 0 (fronto-parallel planes only) and at least one counted evaluation
    assert out["n_eval"] >= int(out["raw_valid"].sum())


# ----------------------------------------------------------------------------------------------------------------------
# fragile maps
# ----------------------------------------------------------------------------------------------------------------------
def _random_maps(seed, H=60, W=80):
    rng = np.random.default_rng(seed)
    c1 = rng.uniform(0.0, 0.6, (H, W))
    c2 = c1 * rng.uniform(0.9, 1.6, (H, W))
    # populate the neighbourhood of the thresholds densely so that flips do occur
    c1[::3, ::2] = 0.3 + rng.uniform(-5e-4, 5e-4, c1[::3, ::2].shape)
    c2[1::3, ::2] = 1.2 * np.maximum(c1[1::3, ::2], 1e-6) + rng.uniform(-8e-4, 8e-4, c2[1::3, ::2].shape)
    raw = (rng.uniform(size=(H, W)) > 0.1).astype(np.uint8)
    return dict(depth=np.where(raw != 0, 5.0, 0.0), c1=c1, c2=c2, raw_valid=raw)


def _verdict(maps, prm):
    m = {k: v.copy() for k, v in maps.items()}
    oracle.filter_mask(prm, m)
    return m["reason"], m["fragile_thr"] != 0


def test_threshold_flags_cover_every_verdict_a_small_threshold_move_can_flip_and_not_much_more():
    """O10: |c1 - alpha| < 2e-4 and |c2 - beta c1| < 3e-4 are flagged.  Moving alpha by less than 2e-4, or beta so that
    beta * c1 moves by less than 3e-4, may change the verdict of flagged pixels only; and the flags stay confined to
    the pixels inside those margins (an over-eager flag would hollow out the validity gate)."""
    prm = synth.params(5, 1.0, 50.0, 0.3, 0.3, 30, 1.2, filters=3)
    n_flip = 0
    for seed in range(4):
        maps = _random_maps(seed)
        base, flagged = _verdict(maps, prm)
        for da in (-1.9e-4, 1.9e-4):
            moved, _ = _verdict(maps, dict(prm, alpha_upper=0.3 + da, alpha_lower=0.3 + da))
            diff = moved != base
            n_flip += int(diff.sum())
            assert not (diff & ~flagged).any()
        for db in (-4e-4, 4e-4):   # c1 <= 0.6: beta * c1 moves by at most 2.4e-4 < 3e-4
            moved, _ = _verdict(maps, dict(prm, beta=1.2 + db))
            diff = moved != base
            n_flip += int(diff.sum())
            assert not (diff & ~flagged).any()
        # a move beyond the margin does flip unflagged pixels: the margins are not vacuous
        far, _ = _verdict(maps, dict(prm, alpha_upper=0.3 + 4e-3, alpha_lower=0.3 + 4e-3))
        assert ((far != base) & ~flagged).any()
        # confinement: nothing outside the margins is flagged, nothing raw-invalid is flagged
        raw = maps["raw_valid"] != 0
        inside = (np.abs(maps["c1"] - 0.3) < 2e-4) | (np.abs(maps["c2"] - 1.2 * np.maximum(maps["c1"], 1e-6)) < 3e-4)
        assert not (flagged & ~(inside & raw)).any()
        assert flagged.mean() < 0.25
    assert n_flip > 20
    # filters off: nothing is flagged
    _, none = _verdict(_random_maps(9), dict(prm, filters=0))
    assert not none.any()


def _finite_pattern(cams, fams, prm, imgs):
    cost, n_eval, frag = oracle.sweep(cams, 0, fams, prm, imgs)
    return np.isfinite(cost), frag != 0


def test_geometric_flags_cover_every_validity_a_small_geometric_move_can_flip():
    """O10: a window sample within 1e-3 px of a view image border, within 1e-5 rad of a field-of-view limit, or a
    range within 1e-6 (relative) of range_max flags the pixel.  Three rigs are built so that one sample sits inside
    one of those margins; moving the limit by less than the margin must flip that sample's validity, and may change
    which (pixel, plane) costs are finite at flagged pixels only."""
    kw = dict(width=44, height=36, fx=17.0, fy=17.0, cx=21.7, cy=18.2, xi=0.95, k1=-0.03, fov_max_deg=160.0)
    cams = [synth.camera(**kw), synth.camera(centre=(0.35, 0.0, 0.0), yaw_deg=6, **kw),
            synth.camera(centre=(-0.3, 0.05, 0.02), yaw_deg=-4, **kw)]
    fams = [synth.family((0, 0, 1), 10, 0.6, 12.0, "inverse"), synth.family((0, 1, 0), 3, 1.0, 2.0, "linear")]
    scene = synth.scene_boxes(seed=4, n_boxes=5)
    imgs = [synth.render_camera(c, scene).astype(np.float64) for c in cams]
    prm = synth.params(3, synth.VAR_FLOOR_U8, 40.0)
    s, d, f, n = oracle.plane_table(fams)
    px, py, k = 30, 21, 6
    r = oracle.back_project(cams[0], px, py)
    t0 = d[k] / r[2]                                         # range of pixel (30,21) to fronto plane 6
    cases = []   # (base cameras, base params, [(moved cameras, moved params)], validity of the constructed sample)
    nrm = (0, 0, 1)
    # (a) range cap 3e-7 (relative) beyond that range; moved by -+0.9e-6
    near = dict(prm, range_max=t0 * (1.0 + 3e-7))
    cases.append((cams, near, [(cams, dict(near, range_max=near["range_max"] * (1.0 + m))) for m in (-0.9e-6, 0.9e-6)],
                  lambda c, q: oracle.warp_pixel(c[0], c[1], nrm, d[k], q["range_max"], px, py) is not None))
    # (b) field of view of view 1 ends 3e-6 rad beyond the direction of that sample; moved by -+0.9e-5 rad
    R, T = oracle.relative_pose(cams[0], cams[1])
    Xv = R @ (t0 * r) + T
    th = math.atan2(math.hypot(Xv[0], Xv[1]), Xv[2])
    fov = lambda half: [cams[0], dict(cams[1], fov_max_deg=2.0 * math.degrees(half)), cams[2]]
    cases.append((fov(th + 3e-6), prm, [(fov(th + 3e-6 + m), prm) for m in (-0.9e-5, 0.9e-5)],
                  lambda c, q: oracle.warp_pixel(c[0], c[1], nrm, d[k], q["range_max"], px, py) is not None))
    # (c) principal point of view 2 shifted so that the sample lands 3e-4 px inside the last admissible column
    #     (u' = W - 1 - 3e-4: the projection is linear in cx); moved by -+0.9e-3 px
    uv = oracle.warp_pixel(cams[0], cams[2], nrm, d[k], 40.0, px, py)
    assert uv is not None
    shift = (cams[2]["width"] - 1 - 3e-4) - uv[0]
    col = lambda dx: [cams[0], cams[1], dict(cams[2], cx=cams[2]["cx"] + shift + dx)]
    cases.append((col(0.0), prm, [(col(m), prm) for m in (-0.9e-3, 0.9e-3)],
                  lambda c, q: oracle.warp_pixel(c[0], c[2], nrm, d[k], q["range_max"], px, py) is not None))
    n_diff = 0
    for base_cams, base_prm, moves, sample_ok in cases:
        base, flagged = _finite_pattern(base_cams, fams, base_prm, imgs)
        assert flagged[py, px] and base.any() and flagged.mean() < 0.5
        assert sample_ok(base_cams, base_prm)
        assert [sample_ok(mc, mp) for mc, mp in moves].count(False) == 1     # one of the two moves crosses the limit
        for mc, mp in moves:
            moved, _ = _finite_pattern(mc, fams, mp, imgs)
            diff = (moved != base).any(axis=0)
            n_diff += int(diff.sum())
            assert not (diff & ~flagged).any()
    assert n_diff > 0
    # a larger move reaches unflagged pixels: the flags are not simply "everything that can ever change"
    base, flagged = _finite_pattern(cams, fams, dict(prm, range_max=t0), imgs)
    far, _ = _finite_pattern(cams, fams, dict(prm, range_max=t0 * 1.2), imgs)
    assert ((far != base).any(axis=0) & ~flagged).any()


def test_compare_counts_ties_and_fragile_pixels_as_documented():
    """oracle/compare.py: a differing index is excused only when it is a tie in the ORACLE's cost vector (2e-4); a
    validity mismatch is excused only on pixels the oracle flags (geometry, thresholds, argmin ties)."""
    cfg = synth.make_config(1)
    p = dict(cfg["params"], alpha_upper=0.3, alpha_lower=0.3, beta=1.2, filters=3, horizon_row=24)
    ref = oracle.compute_depth(cfg["cams"], 0, cfg["families"], p, synth.render_frame(cfg), keep_cost=True)

    def as_test(r):
        return dict(depth=r["depth"].astype(np.float32), best_cost=r["c1"].astype(np.float32),
                    second_cost=r["c2"].astype(np.float32), plane_index=r["kbest"].astype(np.int16),
                    valid_reason=r["reason"].copy())

    st = oracle.compare.compare_maps(ref, as_test(ref), ref["cost"])
    assert st["index_exact_frac"] == 1.0 and st["valid_mismatch_total"] == 0 and st["max_dc2"] < 1e-6
    valid = ref["reason"] == 0
    k = ref["kbest"]
    vol = ref["cost"]
    ys, xs = np.nonzero(valid & (k > 0) & (k < vol.shape[0] - 1))
    up = vol[k[ys, xs] + 1, ys, xs] - vol[k[ys, xs], ys, xs]
    tie_px = [(y, x) for y, x, u in zip(ys, xs, up) if u <= 1e-4][:5]
    far_px = [(y, x) for y, x, u in zip(ys, xs, up) if np.isfinite(u) and u > 1e-3][:5]
    assert tie_px and far_px
    t = as_test(ref)
    for (y, x) in tie_px + far_px:
        t["plane_index"][y, x] += 1
    st = oracle.compare.compare_maps(ref, t, ref["cost"])
    n_valid = int(valid.sum())
    assert round((1.0 - st["index_exact_frac"]) * n_valid) == len(tie_px) + len(far_px)
    assert round((1.0 - st["index_match_frac"]) * n_valid) == len(far_px)     # only the ties are excused
    # validity flipped on one unflagged and one flagged pixel: only the first is counted.  An argmin tie
    # (|c1 - c2raw| < 2e-4) excuses a pixel only where the test really chose another plane.
    with np.errstate(invalid="ignore"):
        tie = (ref["raw_valid"] != 0) & (np.abs(ref["c1"] - ref["c2raw"]) < oracle.compare.TIE_TOL)
    flagged = (ref["fragile_geom"] != 0) | (ref["fragile_thr"] != 0)
    t = as_test(ref)
    y0, x0 = [int(v[0]) for v in np.nonzero(valid & ~flagged & ~tie)]
    y1, x1 = [int(v[0]) for v in np.nonzero(valid & flagged)]
    t["valid_reason"][y0, x0] = 2
    t["valid_reason"][y1, x1] = 2
    st = oracle.compare.compare_maps(ref, t, ref["cost"])
    assert st["valid_mismatch_total"] == 2 and st["valid_mismatch_nonfragile"] == 1
    assert abs(st["fragile_frac"] - flagged.mean()) < 1e-12
    ty, tx = [v[:2] for v in np.nonzero(valid & tie & ~flagged)]
    assert len(ty) == 2
    t = as_test(ref)
    t["valid_reason"][ty[0], tx[0]] = 3                       # same plane, other verdict: counted
    t["valid_reason"][ty[1], tx[1]] = 3                       # another plane at a tie, other verdict: excused
    t["plane_index"][ty[1], tx[1]] += 1 if ref["kbest"][ty[1], tx[1]] == 0 else -1
    st = oracle.compare.compare_maps(ref, t, ref["cost"])
    assert st["valid_mismatch_total"] == 2 and st["valid_mismatch_nonfragile"] == 1
    assert st["tie_frac_of_raw"] > 0.05                       # C1: about 9 % of the raw-valid pixels are ties
    # the second-best gate sees a wrong second cost on a pixel that is not a tie
    t = as_test(ref)
    t["second_cost"][y0, x0] += 5e-4
    assert oracle.compare.compare_maps(ref, t, ref["cost"])["max_dc2"] > 4e-4
