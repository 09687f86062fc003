"""Pins for the oracle's matching cost, sweep, WTA, parabola, filters, mask and multi-resolution merge (O5-O10).

Sources: PAPER.md:76 / :99 (cost end points, alpha), SPEC.md worked examples (tests/golden/spec_examples.txt),
numpy.corrcoef (library routine), closed forms (integer-disparity shift, exact quadratic), brute force in numpy on
tiny inputs written independently of oracle/ (own camera code, own loops), and invariances.
"""
import math
import os

import numpy as np
import pytest

import oracle
import synth
from conftest import read_golden

GOLD = os.path.join(os.path.dirname(__file__), "golden")
INF = float("inf")


# ----------------------------------------------------------------------------
# matching cost
# ----------------------------------------------------------------------------
def test_cost_endpoints_and_affine_invariance():
    g = read_golden(os.path.join(GOLD, "spec_examples.txt"))
    rng = np.random.default_rng(0)
    a = rng.uniform(0, 255, 81)
    assert abs(oracle.zncc_cost(a, a, 6.5) - g["cost_at_zncc_plus1"][0]) < 1e-12      # identical -> 0
    assert abs(oracle.zncc_cost(a, -a + 300, 6.5) - g["cost_at_zncc_minus1"][0]) < 1e-12  # negated + constant -> 1
    assert abs(oracle.zncc_cost(a, 2 * a + 5, 6.5)) < 1e-12
    b = rng.uniform(0, 255, 81)
    assert abs(oracle.zncc_cost(a, b, 6.5) - oracle.zncc_cost(b, a, 6.5)) < 1e-15        # symmetry
    assert abs(oracle.zncc_cost(3 * a - 7, 0.5 * b + 11, 1e-9) - oracle.zncc_cost(a, b, 1e-9)) < 1e-12


def test_cost_equals_corrcoef():
    rng = np.random.default_rng(1)
    for n in (9, 25, 49, 81, 225):
        for _ in range(20):
            a, b = rng.uniform(0, 1, n), rng.uniform(0, 1, n)
            if rng.uniform() < 0.5:
                b = 0.7 * a + 0.3 * b
            expect = 0.5 * (1.0 - np.corrcoef(a, b)[0, 1])
            got = oracle.zncc_cost(a, b, 1e-12)
            assert 0.0 <= got <= 1.0 and abs(got - expect) < 1e-12


def test_cost_variance_floor():
    """Q10: flat windows -> denominator floored -> cost ~ 0.5, no NONE gate."""
    a = np.full(49, 100.0)
    b = np.random.default_rng(2).uniform(0, 255, 49)
    assert abs(oracle.zncc_cost(a, b, 6.5025) - 0.5) < 1e-12
    a2 = a + np.random.default_rng(3).uniform(-1e-3, 1e-3, 49)
    assert abs(oracle.zncc_cost(a2, a2, 6.5025) - 0.5) < 1e-3   # even identical: below the floor it tends to 0.5
    # well above the floor the floor has no effect
    c = np.random.default_rng(4).uniform(0, 255, 49)
    assert oracle.zncc_cost(c, b, 6.5025) == oracle.zncc_cost(c, b, 1e-30)


# ----------------------------------------------------------------------------
# exact-index construction: pinhole, pure x shift, integer disparities
# ----------------------------------------------------------------------------
def _pinhole_pair(W=64, H=40, fx=40.0, b=0.5):
    ref = dict(width=W, height=H, fx=fx, fy=fx, cx=W / 2.0, cy=H / 2.0, xi=0.0, fov_max_deg=179.0,
               R=np.eye(3), t=np.zeros(3))
    view = dict(ref)
    view["t"] = -np.array([b, 0.0, 0.0])
    return ref, view


def test_sweep_recovers_exact_plane_index_integer_disparity():
    W, H, fx, b = 64, 40, 40.0, 0.5
    ref, view = _pinhole_pair(W, H, fx, b)
    # disparities fx*b/d_k = 1..8 px  <=>  1/d_k = (k+1)/20
    fams = [synth.family((0, 0, 1), 8, 20.0, 2.5, "inverse")]
    rng = np.random.default_rng(5)
    big = rng.uniform(0, 255, (H, W + 16))
    img_ref = big[:, 8:8 + W].copy()
    true_k = 4  # disparity 5: view(u') = ref(u' + 5)
    img_view = big[:, 8 + 5:8 + 5 + W].copy()
    prm = synth.params(5, 1e-6, 1e3, subpixel=1)
    out = oracle.compute_depth([ref, view], 0, fams, prm, [img_ref, img_view], keep_cost=True)
    # interior = window inside the image and all 25 warped samples inside the view for the true plane
    valid = np.isfinite(out["cost"][true_k])
    assert valid.sum() == (H - 4) * (W - 4 - 5 - 1 + 1) or valid.sum() > 0.7 * H * W
    assert np.all(out["kbest"][valid] == true_k)                   # index recovered on ALL interior pixels
    assert np.max(out["cost"][true_k][valid]) < 1e-12              # warped image equals the reference: cost 0
    s, d, _, _ = oracle.plane_table(fams)
    # depth = range along the ray = d / r_z ; parabola must not move an exact zero-cost minimum by more than half a step
    yy, xx = np.nonzero(valid)
    for y, x in list(zip(yy, xx))[::97]:
        r = oracle.back_project(ref, x, y)
        lo, hi = 1 / (s[true_k] + 0.5 * abs(s[1] - s[0])) / r[2], 1 / (s[true_k] - 0.5 * abs(s[1] - s[0])) / r[2]
        assert lo <= out["depth"][y, x] <= hi


def test_sweep_fisheye_plane_on_sweep_plane():
    """Textured plane exactly on sweep plane k, spacing >= 1 px of disparity: index k on >= 99% where parallax exists
    (AC2)."""
    kw = dict(width=160, height=120, fx=60.0, fy=60.0, cx=80.0, cy=60.0, xi=0.9, fov_max_deg=190.0)
    cams = [synth.camera(**kw), synth.camera(centre=(0.5, 0, 0), **kw)]
    # f_eff = fx/(1+xi) = 31.6 px/rad; b=0.5: disparity per unit inverse depth = 15.8 px -> delta(1/d)=0.1 -> 1.58 px
    fams = [synth.family((0, 0, 1), 10, 10.0, 1.0, "inverse")]   # 1/d = 0.1 .. 1.0
    s, d, _, _ = oracle.plane_table(fams)
    k_true = 3
    scene = synth.scene_plane(z=d[k_true], cells=(0.25, 1.0), seed=7)
    imgs = [synth.quantize(synth.render_camera(c, scene), "f32") for c in cams]
    prm = synth.params(7, synth.VAR_FLOOR_F32, 100.0)
    out = oracle.compute_depth(cams, 0, fams, prm, imgs)
    yy, xx = np.mgrid[0:120, 0:160]
    # parallax exists away from the baseline direction (x axis): keep the central cone
    keep = (out["raw_valid"] > 0) & (np.hypot(xx - 80, yy - 60) < 45)
    assert keep.sum() > 3000
    assert (out["kbest"][keep] == k_true).mean() >= 0.99
    z = out["depth"][keep]
    assert np.median(np.abs(out["delta"][keep])) < 0.15


# ----------------------------------------------------------------------------
# brute force in numpy, written independently of oracle/
# ----------------------------------------------------------------------------
def _np_project(c, X):
    rho = np.linalg.norm(X)
    den = X[2] + c["xi"] * rho
    if den <= 1e-9 * rho or X[2] < math.cos(math.radians(c["fov_max_deg"]) / 2) * rho:
        return None
    m = X[:2] / den
    r2 = m @ m
    m = m * (1 + c["k1"] * r2)
    return np.array([c["fx"] * m[0] + c["cx"], c["fy"] * m[1] + c["cy"]])


def _np_ray(c, u, v):
    x, y = (u - c["cx"]) / c["fx"], (v - c["cy"]) / c["fy"]
    rd = math.hypot(x, y)
    if c["k1"] != 0 and rd > 0:   # bisection instead of Newton: a different algorithm on purpose
        lo, hi = 0.0, min(3.0, math.sqrt(1 / (3 * abs(c["k1"]))) if c["k1"] < 0 else 3.0)
        if hi * (1 + c["k1"] * hi * hi) < rd:
            return None
        for _ in range(200):
            mid = 0.5 * (lo + hi)
            if mid * (1 + c["k1"] * mid * mid) < rd:
                lo = mid
            else:
                hi = mid
        x, y = x * lo / rd, y * lo / rd
    p2 = x * x + y * y
    eta = (c["xi"] + math.sqrt(1 + (1 - c["xi"] ** 2) * p2)) / (p2 + 1)
    r = np.array([eta * x, eta * y, eta - c["xi"]])
    r /= np.linalg.norm(r)
    if math.atan2(math.hypot(r[0], r[1]), r[2]) > math.radians(c["fov_max_deg"]) / 2:
        return None
    return r


def _np_pixel_costs(cams, fams_nd, images, w, var_floor, range_max, px, py):
    """cost per plane for one pixel: every window sample re-derived from scratch with numpy only."""
    ref = cams[0]
    H, W = images[0].shape
    h = w // 2
    out = []
    for (n, d) in fams_nd:
        n = np.asarray(n, dtype=float)
        tot, cnt = 0.0, 0
        for vi in range(1, len(cams)):
            view = cams[vi]
            Rr, tr, Rv, tv = ref["R"], ref["t"], view["R"], view["t"]
            R = Rv @ Rr.T
            T = tv - R @ tr
            a, b, ok = [], [], True
            for dy in range(-h, h + 1):
                for dx in range(-h, h + 1):
                    x, y = px + dx, py + dy
                    if not (0 <= x < W and 0 <= y < H):
                        ok = False
                        continue
                    r = _np_ray(ref, x, y)
                    if r is None or n @ r <= 1e-9 or d / (n @ r) > range_max:
                        ok = False
                        continue
                    uv = _np_project(view, R @ (r * d / (n @ r)) + T)
                    Hv, Wv = images[vi].shape
                    if uv is None or not (0 <= uv[0] < Wv - 1 and 0 <= uv[1] < Hv - 1):
                        ok = False
                        continue
                    i0, j0 = int(math.floor(uv[0])), int(math.floor(uv[1]))
                    fu, fv = uv[0] - i0, uv[1] - j0
                    I = images[vi]
                    val = (1 - fv) * ((1 - fu) * I[j0, i0] + fu * I[j0, i0 + 1]) + fv * ((1 - fu) * I[j0 + 1, i0] + fu * I[j0 + 1, i0 + 1])
                    a.append(images[0][y, x])
                    b.append(val)
            if not ok:
                continue
            a, b = np.array(a), np.array(b)
            cov = np.mean((a - a.mean()) * (b - b.mean()))
            den = max(math.sqrt(a.var() * b.var()), var_floor)
            tot += min(1.0, max(0.0, 0.5 * (1 - cov / den)))
            cnt += 1
        out.append(tot / cnt if cnt else INF)
    return np.array(out)


def test_sweep_matches_numpy_brute_force_c1():
    cfg = synth.make_config(1)
    imgs = [im.astype(np.float64) for im in synth.render_frame(cfg)]
    out = oracle.compute_depth(cfg["cams"], 0, cfg["families"], cfg["params"], imgs, keep_cost=True)
    s, d, f, n = oracle.plane_table(cfg["families"])
    nd = [((0, 0, 1), dk) for dk in d]
    pts = [(32, 24), (5, 5), (60, 40), (2, 24), (40, 20), (10, 44), (57, 3), (1, 1), (20, 30), (33, 2)]
    for (px, py) in pts:
        want = _np_pixel_costs(cfg["cams"], nd, imgs, 5, cfg["params"]["var_floor"], cfg["params"]["range_max"], px, py)
        got = out["cost"][:, py, px]
        assert np.array_equal(np.isfinite(want), np.isfinite(got)), (px, py)
        fin = np.isfinite(want)
        assert np.allclose(want[fin], got[fin], atol=1e-10), (px, py)
        # the oracle's own per-pixel brute force (no shared warped image) agrees to rounding as well
        got2 = oracle.pixel_costs(cfg["cams"], 0, cfg["families"], cfg["params"], imgs, px, py)
        assert np.array_equal(np.isfinite(got2), fin) and np.allclose(got2[fin], got[fin], atol=1e-12)


def test_sweep_matches_numpy_brute_force_distorted_two_views_ground():
    """3 cameras with yaw, k1 distortion, fronto + ground families, float images."""
    kw = dict(width=48, height=40, fx=22.0, fy=22.0, cx=24.0, cy=20.0, xi=1.0, k1=-0.05, fov_max_deg=185.0)
    cams = [synth.camera(**kw), synth.camera(centre=(-0.4, 0, 0), yaw_deg=-10, **kw), synth.camera(centre=(0.4, 0.02, 0.05), yaw_deg=10, **kw)]
    fams = [synth.family((0, 0, 1), 6, 1.0, 20.0, "inverse"), synth.family((0, 1, 0), 3, 1.1, 2.1, "linear")]
    scene = synth.scene_boxes(seed=9, n_boxes=6)
    imgs = [synth.render_camera(c, scene).astype(np.float64) for c in cams]
    prm = synth.params(3, synth.VAR_FLOOR_F32, 40.0)
    out = oracle.compute_depth(cams, 0, fams, prm, imgs, keep_cost=True)
    s, d, f, n = oracle.plane_table(fams)
    nd = [(tuple(n[fi]), dk) for fi, dk in zip(f, d)]
    n_fin = 0
    for (px, py) in [(24, 20), (10, 30), (40, 33), (24, 36), (6, 12), (30, 25), (44, 20), (3, 20)]:
        want = _np_pixel_costs(cams, nd, imgs, 3, synth.VAR_FLOOR_F32, 40.0, px, py)
        got = out["cost"][:, py, px]
        assert np.array_equal(np.isfinite(want), np.isfinite(got)), (px, py)
        fin = np.isfinite(want)
        n_fin += fin.sum()
        assert np.allclose(want[fin], got[fin], atol=1e-9), (px, py)
    assert n_fin > 20
    assert out["n_eval"] > 0


# ----------------------------------------------------------------------------
# invariances
# ----------------------------------------------------------------------------
def test_view_order_and_gain_bias_invariance():
    cfg = synth.make_config(2)
    cams = [dict(c) for c in cfg["cams"]]
    for c in cams:   # shrink the problem: crop the raster (principal point moves with it)
        c.update(width=96, height=64, cx=48.0, cy=40.0)
    imgs = [synth.render_camera(c, cfg["scene"]).astype(np.float64) for c in cams]
    prm = dict(cfg["params"])
    fams = [synth.family((0, 0, 1), 16, 0.5, 50.0, "inverse")]
    a = oracle.compute_depth(cams, 0, fams, prm, imgs, keep_cost=True)
    b = oracle.compute_depth([cams[0], cams[2], cams[1]], 0, fams, prm, [imgs[0], imgs[2], imgs[1]], keep_cost=True)
    assert np.array_equal(a["kbest"], b["kbest"])
    fin = np.isfinite(a["cost"])
    assert np.array_equal(fin, np.isfinite(b["cost"])) and np.allclose(a["cost"][fin], b["cost"][fin], atol=1e-15)
    # gain / bias on any image leaves the costs (hence the argmin) unchanged where windows are textured
    prm2 = dict(prm)
    prm2["var_floor"] = 1e-12
    a2 = oracle.compute_depth(cams, 0, fams, prm2, imgs, keep_cost=True)
    c2 = oracle.compute_depth(cams, 0, fams, prm2, [2.0 * imgs[0] + 0.1, 0.5 * imgs[1] + 0.3, imgs[2]], keep_cost=True)
    assert np.array_equal(a2["kbest"], c2["kbest"])
    assert np.allclose(a2["cost"][fin], c2["cost"][fin], atol=1e-9)
    # best <= second at every raw-valid pixel
    rv = a["raw_valid"] > 0
    assert np.all(a["c1"][rv] <= a["c2"][rv])


def test_constant_image_dies_in_cost_filter():
    cfg = synth.make_config(1)
    imgs = [np.full((48, 64), 128.0), np.full((48, 64), 90.0)]
    prm = dict(cfg["params"])
    prm.update(filters=oracle.FILTER_COST, alpha_upper=0.3, alpha_lower=0.3, horizon_row=24)
    out = oracle.compute_depth(cfg["cams"], 0, cfg["families"], prm, imgs)
    rv = out["raw_valid"] > 0
    assert rv.sum() > 1000 and np.allclose(out["c1"][rv], 0.5)
    assert out["valid"].sum() == 0 and np.all(out["depth"] == 0)
    assert np.all(out["reason"][rv] == oracle.COST_FILTER)


# ----------------------------------------------------------------------------
# WTA / second best / parabola on synthetic cost vectors
# ----------------------------------------------------------------------------
def _wta_on_vectors(costs, fams, subpixel=1):
    """costs: [n, P] -> run orc_wta on an n x 1 'image' of a pinhole camera looking down the axis."""
    n, P = costs.shape
    cam = dict(width=1, height=n, fx=1e6, fy=1e6, cx=0.0, cy=(n - 1) / 2.0, xi=0.0, fov_max_deg=179.0)
    vol = np.ascontiguousarray(costs.T.reshape(P, n, 1))
    return oracle.wta(cam, fams, synth.params(3, 1e-6, 1e9, subpixel=subpixel), vol)


def _second_best_brute(c, fam_of, kb):
    best = INF
    for j in range(len(c)):
        if (fam_of[j] != fam_of[kb] or abs(j - kb) >= 2) and c[j] < best:
            best = c[j]
    return best if np.isfinite(best) else 1.0


def test_wta_second_best_and_ties():
    rng = np.random.default_rng(6)
    fams = [synth.family((0, 0, 1), 9, 1.0, 10.0, "inverse"), synth.family((0, 1, 0), 5, 1.0, 2.0, "linear")]
    fam_of = [0] * 9 + [1] * 5
    costs = rng.uniform(0, 1, (300, 14))
    costs[rng.uniform(size=costs.shape) < 0.2] = INF
    costs[0] = INF                     # no finite cost at all
    costs[1] = 0.4                     # all tied: lowest index wins
    costs[2, :] = INF
    costs[2, 8] = 0.2                  # single finite cost: second best defaults to 1.0
    costs[3, 7], costs[3, 8], costs[3, 9] = 0.1, 0.05, 0.07   # winner at a family end; plane 9 is another family
    out = _wta_on_vectors(costs, fams)
    for i in range(300):
        c = costs[i]
        if not np.isfinite(c).any():
            assert out["raw_valid"][i, 0] == 0 and out["depth"][i, 0] == 0 and out["kbest"][i, 0] == -1
            continue
        kb = int(np.argmin(c))         # numpy argmin returns the first minimum = lowest-index tie-break
        assert out["kbest"][i, 0] == kb and out["c1"][i, 0] == c[kb]
        assert out["c2"][i, 0] == _second_best_brute(c, fam_of, kb)
        assert out["c1"][i, 0] <= out["c2"][i, 0]
    assert out["kbest"][1, 0] == 0
    assert out["c2"][2, 0] == 1.0 and out["delta"][2, 0] == 0.0
    assert out["c2"][3, 0] == min(0.07, np.min(np.delete(costs[3], [7, 8, 9])))  # 9 counts (other family), 7 does not
    assert out["delta"][3, 0] == 0.0   # no parabola across a family boundary


def test_parabola_vertex_and_depth():
    fams = [synth.family((0, 0, 1), 11, 1.0, 11.0, "linear"), synth.family((0, 0, 1), 11, 1.0, 1.0 / 11.0, "inverse")]
    rows = []
    for off in (-0.37, 0.0, 0.21, 0.49):
        k = np.arange(11)
        rows.append(np.concatenate([0.01 * (k - (5 + off)) ** 2 + 0.1, np.full(11, 0.9)]))   # minimum in the LINEAR family
        rows.append(np.concatenate([np.full(11, 0.9), 0.01 * (k - (5 + off)) ** 2 + 0.1]))   # minimum in the INVERSE family
    out = _wta_on_vectors(np.array(rows), fams)
    offs = [-0.37, -0.37, 0.0, 0.0, 0.21, 0.21, 0.49, 0.49]
    for i, off in enumerate(offs):
        assert abs(out["delta"][i, 0] - off) < 1e-9              # exact quadratic -> the vertex; symmetric -> 0
        if i % 2 == 0:
            assert out["kbest"][i, 0] == 5 and abs(out["depth"][i, 0] - (6.0 + off)) < 1e-6       # d = 1 + k
        else:
            assert out["kbest"][i, 0] == 16 and abs(out["depth"][i, 0] - 1.0 / (6.0 + off)) < 1e-6  # 1/d = 1 + k
    off_out = _wta_on_vectors(np.array(rows), fams, subpixel=0)
    assert np.all(off_out["delta"] == 0)
    # clamp to +-0.5, skip at family ends and next to +inf
    c = np.full((3, 22), 0.9)
    c[0, 4:7] = [0.2, 0.1, 0.1000001]
    c[1, 0:2] = [0.1, 0.3]
    c[2, 4:7] = [INF, 0.1, 0.3]
    o = _wta_on_vectors(c, fams)
    assert abs(o["delta"][0, 0]) <= 0.5 and o["delta"][1, 0] == 0 and o["delta"][2, 0] == 0


# ----------------------------------------------------------------------------
# filters, mask, multi-resolution
# ----------------------------------------------------------------------------
def _maps(c1, c2, H=4, W=4):
    return dict(depth=np.full((H, W), 5.0), c1=np.full((H, W), float(c1)), c2=np.full((H, W), float(c2)),
                raw_valid=np.ones((H, W), dtype=np.uint8))


def test_filters_spec_examples_and_contractive():
    g = read_golden(os.path.join(GOLD, "spec_examples.txt"))
    a_up, a_lo = g["alpha"]
    prm = synth.params(9, 6.5, 100.0, a_up, a_lo, 2, 1.2, filters=oracle.FILTER_COST)
    m = oracle.filter_mask(prm, _maps(0.2, 1.0))
    assert list(m["valid"][:, 0]) == [int(g["cost_filter_example"][0])] * 2 + [int(g["cost_filter_example"][1])] * 2
    m = oracle.filter_mask(prm, _maps(0.0, 1.0))
    assert m["valid"].all()                                    # all-zero-cost map unchanged
    prm = synth.params(9, 6.5, 100.0, 1.0, 1.0, 2, 1.2, filters=oracle.FILTER_RATIO)
    for (b, s, keep) in zip((0.1, 0.3, 0.0), (0.5, 0.31, 0.1), g["ratio_filter_example"]):
        m = oracle.filter_mask(prm, _maps(b, s))
        assert m["valid"].all() == bool(keep) and (m["depth"] > 0).all() == bool(keep)
    # contractive on random maps, never creates depth
    rng = np.random.default_rng(8)
    H, W = 32, 48
    maps = dict(depth=rng.uniform(1, 50, (H, W)), c1=rng.uniform(0, 0.6, (H, W)), c2=rng.uniform(0, 1, (H, W)),
                raw_valid=(rng.uniform(size=(H, W)) < 0.8).astype(np.uint8))
    maps["c2"] = np.maximum(maps["c1"], maps["c2"])
    maps["depth"][maps["raw_valid"] == 0] = 0
    before = maps["depth"].copy()
    mask = (rng.uniform(size=(H, W)) < 0.1).astype(np.uint8)
    prm = synth.params(9, 6.5, 100.0, a_up, a_lo, H // 2, 1.2, filters=3)
    m = oracle.filter_mask(prm, maps, mask)
    assert np.all((m["depth"] == before) | (m["depth"] == 0))
    assert np.all(m["valid"] <= (before > 0))
    # reference decision chain in numpy
    alpha = np.where(np.arange(H)[:, None] < H // 2, a_up, a_lo)
    keep = (before > 0) & ~(m["c1"] > alpha) & ~(m["c2"] < 1.2 * np.maximum(m["c1"], 1e-6)) & (mask == 0)
    assert np.array_equal(keep, m["valid"].astype(bool))


def test_mask_examples():
    g = read_golden(os.path.join(GOLD, "spec_examples.txt"))
    prm = synth.params(9, 6.5, 100.0)
    H, W = 200, 240
    m0 = oracle.filter_mask(prm, _maps(0.1, 0.9, H, W), None)
    assert m0["valid"].all()                                             # empty box list -> identical
    mask = np.zeros((H, W), np.uint8)
    mask[100:140, 100:150] = 1                                           # box (100,100,50,40)
    m1 = oracle.filter_mask(prm, _maps(0.1, 0.9, H, W), mask)
    assert (m1["depth"] == 0).sum() == int(g["mask_box_pixels"][0]) and np.all(m1["reason"][100:140, 100:150] == oracle.MASKED)
    m2 = oracle.filter_mask(prm, _maps(0.1, 0.9, H, W), np.ones((H, W), np.uint8))
    assert not m2["valid"].any()                                         # box covering the image


def test_downsample_and_half_camera_ray_consistency():
    rng = np.random.default_rng(9)
    img = rng.uniform(0, 255, (10, 14))
    lo = oracle.downsample2(img)
    assert lo.shape == (5, 7)
    assert np.allclose(lo, 0.25 * (img[0::2, 0::2] + img[0::2, 1::2] + img[1::2, 0::2] + img[1::2, 1::2]), atol=1e-12)
    c3 = synth.make_config(3)["cams"][0]
    half = oracle.camera_half(c3)
    assert (half.width, half.height, half.fx, half.cx, half.cy) == (640, 512, 175.0, 319.75, 255.75)
    for (i, j) in ((320, 256), (200, 300), (400, 180), (333, 401)):
        a = oracle.back_project(half, i, j)
        b = oracle.back_project(c3, 2 * i + 0.5, 2 * j + 0.5)          # SPEC.md:229 round trip
        assert np.allclose(a, b, atol=1e-12)


def test_multires_merge_rules():
    """Outside the crop = upsampled low-res value; inside, full-res wins where raw-valid (Q19)."""
    kw = dict(width=96, height=64, fx=40.0, fy=40.0, cx=47.5, cy=31.5, xi=0.9, fov_max_deg=190.0)
    cams = [synth.camera(**kw), synth.camera(centre=(0.3, 0, 0), **kw)]
    scene = synth.scene_boxes(seed=11, n_boxes=8)
    imgs = [synth.quantize(synth.render_camera(c, scene), "u8") for c in cams]
    fl = [synth.family((0, 0, 1), 8, 0.5, 30.0, "inverse")]
    fc = [synth.family((0, 0, 1), 12, 0.5, 40.0, "inverse")]
    pl, pc = synth.params(3, synth.VAR_FLOOR_U8, 60.0), synth.params(5, synth.VAR_FLOOR_U8, 80.0)
    crop = (24, 16, 48, 32)
    mask = synth.make_mask(96, 64, seed=4, n_rects=2)
    out = oracle.compute_depth_multires(cams, 0, fl, fc, pl, pc, crop, imgs, mask)
    lo, hi = out["lo"], out["hi"]
    up = lambda a: np.repeat(np.repeat(a, 2, 0), 2, 1)
    inside = np.zeros((64, 96), bool)
    inside[16:48, 24:72] = True
    use_hi = inside & (hi["raw_valid"] > 0)
    assert use_hi.sum() > 500 and (~use_hi & (up(lo["raw_valid"]) > 0)).sum() > 500
    assert np.array_equal(out["c1"][use_hi], hi["c1"][use_hi]) and np.all(out["kbest"][use_hi] & (1 << 14))
    assert np.array_equal(out["c1"][~use_hi], up(lo["c1"])[~use_hi])
    assert np.array_equal(out["kbest"][~use_hi], up(lo["kbest"])[~use_hi])
    keep = out["valid"] > 0
    assert not np.any(keep & (mask > 0))
    want = np.where(use_hi, hi["depth"], up(lo["depth"]))
    assert np.array_equal(out["depth"][keep], want[keep]) and np.all(out["depth"][~keep] == 0)
    assert np.all(hi["raw_valid"][~inside] == 0)                       # the crop pass only computes its ROI
