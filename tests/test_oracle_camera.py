"""Pins for the oracle's camera model and plane-induced warp (O1-O4).

Each test checks oracle/ against something other than itself: values printed in
SPEC.md / SURVEY.md (tests/golden), closed forms (pinhole, stereographic, homography),
invariants (unit norm, round trip, scale invariance), and the synthetic generator's
independently written camera simulator.
"""
import math
import os

import numpy as np
import pytest

import oracle
import synth
from conftest import read_golden

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def cam(**kw):
    base = dict(width=1024, height=544, fx=400.0, fy=400.0, cx=512.0, cy=272.0, xi=1.0, fov_max_deg=360.0)
    base.update(kw)
    return base


def test_spec_printed_examples():
    g = read_golden(os.path.join(GOLD, "spec_examples.txt"))
    uv = oracle.project(cam(xi=0.0), [1, 0, 1])
    assert np.allclose(uv, g["project_pinhole_example"], atol=1e-9)
    uv = oracle.project(cam(xi=1.0), [1, 0, 1])
    assert abs(uv[0] - g["project_xi1_example"][0]) < 0.005 and abs(uv[1] - 272) < 1e-9  # printed to 2 decimals
    # closed form of the same example: x/|X| = 1/sqrt2, denominator 1/sqrt2 + 1
    assert abs(uv[0] - (400.0 * (1 / math.sqrt(2)) / (1 / math.sqrt(2) + 1) + 512.0)) < 1e-9
    for xi in (0.0, 0.5, 1.0, 1.7):
        assert np.allclose(oracle.back_project(cam(xi=xi), 512, 272), g["backproject_principal"], atol=1e-12)
        assert np.allclose(oracle.project(cam(xi=xi), [0, 0, 5]), [512, 272], atol=1e-12)


def test_pinhole_reduction():
    c = cam(xi=0.0)
    rng = np.random.default_rng(0)
    for _ in range(50):
        u, v = rng.uniform(0, 1023), rng.uniform(0, 543)
        x, y = (u - 512) / 400, (v - 272) / 400
        expect = np.array([x, y, 1.0]) / math.sqrt(x * x + y * y + 1)
        assert np.allclose(oracle.back_project(c, u, v), expect, atol=1e-12)
        X = rng.uniform(-3, 3, 3)
        X[2] = abs(X[2]) + 0.5
        assert np.allclose(oracle.project(c, X), [400 * X[0] / X[2] + 512, 400 * X[1] / X[2] + 272], atol=1e-9)


def test_stereographic_closed_form():
    """xi = 1: theta = 2 atan(rho)."""
    c = cam(xi=1.0)
    for rho in (0.0, 0.1, 0.5, 0.9, 1.0):
        r = oracle.back_project(c, 512 + 400 * rho, 272)
        theta = math.atan2(math.hypot(r[0], r[1]), r[2])
        assert abs(theta - 2 * math.atan(rho)) < 1e-12


def test_eq1_unit_norm_and_roundtrip():
    rng = np.random.default_rng(1)
    cams = [cam(xi=0.9), cam(xi=1.0, k1=-0.05, fx=350, fy=350, cx=640, cy=512, width=1280, height=1024, fov_max_deg=185),
            cam(xi=1.2, k1=-0.03, k2=0.002, p1=0.001, p2=-0.0015, fov_max_deg=170), cam(xi=0.0, k1=0.02)]
    for c in cams:
        n_ok = 0
        for _ in range(200):
            u, v = rng.uniform(0, c["width"] - 1), rng.uniform(0, c["height"] - 1)
            r = oracle.back_project(c, u, v)
            if r is None:
                continue
            n_ok += 1
            assert abs(np.linalg.norm(r) - 1) < 1e-12
            for lam in (0.11, 3.7, 250.0):
                uv = oracle.project(c, lam * r)
                assert uv is not None and np.hypot(uv[0] - u, uv[1] - v) < 1e-5
        assert n_ok > 20


def test_projection_scale_invariance_and_fov():
    c = cam(xi=1.0, k1=-0.05, fov_max_deg=185)
    X = np.array([0.4, -0.2, 0.7])
    assert np.allclose(oracle.project(c, X), oracle.project(c, 17.0 * X), atol=1e-9)
    # theta just inside / outside 92.5 degrees
    for th, ok in ((92.4, True), (92.6, False)):
        t = math.radians(th)
        assert (oracle.project(c, [math.sin(t), 0, math.cos(t)]) is not None) == ok
    # pixel outside the FOV circle is NONE in back-projection too
    g = read_golden(os.path.join(GOLD, "survey_spot_values.txt"))
    c3 = synth.make_config(3)["cams"][0]
    radius = g["c3_circle_radius"][0]
    assert oracle.back_project(c3, 640 + radius - 1.0, 512) is not None
    assert oracle.back_project(c3, 640 + radius + 1.0, 512) is None
    assert oracle.back_project(c3, 0, 0) is None  # beyond the invertible range of the k1 polynomial


def test_c3_infov_pixel_count():
    g = read_golden(os.path.join(GOLD, "survey_spot_values.txt"))
    c3 = oracle.make_camera(synth.make_config(3)["cams"][0])
    # radius of the theta_max circle by bisection on the oracle itself, then count lattice points (independent of FOV code)
    lo, hi = 300.0, 400.0
    for _ in range(60):
        mid = 0.5 * (lo + hi)
        if oracle.back_project(c3, 640 + mid, 512) is not None:
            lo = mid
        else:
            hi = mid
    assert abs(lo - g["c3_circle_radius"][0]) < 0.06
    yy, xx = np.mgrid[0:1024, 0:1280]
    count = int(((xx - 640.0) ** 2 + (yy - 512.0) ** 2 <= lo * lo).sum())
    assert count == int(g["c3_infov_pixels"][0])


def test_synth_camera_simulator_agrees():
    """The generator's independently written ray function must agree with the oracle's Eq. 1 (cross pin)."""
    rng = np.random.default_rng(2)
    for idx in (1, 2, 3):
        cfg = synth.make_config(idx)
        for c in cfg["cams"][:1]:
            for _ in range(300):
                u, v = rng.uniform(0, c["width"] - 1), rng.uniform(0, c["height"] - 1)
                a, b = synth.pixel_ray(c, u, v), oracle.back_project(c, u, v)
                assert (a is None) == (b is None)
                if a is not None:
                    assert np.allclose(a, b, atol=1e-12)
    c = cam(xi=1.2, k1=-0.03, k2=0.002, p1=0.001, p2=-0.0015, fov_max_deg=170)
    for _ in range(200):
        u, v = rng.uniform(0, 1023), rng.uniform(0, 543)
        a, b = synth.pixel_ray(c, u, v), oracle.back_project(c, u, v)
        assert (a is None) == (b is None)
        if a is not None:
            assert np.allclose(a, b, atol=1e-11)


def test_relative_pose_and_se3():
    cfg = synth.make_config(2)
    ref, left, right = cfg["cams"]
    R, T = oracle.relative_pose(ref, right)
    # right camera centre is (0.4,0,0) in the ref frame: it must map to the origin of the view frame
    assert np.allclose(R @ np.array([0.4, 0, 0]) + T, 0, atol=1e-12)
    assert np.allclose(R @ R.T, np.eye(3), atol=1e-12) and abs(np.linalg.det(R) - 1) < 1e-12
    # yaw +10 deg turns the optical axis toward +x: the view's z axis expressed in the ref frame
    axis = R.T @ np.array([0, 0, 1.0])
    assert abs(axis[0] - math.sin(math.radians(10))) < 1e-12 and abs(axis[2] - math.cos(math.radians(10))) < 1e-12
    R2, T2 = oracle.relative_pose(ref, ref)
    assert np.allclose(R2, np.eye(3)) and np.allclose(T2, 0)


def test_survey_spot_values():
    g = read_golden(os.path.join(GOLD, "survey_spot_values.txt"))
    c1 = synth.make_config(1)
    s, d, f, n = oracle.plane_table(c1["families"])
    assert abs((s[0] - s[1]) - g["c1_planes"][0]) < 1e-6
    assert np.allclose([d[0], d[27], d[28], d[31]], g["c1_planes"][1:], rtol=2e-6)
    r = oracle.back_project(c1["cams"][0], 40, 20)
    assert np.allclose(r, g["c1_ray_40_20"], atol=1e-6)
    assert abs(d[27] / r[2] - g["c1_range_k27"][0]) < 1e-5
    uv = oracle.warp_pixel(c1["cams"][0], c1["cams"][1], [0, 0, 1], d[27], 100.0, 40, 20)
    assert np.allclose(uv, g["c1_warp_k27"], atol=1e-5)
    c3 = synth.make_config(3)["cams"]
    r = oracle.back_project(c3[0], 800, 600)
    assert np.allclose(r, g["c3_ray_800_600"], atol=1e-6)
    assert abs(math.degrees(math.acos(r[2])) - g["c3_theta_deg"][0]) < 1e-3
    assert abs(10.0 / r[2] - g["c3_range_d10"][0]) < 1e-5
    assert np.allclose(oracle.warp_pixel(c3[0], c3[2], [0, 0, 1], 10.0, 100.0, 800, 600), g["c3_warp_d10_right"], atol=1e-5)
    r = oracle.back_project(c3[0], 800, 800)
    assert abs(1.6 / r[1] - g["c3_range_ground"][0]) < 1e-5
    assert np.allclose(oracle.warp_pixel(c3[0], c3[2], [0, 1, 0], 1.6, 100.0, 800, 800), g["c3_warp_ground_right"], atol=1e-5)


def test_plane_table_examples():
    g = read_golden(os.path.join(GOLD, "spec_examples.txt"))
    s, d, f, n = oracle.plane_table([synth.family((0, 0, 1), 2, 2.0, 60.0, "inverse")])
    assert np.allclose(d, g["planes_two"])
    s, d, f, n = oracle.plane_table([synth.family((0, 0, 2), 64, 0.5, 50, "inverse"), synth.family((0, 3, 0), 30, 1.1, 2.1, "linear")])
    assert len(d) == int(g["planes_paper_total"][0])
    assert np.allclose(n, [[0, 0, 1], [0, 1, 0]])
    assert np.allclose(np.diff(1 / d[:64]), np.diff(1 / d[:64])[0]) and np.allclose(np.diff(d[64:]), 1.0 / 29)
    assert list(f[:64]) == [0] * 64 and list(f[64:]) == [1] * 30
    s, d, f, n = oracle.plane_table([synth.family((0, 1, 0), 3, 1.1, 2.1, "linear")])
    assert np.allclose(d, [1.1, 1.6, 2.1])  # SPEC.md:186 band of +-0.5 m around the estimate


def test_warp_identity_and_translation():
    c = cam(xi=0.9, width=200, height=160, fx=80, fy=80, cx=100, cy=80, fov_max_deg=200)
    # identity pose, same camera: warp(p) = p for every plane with positive intersection depth
    for (u, v) in ((40, 50), (100, 80), (150.5, 33.25)):
        for d in (0.7, 5.0, 40.0):
            assert np.allclose(oracle.warp_pixel(c, c, [0, 0, 1], d, 1e3, u, v), [u, v], atol=1e-9)
    # ray parallel to / facing away from the plane -> NONE
    assert oracle.warp_pixel(c, c, [0, -1, 0], 1.0, 1e3, 100, 120) is None
    # pinhole, pure x translation, fronto plane: u' = u - fx b / d
    p = cam(xi=0.0, width=200, height=160, fx=80, fy=80, cx=100, cy=80)
    q = dict(p)
    q["R"], q["t"] = np.eye(3), -np.array([0.25, 0, 0])
    for d in (2.0, 8.0):
        uv = oracle.warp_pixel(p, q, [0, 0, 1], d, 1e3, 120, 70)
        assert np.allclose(uv, [120 - 80 * 0.25 / d, 70], atol=1e-10)
    # beyond range_max -> NONE
    assert oracle.warp_pixel(p, q, [0, 0, 1], 50.0, 40.0, 120, 70) is None


def test_warp_equals_homography_for_pinhole():
    """xi = 0, no distortion: the mapping is the homography K_v (R + T n^T / d) K_ref^-1."""
    rng = np.random.default_rng(3)
    ref = cam(xi=0.0, width=320, height=240, fx=210, fy=200, cx=158, cy=121)
    view = cam(xi=0.0, width=320, height=240, fx=190, fy=205, cx=163, cy=118)
    ang = 0.12
    Rv = np.array([[math.cos(ang), 0, -math.sin(ang)], [0, 1, 0], [math.sin(ang), 0, math.cos(ang)]]) @ \
        np.array([[1, 0, 0], [0, math.cos(0.05), -math.sin(0.05)], [0, math.sin(0.05), math.cos(0.05)]])
    view["R"], view["t"] = Rv, np.array([-0.3, 0.05, 0.1])
    ref["R"], ref["t"] = np.eye(3), np.zeros(3)
    K = lambda c: np.array([[c["fx"], 0, c["cx"]], [0, c["fy"], c["cy"]], [0, 0, 1.0]])
    for n, d in (((0, 0, 1), 4.0), ((0, 0.6, 0.8), 3.0), ((0, 1, 0), 1.5)):
        n = np.array(n, dtype=float)
        Hm = K(view) @ (Rv + np.outer(view["t"], n) / d) @ np.linalg.inv(K(ref))
        hits = 0
        for _ in range(100):
            u, v = rng.uniform(0, 319), rng.uniform(0, 239)
            uv = oracle.warp_pixel(ref, view, n, d, 1e3, u, v)
            h = Hm @ np.array([u, v, 1.0])
            if uv is not None:
                hits += 1
                assert np.allclose(uv, h[:2] / h[2], atol=1e-8)
        assert hits > 10


def test_ray_homography_identity():
    """X' is proportional to R r + T (n.r)/d for fisheye cameras too, i.e. the warp only needs rays."""
    cfg = synth.make_config(2)
    ref, _, right = cfg["cams"]
    R, T = oracle.relative_pose(ref, right)
    n, d = np.array([0, 0, 1.0]), 6.0
    for (u, v) in ((100, 90), (200, 150), (160, 128)):
        r = oracle.back_project(ref, u, v)
        Xp = R @ r + T * (n @ r) / d
        assert np.allclose(oracle.project(right, Xp), oracle.warp_pixel(ref, right, n, d, 1e3, u, v), atol=1e-9)
