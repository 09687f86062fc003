"""Pins of the TSDF part of the oracle (oracle/fsw_tsdf_oracle.c; run with -m "not gpu").

What fixes it without the oracle's own code: the worked examples of Eq. 2 (SPEC.md integrate:
fresh voxel -> D = 1, w = 1; D = 0.5, w = 2 -> 2/3; eta = -2 mu untouched), the running-average identity and the weight
cap as a numpy recursion, the blocks of one pixel's segment against numpy sample points built with the test suite's
own ray code (bisection undistortion), a textured-free plane scene whose zero crossing must sit on the plane, and the
"at least 3 observations" gate of PAPER.md:180.
"""
import math

import numpy as np

import oracle
import oracle.tsdf as T
import synth
from test_oracle_sweep import _np_ray

VS, MU = 0.05, 0.2


def _pinhole(W=64, H=48, f=40.0):
    return dict(width=W, height=H, fx=f, fy=f, cx=W / 2.0, cy=H / 2.0, xi=0.0, k1=0.0, fov_max_deg=170.0,
                R=np.eye(3), t=np.zeros(3))


def _voxel_index(vol, X):
    """flat index of the voxel that contains the world point X"""
    v = np.floor(np.asarray(X) / VS).astype(int)
    b = v // 8
    l = v - b * 8
    s = ((b[2] - vol.b0[2]) * vol.nb[1] + (b[1] - vol.b0[1])) * vol.nb[0] + (b[0] - vol.b0[0])
    return int(s), int(s * 512 + (l[2] * 8 + l[1]) * 8 + l[0])


def test_eq2_worked_examples_and_running_average():
    cam = _pinhole()
    vol = T.Volume(VS, MU, 100, [-4, -4, 0], [8, 8, 8])
    X = np.array([0.025, 0.025, 1.025])                 # a voxel centre almost on the optical axis
    rng_x = float(np.linalg.norm(X))
    s, v = _voxel_index(vol, X)
    vol.allocated[s] = 1
    depth = np.full((48, 64), rng_x + 5 * MU)           # eta = 5 mu everywhere near the axis: clamp at 1
    n, _ = vol.integrate(cam, np.eye(3), np.zeros(3), depth)
    assert n > 0 and vol.D[v] == 1.0 and vol.W[v] == 1.0             # fresh voxel, eta >= mu -> D = 1, w = 1
    vol.D[v], vol.W[v] = 0.5, 2.0
    vol.integrate(cam, np.eye(3), np.zeros(3), depth)
    assert abs(vol.D[v] - 2.0 / 3.0) < 1e-15 and vol.W[v] == 3.0     # (2 * 0.5 + 1) / 3
    before = (vol.D[v], vol.W[v])
    vol.integrate(cam, np.eye(3), np.zeros(3), np.full((48, 64), rng_x - 2 * MU))
    assert (vol.D[v], vol.W[v]) == before                            # eta = -2 mu: untouched
    vol.integrate(cam, np.eye(3), np.zeros(3), np.full((48, 64), rng_x - 0.999 * MU))
    assert vol.W[v] == 4.0                                           # eta just above -mu: updated
    # running average of clamped samples, then the weight cap (numpy recursion)
    vol2 = T.Volume(VS, MU, 4, [-4, -4, 0], [8, 8, 8])
    vol2.allocated[s] = 1
    etas = np.array([0.5, -0.3, 2.0, 0.1, -0.9, 0.7, 0.25]) * MU
    Dn, wn, samples = 0.0, 0.0, []
    for e in etas:
        vol2.integrate(cam, np.eye(3), np.zeros(3), np.full((48, 64), rng_x + e))
        samples.append(min(1.0, e / MU))
        Dn = (wn * Dn + samples[-1]) / (wn + 1.0)
        wn = min(wn + 1.0, 4.0)
        assert abs(vol2.D[v] - Dn) < 1e-12 and vol2.W[v] == wn
        if len(samples) <= 4:
            assert abs(vol2.D[v] - np.mean(samples)) < 1e-12         # un-capped: the plain mean
        assert abs(vol2.D[v]) <= 1.0
    assert vol2.obs[s] == len(etas)


def test_allocation_is_the_blocks_of_the_sampled_segment():
    cam = dict(width=80, height=60, fx=30.0, fy=30.0, cx=39.6, cy=30.2, xi=0.9, k1=-0.03, fov_max_deg=175.0)
    yaw = math.radians(20.0)
    R = np.array([[math.cos(yaw), 0, -math.sin(yaw)], [0, 1, 0], [math.sin(yaw), 0, math.cos(yaw)]])
    C = np.array([0.3, -0.2, 0.1])
    t = -R @ C
    b0, nb = T.box_for((0, 0, 1.6), (8.0, 8.0, 6.4), VS)
    edge = 8 * VS
    multi = False
    for (px, py, d) in [(40, 30, 2.0), (58, 22, 1.3), (22, 40, 3.1), (20, 20, 0.25)]:
        vol = T.Volume(VS, MU, 100, b0, nb)
        depth = np.zeros((60, 80))
        depth[py, px] = d
        n_new, _ = vol.allocate(cam, R, t, depth)
        r = _np_ray(dict(cam, R=np.eye(3), t=np.zeros(3)), px, py)        # independent ray code (bisection)
        n = math.ceil(2 * MU / (0.5 * edge))
        want = set()
        for i in range(n + 1):
            X = R.T @ ((d - MU + i * 2 * MU / n) * r - t)
            b = np.floor(X / edge).astype(int)
            if all(b0[a] <= b[a] < b0[a] + nb[a] for a in range(3)):
                want.add(tuple(b))
        got = set()
        for s in np.nonzero(vol.allocated)[0]:
            bz, rem = divmod(int(s), nb[0] * nb[1])
            by, bx = divmod(rem, nb[0])
            got.add((bx + b0[0], by + b0[1], bz + b0[2]))
        assert got == want and n_new == len(want) and len(want) >= 1
        multi = multi or len(want) >= 2
        # every allocated block is crossed by the segment (dense sampling), and the blocks form a connected chain
        fine = {tuple(np.floor((R.T @ ((d - MU + f * 2 * MU) * r - t)) / edge).astype(int)) for f in np.linspace(0, 1, 2001)}
        assert got <= fine
    assert multi      # some segment crosses a block face
    # nothing valid -> nothing allocated; a segment wholly outside the local map -> nothing allocated
    vol = T.Volume(VS, MU, 100, b0, nb)
    assert vol.allocate(cam, R, t, np.zeros((60, 80)))[0] == 0
    far = np.zeros((60, 80))
    far[30, 40] = 30.0
    assert vol.allocate(cam, R, t, far)[0] == 0 and vol.allocated.sum() == 0


def _plane_depth(cam, R, t, z_plane):
    """range along every pixel ray to the world plane z = z_plane (0 where the ray misses it)"""
    H, W = cam["height"], cam["width"]
    d = np.zeros((H, W))
    C = -R.T @ t
    for y in range(H):
        for x in range(W):
            r = oracle.back_project(dict(cam, R=np.eye(3), t=np.zeros(3)), x, y)
            if r is None:
                continue
            rw = R.T @ r
            if rw[2] > 1e-6:
                s = (z_plane - C[2]) / rw[2]
                if 0 < s < 20:
                    d[y, x] = s
    return d


def test_plane_scene_zero_crossing_and_observation_gate():
    cam = dict(width=96, height=72, fx=40.0, fy=40.0, cx=47.5, cy=35.5, xi=0.8, k1=-0.02, fov_max_deg=150.0)
    z_plane = 2.0
    b0, nb = T.box_for((0, 0, 1.6), (4.0, 4.0, 3.2), VS)
    vol = T.Volume(VS, MU, 100, b0, nb)
    poses = [np.array([0.0, 0.0, 0.0]), np.array([0.3, 0.0, 0.0]), np.array([-0.2, 0.2, 0.1])]
    counts = []
    for C in poses:
        R, t = np.eye(3), -C
        depth = _plane_depth(cam, R, t, z_plane)
        assert (depth > 0).sum() > 2000
        vol.allocate(cam, R, t, depth)
        vol.integrate(cam, R, t, depth)
        counts.append(vol.extract(min_obs=3)[1])
    assert counts[0] == 0 and counts[1] == 0 and counts[2] > 100     # "at least 3 observations"
    D, Wt, obs, alloc = vol.dense()
    assert np.abs(D).max() <= 1.0 and Wt.max() <= 3.0
    zc = (np.arange(D.shape[0]) + b0[2] * 8 + 0.5) * VS
    seen = Wt > 0
    front = seen & (zc[:, None, None] < z_plane - 2 * VS)
    back = seen & (zc[:, None, None] > z_plane + 2 * VS)
    assert front.sum() > 1000 and back.sum() > 1000
    assert (D[front] > 0).all() and (D[back] < 0).all()              # positive outside, negative inside
    pts3, n3 = vol.extract(min_obs=3)
    pts0, n0 = vol.extract(min_obs=0)
    assert n0 >= n3 > 0
    assert np.abs(pts3[:, 2] - z_plane).max() < VS and np.sqrt(np.mean((pts3[:, 2] - z_plane) ** 2)) < VS / 2
    assert {tuple(np.round(p, 9)) for p in pts3} <= {tuple(np.round(p, 9)) for p in pts0}
