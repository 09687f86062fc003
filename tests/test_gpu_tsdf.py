"""-m gpu: the TSDF consumer (fsw_tsdf_*) against its oracle on the same seeded inputs.

Gates: allocated blocks equal except where a segment sample lies within 1e-4 block edges of a block face (flagged by the
oracle); observation counts w(X) bit-exact and D(X) within 1e-4 on voxels the oracle does not flag (a nearest-pixel
rounding, the eta >= -mu test or a field-of-view test closer to its threshold than float arithmetic resolves);
per-block observation counts equal on blocks without flagged voxels; extracted points matched to the oracle's within
1 mm.  Ground-truth range maps of the generator's ray caster are the depth input (the sweep's own maps in the last test).
"""
import math

import numpy as np
import pytest

import oracle
import oracle.tsdf as OT
import synth

pytestmark = pytest.mark.gpu

# the ABI takes voxel size and truncation distance as floats: the oracle gets the same (float-rounded) values, or the
# number of segment samples n = ceil(2 mu / (edge / 2)) of reading T2 can differ where that ratio is an integer
VS, MU = float(np.float32(0.05)), float(np.float32(0.2))
OFFSET = np.array([0.137, 0.093, 0.211])


def _yaw(deg):
    a = math.radians(deg)
    return np.array([[math.cos(a), 0.0, -math.sin(a)], [0.0, 1.0, 0.0], [math.sin(a), 0.0, math.cos(a)]])


def _frames():
    """three poses of a fisheye camera in a box scene, with the generator's exact ranges as depth maps"""
    cam = synth.camera(width=160, height=120, fx=55.0, fy=55.0, cx=79.6, cy=60.3, xi=0.9, k1=-0.03, fov_max_deg=170.0)
    scene = synth.scene_boxes(seed=21, n_boxes=12)
    out = []
    for C, yaw in (((0.0, 0.0, 0.0), 0.0), ((0.25, -0.05, 0.4), 12.0), ((-0.3, 0.05, 0.8), -9.0)):
        c = dict(cam, R=_yaw(yaw), t=-_yaw(yaw) @ np.array(C))
        img, rng = synth.render_camera(c, scene, want_range=True)
        d = np.where((rng > 0) & (rng < 12.0), rng, 0.0).astype(np.float32)
        # the map frame is the scene frame moved by OFFSET, so that the axis-aligned faces of the scene (the ground
        # at y = 1.6 m = 4 block edges) do not lie exactly on block faces, where every block would be a fragile one
        out.append((dict(c, t=-_yaw(yaw) @ (np.array(C) + OFFSET)), d))
    return cam, out


def test_allocate_integrate_extract_against_oracle():
    import torch
    from paper_1809_06132_b200.tsdf import TsdfVolume
    cam, frames = _frames()
    centre, size = tuple(np.array([0.0, 0.0, 3.0]) + OFFSET), (8.0, 4.0, 8.0)
    vol = TsdfVolume(VS, MU, 100, size, centre)
    b0, nb = vol.box()
    assert (b0, nb) == OT.box_for(centre, size, VS)
    ref = OT.Volume(VS, MU, 100, b0, nb)
    frag_b = np.zeros(ref.allocated.size, np.uint8)
    frag_v = np.zeros(ref.D.size, np.uint8)
    for c, d in frames:
        vol.integrate(c, c["R"], c["t"], torch.from_numpy(d).cuda())
        st = vol.stats()
        n_new, fb = ref.allocate(c, c["R"], c["t"], d, want_fragile=True)
        n_upd, fv = ref.integrate(c, c["R"], c["t"], d, want_fragile=True)
        frag_b |= fb
        frag_v |= fv
        assert abs(st["n_new_blocks"] - n_new) <= max(2, fb.sum()) and st["n_visible_blocks"] >= st["n_new_blocks"] > 0
        # a flagged block may exist on one side only: the voxel counts differ by what those blocks hold
        assert abs(st["n_voxels_updated"] - n_upd) <= 0.002 * n_upd + frag_v.sum() + 512 * int(fb.sum())
    D, Wt, obs, alloc = vol.download()
    rD, rW, robs, ralloc = ref.dense()
    fb3 = frag_b.reshape(alloc.shape) != 0
    assert ralloc.sum() > 400 and not ((alloc != ralloc) & ~fb3).any()          # allocation: equal off the flagged blocks
    both = (alloc != 0) & (ralloc != 0)
    up = lambda a: np.repeat(np.repeat(np.repeat(a, 8, axis=0), 8, axis=1), 8, axis=2)
    nbx, nby, nbz = nb
    fv3 = frag_v.reshape(nbz, nby, nbx, 8, 8, 8).transpose(0, 3, 1, 4, 2, 5).reshape(D.shape) != 0
    ok = up(both & ~fb3) & ~fv3        # a flagged block may have been allocated a frame earlier on one side
    assert ok.sum() > 100000 and (rW[ok] > 0).sum() > 50000
    bad = ok & (Wt != rW.astype(np.float32))
    print("tsdf parity: %d voxels compared, %d weight mismatches, flagged voxels %.4f, flagged blocks %.4f" % (
        ok.sum(), bad.sum(), fv3.mean(), fb3.mean()))
    assert np.array_equal(Wt[ok], rW[ok].astype(np.float32))                   # observation counts: exact
    assert np.abs(D[ok] - rD[ok]).max() <= 1e-4 and np.abs(D).max() <= 1.0
    # per-block observation counts: a block counts a frame when any of its voxels was updated, so the two sides may
    # differ only in a block that holds a flagged voxel (almost every block holds one after three frames), and rarely
    has_flag = fv3.reshape(nbz, 8, nby, 8, nbx, 8).any(axis=(1, 3, 5))
    cmp_blocks = both & ~fb3
    differ = cmp_blocks & (obs != robs)
    assert cmp_blocks.sum() > 300 and robs[cmp_blocks].max() == 3 and not (differ & ~has_flag).any()
    assert differ.sum() <= 0.01 * cmp_blocks.sum()
    assert fv3.mean() < 0.005 and fb3.mean() < 0.02                               # the flags excuse little
    # points of the map: "at least 3 observations"
    from scipy.spatial import cKDTree
    for min_obs in (3, 1):
        pts, n = vol.extract_points(min_obs)
        rp, rn = ref.extract(min_obs)
        origin = np.array(b0) * 8 * VS
        assert rn > 200 and abs(n - rn) <= 0.02 * rn
        dist, _ = cKDTree(rp - origin).query(pts.cpu().numpy())
        assert (dist < 1e-3).mean() > 0.98
    assert vol.extract_points(3)[1] < vol.extract_points(1)[1]
    # every extracted point lies within mu of a surface the generator reports (the input ranges are exact)
    vol.close()


def test_recentre_frees_the_blocks_that_leave_and_keeps_the_rest():
    import torch
    from paper_1809_06132_b200.tsdf import TsdfVolume
    cam, frames = _frames()
    centre, size = tuple(np.array([0.0, 0.0, 3.0]) + OFFSET), (8.0, 4.0, 8.0)
    vol = TsdfVolume(VS, MU, 100, size, centre)
    for c, d in frames[:2]:
        vol.integrate(c, c["R"], c["t"], torch.from_numpy(d).cuda())
    D0, W0, obs0, al0 = vol.download()
    b0, nb = vol.box()
    shift = 3                                              # blocks along +x
    vol.recentre((centre[0] + shift * 8 * VS, centre[1], centre[2]))
    b1, _ = vol.box()
    assert b1 == [b0[0] + shift, b0[1], b0[2]]
    assert vol.stats()["n_blocks_freed"] == int(al0[:, :, :shift].sum()) > 0
    D1, W1, obs1, al1 = vol.download()
    assert np.array_equal(al1[:, :, :-shift], al0[:, :, shift:]) and not al1[:, :, -shift:].any()
    assert np.array_equal(D1[:, :, :-8 * shift], D0[:, :, 8 * shift:]) and np.array_equal(W1[:, :, :-8 * shift], W0[:, :, 8 * shift:])
    assert np.array_equal(obs1[:, :, :-shift], obs0[:, :, shift:])
    # integrating again allocates fresh (cleared) blocks in the slots that were freed, and matches an oracle that
    # carries the kept content over
    c, d = frames[2]
    vol.integrate(c, c["R"], c["t"], torch.from_numpy(d).cuda())
    ref = OT.Volume(VS, MU, 100, b1, nb)
    nbx, nby, nbz = nb
    def block_major(a):   # [nz*8, ny*8, nx*8] -> flat block-major
        return a.reshape(nbz, 8, nby, 8, nbx, 8).transpose(0, 2, 4, 1, 3, 5).reshape(-1)
    ref.allocated[:] = al1.reshape(-1)
    ref.D[:] = block_major(D1.astype(np.float64))
    ref.W[:] = block_major(W1.astype(np.float64))
    ref.obs[:] = obs1.reshape(-1)
    _, fb = ref.allocate(c, c["R"], c["t"], d, want_fragile=True)
    _, fv = ref.integrate(c, c["R"], c["t"], d, want_fragile=True)
    D2, W2, obs2, al2 = vol.download()
    rD, rW, robs, ralloc = ref.dense()
    fb3 = fb.reshape(al2.shape) != 0
    assert not ((al2 != ralloc) & ~fb3).any()
    fv3 = fv.reshape(nbz, nby, nbx, 8, 8, 8).transpose(0, 3, 1, 4, 2, 5).reshape(D2.shape) != 0
    up = lambda a: np.repeat(np.repeat(np.repeat(a, 8, axis=0), 8, axis=1), 8, axis=2)
    ok = up((al2 != 0) & (ralloc != 0) & ~fb3) & ~fv3
    assert np.array_equal(W2[ok], rW[ok].astype(np.float32)) and np.abs(D2[ok] - rD[ok]).max() <= 1e-4
    vol.close()


def test_paper_scale_local_map_fed_by_the_sweep():
    """The pipeline of PAPER.md:65-67 on one device: the depth map the sweep kernel wrote (C3, filters on) goes straight
    into a 60 m x 60 m x 3.2 m local map at 0.05 m (180 000 blocks, 737 MB); sizes, counters and timing only."""
    import torch
    import paper_1809_06132_b200 as fsw
    from paper_1809_06132_b200.tsdf import TsdfVolume
    cfg = synth.make_config(3)
    images = synth.render_frame(cfg, 0)
    rig = fsw.Rig(cfg["cams"], 0)
    ctx = fsw.Context(rig, 0)
    planes = fsw.PlaneSet(cfg["families"])
    out = ctx.compute_depth(planes, cfg["params"], [torch.from_numpy(im).cuda() for im in images])
    ref_cam = cfg["cams"][0]
    # the rig frame has y down: a box of 60 x 3.2 x 60 m (x, y = height, z) around the vehicle
    vol = TsdfVolume(0.05, 0.2, 100, (60.0, 3.2, 60.0), (0.0, 0.0, 0.0))
    assert vol.box()[1] == [150, 8, 150]
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    vol.integrate(ref_cam, ref_cam["R"], ref_cam["t"], out["depth"])
    torch.cuda.synchronize()
    ev0.record()
    for _ in range(5):
        vol.integrate(ref_cam, ref_cam["R"], ref_cam["t"], out["depth"])
    ev1.record()
    torch.cuda.synchronize()
    st = vol.stats()
    ms = ev0.elapsed_time(ev1) / 5
    n_valid = int((out["depth"] > 0).sum())
    print("tsdf: %d valid depths -> %d blocks, %d voxels updated per frame, %.3f ms per frame (%.1f GB/s of block traffic)" % (
        n_valid, st["n_visible_blocks"], st["n_voxels_updated"], ms, st["n_visible_blocks"] * 8192 / ms / 1e6))
    assert st["n_frames"] == 6 and st["n_new_blocks"] == 0 and 1000 < st["n_visible_blocks"] < 180000
    assert st["n_voxels_updated"] > 10 * st["n_visible_blocks"]
    pts, n = vol.extract_points(3)
    assert n > 1000
    vol.close()
