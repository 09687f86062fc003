"""Host logic of the tile schedule (S0; fsw_plan_schedule, no device): run with -m "not gpu".

What fixes the plan without the library's own code: tiles the image circle or the region of interest cannot reach carry
no weight and come last; above the horizon a ground-parallel family adds nothing, so a tile of the lower image half
weighs more than its mirror image in the upper half by about the share of ground planes; weights scale with the number
of planes; the chosen number of whole tiles is never worse, under the same list-scheduling model replayed here in
numpy, than sweeping everything whole or everything in halves; long queues are not split and keep the
centre-first order.
"""
import heapq
import math

import numpy as np
import pytest

import paper_1809_06132_b200 as fsw
import synth


def _rig_planes(idx):
    cfg = synth.make_config(idx)
    return cfg, fsw.Rig(cfg["cams"], 0), fsw.PlaneSet(cfg["families"])


def _makespan(weights, n_live, n_whole, n_sets, slots):
    """list scheduling in queue order: whole tiles, then two items of 0.6 w + 0.5 per halved tile (fsw_api.cu)"""
    load = [0.0] * slots
    heapq.heapify(load)
    items = [w for w in weights[:n_whole] for _ in range(n_sets)]
    items += [0.6 * w + 0.5 for w in weights[n_whole:n_live] for _ in range(2 * n_sets)]
    for w in items:
        heapq.heappush(load, heapq.heappop(load) + w)
    return max(load)


def test_weights_follow_the_geometry_of_config_5():
    cfg, rig, planes = _rig_planes(5)
    plan = fsw.plan_schedule(rig, planes, cfg["params"], n_sets=1, n_blocks=148)
    cam = cfg["cams"][0]
    W, H = cam["width"], cam["height"]
    tw, th = plan["tile_w"], plan["tile_h"]
    assert (tw, th) == (64, 40) and plan["n_tiles_x"] == math.ceil(W / tw) and plan["n_tiles"] == plan["n_tiles_x"] * math.ceil(H / th)
    order, weight = plan["tile_order"], plan["tile_weight"]
    assert sorted(order.tolist()) == list(range(plan["n_tiles"]))                 # a permutation of the tiles
    assert plan["by_weight"] == 1 and (np.diff(weight) <= 0).all()                # heaviest first
    assert (weight[:plan["n_live"]] > 0).all() and (weight[plan["n_live"]:] == 0).all()
    w_of = np.zeros(plan["n_tiles"])
    w_of[order] = weight
    grid = w_of.reshape(-1, plan["n_tiles_x"])
    # tiles whose nearest point (with the window's halo) is outside the image circle carry nothing
    th_max = 0.5 * math.radians(cam["fov_max_deg"])
    ru = math.sin(th_max) / (math.cos(th_max) + cam["xi"])
    rd = ru * (1 + cam.get("k1", 0.0) * ru * ru) * 1.02
    for ty in range(grid.shape[0]):
        for tx in range(grid.shape[1]):
            x0, y0 = tx * tw, ty * th
            nx = max(x0 - 4 - cam["cx"], cam["cx"] - (x0 + tw - 1 + 4), 0.0) / cam["fx"]
            ny = max(y0 - 4 - cam["cy"], cam["cy"] - (y0 + th - 1 + 4), 0.0) / cam["fy"]
            assert (grid[ty, tx] > 0) == (nx * nx + ny * ny <= rd * rd), (tx, ty)
    # centre column: a tile well below the principal point sees both families, its mirror image above only the
    # fronto-parallel one (the ground-parallel planes face no ray above the horizon)
    n_fronto, n_ground = (f["n_planes"] for f in cfg["families"])
    tx = int(cam["cx"] // tw)
    ty_c = int(cam["cy"] // th)
    up, down = grid[ty_c - 4, tx], grid[ty_c + 4, tx]
    assert abs(up - (n_fronto + 2)) < 0.5                       # every fronto plane in range for every ray, + S1 / epilogue
    assert n_fronto + 2 + 0.3 * n_ground < down <= n_fronto + n_ground + 2.01
    # the split: some tiles whole (the heavy head of the queue), the rest in halves; never worse than either extreme
    n_whole = plan["n_whole_slots"]
    assert 0 < n_whole < plan["n_tiles"] and n_whole + plan["n_halved_slots"] == plan["n_tiles"]
    m = _makespan(weight.tolist(), plan["n_live"], n_whole, 1, 148)
    assert m <= _makespan(weight.tolist(), plan["n_live"], plan["n_live"], 1, 148) * 1.0001
    assert m <= _makespan(weight.tolist(), plan["n_live"], 0, 1, 148) * 1.0001
    for other in range(0, plan["n_live"] + 1, 7):
        assert m <= _makespan(weight.tolist(), plan["n_live"], other, 1, 148) * 1.002, other


def test_long_queues_are_not_split_and_weights_scale_with_planes():
    cfg, rig, planes = _rig_planes(5)
    one = fsw.plan_schedule(rig, planes, cfg["params"], n_sets=1)
    eight = fsw.plan_schedule(rig, planes, cfg["params"], n_sets=8)
    assert eight["by_weight"] == 0 and eight["n_halved_slots"] == 0 and eight["n_whole_slots"] == 8 * eight["n_tiles"]
    assert eight["n_live"] == one["n_live"]
    # centre-first order: the first tile of the long queue contains (or touches) the principal point
    cam = cfg["cams"][0]
    t0 = int(eight["tile_order"][0])
    tx, ty = t0 % eight["n_tiles_x"], t0 // eight["n_tiles_x"]
    assert abs((tx + 0.5) * 64 - cam["cx"]) <= 64 and abs((ty + 0.5) * 40 - cam["cy"]) <= 40
    assert (eight["tile_weight"][:eight["n_live"]] > 0).all() and (eight["tile_weight"][eight["n_live"]:] == 0).all()
    # half as many fronto-parallel planes: the weight of a tile above the horizon drops by that many passes
    fams = [dict(cfg["families"][0], n_planes=cfg["families"][0]["n_planes"] // 2), cfg["families"][1]]
    fewer = fsw.plan_schedule(rig, fsw.PlaneSet(fams), cfg["params"], n_sets=1)
    w1 = np.zeros(one["n_tiles"]); w1[one["tile_order"]] = one["tile_weight"]
    w2 = np.zeros(one["n_tiles"]); w2[fewer["tile_order"]] = fewer["tile_weight"]
    tile = int(cam["cy"] // 40 - 4) * one["n_tiles_x"] + int(cam["cx"] // 64)
    assert abs((w1[tile] - w2[tile]) - cfg["families"][0]["n_planes"] // 2) < 0.5
    # a region of interest: tiles outside it carry nothing
    p = dict(cfg["params"], roi=(448, 400, 320, 240))
    roi = fsw.plan_schedule(rig, planes, p, n_sets=1)
    wr = np.zeros(roi["n_tiles"]); wr[roi["tile_order"]] = roi["tile_weight"]
    g = wr.reshape(-1, roi["n_tiles_x"])
    assert g[10:16, 7:12].min() > 0 and g[:10].max() == 0 and g[16:].max() == 0 and g[:, :7].max() == 0 and g[:, 12:].max() == 0
    assert roi["n_live"] < one["n_live"]


def test_plan_rejects_bad_arguments():
    cfg, rig, planes = _rig_planes(1)
    with pytest.raises(fsw.FswError):
        fsw.plan_schedule(rig, planes, cfg["params"], n_sets=0)
    with pytest.raises(fsw.FswError):
        fsw.plan_schedule(rig, planes, cfg["params"], n_blocks=0)
    with pytest.raises(fsw.FswError):
        fsw.plan_schedule(rig, planes, dict(cfg["params"], window=4))
    small = fsw.plan_schedule(rig, planes, cfg["params"], n_sets=1, n_blocks=148)
    assert small["n_live"] >= 1 and small["n_whole_slots"] + small["n_halved_slots"] == small["n_tiles"]
