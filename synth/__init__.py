"""Seeded synthetic inputs for the fisheye plane-sweep path.

INPUT GENERATION ONLY.  This module renders the fisheye frame sets, masks and
rig / plane-set / parameter *descriptions* of BASELINE.json's five configs (the
recipe is in DESIGN.md, "Input recipe").  It holds none of the plane-sweep
method: no warp, no matching cost, no WTA, no filters.  Both the CPU oracle and
the CUDA path consume what it returns; neither is imported here.

The paper's own sequences are private; these synthetic frame
sets take their shapes (multi-fisheye rig, forward-facing street scenes,
~1 MP grayscale, ~100 planes, 9x9 / 7x7 windows) and stand in for them.
"""
from __future__ import annotations

import ctypes
import math
import os
import subprocess
from functools import lru_cache

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "synth_core.c")
_LIB = os.path.join(_HERE, "libsynth_core.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile synth_core.c -> libsynth_core.so (gcc, OpenMP)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp",
                               "-ffp-contract=off", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB)
        dp = ctypes.POINTER(ctypes.c_double)
        fp = ctypes.POINTER(ctypes.c_float)
        lib.synth_hash4.restype = ctypes.c_uint32
        lib.synth_hash4.argtypes = [ctypes.c_uint32] * 4
        lib.synth_pixel_ray.restype = ctypes.c_int
        lib.synth_pixel_ray.argtypes = [dp, ctypes.c_double, ctypes.c_double, dp]
        lib.synth_render.restype = ctypes.c_int
        lib.synth_render.argtypes = [dp, ctypes.c_int, ctypes.c_int, dp, dp, ctypes.c_int, dp, dp,
                                     ctypes.c_uint32, ctypes.c_int, ctypes.c_double, ctypes.c_double,
                                     ctypes.c_uint32, fp, fp]
        _lib = lib
    return _lib


def _dp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


# ----------------------------------------------------------------------------
# counter-based random numbers
# ----------------------------------------------------------------------------
def hash4(a: int, b: int, c: int, d: int) -> int:
    return int(_load().synth_hash4(a & 0xFFFFFFFF, b & 0xFFFFFFFF, c & 0xFFFFFFFF, d & 0xFFFFFFFF))


def uniform(seed: int, stream: int, i: int, j: int = 0, lo: float = 0.0, hi: float = 1.0) -> float:
    return lo + (hi - lo) * ((hash4(seed, stream, i, j) + 0.5) / 4294967296.0)


# ----------------------------------------------------------------------------
# rig helpers (descriptions only)
# ----------------------------------------------------------------------------
def yaw_rig_to_cam(psi_deg: float) -> np.ndarray:
    """rig->camera rotation of a camera yawed by psi about +y (down); psi>0 turns the axis toward +x."""
    p = math.radians(psi_deg)
    c, s = math.cos(p), math.sin(p)
    r_cam_to_rig = np.array([[c, 0.0, s], [0.0, 1.0, 0.0], [-s, 0.0, c]])
    return r_cam_to_rig.T.copy()


def camera(width, height, fx, fy, cx, cy, xi, k1=0.0, k2=0.0, p1=0.0, p2=0.0, fov_max_deg=180.0,
           centre=(0.0, 0.0, 0.0), yaw_deg=0.0) -> dict:
    """Camera description.  Extrinsic is rig->camera: X_cam = R X_rig + t, t = -R C."""
    R = yaw_rig_to_cam(yaw_deg)
    C = np.asarray(centre, dtype=np.float64)
    return dict(width=int(width), height=int(height), fx=float(fx), fy=float(fy), cx=float(cx), cy=float(cy),
                xi=float(xi), k1=float(k1), k2=float(k2), p1=float(p1), p2=float(p2),
                fov_max_deg=float(fov_max_deg), R=R, t=-R @ C)


def family(normal, n_planes, d_first, d_last, spacing) -> dict:
    assert spacing in ("inverse", "linear")
    return dict(normal=[float(x) for x in normal], n_planes=int(n_planes), d_first=float(d_first),
                d_last=float(d_last), spacing=spacing)


def params(window, var_floor, range_max, alpha_upper=1.0, alpha_lower=1.0, horizon_row=0, beta=1.0,
           subpixel=1, filters=0, depth_kind=0, roi=None) -> dict:
    return dict(window=int(window), var_floor=float(var_floor), range_max=float(range_max),
                alpha_upper=float(alpha_upper), alpha_lower=float(alpha_lower), horizon_row=int(horizon_row),
                beta=float(beta), subpixel=int(subpixel), filters=int(filters), depth_kind=int(depth_kind),
                roi=None if roi is None else tuple(int(x) for x in roi))


FILTER_COST = 1
FILTER_RATIO = 2
VAR_FLOOR_U8 = 6.5025   # (0.01*255)^2, SURVEY 8(c) Q10
VAR_FLOOR_F32 = 1e-4    # (0.01)^2


# ----------------------------------------------------------------------------
# scenes (lists of textured boxes)
# ----------------------------------------------------------------------------
BIG = 1.0e4


def _tex(base, contrast, cells, ident):
    c = list(cells) + [0.0] * (3 - len(cells))
    return [base, contrast, c[0], c[1], c[2], float(ident)]


def scene_plane(z=4.0, cells=(0.6, 2.4), seed=1) -> dict:
    boxes = [[-BIG, -BIG, z, BIG, BIG, z + 1.0]]
    tex = [_tex(0.5, 0.45, cells, 1)]
    return dict(boxes=np.array(boxes, dtype=np.float64), tex=np.array(tex, dtype=np.float64), seed=seed,
                sky=0.5, noise_sigma=0.0, supersample=3)


def scene_boxes(seed=2, n_boxes=20, ground_y=1.6) -> dict:
    boxes = [[-BIG, ground_y, -BIG, BIG, ground_y + 1.0, BIG]]
    tex = [_tex(0.45, 0.35, (0.25, 1.0, 4.0), 1)]
    for i in range(n_boxes):
        edge = uniform(seed, 11, i, 0, 1.0, 4.0)
        dist = uniform(seed, 12, i, 0, 3.0, 30.0)
        az = math.radians(uniform(seed, 13, i, 0, -80.0, 80.0))
        x, z = dist * math.sin(az), dist * math.cos(az)
        boxes.append([x - edge / 2, ground_y - edge, z - edge / 2, x + edge / 2, ground_y, z + edge / 2])
        tex.append(_tex(uniform(seed, 14, i, 0, 0.3, 0.7), uniform(seed, 15, i, 0, 0.3, 0.5), (0.2, 0.8), 2 + i))
    return dict(boxes=np.array(boxes, dtype=np.float64), tex=np.array(tex, dtype=np.float64), seed=seed,
                sky=0.5, noise_sigma=0.01, supersample=3)


def scene_street(seed=3, n_cars=40, ground_y=1.6, z_start=-20.0, z_end=260.0) -> dict:
    """Procedural urban street: ground, facades at 6-15 m lateral in 10-30 m segments, 40 car boxes."""
    boxes = [[-BIG, ground_y, -BIG, BIG, ground_y + 1.0, BIG]]
    tex = [_tex(0.40, 0.35, (0.15, 0.6, 2.4), 1)]
    ident = 2
    for side in (-1.0, 1.0):
        z, j = z_start, 0
        while z < z_end:
            seg = uniform(seed, 21 + int(side > 0), j, 0, 10.0, 30.0)
            lat = uniform(seed, 23 + int(side > 0), j, 0, 6.0, 15.0)
            hgt = uniform(seed, 25 + int(side > 0), j, 0, 6.0, 20.0)
            x0, x1 = (lat, lat + 2.0) if side > 0 else (-lat - 2.0, -lat)
            boxes.append([x0, ground_y - hgt, z, x1, ground_y, z + seg])
            tex.append(_tex(uniform(seed, 27, ident, 0, 0.3, 0.7), uniform(seed, 28, ident, 0, 0.25, 0.5),
                            (0.2, 0.8, 3.2), ident))
            ident += 1
            z += seg
            j += 1
    for i in range(n_cars):
        side = 1.0 if uniform(seed, 31, i) < 0.5 else -1.0
        lat = side * uniform(seed, 32, i, 0, 2.0, 5.0)
        zc = uniform(seed, 33, i, 0, 5.0, 150.0)
        boxes.append([lat - 0.9, ground_y - 1.5, zc - 2.25, lat + 0.9, ground_y, zc + 2.25])
        tex.append(_tex(uniform(seed, 34, i, 0, 0.25, 0.75), uniform(seed, 35, i, 0, 0.3, 0.5), (0.12, 0.5), ident))
        ident += 1
    return dict(boxes=np.array(boxes, dtype=np.float64), tex=np.array(tex, dtype=np.float64), seed=seed,
                sky=0.5, noise_sigma=0.0, supersample=3)


# ----------------------------------------------------------------------------
# rendering
# ----------------------------------------------------------------------------
def cam_array(cam: dict) -> np.ndarray:
    return np.array([cam["fx"], cam["fy"], cam["cx"], cam["cy"], cam["xi"], cam["k1"], cam["k2"], cam["p1"],
                     cam["p2"], math.radians(cam["fov_max_deg"]) / 2.0], dtype=np.float64)


def pixel_ray(cam: dict, u: float, v: float):
    """Unit ray of pixel (u,v) by the generator's own camera simulator; None if outside the FOV."""
    r = np.zeros(3)
    ok = _load().synth_pixel_ray(_dp(cam_array(cam)), float(u), float(v), _dp(r))
    return r if ok else None


def render_camera(cam: dict, scene: dict, rig_position=(0.0, 0.0, 0.0), noise_seed=0, want_range=False):
    """Ray-cast one camera of a rig whose frame is axis-aligned with the world at rig_position.
    Returns float32 [H,W] in [0,1] (and the ground-truth range along the pixel-centre ray)."""
    lib = _load()
    W, H = cam["width"], cam["height"]
    R = np.asarray(cam["R"], dtype=np.float64)
    t = np.asarray(cam["t"], dtype=np.float64)
    R_wc = np.ascontiguousarray(R.T)                      # camera -> rig (= world) rotation
    C_w = np.ascontiguousarray(np.asarray(rig_position, dtype=np.float64) + (-R.T @ t))
    img = np.empty((H, W), dtype=np.float32)
    rng = np.empty((H, W), dtype=np.float32) if want_range else None
    boxes = np.ascontiguousarray(scene["boxes"], dtype=np.float64)
    tex = np.ascontiguousarray(scene["tex"], dtype=np.float64)
    ca = cam_array(cam)
    lib.synth_render(_dp(ca), W, H, _dp(R_wc), _dp(C_w), boxes.shape[0], _dp(boxes), _dp(tex),
                     int(scene["seed"]), int(scene["supersample"]), float(scene["sky"]),
                     float(scene["noise_sigma"]), int(noise_seed) & 0xFFFFFFFF,
                     img.ctypes.data_as(ctypes.POINTER(ctypes.c_float)),
                     rng.ctypes.data_as(ctypes.POINTER(ctypes.c_float)) if want_range else None)
    return (img, rng) if want_range else img


def quantize(img: np.ndarray, dtype: str) -> np.ndarray:
    if dtype == "u8":
        return np.clip(np.floor(img.astype(np.float64) * 255.0 + 0.5), 0, 255).astype(np.uint8)
    return np.ascontiguousarray(img, dtype=np.float32)


def render_frame(cfg: dict, frame: int = 0):
    """All images of one synchronized frame set of a config, in rig order (u8 or f32 per cfg['dtype'])."""
    pos = (0.0, 0.0, cfg.get("step_m", 0.0) * frame)
    out = []
    for ci, cam in enumerate(cfg["cams"]):
        img = render_camera(cam, cfg["scene"], pos, noise_seed=cfg["scene"]["seed"] * 1000 + 16 * frame + ci)
        out.append(quantize(img, cfg["dtype"]))
    return out


def make_mask(width: int, height: int, seed: int, n_rects: int = 8) -> np.ndarray:
    """Seeded binary mask of n random rectangles (stand-in for detector boxes)."""
    m = np.zeros((height, width), dtype=np.uint8)
    for i in range(n_rects):
        w = int(uniform(seed, 41, i, 0, 40.0, 300.0))
        h = int(uniform(seed, 42, i, 0, 40.0, 200.0))
        w, h = min(w, width), min(h, height)
        x0 = int(uniform(seed, 43, i, 0, 0.0, float(width - w + 1)))
        y0 = int(uniform(seed, 44, i, 0, 0.0, float(height - h + 1)))
        m[y0:y0 + h, x0:x0 + w] = 1
    return m


# ----------------------------------------------------------------------------
# BASELINE.json configs[0..4]  (C1..C5); values marked (+) are this repo's choices, see DESIGN.md
# ----------------------------------------------------------------------------
def _street_rig():
    kw = dict(width=1280, height=1024, fx=350.0, fy=350.0, cx=640.0, cy=512.0, xi=1.0, k1=-0.05, fov_max_deg=185.0)
    return [camera(**kw), camera(centre=(-0.5, 0, 0), **kw), camera(centre=(0.5, 0, 0), **kw)]


def _paper_rig():
    """The shape of the paper's own workload: five fisheye cameras of 1024 x 544, the reference
    in the middle and four matching views with rotated optical axes (values are this generator's, not the paper's:
    its calibration is not published)."""
    kw = dict(width=1024, height=544, fx=285.0, fy=285.0, cx=512.0, cy=272.0, xi=1.0, k1=-0.05, fov_max_deg=185.0)
    return [camera(**kw), camera(centre=(-0.6, 0.0, 0.0), yaw_deg=-12.0, **kw), camera(centre=(0.6, 0.0, 0.0), yaw_deg=12.0, **kw),
            camera(centre=(-0.25, -0.3, 0.1), yaw_deg=-4.0, **kw), camera(centre=(0.25, -0.3, 0.1), yaw_deg=4.0, **kw)]


def _half_camera(c: dict) -> dict:
    """The camera of the 2x2-box-downsampled image (pixel centres at integers: f/2, c' = (c - 0.5)/2)."""
    h = dict(c)
    h.update(width=c["width"] // 2, height=c["height"] // 2, fx=c["fx"] / 2.0, fy=c["fy"] / 2.0,
             cx=(c["cx"] - 0.5) / 2.0, cy=(c["cy"] - 0.5) / 2.0)
    return h


def make_config(index: int, cameras=None) -> dict:
    """index = 1..5 for C1..C5 (BASELINE.json configs[index-1]); 6..8 = the paper's own workload shapes (
    PAPER.md:76, :88-90, :224, :249), each a stream of 32 frame sets of the five-camera rig (4 matching views):
      6  "P"   full resolution 1024 x 544, 64 fronto-parallel + 30 ground-parallel planes, 9 x 9 ZNCC (the 50 ms case)
      7  "PM"  multi-scale: 512 x 272 full field of view with 7 x 7 + the 572 x 332 centre crop at full resolution with
               9 x 9, the same 64 + 30 planes in both passes (the 36 ms case)
      8  "PH"  half resolution 512 x 272, 7 x 7 (the 16 ms case); the cameras are those of the downsampled images
    cameras: optional list of camera indices (the reference first) selecting a sub-rig, e.g. (0, 1, 2) for the
    three-camera configuration of PAPER.md:280, :294."""
    if index in (6, 7, 8):
        cfg = _paper_config(index)
        if cameras is not None:
            assert cameras[0] == 0, "the reference camera comes first"
            cfg = dict(cfg, cams=[cfg["cams"][i] for i in cameras], cameras=tuple(cameras),
                       name=cfg["name"] + "%d" % len(cameras))
        return cfg
    assert cameras is None
    return _baseline_config(index)


def _paper_config(index: int) -> dict:
    fams = [family((0, 0, 1), 64, 0.5, 50.0, "inverse"), family((0, 1, 0), 30, 1.1, 2.1, "linear")]
    fil = FILTER_COST | FILTER_RATIO
    if index == 7:
        return dict(name="PM", dtype="u8", ref_index=0, cams=_paper_rig(), n_frames=32, step_m=0.5, mask_seed=None,
                    families_low=fams, families_crop=fams,
                    params_low=params(7, VAR_FLOOR_U8, 100.0, 0.05, 0.3, 272, 1.2, filters=fil),
                    params_crop=params(9, VAR_FLOOR_U8, 100.0, 0.05, 0.3, 272, 1.2, filters=fil),
                    crop=((1024 - 572) // 2, (544 - 332) // 2, 572, 332), scene=scene_street(seed=3))
    if index == 8:
        return dict(name="PH", dtype="u8", ref_index=0, cams=[_half_camera(c) for c in _paper_rig()], n_frames=32,
                    step_m=0.5, mask_seed=None, families=fams,
                    params=params(7, VAR_FLOOR_U8, 100.0, 0.05, 0.3, 136, 1.2, filters=fil), scene=scene_street(seed=3))
    return _baseline_config(6)


def _baseline_config(index: int) -> dict:
    if index == 6:
        return dict(name="P", dtype="u8", ref_index=0, cams=_paper_rig(), n_frames=32, step_m=0.5, mask_seed=None,
                    families=[family((0, 0, 1), 64, 0.5, 50.0, "inverse"), family((0, 1, 0), 30, 1.1, 2.1, "linear")],
                    params=params(9, VAR_FLOOR_U8, 100.0, 0.05, 0.3, 272, 1.2, filters=FILTER_COST | FILTER_RATIO),
                    scene=scene_street(seed=3))
    if index == 1:
        kw = dict(width=64, height=48, fx=30.0, fy=30.0, cx=32.0, cy=24.0, xi=0.9, fov_max_deg=200.0)
        return dict(name="C1", dtype="u8", ref_index=0,
                    cams=[camera(**kw), camera(centre=(0.3, 0, 0), **kw)],
                    families=[family((0, 0, 1), 32, 0.5, 50.0, "inverse")],
                    params=params(5, VAR_FLOOR_U8, 100.0),
                    scene=scene_plane(4.0, (0.6, 2.4), seed=1))
    if index == 2:
        kw = dict(width=320, height=256, fx=160.0, fy=160.0, cx=160.0, cy=128.0, xi=1.0, fov_max_deg=185.0)
        return dict(name="C2", dtype="f32", ref_index=0,
                    cams=[camera(**kw), camera(centre=(-0.4, 0, 0), yaw_deg=-10.0, **kw),
                          camera(centre=(0.4, 0, 0), yaw_deg=10.0, **kw)],
                    families=[family((0, 0, 1), 64, 0.5, 50.0, "inverse")],
                    params=params(7, VAR_FLOOR_F32, 100.0),
                    scene=scene_boxes(seed=2))
    if index in (3, 4, 5):
        cams = _street_rig()
        fil = FILTER_COST | FILTER_RATIO
        if index == 3:
            return dict(name="C3", dtype="u8", ref_index=0, cams=cams,
                        families=[family((0, 0, 1), 96, 0.5, 50.0, "inverse"),
                                  family((0, 1, 0), 32, 1.1, 2.1, "linear")],
                        params=params(9, VAR_FLOOR_U8, 100.0, 0.05, 0.3, 512, 1.2, filters=fil),
                        scene=scene_street(seed=3))
        if index == 4:
            return dict(name="C4", dtype="u8", ref_index=0, cams=cams,
                        families_low=[family((0, 0, 1), 96, 0.5, 50.0, "inverse")],
                        families_crop=[family((0, 0, 1), 192, 0.5, 80.0, "inverse")],
                        params_low=params(7, VAR_FLOOR_U8, 100.0, 0.05, 0.3, 512, 1.2, filters=fil),
                        params_crop=params(9, VAR_FLOOR_U8, 160.0, 0.05, 0.3, 512, 1.2, filters=fil),
                        crop=(384, 256, 512, 512), mask_seed=4,
                        scene=scene_street(seed=3))
        return dict(name="C5", dtype="u8", ref_index=0, cams=cams, n_frames=32, step_m=0.5, mask_seed=5,
                    families=[family((0, 0, 1), 192, 0.5, 50.0, "inverse"),
                              family((0, 1, 0), 64, 1.1, 2.1, "linear")],
                    params=params(9, VAR_FLOOR_U8, 100.0, 0.05, 0.3, 512, 1.2, filters=fil),
                    scene=scene_street(seed=3))
    raise ValueError("config index must be 1..8")


@lru_cache(maxsize=8)
def cached_frame(index: int, frame: int = 0):
    cfg = make_config(index)
    return tuple(render_frame(cfg, frame))
