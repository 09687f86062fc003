"""ctypes wrapper of the CPU ORACLE (oracle/fsw_oracle.c) -- TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It shares no code with paper_1809_06132_b200 (the CUDA
path) and does not import it.  Everything numerical happens in the C file; this module
marshals numpy arrays and sequences the C calls in the order SURVEY 8(c) O4..O10 gives:
sweep -> wta -> (merge) -> filters -> mask.
"""
from __future__ import annotations

import ctypes
import math
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "fsw_oracle.c")
_SRC_TSDF = os.path.join(_HERE, "fsw_tsdf_oracle.c")
_HDR = os.path.join(_HERE, "fsw_oracle.h")
_LIB = os.path.join(_HERE, "libfsw_oracle.so")
_lib = None

INVERSE, LINEAR = 0, 1
FILTER_COST, FILTER_RATIO = 1, 2
OK, NO_PLANE, COST_FILTER, RATIO_FILTER, MASKED = 0, 1, 2, 3, 4


class Camera(ctypes.Structure):
    _fields_ = [("width", ctypes.c_int32), ("height", ctypes.c_int32),
                ("fx", ctypes.c_double), ("fy", ctypes.c_double), ("cx", ctypes.c_double), ("cy", ctypes.c_double),
                ("xi", ctypes.c_double),
                ("k1", ctypes.c_double), ("k2", ctypes.c_double), ("p1", ctypes.c_double), ("p2", ctypes.c_double),
                ("theta_max", ctypes.c_double), ("R", ctypes.c_double * 9), ("t", ctypes.c_double * 3)]


class Family(ctypes.Structure):
    _fields_ = [("normal", ctypes.c_double * 3), ("n_planes", ctypes.c_int32), ("spacing", ctypes.c_int32),
                ("d_first", ctypes.c_double), ("d_last", ctypes.c_double)]


class Params(ctypes.Structure):
    _fields_ = [("window", ctypes.c_int32), ("subpixel", ctypes.c_int32), ("filters", ctypes.c_int32),
                ("depth_kind", ctypes.c_int32),
                ("roi_x0", ctypes.c_int32), ("roi_y0", ctypes.c_int32), ("roi_w", ctypes.c_int32), ("roi_h", ctypes.c_int32),
                ("horizon_row", ctypes.c_int32),
                ("alpha_upper", ctypes.c_double), ("alpha_lower", ctypes.c_double), ("beta", ctypes.c_double),
                ("var_floor", ctypes.c_double), ("range_max", ctypes.c_double), ("best_k", ctypes.c_int32)]


def build(force: bool = False) -> str:
    newest = max(os.path.getmtime(_SRC), os.path.getmtime(_SRC_TSDF), os.path.getmtime(_HDR))
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < newest:
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
                               "-Wall", "-o", tmp, _SRC, _SRC_TSDF, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_LIB)
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int32)
        bp = ctypes.POINTER(ctypes.c_uint8)
        cam, fam, prm = ctypes.POINTER(Camera), ctypes.POINTER(Family), ctypes.POINTER(Params)
        I, D = ctypes.c_int, ctypes.c_double
        L.orc_project.argtypes = [cam, dp, dp]
        L.orc_back_project.argtypes = [cam, D, D, dp]
        L.orc_pixel_theta.argtypes = [cam, D, D]
        L.orc_pixel_theta.restype = D
        L.orc_relative_pose.argtypes = [cam, cam, dp, dp]
        L.orc_relative_pose.restype = None
        L.orc_plane_table.argtypes = [fam, I, dp, dp, ip, dp]
        L.orc_warp_pixel.argtypes = [cam, cam, dp, D, D, D, D, dp]
        L.orc_bilinear.argtypes = [dp, I, I, D, D]
        L.orc_bilinear.restype = D
        L.orc_zncc_cost.argtypes = [dp, dp, I, D]
        L.orc_zncc_cost.restype = D
        L.orc_sweep.argtypes = [cam, I, I, fam, I, prm, ctypes.POINTER(dp), dp, ctypes.POINTER(ctypes.c_int64), bp]
        L.orc_pixel_costs.argtypes = [cam, I, I, fam, I, prm, ctypes.POINTER(dp), I, I, dp]
        L.orc_wta.argtypes = [cam, fam, I, prm, dp, dp, dp, dp, dp, ip, dp, dp, bp]
        L.orc_filter_mask.argtypes = [I, I, prm, bp, bp, dp, dp, dp, bp, bp]
        L.orc_filter_continuity.argtypes = [dp, I, I, I, D, D, bp, dp, bp]
        L.orc_downsample2.argtypes = [dp, I, I, dp]
        L.orc_camera_half.argtypes = [cam, cam]
        L.orc_camera_half.restype = None
        L.orc_merge.argtypes = [I, I, I, I, I, I, dp, dp, dp, ip, bp, dp, dp, dp, ip, bp, dp, dp, dp, ip, bp]
        L.orc_num_threads.restype = I
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _ip(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_int32))


def _bp(a):
    return None if a is None else a.ctypes.data_as(ctypes.POINTER(ctypes.c_uint8))


# ----------------------------------------------------------------------------
# description -> C struct
# ----------------------------------------------------------------------------
def make_camera(c) -> Camera:
    if isinstance(c, Camera):
        return c
    out = Camera()
    out.width, out.height = int(c["width"]), int(c["height"])
    for k in ("fx", "fy", "cx", "cy", "xi"):
        setattr(out, k, float(c[k]))
    for k in ("k1", "k2", "p1", "p2"):
        setattr(out, k, float(c.get(k, 0.0)))
    out.theta_max = math.radians(float(c.get("fov_max_deg", 360.0))) / 2.0
    R = np.asarray(c.get("R", np.eye(3)), dtype=np.float64).reshape(9)
    t = np.asarray(c.get("t", np.zeros(3)), dtype=np.float64).reshape(3)
    out.R = (ctypes.c_double * 9)(*R)
    out.t = (ctypes.c_double * 3)(*t)
    return out


def make_cameras(cams):
    arr = (Camera * len(cams))()
    for i, c in enumerate(cams):
        arr[i] = make_camera(c)
    return arr


def make_families(fams):
    arr = (Family * len(fams))()
    for i, f in enumerate(fams):
        arr[i].normal = (ctypes.c_double * 3)(*[float(x) for x in f["normal"]])
        arr[i].n_planes = int(f["n_planes"])
        arr[i].spacing = INVERSE if f["spacing"] in ("inverse", INVERSE) else LINEAR
        arr[i].d_first, arr[i].d_last = float(f["d_first"]), float(f["d_last"])
    return arr


def make_params(p) -> Params:
    out = Params()
    out.window, out.subpixel = int(p["window"]), int(p.get("subpixel", 1))
    out.filters, out.depth_kind = int(p.get("filters", 0)), int(p.get("depth_kind", 0))
    roi = p.get("roi")
    if roi is None:
        out.roi_x0 = out.roi_y0 = 0
        out.roi_w = out.roi_h = 0
    else:
        out.roi_x0, out.roi_y0, out.roi_w, out.roi_h = [int(x) for x in roi]
    out.horizon_row = int(p.get("horizon_row", 0))
    out.alpha_upper, out.alpha_lower = float(p.get("alpha_upper", 1.0)), float(p.get("alpha_lower", 1.0))
    out.beta, out.var_floor = float(p.get("beta", 1.0)), float(p["var_floor"])
    out.range_max = float(p["range_max"])
    out.best_k = int(p.get("best_k", 0))
    return out


# ----------------------------------------------------------------------------
# O1..O3 scalars
# ----------------------------------------------------------------------------
def project(cam, X):
    uv = np.zeros(2)
    Xa = np.ascontiguousarray(X, dtype=np.float64)
    ok = _load().orc_project(ctypes.byref(make_camera(cam)), _dp(Xa), _dp(uv))
    return uv if ok else None


def back_project(cam, u, v):
    r = np.zeros(3)
    ok = _load().orc_back_project(ctypes.byref(make_camera(cam)), float(u), float(v), _dp(r))
    return r if ok else None


def pixel_theta(cam, u, v):
    return float(_load().orc_pixel_theta(ctypes.byref(make_camera(cam)), float(u), float(v)))


def relative_pose(ref, view):
    R, T = np.zeros(9), np.zeros(3)
    _load().orc_relative_pose(ctypes.byref(make_camera(ref)), ctypes.byref(make_camera(view)), _dp(R), _dp(T))
    return R.reshape(3, 3), T


def plane_table(fams):
    fa = make_families(fams)
    P = _load().orc_plane_table(fa, len(fams), None, None, None, None)
    s, d, f, n = np.zeros(P), np.zeros(P), np.zeros(P, dtype=np.int32), np.zeros(3 * len(fams))
    _load().orc_plane_table(fa, len(fams), _dp(s), _dp(d), _ip(f), _dp(n))
    return s, d, f, n.reshape(-1, 3)


def warp_pixel(ref, view, normal, d, range_max, u, v):
    uv = np.zeros(2)
    n = np.ascontiguousarray(normal, dtype=np.float64)
    ok = _load().orc_warp_pixel(ctypes.byref(make_camera(ref)), ctypes.byref(make_camera(view)), _dp(n), float(d),
                                float(range_max), float(u), float(v), _dp(uv))
    return uv if ok else None


def bilinear(img, u, v):
    a = np.ascontiguousarray(img, dtype=np.float64)
    return float(_load().orc_bilinear(_dp(a), a.shape[1], a.shape[0], float(u), float(v)))


def zncc_cost(a, b, var_floor):
    a = np.ascontiguousarray(a, dtype=np.float64).ravel()
    b = np.ascontiguousarray(b, dtype=np.float64).ravel()
    assert a.size == b.size
    return float(_load().orc_zncc_cost(_dp(a), _dp(b), a.size, float(var_floor)))


# ----------------------------------------------------------------------------
# O4..O8 maps
# ----------------------------------------------------------------------------
def _images_f64(images):
    imgs = [np.ascontiguousarray(im, dtype=np.float64) for im in images]
    ptrs = (ctypes.POINTER(ctypes.c_double) * len(imgs))(*[_dp(im) for im in imgs])
    return imgs, ptrs


def sweep(cams, ref_index, fams, params, images, want_fragile=True):
    """Cost volume [P,H,W] (float64, +inf = undefined), N_eval, geometric fragility map."""
    ca, fa, pr = make_cameras(cams), make_families(fams), make_params(params)
    imgs, ptrs = _images_f64(images)
    H, W = ca[ref_index].height, ca[ref_index].width
    P = _load().orc_plane_table(fa, len(fams), None, None, None, None)
    cost = np.empty((P, H, W), dtype=np.float64)
    n_eval = ctypes.c_int64(0)
    frag = np.zeros((H, W), dtype=np.uint8) if want_fragile else None
    rc = _load().orc_sweep(ca, len(cams), ref_index, fa, len(fams), ctypes.byref(pr), ptrs, _dp(cost),
                           ctypes.byref(n_eval), _bp(frag))
    if rc < 0:
        raise ValueError("orc_sweep rejected its arguments")
    return cost, int(n_eval.value), frag


def pixel_costs(cams, ref_index, fams, params, images, px, py):
    ca, fa, pr = make_cameras(cams), make_families(fams), make_params(params)
    imgs, ptrs = _images_f64(images)
    P = _load().orc_plane_table(fa, len(fams), None, None, None, None)
    out = np.empty(P, dtype=np.float64)
    _load().orc_pixel_costs(ca, len(cams), ref_index, fa, len(fams), ctypes.byref(pr), ptrs, int(px), int(py), _dp(out))
    return out


def wta(ref_cam, fams, params, cost):
    rc, fa, pr = make_camera(ref_cam), make_families(fams), make_params(params)
    P, H, W = cost.shape
    out = dict(depth=np.empty((H, W)), c1=np.empty((H, W)), c2=np.empty((H, W)), c2raw=np.empty((H, W)),
               kbest=np.empty((H, W), dtype=np.int32), delta=np.empty((H, W)), pden=np.empty((H, W)),
               raw_valid=np.empty((H, W), dtype=np.uint8))
    cost = np.ascontiguousarray(cost, dtype=np.float64)
    _load().orc_wta(ctypes.byref(rc), fa, len(fams), ctypes.byref(pr), _dp(cost), _dp(out["depth"]), _dp(out["c1"]),
                    _dp(out["c2"]), _dp(out["c2raw"]), _ip(out["kbest"]), _dp(out["delta"]), _dp(out["pden"]),
                    _bp(out["raw_valid"]))
    return out


def filter_mask(params, maps, mask=None):
    """Applies S9 + S11 to maps (dict from wta/merge) in place; adds 'reason', 'valid', 'fragile_thr'."""
    pr = make_params(params)
    H, W = maps["depth"].shape
    reason = np.zeros((H, W), dtype=np.uint8)
    frag = np.zeros((H, W), dtype=np.uint8)
    m = None if mask is None else np.ascontiguousarray(mask, dtype=np.uint8)
    _load().orc_filter_mask(W, H, ctypes.byref(pr), _bp(m), _bp(maps["raw_valid"]), _dp(maps["c1"]), _dp(maps["c2"]),
                            _dp(maps["depth"]), _bp(reason), _bp(frag))
    maps["reason"], maps["valid"], maps["fragile_thr"] = reason, (reason == 0).astype(np.uint8), frag
    return maps


def filter_continuity(depth, window=5, gamma=0.5, delta=0.3, mask=None):
    """Local depth-continuity filter (third filter; reading Q25) followed by the mask.
    depth: H x W, 0 = invalid.  -> (filtered depth float64, reason uint8)."""
    a = np.ascontiguousarray(depth, dtype=np.float64)
    H, W = a.shape
    out = np.empty((H, W), dtype=np.float64)
    reason = np.zeros((H, W), dtype=np.uint8)
    m = None if mask is None else np.ascontiguousarray(mask, dtype=np.uint8)
    rc = _load().orc_filter_continuity(_dp(a), W, H, int(window), float(gamma), float(delta), _bp(m), _dp(out), _bp(reason))
    if rc != 0:
        raise ValueError("filter_continuity: window must be odd and >= 3")
    return out, reason


def downsample2(img):
    a = np.ascontiguousarray(img, dtype=np.float64)
    H, W = a.shape
    out = np.empty((H // 2, W // 2), dtype=np.float64)
    _load().orc_downsample2(_dp(a), W, H, _dp(out))
    return out


def camera_half(cam) -> Camera:
    out = Camera()
    _load().orc_camera_half(ctypes.byref(make_camera(cam)), ctypes.byref(out))
    return out


def merge(W, H, crop, lo, hi):
    out = dict(depth=np.empty((H, W)), c1=np.empty((H, W)), c2=np.empty((H, W)),
               kbest=np.empty((H, W), dtype=np.int32), raw_valid=np.empty((H, W), dtype=np.uint8))
    x0, y0, cw, ch = [int(v) for v in crop]
    _load().orc_merge(W, H, x0, y0, cw, ch, _dp(lo["depth"]), _dp(lo["c1"]), _dp(lo["c2"]), _ip(lo["kbest"]),
                      _bp(lo["raw_valid"]), _dp(hi["depth"]), _dp(hi["c1"]), _dp(hi["c2"]), _ip(hi["kbest"]),
                      _bp(hi["raw_valid"]), _dp(out["depth"]), _dp(out["c1"]), _dp(out["c2"]), _ip(out["kbest"]),
                      _bp(out["raw_valid"]))
    return out


def num_threads() -> int:
    return int(_load().orc_num_threads())


# ----------------------------------------------------------------------------
# whole path, single resolution and multi-resolution
# ----------------------------------------------------------------------------
def compute_depth(cams, ref_index, fams, params, images, mask=None, keep_cost=False):
    """S1..S9, S11 for one synchronized frame set.  Returns the map dict (+ 'n_eval', 'fragile_geom', 'cost')."""
    cost, n_eval, frag = sweep(cams, ref_index, fams, params, images)
    maps = wta(cams[ref_index], fams, params, cost)
    filter_mask(params, maps, mask)
    maps["n_eval"], maps["fragile_geom"] = n_eval, frag
    if keep_cost:
        maps["cost"] = cost
    return maps


def compute_depth_multires(cams, ref_index, fams_low, fams_crop, params_low, params_crop, crop, images, mask=None,
                           keep_cost=False):
    """S10: half-resolution full-FOV pass + full-resolution crop pass, merged, then filters (params_crop) and mask
    (reading Q20).  With params_crop['filter_before_merge'] the other order of Q20 (reading Q27): each pass is filtered
    on its own (the half-resolution one with params_low, whose horizon_row counts half-resolution rows), then inside
    the crop the full-resolution estimate wins where it SURVIVED its filters, else the surviving upsampled one; then
    the mask."""
    cams_c = [make_camera(c) for c in cams]
    cams_lo = [camera_half(c) for c in cams_c]
    imgs_lo = [downsample2(im) for im in images]
    cost_lo, n_lo, frag_lo = sweep(cams_lo, ref_index, fams_low, params_low, imgs_lo)
    lo = wta(cams_lo[ref_index], fams_low, params_low, cost_lo)
    p_hi = dict(params_crop)
    p_hi["roi"] = tuple(crop)
    cost_hi, n_hi, frag_hi = sweep(cams_c, ref_index, fams_crop, p_hi, images)
    hi = wta(cams_c[ref_index], fams_crop, p_hi, cost_hi)
    H, W = cams_c[ref_index].height, cams_c[ref_index].width
    up = lambda a: np.repeat(np.repeat(a, 2, axis=0), 2, axis=1)[:H, :W]
    if params_crop.get("filter_before_merge"):
        filter_mask(params_low, lo)
        filter_mask(p_hi, hi)
        x0, y0, cw, ch = [int(v) for v in crop]
        in_crop = np.zeros((H, W), dtype=bool)
        in_crop[y0:y0 + ch, x0:x0 + cw] = True
        pad = lambda a, fill: np.pad(up(a), ((0, H - up(a).shape[0]), (0, W - up(a).shape[1])), constant_values=fill)
        lo_valid, lo_raw = pad(lo["valid"], 0) != 0, pad(lo["raw_valid"], 0) != 0
        hi_valid, hi_raw = in_crop & (hi["valid"] != 0), in_crop & (hi["raw_valid"] != 0)
        # where the values come from: a surviving estimate first (full resolution before half resolution), else the
        # estimate the other order would have taken (it says why the pixel is invalid)
        from_hi = hi_valid | (~lo_valid & hi_raw)
        from_lo = ~from_hi & lo_raw
        maps = {}
        for key, fill in (("depth", 0.0), ("c1", np.inf), ("c2", np.inf)):
            maps[key] = np.where(from_hi, hi[key], np.where(from_lo, pad(lo[key], fill), fill))
        maps["kbest"] = np.where(from_hi, hi["kbest"] | (1 << 14), np.where(from_lo, pad(lo["kbest"], -1), -1)).astype(np.int32)
        maps["raw_valid"] = (from_hi | from_lo).astype(np.uint8)
        reason = np.where(from_hi, hi["reason"], np.where(from_lo, pad(lo["reason"], NO_PLANE), NO_PLANE)).astype(np.uint8)
        if mask is not None:
            masked = (reason == OK) & (np.asarray(mask) != 0)
            reason[masked] = MASKED
        maps["depth"] = np.where(reason == OK, maps["depth"], 0.0)
        maps["reason"], maps["valid"] = reason, (reason == OK).astype(np.uint8)
        maps["fragile_thr"] = (pad(lo["fragile_thr"], 0) | hi["fragile_thr"]).astype(np.uint8)
    else:
        maps = merge(W, H, crop, lo, hi)
        filter_mask(params_crop, maps, mask)
    if params_crop.get("upsample_plane"):
        # alternative of reading Q18 (reading Q28): a pixel that takes the half-resolution estimate intersects ITS OWN
        # ray with the refined plane the half-resolution pixel chose: range = d* / (n.r); outside the field of view or
        # not facing the plane -> invalid (NO_PLANE).  Costs and index stay the copied ones.
        s_lo, d_lo, f_lo, n_lo_fam = plane_table(fams_low)
        depth_kind = int(params_crop.get("depth_kind", 0))
        ys, xs = np.nonzero((maps["kbest"] >= 0) & ((maps["kbest"] >> 14) == 0))
        for y, x in zip(ys, xs):
            yl, xl = y >> 1, x >> 1
            k = int(lo["kbest"][yl, xl])
            sk = s_lo[k]
            if lo["delta"][yl, xl] != 0.0:
                sk = sk + lo["delta"][yl, xl] * (s_lo[k + 1] - s_lo[k])
            f = int(f_lo[k])
            d_star = 1.0 / sk if fams_low[f]["spacing"] in ("inverse", INVERSE) else sk
            r = back_project(cams_c[ref_index], float(x), float(y))
            q = -1.0 if r is None else float(n_lo_fam[f] @ r)
            if q > 1e-9:
                if maps["reason"][y, x] == OK:
                    maps["depth"][y, x] = d_star / q * (r[2] if depth_kind == 1 else 1.0)
            else:
                maps["reason"][y, x] = NO_PLANE
                maps["depth"][y, x] = 0.0
        maps["valid"] = (maps["reason"] == OK).astype(np.uint8)
    frag = up(frag_lo)
    frag = np.pad(frag, ((0, H - frag.shape[0]), (0, W - frag.shape[1]))) | frag_hi
    maps.update(n_eval=n_lo + n_hi, fragile_geom=frag, lo=lo, hi=hi)
    if keep_cost:
        maps["cost_lo"], maps["cost_hi"] = cost_lo, cost_hi
    return maps
