"""Thin ctypes binding of libfsw.so (include/fsw.h).  Argument marshalling only: every step of the plane-sweep path
runs in the CUDA kernels behind the C ABI.  PyTorch supplies device memory and the current stream.

There is no CPU fallback: importing works without a GPU (so that the ABI can be checked), but creating a Context
without a CUDA device raises FswError, and a missing libfsw.so that cannot be built raises ImportError.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libfsw.so")

OK, E_INVALID_ARG, E_CONFIG, E_CUDA, E_NOMEM, E_UNSUPPORTED = 0, -1, -2, -3, -4, -5
U8, F32 = 0, 1
INVERSE, LINEAR = 0, 1
FILTER_COST, FILTER_RATIO = 1, 2
DEPTH_RANGE, DEPTH_Z = 0, 1
REASON_OK, REASON_NO_PLANE, REASON_COST_FILTER, REASON_RATIO_FILTER, REASON_MASKED = 0, 1, 2, 3, 4
INDEX_FROM_CROP = 1 << 14
STATIC_SCRATCH_BYTES = 24 << 20

EXPORTS = (
    "fsw_version", "fsw_last_error", "fsw_rig_create", "fsw_rig_destroy", "fsw_rig_relative_pose",
    "fsw_ground_normal_in_ref", "fsw_planeset_create", "fsw_planeset_destroy", "fsw_planeset_size",
    "fsw_planeset_table", "fsw_context_create", "fsw_context_destroy", "fsw_compute_depth",
    "fsw_compute_depth_multires", "fsw_compute_depth_host", "fsw_compute_depth_multires_host",
    "fsw_compute_depth_batch", "fsw_compute_depth_batch_host", "fsw_compute_depth_multires_batch",
    "fsw_compute_depth_multires_batch_host", "fsw_rig_subset",
    "fsw_context_set_timing", "fsw_context_set_split", "fsw_context_set_host_async", "fsw_get_last_counters", "fsw_filter_continuity",
    "fsw_plan_schedule", "fsw_compute_depth_static",
)


class FswError(RuntimeError):
    def __init__(self, code, message):
        super().__init__("fsw error %d: %s" % (code, message))
        self.code = code


class CCamera(ctypes.Structure):
    _fields_ = [("struct_size", ctypes.c_uint32), ("width", ctypes.c_int32), ("height", ctypes.c_int32),
                ("fx", ctypes.c_double), ("fy", ctypes.c_double), ("cx", ctypes.c_double), ("cy", ctypes.c_double),
                ("xi", ctypes.c_double), ("k1", ctypes.c_double), ("k2", ctypes.c_double), ("p1", ctypes.c_double),
                ("p2", ctypes.c_double), ("fov_max_deg", ctypes.c_double), ("R", ctypes.c_double * 9),
                ("t", ctypes.c_double * 3)]


class CFamily(ctypes.Structure):
    _fields_ = [("struct_size", ctypes.c_uint32), ("normal", ctypes.c_double * 3), ("n_planes", ctypes.c_int32),
                ("spacing", ctypes.c_int32), ("d_first", ctypes.c_double), ("d_last", ctypes.c_double)]


class CRect(ctypes.Structure):
    _fields_ = [("x0", ctypes.c_int32), ("y0", ctypes.c_int32), ("w", ctypes.c_int32), ("h", ctypes.c_int32)]


class CParams(ctypes.Structure):
    _fields_ = [("struct_size", ctypes.c_uint32), ("window", ctypes.c_int32), ("subpixel", ctypes.c_int32),
                ("filters_enabled", ctypes.c_int32), ("depth_kind", ctypes.c_int32), ("roi", CRect),
                ("horizon_row", ctypes.c_int32), ("alpha_upper", ctypes.c_float), ("alpha_lower", ctypes.c_float),
                ("beta", ctypes.c_float), ("var_floor", ctypes.c_float), ("range_max", ctypes.c_float),
                ("debug_cost_volume", ctypes.c_void_p), ("best_k", ctypes.c_int32), ("filter_before_merge", ctypes.c_int32),
                ("upsample_plane", ctypes.c_int32), ("reserved_", ctypes.c_int32)]


class CImage(ctypes.Structure):
    _fields_ = [("data", ctypes.c_void_p), ("pitch_bytes", ctypes.c_size_t), ("dtype", ctypes.c_int32)]


class CDepthOut(ctypes.Structure):
    _fields_ = [("struct_size", ctypes.c_uint32),
                ("depth", ctypes.c_void_p), ("depth_pitch", ctypes.c_size_t),
                ("best_cost", ctypes.c_void_p), ("best_cost_pitch", ctypes.c_size_t),
                ("second_cost", ctypes.c_void_p), ("second_cost_pitch", ctypes.c_size_t),
                ("plane_index", ctypes.c_void_p), ("plane_index_pitch", ctypes.c_size_t),
                ("valid_reason", ctypes.c_void_p), ("valid_reason_pitch", ctypes.c_size_t)]


class CCounters(ctypes.Structure):
    _fields_ = [("struct_size", ctypes.c_uint32), ("n_eval", ctypes.c_int64), ("n_raw_valid", ctypes.c_int64),
                ("n_valid", ctypes.c_int64), ("n_launches", ctypes.c_int64), ("sweep_ms", ctypes.c_double),
                ("n_split_launches", ctypes.c_int64)]


_lib = None


def load_library():
    """Loads libfsw.so (building it with nvcc if it is missing) and declares the prototypes of include/fsw.h."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        from . import build as _build
        try:
            _build.build()
        except Exception as exc:  # no silent fallback: the product path needs the CUDA extension
            raise ImportError("libfsw.so is missing and could not be built: %s" % exc) from exc
    L = ctypes.CDLL(LIB_PATH)
    vp, i32, sz = ctypes.c_void_p, ctypes.c_int32, ctypes.c_size_t
    P = ctypes.POINTER
    L.fsw_version.argtypes = [P(i32), P(i32)]
    L.fsw_last_error.restype = ctypes.c_char_p
    L.fsw_rig_create.argtypes = [P(CCamera), i32, i32, P(vp)]
    L.fsw_rig_destroy.argtypes = [vp]
    L.fsw_rig_relative_pose.argtypes = [vp, i32, P(ctypes.c_double), P(ctypes.c_double)]
    L.fsw_ground_normal_in_ref.argtypes = [vp, P(ctypes.c_double), P(ctypes.c_double)]
    L.fsw_planeset_create.argtypes = [P(CFamily), i32, P(vp)]
    L.fsw_planeset_destroy.argtypes = [vp]
    L.fsw_planeset_size.argtypes = [vp, P(i32)]
    L.fsw_planeset_table.argtypes = [vp, P(ctypes.c_double), P(ctypes.c_double), P(i32)]
    L.fsw_context_create.argtypes = [vp, i32, P(vp)]
    L.fsw_context_destroy.argtypes = [vp]
    single = [vp, vp, P(CParams), P(CImage), vp, sz, P(CDepthOut), vp]
    multi = [vp, vp, vp, P(CParams), P(CParams), CRect, P(CImage), vp, sz, P(CDepthOut), vp]
    L.fsw_compute_depth.argtypes = single
    L.fsw_compute_depth_host.argtypes = single
    L.fsw_compute_depth_static.argtypes = single
    L.fsw_compute_depth_multires.argtypes = multi
    batch = [vp, vp, P(CParams), i32, P(CImage), P(vp), sz, P(CDepthOut), vp]
    L.fsw_compute_depth_batch.argtypes = batch
    L.fsw_compute_depth_batch_host.argtypes = batch
    L.fsw_compute_depth_multires_host.argtypes = multi
    multi_batch = [vp, vp, vp, P(CParams), P(CParams), CRect, i32, P(CImage), P(vp), sz, P(CDepthOut), vp]
    L.fsw_compute_depth_multires_batch.argtypes = multi_batch
    L.fsw_compute_depth_multires_batch_host.argtypes = multi_batch
    L.fsw_rig_subset.argtypes = [vp, P(i32), i32, P(vp)]
    L.fsw_context_set_timing.argtypes = [vp, i32]
    L.fsw_context_set_split.argtypes = [vp, i32]
    L.fsw_context_set_host_async.argtypes = [vp, i32]
    L.fsw_get_last_counters.argtypes = [vp, P(CCounters)]
    L.fsw_plan_schedule.argtypes = [vp, vp, P(CParams), i32, i32, i32, P(i32), P(ctypes.c_float), P(CSchedulePlan)]
    for name in EXPORTS:
        if name != "fsw_last_error":
            getattr(L, name).restype = i32
    _lib = L
    return L


def _check(rc):
    if rc != OK:
        raise FswError(rc, load_library().fsw_last_error().decode("utf-8", "replace"))


def version():
    a, b = ctypes.c_int32(), ctypes.c_int32()
    _check(load_library().fsw_version(ctypes.byref(a), ctypes.byref(b)))
    return a.value, b.value


# ---- description dicts -> C structs -----------------------------------------------------------------------------
def make_camera(c) -> CCamera:
    out = CCamera()
    out.struct_size = ctypes.sizeof(CCamera)
    out.width, out.height = int(c["width"]), int(c["height"])
    for k in ("fx", "fy", "cx", "cy", "xi"):
        setattr(out, k, float(c[k]))
    for k in ("k1", "k2", "p1", "p2"):
        setattr(out, k, float(c.get(k, 0.0)))
    out.fov_max_deg = float(c.get("fov_max_deg", 360.0))
    out.R = (ctypes.c_double * 9)(*np.asarray(c.get("R", np.eye(3)), dtype=np.float64).reshape(9))
    out.t = (ctypes.c_double * 3)(*np.asarray(c.get("t", np.zeros(3)), dtype=np.float64).reshape(3))
    return out


def make_family(f) -> CFamily:
    out = CFamily()
    out.struct_size = ctypes.sizeof(CFamily)
    out.normal = (ctypes.c_double * 3)(*[float(x) for x in f["normal"]])
    out.n_planes = int(f["n_planes"])
    sp = f["spacing"]
    out.spacing = INVERSE if sp in ("inverse", INVERSE) else (LINEAR if sp in ("linear", LINEAR) else int(sp))
    out.d_first, out.d_last = float(f["d_first"]), float(f["d_last"])
    return out


class CSchedulePlan(ctypes.Structure):
    _fields_ = [("struct_size", ctypes.c_uint32), ("tile_w", ctypes.c_int32), ("tile_h", ctypes.c_int32),
                ("n_tiles_x", ctypes.c_int32), ("n_tiles", ctypes.c_int32), ("n_live", ctypes.c_int32),
                ("by_weight", ctypes.c_int32), ("n_whole_slots", ctypes.c_int64), ("n_halved_slots", ctypes.c_int64)]


def plan_schedule(rig, planes, params, n_sets=1, n_blocks=148):
    """fsw_plan_schedule (host only): the queue order of the tiles, their estimated weights and the number of
    (tile, frame set) slots FSW_SPLIT_AUTO sweeps whole for a call with n_sets frame sets on n_blocks SMs."""
    import numpy as np
    L = load_library()
    cp = make_params(params)
    plan = CSchedulePlan()
    plan.struct_size = ctypes.sizeof(CSchedulePlan)
    _check(L.fsw_plan_schedule(rig.handle, planes.handle, ctypes.byref(cp), n_sets, n_blocks, 0, None, None, ctypes.byref(plan)))
    order = np.zeros(plan.n_tiles, np.int32)
    weight = np.zeros(plan.n_tiles, np.float32)
    _check(L.fsw_plan_schedule(rig.handle, planes.handle, ctypes.byref(cp), n_sets, n_blocks, plan.n_tiles,
                               order.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)),
                               weight.ctypes.data_as(ctypes.POINTER(ctypes.c_float)), ctypes.byref(plan)))
    out = {name: getattr(plan, name) for name, _ in CSchedulePlan._fields_ if name != "struct_size"}
    out["tile_order"], out["tile_weight"] = order, weight
    return out


def make_params(p, debug_cost_ptr=None) -> CParams:
    out = CParams()
    out.struct_size = ctypes.sizeof(CParams)
    out.window, out.subpixel = int(p["window"]), int(p.get("subpixel", 1))
    out.filters_enabled, out.depth_kind = int(p.get("filters", 0)), int(p.get("depth_kind", 0))
    roi = p.get("roi")
    out.roi = CRect(0, 0, 0, 0) if roi is None else CRect(*[int(x) for x in roi])
    out.horizon_row = int(p.get("horizon_row", 0))
    out.alpha_upper, out.alpha_lower = float(p.get("alpha_upper", 1.0)), float(p.get("alpha_lower", 1.0))
    out.beta, out.var_floor, out.range_max = float(p.get("beta", 1.0)), float(p["var_floor"]), float(p["range_max"])
    out.debug_cost_volume = debug_cost_ptr
    out.best_k, out.filter_before_merge = int(p.get("best_k", 0)), int(p.get("filter_before_merge", 0))
    out.upsample_plane = int(p.get("upsample_plane", 0))
    return out


# ---- handles ------------------------------------------------------------------------------------------------------
class Rig:
    """fsw_rig: calibrated multi-fisheye rig (intrinsics, distortion, mirror parameter, 6-DoF rig->camera poses)."""

    def __init__(self, cams, ref_index=0):
        L = load_library()
        arr = (CCamera * len(cams))(*[make_camera(c) for c in cams])
        h = ctypes.c_void_p()
        _check(L.fsw_rig_create(arr, len(cams), int(ref_index), ctypes.byref(h)))
        self.handle, self.n_cams, self.ref_index = h, len(cams), int(ref_index)
        self.sizes = [(int(c["width"]), int(c["height"])) for c in cams]

    def subset(self, cam_indices):
        """fsw_rig_subset: a rig of the listed cameras (must include the reference, which stays the reference)."""
        idx = [int(i) for i in cam_indices]
        arr = (ctypes.c_int32 * len(idx))(*idx)
        h = ctypes.c_void_p()
        _check(load_library().fsw_rig_subset(self.handle, arr, len(idx), ctypes.byref(h)))
        sub = Rig.__new__(Rig)
        sub.handle, sub.n_cams, sub.ref_index = h, len(idx), idx.index(self.ref_index)
        sub.sizes = [self.sizes[i] for i in idx]
        return sub

    def relative_pose(self, cam):
        R, T = (ctypes.c_double * 9)(), (ctypes.c_double * 3)()
        _check(load_library().fsw_rig_relative_pose(self.handle, int(cam), R, T))
        return np.array(R).reshape(3, 3), np.array(T)

    def ground_normal_in_ref(self, dir_rig=(0.0, 1.0, 0.0)):
        d, o = (ctypes.c_double * 3)(*[float(x) for x in dir_rig]), (ctypes.c_double * 3)()
        _check(load_library().fsw_ground_normal_in_ref(self.handle, d, o))
        return np.array(o)

    def close(self):
        if getattr(self, "handle", None):
            load_library().fsw_rig_destroy(self.handle)
            self.handle = None

    __del__ = close


class PlaneSet:
    """fsw_planeset: families of sweep planes n.X = d_k in the reference-camera frame."""

    def __init__(self, fams):
        L = load_library()
        arr = (CFamily * len(fams))(*[make_family(f) for f in fams])
        h = ctypes.c_void_p()
        _check(L.fsw_planeset_create(arr, len(fams), ctypes.byref(h)))
        self.handle = h
        n = ctypes.c_int32()
        _check(L.fsw_planeset_size(h, ctypes.byref(n)))
        self.n_planes = n.value

    def table(self):
        P = self.n_planes
        s, d, f = (ctypes.c_double * P)(), (ctypes.c_double * P)(), (ctypes.c_int32 * P)()
        _check(load_library().fsw_planeset_table(self.handle, s, d, f))
        return np.array(s), np.array(d), np.array(f)

    def close(self):
        if getattr(self, "handle", None):
            load_library().fsw_planeset_destroy(self.handle)
            self.handle = None

    __del__ = close


def _torch():
    import torch
    return torch


class Context:
    """fsw_context on one CUDA device; owns the library's device scratch."""

    def __init__(self, rig: Rig, device: int = 0):
        L = load_library()
        h = ctypes.c_void_p()
        _check(L.fsw_context_create(rig.handle, int(device), ctypes.byref(h)))
        self.handle, self.rig, self.device = h, rig, int(device)

    def close(self):
        if getattr(self, "handle", None):
            load_library().fsw_context_destroy(self.handle)
            self.handle = None

    __del__ = close

    # -- marshalling helpers -------------------------------------------------------------------------------------
    def _images(self, images, host):
        torch = _torch()
        arr = (CImage * self.rig.n_cams)()
        keep = []
        assert len(images) == self.rig.n_cams, "one image per camera, in rig order"
        for i, im in enumerate(images):
            W, H = self.rig.sizes[i]
            if host:
                if isinstance(im, torch.Tensor):
                    assert not im.is_cuda
                    a = im
                    dt = U8 if a.dtype == torch.uint8 else F32
                    assert a.dtype in (torch.uint8, torch.float32) and tuple(a.shape) == (H, W) and a.stride(1) == 1
                    ptr, pitch = a.data_ptr(), a.stride(0) * a.element_size()
                else:
                    a = np.asarray(im)
                    assert a.dtype in (np.uint8, np.float32) and a.shape == (H, W) and a.strides[1] == a.itemsize
                    dt = U8 if a.dtype == np.uint8 else F32
                    ptr, pitch = a.ctypes.data, a.strides[0]
            else:
                a = im
                assert isinstance(a, torch.Tensor) and a.is_cuda and a.device.index == self.device
                assert a.dtype in (torch.uint8, torch.float32) and tuple(a.shape) == (H, W) and a.stride(1) == 1
                dt = U8 if a.dtype == torch.uint8 else F32
                ptr, pitch = a.data_ptr(), a.stride(0) * a.element_size()
            keep.append(a)
            arr[i] = CImage(ptr, pitch, dt)
        return arr, keep

    def _outputs(self, host, want, out=None):
        torch = _torch()
        W, H = self.rig.sizes[self.rig.ref_index]
        spec = dict(depth=torch.float32, best_cost=torch.float32, second_cost=torch.float32, plane_index=torch.int16,
                    valid_reason=torch.uint8)
        if out is not None:  # caller-owned output tensors (e.g. pinned host buffers reused across calls)
            c = CDepthOut()
            c.struct_size = ctypes.sizeof(CDepthOut)
            assert out.get("depth") is not None, "the depth map is required"
            for name, dt in spec.items():
                t = out.get(name)
                if t is not None:
                    # fsw.h sees pointers and pitches only: type, shape and device are checked here
                    assert t.dtype == dt, "%s must be %s" % (name, dt)
                    assert tuple(t.shape) == (H, W) and t.stride(1) == 1, "%s must be a row-major (H, W) map" % name
                    assert t.is_cuda != host, "%s is on the wrong side (host=%s)" % (name, host)
                    assert host or t.device.index == self.device, "%s is on another GPU than the context" % name
                    setattr(c, name, t.data_ptr())
                    setattr(c, name + "_pitch", t.stride(0) * t.element_size())
            return c, dict(out)
        kw = dict(device="cpu", pin_memory=True) if host else dict(device="cuda:%d" % self.device)
        out, c = {}, CDepthOut()
        c.struct_size = ctypes.sizeof(CDepthOut)
        for name, dt in spec.items():
            if name == "depth" or name in want:
                t = torch.empty((H, W), dtype=dt, **kw)
                out[name] = t
                setattr(c, name, t.data_ptr())
                setattr(c, name + "_pitch", t.stride(0) * t.element_size())
        return c, out

    def _mask(self, mask, host):
        if mask is None:
            return None, 0, None
        torch = _torch()
        W, H = self.rig.sizes[self.rig.ref_index]
        if host and not isinstance(mask, torch.Tensor):
            m = np.ascontiguousarray(mask, dtype=np.uint8)
            assert m.shape == (H, W)
            return m.ctypes.data, m.strides[0], m
        assert mask.dtype == torch.uint8 and tuple(mask.shape) == (H, W) and mask.stride(1) == 1
        assert mask.is_cuda != host and (host or mask.device.index == self.device)
        return mask.data_ptr(), mask.stride(0), mask

    ALL = ("best_cost", "second_cost", "plane_index", "valid_reason")

    # -- the calls of include/fsw.h ---------------------------------------------------------------------------------
    def compute_depth(self, planes: PlaneSet, params, images, mask=None, want=ALL, host=False, debug_cost=False,
                      out=None):
        """fsw_compute_depth (device tensors) / fsw_compute_depth_host (host=True: numpy or CPU tensors).
        Returns a dict of tensors: depth (+ best_cost, second_cost, plane_index, valid_reason as requested)."""
        torch = _torch()
        L = load_library()
        arr, keep = self._images(images, host)
        mptr, mpitch, mkeep = self._mask(mask, host)
        cout, out = self._outputs(host, want, out)
        dbg = None
        if debug_cost:
            assert not host
            W, H = self.rig.sizes[self.rig.ref_index]
            dbg = torch.empty((planes.n_planes, H, W), dtype=torch.float32, device="cuda:%d" % self.device)
            out["cost_volume"] = dbg
        cp = make_params(params, None if dbg is None else dbg.data_ptr())
        stream = torch.cuda.current_stream(self.device).cuda_stream
        fn = L.fsw_compute_depth_host if host else L.fsw_compute_depth
        _check(fn(self.handle, planes.handle, ctypes.byref(cp), arr, mptr, mpitch, ctypes.byref(cout), stream))
        out["_keep"] = (keep, mkeep)
        return out

    def compute_depth_static(self, planes: PlaneSet, params, images, out, mask=None):
        """fsw_compute_depth_static: fsw_compute_depth without any device allocation (scratch in the library's static
        24 MiB array, STATIC_SCRATCH_BYTES).  `out` is required: caller-owned device tensors, so that this wrapper
        allocates nothing on the device either.  Returns `out`."""
        torch = _torch()
        L = load_library()
        assert out is not None, "compute_depth_static writes into caller-owned tensors"
        arr, keep = self._images(images, False)
        mptr, mpitch, mkeep = self._mask(mask, False)
        cout, out = self._outputs(False, (), out)
        cp = make_params(params, None)
        stream = torch.cuda.current_stream(self.device).cuda_stream
        _check(L.fsw_compute_depth_static(self.handle, planes.handle, ctypes.byref(cp), arr, mptr, mpitch,
                                          ctypes.byref(cout), stream))
        out["_keep"] = (keep, mkeep)
        return out

    def compute_depth_batch(self, planes: PlaneSet, params, image_sets, masks=None, want=ALL, host=False, outs=None):
        """fsw_compute_depth_batch / _host: n independent frame sets of the rig in one sweep launch.
        image_sets: list of per-set image lists; masks: list (entries may be None) or None; outs: optional list of
        caller-owned output dicts.  Returns a list of output dicts, one per frame set."""
        torch = _torch()
        L = load_library()
        n, nc = len(image_sets), self.rig.n_cams
        arr = (CImage * (n * nc))()
        keep = []
        for s, images in enumerate(image_sets):
            a, k = self._images(images, host)
            for c in range(nc):
                arr[s * nc + c] = a[c]
            keep.append(k)
        marr, mpitch = None, 0
        if masks is not None and any(m is not None for m in masks):
            marr = (ctypes.c_void_p * n)()
            for s, m in enumerate(masks):
                ptr, pitch, mk = self._mask(m, host)
                marr[s] = ptr
                keep.append(mk)
                if ptr:
                    assert mpitch in (0, pitch), "all masks of a batch share one pitch"
                    mpitch = pitch
        couts = (CDepthOut * n)()
        results = []
        for s in range(n):
            c, o = self._outputs(host, want, None if outs is None else outs[s])
            couts[s] = c
            results.append(o)
        cp = make_params(params)
        stream = torch.cuda.current_stream(self.device).cuda_stream
        fn = L.fsw_compute_depth_batch_host if host else L.fsw_compute_depth_batch
        _check(fn(self.handle, planes.handle, ctypes.byref(cp), n, arr, marr, mpitch, couts, stream))
        results[0]["_keep"] = keep
        return results

    def compute_depth_multires(self, planes_low: PlaneSet, planes_crop: PlaneSet, params_low, params_crop, crop,
                               images, mask=None, want=ALL, host=False, out=None):
        """fsw_compute_depth_multires / _host: the two-scale strategy of PAPER.md:88-90."""
        torch = _torch()
        L = load_library()
        arr, keep = self._images(images, host)
        mptr, mpitch, mkeep = self._mask(mask, host)
        cout, out = self._outputs(host, want, out)
        pl, pc = make_params(params_low), make_params(params_crop)
        stream = torch.cuda.current_stream(self.device).cuda_stream
        fn = L.fsw_compute_depth_multires_host if host else L.fsw_compute_depth_multires
        _check(fn(self.handle, planes_low.handle, planes_crop.handle, ctypes.byref(pl), ctypes.byref(pc),
                  CRect(*[int(x) for x in crop]), arr, mptr, mpitch, ctypes.byref(cout), stream))
        out["_keep"] = (keep, mkeep)
        return out

    def compute_depth_multires_batch(self, planes_low: PlaneSet, planes_crop: PlaneSet, params_low, params_crop, crop,
                                     image_sets, masks=None, want=ALL, host=False, outs=None):
        """fsw_compute_depth_multires_batch / _host: the two-scale strategy for n frame sets in one call."""
        torch = _torch()
        L = load_library()
        n, nc = len(image_sets), self.rig.n_cams
        arr = (CImage * (n * nc))()
        keep = []
        for s, images in enumerate(image_sets):
            a, k = self._images(images, host)
            for c in range(nc):
                arr[s * nc + c] = a[c]
            keep.append(k)
        marr, mpitch = None, 0
        if masks is not None and any(m is not None for m in masks):
            marr = (ctypes.c_void_p * n)()
            for s, m in enumerate(masks):
                ptr, pitch, mk = self._mask(m, host)
                marr[s] = ptr
                keep.append(mk)
                if ptr:
                    assert mpitch in (0, pitch), "all masks of a batch share one pitch"
                    mpitch = pitch
        couts = (CDepthOut * n)()
        results = []
        for s in range(n):
            c, o = self._outputs(host, want, None if outs is None else outs[s])
            couts[s] = c
            results.append(o)
        pl, pc = make_params(params_low), make_params(params_crop)
        stream = torch.cuda.current_stream(self.device).cuda_stream
        fn = L.fsw_compute_depth_multires_batch_host if host else L.fsw_compute_depth_multires_batch
        _check(fn(self.handle, planes_low.handle, planes_crop.handle, ctypes.byref(pl), ctypes.byref(pc),
                  CRect(*[int(x) for x in crop]), n, arr, marr, mpitch, couts, stream))
        if results:
            results[0]["_keep"] = keep
        return results

    def filter_continuity(self, depth, window=5, gamma=0.5, delta=0.3, mask=None, want_reason=True):
        """fsw_filter_continuity: the local depth-continuity filter of PAPER.md:99 + mask on a device depth map.
        Returns dict(depth=..., valid_reason=...) of new device tensors."""
        torch = _torch()
        W, H = self.rig.sizes[self.rig.ref_index]
        assert depth.is_cuda and depth.device.index == self.device, "depth must live on the context's GPU"
        assert depth.dtype == torch.float32 and tuple(depth.shape) == (H, W) and depth.stride(1) == 1
        out = torch.empty((H, W), dtype=torch.float32, device=depth.device)
        reason = torch.empty((H, W), dtype=torch.uint8, device=depth.device) if want_reason else None
        mptr, mpitch, mkeep = self._mask(mask, False)
        stream = torch.cuda.current_stream(self.device).cuda_stream
        fn = load_library().fsw_filter_continuity
        fn.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_size_t, ctypes.c_int32, ctypes.c_double, ctypes.c_double,
                       ctypes.c_void_p, ctypes.c_size_t, ctypes.c_void_p, ctypes.c_size_t, ctypes.c_void_p,
                       ctypes.c_size_t, ctypes.c_void_p]
        _check(fn(self.handle, depth.data_ptr(), depth.stride(0) * 4, int(window), float(gamma), float(delta),
                  mptr, mpitch, out.data_ptr(), out.stride(0) * 4,
                  None if reason is None else reason.data_ptr(), 0 if reason is None else reason.stride(0), stream))
        return dict(depth=out, valid_reason=reason, _keep=(depth, mkeep))

    def last_counters(self):
        c = CCounters()
        c.struct_size = ctypes.sizeof(CCounters)
        _check(load_library().fsw_get_last_counters(self.handle, ctypes.byref(c)))
        return dict(n_eval=c.n_eval, n_raw_valid=c.n_raw_valid, n_valid=c.n_valid, n_launches=c.n_launches,
                    sweep_ms=c.sweep_ms, n_split_launches=c.n_split_launches)

    def set_host_async(self, on=True):
        """fsw_context_set_host_async: host=True calls return without synchronizing their stream."""
        _check(load_library().fsw_context_set_host_async(self.handle, 1 if on else 0))

    def set_split(self, mode="auto"):
        """fsw_context_set_split: plane split of the light tiles of calls with few frame sets ('auto', 'off', 'on')."""
        _check(load_library().fsw_context_set_split(self.handle, {"auto": 0, "off": 1, "on": 2}[mode]))

    def set_timing(self, on=True):
        """fsw_context_set_timing: bracket the sweep kernels of later calls with CUDA events (last_counters()['sweep_ms'])."""
        _check(load_library().fsw_context_set_timing(self.handle, 1 if on else 0))
