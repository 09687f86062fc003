"""ctypes binding of the TSDF consumer of libfsw.so (include/fsw.h, fsw_tsdf_*).  Marshalling only."""
from __future__ import annotations

import ctypes

import numpy as np

from .binding import CCamera, FswError, OK, load_library, make_camera


class CTsdfParams(ctypes.Structure):
    _fields_ = [("struct_size", ctypes.c_uint32), ("voxel_size", ctypes.c_float), ("mu", ctypes.c_float),
                ("w_max", ctypes.c_int32), ("box_size", ctypes.c_float * 3)]


class CTsdfStats(ctypes.Structure):
    _fields_ = [("struct_size", ctypes.c_uint32), ("n_new_blocks", ctypes.c_int64), ("n_visible_blocks", ctypes.c_int64),
                ("n_voxels_updated", ctypes.c_int64), ("n_points", ctypes.c_int64), ("n_blocks_freed", ctypes.c_int64),
                ("n_frames", ctypes.c_int64)]


TSDF_EXPORTS = ("fsw_tsdf_create", "fsw_tsdf_destroy", "fsw_tsdf_last_error", "fsw_tsdf_box", "fsw_tsdf_recentre",
                "fsw_tsdf_integrate", "fsw_tsdf_extract_points", "fsw_tsdf_get_stats", "fsw_tsdf_download")


def _lib():
    L = load_library()
    if not getattr(L, "_tsdf_ready", False):
        vp, i32, sz, P = ctypes.c_void_p, ctypes.c_int32, ctypes.c_size_t, ctypes.POINTER
        dp = P(ctypes.c_double)
        L.fsw_tsdf_create.argtypes = [i32, P(CTsdfParams), dp, P(vp)]
        L.fsw_tsdf_destroy.argtypes = [vp]
        L.fsw_tsdf_last_error.restype = ctypes.c_char_p
        L.fsw_tsdf_box.argtypes = [vp, P(i32), P(i32)]
        L.fsw_tsdf_recentre.argtypes = [vp, dp, vp]
        L.fsw_tsdf_integrate.argtypes = [vp, P(CCamera), dp, dp, vp, sz, vp]
        L.fsw_tsdf_extract_points.argtypes = [vp, i32, vp, i32, vp]
        L.fsw_tsdf_get_stats.argtypes = [vp, P(CTsdfStats)]
        L.fsw_tsdf_download.argtypes = [vp, vp, vp, vp, vp, vp]
        for name in TSDF_EXPORTS:
            if name != "fsw_tsdf_last_error":
                getattr(L, name).restype = i32
        L._tsdf_ready = True
    return L


def _check(rc):
    if rc != OK:
        raise FswError(rc, _lib().fsw_tsdf_last_error().decode("utf-8", "replace"))


def _d3(v, n=3):
    return (ctypes.c_double * n)(*[float(x) for x in np.asarray(v, dtype=np.float64).reshape(n)])


class TsdfVolume:
    """fsw_tsdf: the local TSDF map on one CUDA device."""

    def __init__(self, voxel_size=0.05, mu=0.2, w_max=100, box_size=(60.0, 60.0, 3.0), centre=(0.0, 0.0, 0.0), device=0):
        p = CTsdfParams(ctypes.sizeof(CTsdfParams), float(voxel_size), float(mu), int(w_max), (ctypes.c_float * 3)(*box_size))
        h = ctypes.c_void_p()
        _check(_lib().fsw_tsdf_create(int(device), ctypes.byref(p), _d3(centre), ctypes.byref(h)))
        self.handle, self.device, self.voxel_size = h, int(device), float(voxel_size)

    def close(self):
        if getattr(self, "handle", None):
            _lib().fsw_tsdf_destroy(self.handle)
            self.handle = None

    __del__ = close

    def _stream(self):
        import torch
        return torch.cuda.current_stream(self.device).cuda_stream

    def box(self):
        b0, nb = (ctypes.c_int32 * 3)(), (ctypes.c_int32 * 3)()
        _check(_lib().fsw_tsdf_box(self.handle, b0, nb))
        return list(b0), list(nb)

    def recentre(self, centre):
        _check(_lib().fsw_tsdf_recentre(self.handle, _d3(centre), self._stream()))

    def integrate(self, cam, R, t, depth):
        """depth: CUDA float32 tensor [H, W] of ranges along the pixel rays (0 = invalid)."""
        import torch
        assert depth.is_cuda and depth.device.index == self.device and depth.dtype == torch.float32 and depth.stride(1) == 1
        assert tuple(depth.shape) == (int(cam["height"]), int(cam["width"]))
        c = make_camera(cam)
        _check(_lib().fsw_tsdf_integrate(self.handle, ctypes.byref(c), _d3(R, 9), _d3(t), depth.data_ptr(),
                                         depth.stride(0) * 4, self._stream()))
        self._keep = depth

    def extract_points(self, min_block_observations=3, capacity=1 << 20):
        """-> (points [n, 3] float32 CUDA tensor relative to the box origin, total count)"""
        import torch
        pts = torch.empty((capacity, 3), dtype=torch.float32, device="cuda:%d" % self.device)
        _check(_lib().fsw_tsdf_extract_points(self.handle, int(min_block_observations), pts.data_ptr(), int(capacity), self._stream()))
        n = self.stats()["n_points"]
        return pts[:min(n, capacity)], n

    def stats(self):
        s = CTsdfStats()
        s.struct_size = ctypes.sizeof(CTsdfStats)
        _check(_lib().fsw_tsdf_get_stats(self.handle, ctypes.byref(s)))
        return {k: getattr(s, k) for k, _ in CTsdfStats._fields_ if k != "struct_size"}

    def download(self):
        """dense copies in box order: (tsdf, weight) [nz*8, ny*8, nx*8] float32, (observations, allocated) [nz, ny, nx]"""
        import torch
        _, nb = self.box()
        dev = "cuda:%d" % self.device
        shape = (nb[2] * 8, nb[1] * 8, nb[0] * 8)
        D = torch.empty(shape, dtype=torch.float32, device=dev)
        Wt = torch.empty(shape, dtype=torch.float32, device=dev)
        obs = torch.empty((nb[2], nb[1], nb[0]), dtype=torch.int32, device=dev)
        al = torch.empty((nb[2], nb[1], nb[0]), dtype=torch.uint8, device=dev)
        _check(_lib().fsw_tsdf_download(self.handle, D.data_ptr(), Wt.data_ptr(), obs.data_ptr(), al.data_ptr(), self._stream()))
        torch.cuda.synchronize(self.device)
        return D.cpu().numpy(), Wt.cpu().numpy(), obs.cpu().numpy(), al.cpu().numpy()
