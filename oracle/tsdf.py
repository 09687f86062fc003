"""ctypes wrapper of the TSDF part of the CPU ORACLE (oracle/fsw_tsdf_oracle.c) -- TEST INFRASTRUCTURE.

A `Volume` is the dense local box of PAPER.md:175-176: nb blocks of 8^3 voxels from the integer block origin b0.
"""
from __future__ import annotations

import ctypes
import math

import numpy as np

from . import _load, make_camera, _dp, _bp


class Box(ctypes.Structure):
    _fields_ = [("voxel_size", ctypes.c_double), ("mu", ctypes.c_double), ("w_max", ctypes.c_int32),
                ("b0", ctypes.c_int32 * 3), ("nb", ctypes.c_int32 * 3)]


def box_for(centre, box_size, voxel_size):
    """Block origin and block counts of the local map centred at `centre` (metres), snapped to whole blocks: the
    centre block contains the centre, the box extends ceil(size / edge / 2) ... blocks to either side (reading T6)."""
    edge = 8.0 * voxel_size
    nb = [int(math.ceil(s / edge - 1e-9)) for s in box_size]
    b0 = [int(math.floor(c / edge)) - n // 2 for c, n in zip(centre, nb)]
    return b0, nb


class Volume:
    def __init__(self, voxel_size, mu, w_max, b0, nb):
        self.box = Box(float(voxel_size), float(mu), int(w_max), (ctypes.c_int32 * 3)(*b0), (ctypes.c_int32 * 3)(*nb))
        n = int(nb[0]) * int(nb[1]) * int(nb[2])
        self.nb, self.b0 = [int(v) for v in nb], [int(v) for v in b0]
        self.allocated = np.zeros(n, dtype=np.uint8)
        self.D = np.zeros(n * 512, dtype=np.float64)
        self.W = np.zeros(n * 512, dtype=np.float64)
        self.obs = np.zeros(n, dtype=np.int32)
        L = _load()
        L.orc_tsdf_allocate.restype = ctypes.c_int64
        L.orc_tsdf_integrate.restype = ctypes.c_int64
        L.orc_tsdf_extract.restype = ctypes.c_int64

    def _pose(self, R, t):
        R = np.ascontiguousarray(R, dtype=np.float64).reshape(9)
        t = np.ascontiguousarray(t, dtype=np.float64).reshape(3)
        return R, t

    def allocate(self, cam, R, t, depth, want_fragile=False):
        R, t = self._pose(R, t)
        d = np.ascontiguousarray(depth, dtype=np.float64)
        frag = np.zeros_like(self.allocated) if want_fragile else None
        c = make_camera(cam)
        n = _load().orc_tsdf_allocate(ctypes.byref(self.box), ctypes.byref(c), _dp(R), _dp(t), _dp(d), _bp(self.allocated), _bp(frag))
        return int(n), frag

    def integrate(self, cam, R, t, depth, want_fragile=False):
        R, t = self._pose(R, t)
        d = np.ascontiguousarray(depth, dtype=np.float64)
        frag = np.zeros(self.D.size, dtype=np.uint8) if want_fragile else None
        c = make_camera(cam)
        n = _load().orc_tsdf_integrate(ctypes.byref(self.box), ctypes.byref(c), _dp(R), _dp(t), _dp(d), _bp(self.allocated),
                                       _dp(self.D), _dp(self.W), self.obs.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)), _bp(frag))
        return int(n), frag

    def extract(self, min_obs=3, cap=2000000):
        pts = np.zeros((cap, 3), dtype=np.float64)
        n = _load().orc_tsdf_extract(ctypes.byref(self.box), _bp(self.allocated), _dp(self.D), _dp(self.W),
                                     self.obs.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)), int(min_obs), _dp(pts), int(cap))
        return pts[:min(int(n), cap)], int(n)

    def dense(self):
        """(D, W) as [nz*8, ny*8, nx*8] arrays (voxel order z, y, x) and obs / allocated as [nbz, nby, nbx]."""
        nbx, nby, nbz = self.nb
        def unblock(a):
            a = a.reshape(nbz, nby, nbx, 8, 8, 8)          # bz by bx k j i
            return a.transpose(0, 3, 1, 4, 2, 5).reshape(nbz * 8, nby * 8, nbx * 8)
        return unblock(self.D), unblock(self.W), self.obs.reshape(nbz, nby, nbx), self.allocated.reshape(nbz, nby, nbx)
