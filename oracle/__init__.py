"""CPU oracle for the fused TSDF + asymmetrical colour-volume integration (TEST INFRASTRUCTURE).

Thin ctypes loader around ``oracle/ref_fusion.c`` -- the plain per-voxel loops written from
PAPER.md eq. 5-10 (L91-124) and the TSDF definition of readings A5/A6.  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import
this package; the product path (``paper_1602_06645_b200``) never does, and this package never imports it.

The depth front end and the ICP step are in ``oracle/frontend.py`` (numpy).

Parity pins: tests/test_oracle_*.py (closed forms, fp64 brute force, invariants).  Unpinned by the
paper itself (conventions of this build): the TSDF update (A5/A6), the HD-mapping
reading A11 and the u8 weight encoding A12 -- "parity unpinned" w.r.t. the paper for those.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ref_fusion.c")
_SO = os.path.join(_HERE, "_ref_fusion.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (idempotent).  -ffp-contract=off: no implicit fma; -mfma: fmaf() is the instruction."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-ffp-contract=off", "-mfma", "-shared", "-fPIC", _SRC, "-o", _SO, "-lm"]
        subprocess.run(cmd, check=True)
    return _SO


class RefVol(ctypes.Structure):
    _fields_ = [("nx", ctypes.c_int32), ("ny", ctypes.c_int32), ("nz", ctypes.c_int32), ("r", ctypes.c_int32),
                ("origin", ctypes.c_float * 3), ("extent", ctypes.c_float), ("mu", ctypes.c_float),
                ("w_max", ctypes.c_int32), ("sigma", ctypes.c_float), ("gate", ctypes.c_float), ("variant", ctypes.c_int32)]


# alternative readings (ref_fusion.c), one at a time
VAR_HD_FROM_DEPTH_POINT, VAR_TSDF_ALONG_RAY, VAR_ADDITIVE_WEIGHT = 1, 2, 4


class RefFrame(ctypes.Structure):
    _fields_ = [("depth", ctypes.c_void_p), ("wd", ctypes.c_int32), ("hd", ctypes.c_int32),
                ("rgb", ctypes.c_void_p), ("wh", ctypes.c_int32), ("hh", ctypes.c_int32),
                ("T_world_depth", ctypes.c_float * 16), ("K_depth", ctypes.c_float * 9),
                ("K_rgb", ctypes.c_float * 9), ("T_depth_rgb", ctypes.c_float * 16)]


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_SO)
        P = ctypes.c_void_p
        lib.ref_integrate.restype = ctypes.c_int
        lib.ref_integrate.argtypes = [P, P, P, P, P]
        lib.ref_integrate_sectors.restype = ctypes.c_int
        lib.ref_integrate_sectors.argtypes = [P, P, P, P, P, P, P, P, P]
        lib.ref_threads.restype = ctypes.c_int
        lib.ref_threads.argtypes = []
        lib.ref_integrate_subset.restype = ctypes.c_int
        lib.ref_integrate_subset.argtypes = [P, P, P, ctypes.c_int64, P, P, ctypes.c_int64, P]
        lib.ref_frame_constants.restype = ctypes.c_int
        lib.ref_frame_constants.argtypes = [P, P, P]
        lib.ref_sample_colour.restype = ctypes.c_int
        lib.ref_sample_colour.argtypes = [P, P, P, ctypes.c_int64, P]
        lib.ref_sample_colour_trilinear.restype = ctypes.c_int
        lib.ref_sample_colour_trilinear.argtypes = [P, P, P, ctypes.c_int64, P]
        lib.ref_raycast.restype = ctypes.c_int
        lib.ref_raycast.argtypes = [P, P, P, ctypes.c_int32, ctypes.c_int32, P, P, ctypes.c_float, ctypes.c_float, P, P]
        lib.ref_raycast_trilinear.restype = ctypes.c_int
        lib.ref_raycast_trilinear.argtypes = [P, P, P, ctypes.c_int32, ctypes.c_int32, P, P, ctypes.c_float, ctypes.c_float, P, P]
        _lib = lib
    return _lib


def _f32(a, n):
    a = np.ascontiguousarray(np.asarray(a, dtype=np.float32).reshape(-1))
    assert a.size == n
    return a


class RefVolume:
    """Host-side volume pair driven by the oracle.  Same call shapes as the CUDA binding's Volume."""

    def __init__(self, dims_geo, r, origin, extent, mu, w_max, sigma=0.020, gate=0.8, allocate=True, variant=0):
        self.dims_geo = tuple(int(d) for d in dims_geo)
        self.r = int(r)
        self.dims_col = tuple(d * self.r for d in self.dims_geo)
        self.desc = RefVol(self.dims_geo[0], self.dims_geo[1], self.dims_geo[2], self.r,
                           (ctypes.c_float * 3)(*[float(x) for x in origin]), float(extent), float(mu),
                           int(w_max), float(sigma), float(gate), int(variant))
        nx, ny, nz = self.dims_geo
        if allocate:
            self.geo = np.zeros((nz, ny, nx), dtype=np.uint32)                     # weight 0 = never observed
            self.col = np.zeros((nz * self.r, ny * self.r, nx * self.r), dtype=np.uint32)
        self.counters = []

    def _frame(self, depth, rgb, T_world_depth, K_depth, K_rgb, T_depth_rgb):
        depth = np.ascontiguousarray(depth, dtype=np.uint16)
        rgb = np.ascontiguousarray(rgb, dtype=np.uint8)
        assert depth.ndim == 2 and rgb.ndim == 3 and rgb.shape[2] == 3
        fr = RefFrame()
        fr.depth, fr.hd, fr.wd = depth.ctypes.data, depth.shape[0], depth.shape[1]
        fr.rgb, fr.hh, fr.wh = rgb.ctypes.data, rgb.shape[0], rgb.shape[1]
        fr.T_world_depth[:] = _f32(T_world_depth, 16).tolist()
        fr.K_depth[:] = _f32(K_depth, 9).tolist()
        fr.K_rgb[:] = _f32(K_rgb, 9).tolist()
        fr.T_depth_rgb[:] = _f32(T_depth_rgb, 16).tolist()
        return fr, (depth, rgb)

    def integrate(self, depth, rgb, T_world_depth, K_depth, K_rgb, T_depth_rgb):
        """One frame over both whole volumes.  Returns this frame's counters
        [geo_read, geo_changed, col_read, col_changed]."""
        fr, keep = self._frame(depth, rgb, T_world_depth, K_depth, K_rgb, T_depth_rgb)
        cnt = np.zeros(4, dtype=np.uint64)
        rc = _load().ref_integrate(ctypes.addressof(self.desc), ctypes.addressof(fr),
                                   self.geo.ctypes.data, self.col.ctypes.data, cnt.ctypes.data)
        if rc != 0:
            raise ValueError("ref_integrate: bad arguments")
        self.counters.append(cnt)
        return cnt

    def integrate_sectors(self, depth, rgb, T_world_depth, K_depth, K_rgb, T_depth_rgb):
        """integrate() that also counts the distinct 32-byte sectors (8 consecutive words) holding a read / changed voxel:
        returns [geo_read, geo_changed, col_read, col_changed, geo_sectors_read, geo_sectors_written, col_sectors_read,
        col_sectors_written]."""
        fr, keep = self._frame(depth, rgb, T_world_depth, K_depth, K_rgb, T_depth_rgb)
        cnt = np.zeros(4, dtype=np.uint64)
        maps = [np.zeros((a.size + 7) // 8, np.uint8) for a in (self.geo, self.geo, self.col, self.col)]
        rc = _load().ref_integrate_sectors(ctypes.addressof(self.desc), ctypes.addressof(fr), self.geo.ctypes.data, self.col.ctypes.data,
                                           cnt.ctypes.data, *[m.ctypes.data for m in maps])
        if rc != 0:
            raise ValueError("ref_integrate_sectors: bad arguments")
        self.counters.append(cnt)
        return np.concatenate([cnt, np.array([int(m.sum(dtype=np.uint64)) for m in maps], np.uint64)])

    def integrate_subset(self, geo_idx, geo_words, col_idx, col_words, depth, rgb, T_world_depth, K_depth, K_rgb,
                         T_depth_rgb):
        """One frame applied only to the listed voxels (linear indices; words updated in place)."""
        fr, keep = self._frame(depth, rgb, T_world_depth, K_depth, K_rgb, T_depth_rgb)
        for a, dt in ((geo_idx, np.int64), (col_idx, np.int64), (geo_words, np.uint32), (col_words, np.uint32)):
            assert a.dtype == dt and a.flags.c_contiguous
        rc = _load().ref_integrate_subset(ctypes.addressof(self.desc), ctypes.addressof(fr),
                                          geo_idx.ctypes.data, geo_idx.size, geo_words.ctypes.data,
                                          col_idx.ctypes.data, col_idx.size, col_words.ctypes.data)
        if rc != 0:
            raise ValueError("ref_integrate_subset: bad arguments")

    def sample_colour(self, pts):
        """ref_sample_colour: packed colour words (uint32 [n]) of the colour voxels containing the world points pts [n, 3]."""
        pts = np.ascontiguousarray(pts, dtype=np.float32).reshape(-1, 3)
        out = np.zeros(pts.shape[0], dtype=np.uint32)
        rc = _load().ref_sample_colour(ctypes.addressof(self.desc), self.col.ctypes.data, pts.ctypes.data, pts.shape[0], out.ctypes.data)
        if rc != 0:
            raise ValueError("ref_sample_colour: bad arguments")
        return out

    def sample_colour_trilinear(self, pts):
        """ref_sample_colour_trilinear: trilinearly interpolated colour words (uint32 [n]) at the world points pts [n, 3]."""
        pts = np.ascontiguousarray(pts, dtype=np.float32).reshape(-1, 3)
        out = np.zeros(pts.shape[0], dtype=np.uint32)
        rc = _load().ref_sample_colour_trilinear(ctypes.addressof(self.desc), self.col.ctypes.data, pts.ctypes.data, pts.shape[0], out.ctypes.data)
        if rc != 0:
            raise ValueError("ref_sample_colour_trilinear: bad arguments")
        return out

    def raycast(self, w, h, T_world_cam, K, t_near, t_far):
        """ref_raycast: (depth float32 [h, w] metres, 0 = no surface; rgb uint8 [h, w, 3]) seen by a virtual camera."""
        T, Kc = _f32(T_world_cam, 16), _f32(K, 9)
        depth = np.zeros((h, w), dtype=np.float32)
        rgb = np.zeros((h, w, 3), dtype=np.uint8)
        rc = _load().ref_raycast(ctypes.addressof(self.desc), self.geo.ctypes.data, self.col.ctypes.data, int(w), int(h),
                                 T.ctypes.data, Kc.ctypes.data, float(t_near), float(t_far), depth.ctypes.data, rgb.ctypes.data)
        if rc != 0:
            raise ValueError("ref_raycast: bad arguments")
        return depth, rgb

    def raycast_trilinear(self, w, h, T_world_cam, K, t_near, t_far):
        """ref_raycast_trilinear (reading R7): as raycast(), the TSDF of a sample interpolated from the 8 surrounding voxels."""
        T, Kc = _f32(T_world_cam, 16), _f32(K, 9)
        depth = np.zeros((h, w), dtype=np.float32)
        rgb = np.zeros((h, w, 3), dtype=np.uint8)
        rc = _load().ref_raycast_trilinear(ctypes.addressof(self.desc), self.geo.ctypes.data, self.col.ctypes.data, int(w), int(h),
                                           T.ctypes.data, Kc.ctypes.data, float(t_near), float(t_far), depth.ctypes.data, rgb.ctypes.data)
        if rc != 0:
            raise ValueError("ref_raycast_trilinear: bad arguments")
        return depth, rgb

    def frame_constants(self, T_world_depth, T_depth_rgb):
        dummy_d = np.zeros((1, 1), np.uint16)
        dummy_c = np.zeros((1, 1, 3), np.uint8)
        fr, keep = self._frame(dummy_d, dummy_c, T_world_depth, np.eye(3), np.eye(3), T_depth_rgb)
        out = np.zeros(24, dtype=np.float32)
        _load().ref_frame_constants(ctypes.addressof(self.desc), ctypes.addressof(fr), out.ctypes.data)
        return out[0:9].reshape(3, 3), out[9:12], out[12:21].reshape(3, 3), out[21:24]


# unpack helpers (layout only; used by tests on either side's downloaded state)
def threads() -> int:
    """OpenMP threads the oracle's loops use (omp_get_max_threads)."""
    return int(_load().ref_threads())


def geo_q(words):
    return (words & np.uint32(0xffff)).astype(np.uint16).view(np.int16).astype(np.int32)


def geo_w(words):
    return (words >> np.uint32(16)).astype(np.uint16).view(np.int16).astype(np.int32)


def col_rgb(words):
    return np.stack([(words >> np.uint32(8 * c)) & np.uint32(0xff) for c in range(3)], axis=-1).astype(np.int32)


def col_w(words):
    return (words >> np.uint32(24)).astype(np.int32)
