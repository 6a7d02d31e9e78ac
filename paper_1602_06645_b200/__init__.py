"""paper_1602_06645_b200 -- B200-native fused TSDF + asymmetrical colour-volume integration (arXiv 1602.06645).

Thin ctypes binding over the C ABI declared in ``include/volfusion.h`` (same names, argument marshalling only:
every step of the path runs in the sm_100a kernels of ``csrc/``).  PyTorch is used by callers for device memory and
streams; this module only needs ``data_ptr()`` of CUDA tensors.  There is no CPU fallback: if ``libvolfusion.so`` is
missing or no CUDA device is usable, calls raise.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_ROOT = os.path.dirname(_HERE)
_SRC_DIR = os.path.join(_HERE, "csrc")
_SO = os.path.join(_HERE, "libvolfusion.so")
_lib = None

VOL_OK, VOL_E_ARG, VOL_E_OOM, VOL_E_CUDA, VOL_E_LOST, VOL_E_TOOBIG = 0, -1, -2, -3, -4, -5
VOL_SLAB = 8
VOL_STATS_RAW_BYTES = 128

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "--fmad=false", "-std=c++17",
              "-Xcompiler", "-fPIC,-ffp-contract=off", "-shared"]

EXPORTS = ["vol_create", "vol_integrate", "vol_integrate_host", "vol_raycast", "vol_raycast_trilinear", "vol_sample_colour", "vol_sample_colour_trilinear", "vol_download", "vol_download_voxels", "vol_upload",
           "vol_reset", "vol_info", "vol_shard_layers", "vol_set_counting", "vol_frame_stats", "vol_frame_stats_async", "vol_stats_decode", "vol_set_profiling", "vol_last_kernel_ms",
           "vol_launches_per_frame", "vol_selftest", "vol_destroy", "vol_strerror",
           # include/volfrontend.h
           "vol_frontend_create", "vol_frontend_destroy", "vol_frontend_measure", "vol_frontend_predict_depth", "vol_frontend_predict",
           "vol_frontend_icp_step", "vol_frontend_track", "vol_frontend_track_info", "vol_frontend_maps",
           "vol_icp_step_static"]


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile csrc/volfusion.cu for sm_100a into libvolfusion.so (in-tree; nvcc cross-compiles without a GPU)."""
    srcs = [os.path.join(_SRC_DIR, f) for f in os.listdir(_SRC_DIR)] + [os.path.join(_ROOT, "include", f) for f in os.listdir(os.path.join(_ROOT, "include"))]
    newest = max(os.path.getmtime(s) for s in srcs)
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < newest:
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + [os.path.join(_SRC_DIR, "volfusion.cu"), "-o", _SO]
        subprocess.run(cmd, check=True)
    return _SO


class VolOpts(ctypes.Structure):
    _fields_ = [("sigma_m", ctypes.c_float), ("gate", ctypes.c_float), ("geo_dev", ctypes.c_void_p),
                ("col_dev", ctypes.c_void_p), ("device", ctypes.c_int32), ("shard_rank", ctypes.c_int32),
                ("shard_world", ctypes.c_int32), ("variant", ctypes.c_int32)]


# vol_opts_t.variant: alternative readings of the method (volfusion.h), one at a time
VARIANT_HD_FROM_DEPTH_POINT, VARIANT_TSDF_ALONG_RAY, VARIANT_ADDITIVE_WEIGHT = 1, 2, 4


class VolInfo(ctypes.Structure):
    _fields_ = [("dims_geo", ctypes.c_int32 * 3), ("r", ctypes.c_int32), ("dims_col", ctypes.c_int32 * 3),
                ("local_nz_geo", ctypes.c_int32), ("voxel_geo_m", ctypes.c_float), ("voxel_col_m", ctypes.c_float),
                ("origin_m", ctypes.c_float * 3), ("extent_m", ctypes.c_float), ("trunc_mu_m", ctypes.c_float),
                ("sigma_m", ctypes.c_float), ("gate", ctypes.c_float), ("w_max", ctypes.c_int32),
                ("device", ctypes.c_int32), ("shard_rank", ctypes.c_int32), ("shard_world", ctypes.c_int32),
                ("variant", ctypes.c_int32), ("geo_bytes", ctypes.c_uint64), ("col_bytes", ctypes.c_uint64), ("geo_dev", ctypes.c_void_p),
                ("col_dev", ctypes.c_void_p)]


class VolStats(ctypes.Structure):
    _fields_ = [("geo_read", ctypes.c_uint64), ("geo_changed", ctypes.c_uint64), ("col_read", ctypes.c_uint64),
                ("col_changed", ctypes.c_uint64), ("tiles_total", ctypes.c_uint32), ("tiles_geo", ctypes.c_uint32),
                ("items_col", ctypes.c_uint32), ("cells_col", ctypes.c_uint32),
                ("geo_sectors_read", ctypes.c_uint64), ("geo_sectors_written", ctypes.c_uint64),
                ("col_sectors_read", ctypes.c_uint64), ("col_sectors_written", ctypes.c_uint64),
                ("geo_visited", ctypes.c_uint64), ("col_gated", ctypes.c_uint64), ("geo_skippable", ctypes.c_uint64),
                ("geo_sectors_skippable", ctypes.c_uint64),
                ("subs_geo", ctypes.c_uint32), ("jobs_mark", ctypes.c_uint32)]


def lib():
    """Load libvolfusion.so (building it if the sources are newer) and declare the prototypes."""
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_SO)
        P, I32, I64, F = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_float
        L.vol_create.argtypes = [ctypes.POINTER(P), P, I32, P, F, F, I32, P]
        L.vol_integrate.argtypes = [P, P, I32, I32, P, I32, I32, P, P, P, P, P]
        L.vol_integrate_host.argtypes = L.vol_integrate.argtypes
        L.vol_raycast.argtypes = [P, I32, I32, P, P, F, F, P, P, P]
        L.vol_raycast_trilinear.argtypes = [P, I32, I32, P, P, F, F, P, P, P]
        L.vol_sample_colour.argtypes = [P, P, I64, P, P]
        L.vol_sample_colour_trilinear.argtypes = [P, P, I64, P, P]
        L.vol_download.argtypes = [P, P, ctypes.c_size_t, P, ctypes.c_size_t, P]
        L.vol_download_voxels.argtypes = [P, P, I64, P, P, I64, P, P]
        L.vol_upload.argtypes = [P, P, P, P]
        L.vol_reset.argtypes = [P, P]
        L.vol_info.argtypes = [P, P]
        L.vol_shard_layers.argtypes = [I32, I32, I32, P, I32]
        L.vol_set_counting.argtypes = [P, I32]
        L.vol_frame_stats.argtypes = [P, P, P]
        L.vol_frame_stats_async.argtypes = [P, P, P]
        L.vol_stats_decode.argtypes = [P, P, P]
        L.vol_set_profiling.argtypes = [P, I32]
        L.vol_last_kernel_ms.argtypes = [P, P]
        L.vol_launches_per_frame.argtypes = [P]
        L.vol_selftest.argtypes = [P, I32]
        L.vol_destroy.argtypes = [P]
        L.vol_destroy.restype = None
        L.vol_strerror.argtypes = [ctypes.c_int]
        L.vol_strerror.restype = ctypes.c_char_p
        L.vol_frontend_create.argtypes = [ctypes.POINTER(P), I32, I32, I32, P]
        L.vol_frontend_destroy.argtypes = [P]
        L.vol_frontend_destroy.restype = None
        L.vol_frontend_measure.argtypes = [P, P, P, P]
        L.vol_frontend_predict_depth.argtypes = [P, P, P, I32, P]
        L.vol_frontend_predict.argtypes = [P, P, P, P, F, F, P]
        L.vol_frontend_icp_step.argtypes = [P, I32, P, P, P]
        L.vol_frontend_track.argtypes = [P, P, P, P, P, P, P]
        L.vol_frontend_track_info.argtypes = [P, P, P, P]
        L.vol_frontend_maps.argtypes = [P, I32, I32, P, P, P, P]
        L.vol_icp_step_static.argtypes = [P, P, P, P, I32, I32, P, P, F, F, P, P]
        for name in EXPORTS:
            if name not in ("vol_destroy", "vol_strerror", "vol_frontend_destroy"):
                getattr(L, name).restype = ctypes.c_int
        _lib = L
    return _lib


class VolError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        super().__init__(f"{where}: {lib().vol_strerror(code).decode()} ({code})")


def _check(rc: int, where: str):
    if rc != VOL_OK:
        raise VolError(rc, where)


def _f32(a, n):
    a = np.ascontiguousarray(np.asarray(a, dtype=np.float32).reshape(-1))
    if a.size != n:
        raise ValueError(f"expected {n} floats, got {a.size}")
    return a


def _dev_ptr(t):
    """Device pointer of a CUDA tensor (anything with .data_ptr() and .is_cuda) or a raw int address."""
    if isinstance(t, int):
        return t
    if not getattr(t, "is_cuda", False):
        raise TypeError("expected a CUDA tensor (or an int device address)")
    if not t.is_contiguous():
        raise ValueError("CUDA tensor must be contiguous")
    return t.data_ptr()


def _stream_ptr(stream):
    if stream is None:
        return None
    return getattr(stream, "cuda_stream", stream)


def shard_layers(nz: int, shard_rank: int, shard_world: int):
    """vol_shard_layers: the geometry layers (global indices, storage order) that rank `shard_rank` of `shard_world` owns."""
    n = lib().vol_shard_layers(int(nz), int(shard_rank), int(shard_world), None, 0)
    _check(min(n, 0), "vol_shard_layers")
    out = np.empty(n, dtype=np.int32)
    _check(min(lib().vol_shard_layers(int(nz), int(shard_rank), int(shard_world), out.ctypes.data, n), 0), "vol_shard_layers")
    return out


def selftest(exhaustive: bool = False):
    """vol_selftest: (reciprocal, TSDF-quotient, colour-quotient) mismatches of the branch-free exact arithmetic; all must be 0."""
    out = (ctypes.c_uint64 * 3)()
    _check(lib().vol_selftest(out, int(exhaustive)), "vol_selftest")
    return int(out[0]), int(out[1]), int(out[2])


class Volume:
    """A geometry (TSDF) volume and its asymmetrical colour volume on one GPU (or one z-slab shard of them)."""

    def __init__(self, dims_geo, r, origin, extent, mu, w_max, sigma=0.0, gate=0.0, device=-1, shard_rank=0,
                 shard_world=1, geo_dev=None, col_dev=None, variant=0):
        self._h = ctypes.c_void_p()
        dims = (ctypes.c_int32 * 3)(*[int(d) for d in dims_geo])
        org = (ctypes.c_float * 3)(*[float(x) for x in origin])
        opts = VolOpts(float(sigma), float(gate), geo_dev, col_dev, int(device), int(shard_rank), int(shard_world), int(variant))
        rc = lib().vol_create(ctypes.byref(self._h), dims, int(r), org, float(extent), float(mu), int(w_max), ctypes.byref(opts))
        if rc != VOL_OK:
            self._h = ctypes.c_void_p()
        _check(rc, "vol_create")
        self.info = self._info()

    def _info(self) -> VolInfo:
        o = VolInfo()
        _check(lib().vol_info(self._h, ctypes.byref(o)), "vol_info")
        return o

    def _mats(self, T_world_depth, K_depth, K_rgb, T_depth_rgb):
        return (_f32(T_world_depth, 16), _f32(K_depth, 9), _f32(K_rgb, 9), _f32(T_depth_rgb, 16))

    def integrate(self, depth_dev, wd, hd, rgb_dev, wh, hh, T_world_depth, K_depth, K_rgb, T_depth_rgb, stream=None):
        """vol_integrate: fuse one frame whose images are already resident on the device."""
        T, Kd, Kh, Tc = self._mats(T_world_depth, K_depth, K_rgb, T_depth_rgb)
        _check(lib().vol_integrate(self._h, _dev_ptr(depth_dev), wd, hd, _dev_ptr(rgb_dev), wh, hh, T.ctypes.data,
                                   Kd.ctypes.data, Kh.ctypes.data, Tc.ctypes.data, _stream_ptr(stream)), "vol_integrate")

    def integrate_host(self, depth, rgb, T_world_depth, K_depth, K_rgb, T_depth_rgb, stream=None):
        """vol_integrate_host: images are host arrays (numpy uint16 [hd,wd] / uint8 [hh,wh,3], or pinned CPU tensors)."""
        T, Kd, Kh, Tc = self._mats(T_world_depth, K_depth, K_rgb, T_depth_rgb)
        if isinstance(depth, np.ndarray):
            assert depth.dtype == np.uint16 and depth.flags.c_contiguous and rgb.dtype == np.uint8 and rgb.flags.c_contiguous
            dp, cp = depth.ctypes.data, rgb.ctypes.data
        else:                                           # CPU torch tensors (pinned)
            assert not depth.is_cuda and not rgb.is_cuda and depth.is_contiguous() and rgb.is_contiguous()
            dp, cp = depth.data_ptr(), rgb.data_ptr()
        hd, wd = int(depth.shape[0]), int(depth.shape[1])
        hh, wh = int(rgb.shape[0]), int(rgb.shape[1])
        _check(lib().vol_integrate_host(self._h, dp, wd, hd, cp, wh, hh, T.ctypes.data, Kd.ctypes.data, Kh.ctypes.data,
                                        Tc.ctypes.data, _stream_ptr(stream)), "vol_integrate_host")

    def raycast(self, w, h, T_world_cam, K, t_near, t_far, depth_dev, rgb_dev=None, stream=None):
        """vol_raycast: depth_dev = CUDA float32 tensor of w*h elements, rgb_dev = CUDA uint8 tensor of w*h*3 (or None)."""
        T, Kc = _f32(T_world_cam, 16), _f32(K, 9)
        _check(lib().vol_raycast(self._h, int(w), int(h), T.ctypes.data, Kc.ctypes.data, float(t_near), float(t_far),
                                 _dev_ptr(depth_dev), None if rgb_dev is None else _dev_ptr(rgb_dev), _stream_ptr(stream)), "vol_raycast")

    def raycast_trilinear(self, w, h, T_world_cam, K, t_near, t_far, depth_dev, rgb_dev=None, stream=None):
        """vol_raycast_trilinear: as raycast(), the TSDF of a sample interpolated from the 8 surrounding voxels (reading R7)."""
        T, Kc = _f32(T_world_cam, 16), _f32(K, 9)
        _check(lib().vol_raycast_trilinear(self._h, int(w), int(h), T.ctypes.data, Kc.ctypes.data, float(t_near), float(t_far),
                                           _dev_ptr(depth_dev), None if rgb_dev is None else _dev_ptr(rgb_dev), _stream_ptr(stream)),
               "vol_raycast_trilinear")

    def sample_colour(self, points_dev, n, words_dev, stream=None):
        """vol_sample_colour: points_dev = CUDA float32 tensor [n, 3] (world), words_dev = CUDA int32/uint32 tensor [n]."""
        _check(lib().vol_sample_colour(self._h, _dev_ptr(points_dev), int(n), _dev_ptr(words_dev), _stream_ptr(stream)), "vol_sample_colour")

    def sample_colour_trilinear(self, points_dev, n, words_dev, stream=None):
        """vol_sample_colour_trilinear: same arguments as sample_colour; trilinear interpolation over observed voxels."""
        _check(lib().vol_sample_colour_trilinear(self._h, _dev_ptr(points_dev), int(n), _dev_ptr(words_dev), _stream_ptr(stream)),
               "vol_sample_colour_trilinear")

    def download(self, stream=None):
        """vol_download: (geo uint32 [local_nz, Ny, Nx], col uint32 [r*local_nz, r*Ny, r*Nx]) of this shard."""
        i = self.info
        geo = np.empty((i.local_nz_geo, i.dims_geo[1], i.dims_geo[0]), dtype=np.uint32)
        col = np.empty((i.local_nz_geo * i.r, i.dims_col[1], i.dims_col[0]), dtype=np.uint32)
        _check(lib().vol_download(self._h, geo.ctypes.data, geo.nbytes, col.ctypes.data, col.nbytes, _stream_ptr(stream)), "vol_download")
        return geo, col

    def download_voxels(self, geo_idx, col_idx, stream=None):
        geo_idx = np.ascontiguousarray(geo_idx, dtype=np.int64)
        col_idx = np.ascontiguousarray(col_idx, dtype=np.int64)
        gw, cw = np.empty(geo_idx.size, np.uint32), np.empty(col_idx.size, np.uint32)
        _check(lib().vol_download_voxels(self._h, geo_idx.ctypes.data, geo_idx.size, gw.ctypes.data, col_idx.ctypes.data,
                                         col_idx.size, cw.ctypes.data, _stream_ptr(stream)), "vol_download_voxels")
        return gw, cw

    def upload(self, geo=None, col=None, stream=None):
        for a, nb in ((geo, self.info.geo_bytes), (col, self.info.col_bytes)):
            if a is not None:
                assert a.dtype == np.uint32 and a.flags.c_contiguous and a.nbytes == nb
        _check(lib().vol_upload(self._h, None if geo is None else geo.ctypes.data, None if col is None else col.ctypes.data,
                                _stream_ptr(stream)), "vol_upload")

    def reset(self, stream=None):
        _check(lib().vol_reset(self._h, _stream_ptr(stream)), "vol_reset")

    def set_counting(self, on: bool):
        _check(lib().vol_set_counting(self._h, int(on)), "vol_set_counting")

    def frame_stats(self, stream=None) -> VolStats:
        s = VolStats()
        _check(lib().vol_frame_stats(self._h, ctypes.byref(s), _stream_ptr(stream)), "vol_frame_stats")
        return s

    def frame_stats_async(self, raw_host, stream=None):
        """vol_frame_stats_async: raw_host = pinned CPU tensor of >= VOL_STATS_RAW_BYTES; filled in stream order, no synchronisation."""
        assert not raw_host.is_cuda and raw_host.is_pinned() and raw_host.numel() * raw_host.element_size() >= VOL_STATS_RAW_BYTES
        _check(lib().vol_frame_stats_async(self._h, raw_host.data_ptr(), _stream_ptr(stream)), "vol_frame_stats_async")

    def decode_stats(self, raw_host) -> VolStats:
        """vol_stats_decode of a record written by frame_stats_async (after the stream has passed it)."""
        s = VolStats()
        _check(lib().vol_stats_decode(self._h, raw_host.data_ptr(), ctypes.byref(s)), "vol_stats_decode")
        return s

    def set_profiling(self, on: bool):
        _check(lib().vol_set_profiling(self._h, int(on)), "vol_set_profiling")

    def last_kernel_ms(self):
        ms = (ctypes.c_float * 3)()
        _check(lib().vol_last_kernel_ms(self._h, ms), "vol_last_kernel_ms")
        return [float(x) for x in ms]

    def launches_per_frame(self) -> int:
        return int(lib().vol_launches_per_frame(self._h))

    def close(self):
        if getattr(self, "_h", None) is not None and self._h:
            lib().vol_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()


class FrontendOpts(ctypes.Structure):
    _fields_ = [("sigma_s_px", ctypes.c_float), ("sigma_r_m", ctypes.c_float), ("dist_m", ctypes.c_float),
                ("cos_min", ctypes.c_float), ("device", ctypes.c_int32), ("cond_min", ctypes.c_float),
                ("trilinear_prediction", ctypes.c_int32)]


ICP_SUMS = 29


ICP_STATIC_MAX_BLOCKS = 8192


def icp_step_static(V, N, Vp, Np, w, h, K, T_pred_cur, sums_out, dist_m=0.0, cos_min=0.0, stream=None):
    """vol_icp_step_static: one F5 step without any allocation.  V, N, Vp, Np: CUDA float32 tensors of w*h*4 (x, y, z, 0);
    K: intrinsics of this level; sums_out: CUDA float64 tensor of ICP_SUMS, written in stream order (asynchronous)."""
    Kc, T = _f32(K, 9), _f32(T_pred_cur, 16)
    _check(lib().vol_icp_step_static(_dev_ptr(V), _dev_ptr(N), _dev_ptr(Vp), _dev_ptr(Np), int(w), int(h), Kc.ctypes.data, T.ctypes.data,
                                     float(dist_m), float(cos_min), _dev_ptr(sums_out), _stream_ptr(stream)), "vol_icp_step_static")


class Frontend:
    """include/volfrontend.h: depth front end (bilateral filter, vertex / normal map pyramid) and ICP tracking against a
    ray-cast prediction -- the measured and predicted map pyramids of one image size on one GPU."""

    def __init__(self, w, h, levels=3, sigma_s_px=0.0, sigma_r_m=0.0, dist_m=0.0, cos_min=0.0, device=-1, cond_min=0.0, trilinear_prediction=False):
        self._h = ctypes.c_void_p()
        self.w, self.h, self.levels = int(w), int(h), int(levels)
        opts = FrontendOpts(float(sigma_s_px), float(sigma_r_m), float(dist_m), float(cos_min), int(device), float(cond_min), int(bool(trilinear_prediction)))
        rc = lib().vol_frontend_create(ctypes.byref(self._h), self.w, self.h, self.levels, ctypes.byref(opts))
        if rc != VOL_OK:
            self._h = ctypes.c_void_p()
        _check(rc, "vol_frontend_create")

    def measure(self, depth_dev, K, stream=None):
        """vol_frontend_measure: depth_dev = CUDA tensor of w*h uint16 millimetres (any 2-byte dtype)."""
        Kc = _f32(K, 9)
        _check(lib().vol_frontend_measure(self._h, _dev_ptr(depth_dev), Kc.ctypes.data, _stream_ptr(stream)), "vol_frontend_measure")

    def predict_depth(self, depth_m_dev, K, filter=False, stream=None):
        """vol_frontend_predict_depth: depth_m_dev = CUDA float32 tensor of w*h metres; filter=True for ray-cast maps (F8)."""
        Kc = _f32(K, 9)
        _check(lib().vol_frontend_predict_depth(self._h, _dev_ptr(depth_m_dev), Kc.ctypes.data, int(bool(filter)), _stream_ptr(stream)),
               "vol_frontend_predict_depth")

    def predict(self, volume, T_world_cam, K, t_near, t_far, stream=None):
        """vol_frontend_predict: ray-cast `volume` from T_world_cam and build the predicted maps."""
        T, Kc = _f32(T_world_cam, 16), _f32(K, 9)
        _check(lib().vol_frontend_predict(self._h, volume._h, T.ctypes.data, Kc.ctypes.data, float(t_near), float(t_far), _stream_ptr(stream)),
               "vol_frontend_predict")

    def icp_step(self, level, T_pred_cur, stream=None):
        """vol_frontend_icp_step: (A [6,6], b [6], sum r^2, count) of one linearised step at `level`."""
        T = _f32(T_pred_cur, 16)
        s = np.zeros(ICP_SUMS, np.float64)
        _check(lib().vol_frontend_icp_step(self._h, int(level), T.ctypes.data, s.ctypes.data, _stream_ptr(stream)), "vol_frontend_icp_step")
        A = np.zeros((6, 6))
        A[np.triu_indices(6)] = s[:21]
        A = A + np.triu(A, 1).T
        return A, s[21:27].copy(), float(s[27]), int(s[28])

    def track(self, T_init=None, iterations=(10, 5, 4), stream=None):
        """vol_frontend_track: (T_pred_cur float32 [4,4], rms, count); raises VolError(VOL_E_LOST) when tracking is lost."""
        it = np.ascontiguousarray(np.asarray(iterations, np.int32))
        assert it.size == self.levels
        Ti = None if T_init is None else _f32(T_init, 16)
        out = np.zeros(16, np.float32)
        rms, cnt = ctypes.c_double(0.0), ctypes.c_int64(0)
        _check(lib().vol_frontend_track(self._h, None if Ti is None else Ti.ctypes.data, it.ctypes.data, out.ctypes.data,
                                        ctypes.byref(rms), ctypes.byref(cnt), _stream_ptr(stream)), "vol_frontend_track")
        return out.reshape(4, 4), rms.value, cnt.value

    def track_info(self):
        """vol_frontend_track_info: (status, level, conditioning) of the last step of the most recent track()."""
        st, lv, cond = ctypes.c_int32(0), ctypes.c_int32(0), ctypes.c_double(0.0)
        _check(lib().vol_frontend_track_info(self._h, ctypes.byref(st), ctypes.byref(lv), ctypes.byref(cond)), "vol_frontend_track_info")
        return st.value, lv.value, cond.value

    def maps(self, which, level, stream=None):
        """vol_frontend_maps: (D [h,w], V [h,w,3], N [h,w,3]) float32 of one level; which = 0 measured, 1 predicted."""
        wl, hl = self.w >> level, self.h >> level
        D, V, N = np.zeros((hl, wl), np.float32), np.zeros((hl, wl, 3), np.float32), np.zeros((hl, wl, 3), np.float32)
        _check(lib().vol_frontend_maps(self._h, int(which), int(level), D.ctypes.data, V.ctypes.data, N.ctypes.data, _stream_ptr(stream)),
               "vol_frontend_maps")
        return D, V, N

    def close(self):
        if self._h:
            lib().vol_frontend_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
