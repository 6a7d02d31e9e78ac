"""Seeded synthetic RGB-D input generator (HARNESS ONLY).

This module is the one piece shared by the CPU oracle (``oracle/``) and the CUDA
path (``paper_1602_06645_b200/``): it produces the *inputs* -- depth frames
(uint16 mm, 0 = invalid), RGB8 frames, poses and calibration -- and holds none of
the method's arithmetic.  Neither ``oracle`` nor the CUDA package is imported here.

The five configurations are the ones of BASELINE.json ``configs`` (restated in
SURVEY.md section 8(d)); they are synthetic stand-ins for the paper's handheld
Kinect + HD-camera scans of a lunch bag and a backpack, which are
not public.  Recipe and conventions: DESIGN.md "Synthetic inputs".

Conventions
-----------
* Camera frame: x right, y down, z forward.  Pixel (x, y) <-> ray
  ((x-cx)/fx, (y-cy)/fy, 1); pixel centres sit at integer coordinates.
* ``T_a_b`` maps b-coordinates to a-coordinates (row-major 4x4, float32).
* Depth = z-depth of the nearest analytic hit + noise, ``clip(rint(1000 z), 1, 65535)``,
  misses and dropouts are 0.  RGB = albedo texture at the hit point, no shading.
* Seeds: ``numpy.random.default_rng(160206645 + 1000*cfg + frame)``.
"""
from __future__ import annotations

import ctypes
import dataclasses
import os
import subprocess
from typing import Callable, Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "_render.so")
_SRC = os.path.join(_HERE, "render.c")
_lib = None

SEED0 = 160206645
MAX_RANGE_M = 8.0      # hits beyond the sensor's range read as invalid (0)

PRIM_SPHERE, PRIM_BOX, PRIM_PLANE, PRIM_CYLINDER, PRIM_TORUS = 0, 1, 2, 3, 4
TEX_CONST, TEX_CHECKER, TEX_NOISE, TEX_STRIPES = 0, 1, 2, 3


def build(force: bool = False) -> str:
    """Compile synth/render.c with gcc (idempotent)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-ffp-contract=off", "-shared", "-fPIC", _SRC, "-o", _SO, "-lm"]
        subprocess.run(cmd, check=True)
    return _SO


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_SO)
        lib.synth_render.restype = ctypes.c_int
        lib.synth_render.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p,
                                     ctypes.c_int, ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
        _lib = lib
    return _lib


def prim(ptype, tex, seed, centre, size, scale=1.0, colour=(128, 128, 128)):
    p = np.zeros(16, dtype=np.float64)
    p[0], p[1], p[2] = ptype, tex, seed
    p[3:6] = centre
    s = list(size) + [0.0] * (3 - len(size))
    p[6:9] = s
    p[9] = scale
    p[10:13] = colour
    return p


def render(prims: np.ndarray, K: np.ndarray, T_world_cam: np.ndarray, w: int, h: int,
           want_depth: bool, want_rgb: bool, bg=(128, 128, 128)):
    """Ray-cast ``prims`` from one camera.  Returns (z-depth float32 [h,w] | None, rgb8 [h,w,3] | None)."""
    lib = _load()
    prims = np.ascontiguousarray(prims, dtype=np.float64).reshape(-1, 16)
    K = np.asarray(K, dtype=np.float64)
    k4 = np.array([K[0, 0], K[1, 1], K[0, 2], K[1, 2]], dtype=np.float64)
    T = np.ascontiguousarray(T_world_cam, dtype=np.float64)
    depth = np.empty((h, w), dtype=np.float32) if want_depth else None
    rgb = np.empty((h, w, 3), dtype=np.uint8) if want_rgb else None
    bgc = np.array(bg, dtype=np.uint8)
    rc = lib.synth_render(prims.ctypes.data, prims.shape[0], k4.ctypes.data, T.ctypes.data, w, h,
                          depth.ctypes.data if want_depth else None,
                          rgb.ctypes.data if want_rgb else None, bgc.ctypes.data)
    assert rc == 0
    return depth, rgb


# ----------------------------------------------------------------------------------------------
# poses
# ----------------------------------------------------------------------------------------------

def look_at(eye, target, up=(0.0, 0.0, 1.0)) -> np.ndarray:
    """T_world_cam (float64 4x4): camera z looks from ``eye`` to ``target``; x right, y down."""
    eye = np.asarray(eye, dtype=np.float64)
    f = np.asarray(target, dtype=np.float64) - eye
    f /= np.linalg.norm(f)
    r = np.cross(f, np.asarray(up, dtype=np.float64))
    r /= np.linalg.norm(r)
    d = np.cross(f, r)
    T = np.eye(4)
    T[:3, 0], T[:3, 1], T[:3, 2], T[:3, 3] = r, d, f, eye
    return T


def rot_axis(axis, ang) -> np.ndarray:
    a = np.asarray(axis, dtype=np.float64)
    a = a / np.linalg.norm(a)
    Kx = np.array([[0, -a[2], a[1]], [a[2], 0, -a[0]], [-a[1], a[0], 0]])
    return np.eye(3) + np.sin(ang) * Kx + (1 - np.cos(ang)) * (Kx @ Kx)


def intrinsics(f, cx, cy) -> np.ndarray:
    return np.array([[f, 0, cx], [0, f, cy], [0, 0, 1]], dtype=np.float32)


def rigid32(T64: np.ndarray) -> np.ndarray:
    """Re-orthonormalise in float64 (SVD) and round once to float32."""
    T = np.array(T64, dtype=np.float64)
    U, _, Vt = np.linalg.svd(T[:3, :3])
    T[:3, :3] = U @ Vt
    T[3] = [0, 0, 0, 1]
    return T.astype(np.float32)


# ----------------------------------------------------------------------------------------------
# configurations
# ----------------------------------------------------------------------------------------------

@dataclasses.dataclass
class Config:
    cfg: int
    name: str
    dims_geo: tuple
    r: int
    origin: np.ndarray            # float32[3], world position of the volume corner
    extent: float                 # metres along x; voxel = extent / dims_geo[0] (cubic)
    mu: float
    w_max: int
    wd: int
    hd: int
    wh: int
    hh: int
    K_depth: np.ndarray
    K_rgb: np.ndarray
    T_depth_rgb: np.ndarray       # float32 4x4: RGB-camera coords -> depth-camera coords
    n_frames: int
    prims: np.ndarray
    pose: Callable[[int], np.ndarray]   # frame -> T_world_depth float64
    noise: Callable[[np.ndarray], np.ndarray]   # z -> sigma(z) metres
    dropout: float
    bg: tuple = (128, 128, 128)
    sigma: float = 0.020
    gate: float = 0.8

    @property
    def dims_col(self):
        return tuple(int(d) * self.r for d in self.dims_geo)

    @property
    def voxel(self) -> float:
        return float(np.float32(self.extent) / np.float32(self.dims_geo[0]))

    def scaled(self, n_geo: int, r: Optional[int] = None, keep_mu: bool = False) -> "Config":
        """Same scene, cameras and extent with a coarser (cubic) grid: parity-test sized variants."""
        c = dataclasses.replace(self)
        c.dims_geo = (n_geo, n_geo, n_geo)
        if r is not None:
            c.r = r
        if not keep_mu:
            c.mu = float(np.float32(3.0) * np.float32(c.extent) / np.float32(n_geo)) if self.cfg != 5 else self.mu
        c.name = f"{self.name}@{n_geo}r{c.r}"
        return c


def _kinect_pair():
    Kd = intrinsics(525.0, 319.5, 239.5)
    Kh = intrinsics(1050.0, 959.5, 539.5)
    return 640, 480, 1920, 1080, Kd, Kh


def _t_depth_rgb():
    T = np.eye(4, dtype=np.float32)
    T[0, 3] = 0.025            # RGB camera sits 25 mm to the right of the depth camera (reading A10)
    return T


def _rng(cfg: int, frame: int):
    return np.random.default_rng(SEED0 + 1000 * cfg + frame)


def config(cfg: int, r: Optional[int] = None) -> Config:
    """BASELINE.json configs, numbered 1..5 as in SURVEY.md section 8(d)."""
    if cfg == 1:
        n, ext = 64, 1.0
        centre = np.array([0.0, 0.0, 1.5])
        prims = np.stack([prim(PRIM_SPHERE, TEX_CHECKER, 11, centre, (0.3,), scale=8.0)])
        yaws = np.deg2rad([-10.0, -5.0, 0.0, 5.0, 10.0])

        def pose(i):
            R = rot_axis((0, 1, 0), yaws[i])
            T = np.eye(4)
            T[:3, :3] = R
            T[:3, 3] = centre + R @ (np.zeros(3) - centre)
            return T
        return Config(1, "cfg1", (n, n, n), r or 2, (centre - ext / 2).astype(np.float32), ext,
                      3.0 * ext / n, 128, 160, 120, 320, 240,
                      intrinsics(131.25, 79.5, 59.5), intrinsics(262.5, 159.5, 119.5), _t_depth_rgb(),
                      5, prims, pose, lambda z: np.full_like(z, 1e-3), 0.0)
    wd, hd, wh, hh, Kd, Kh = _kinect_pair()
    quad = lambda z: 1.5e-3 * z * z
    if cfg == 2:
        n, ext = 256, 2.0
        prims = np.stack([
            prim(PRIM_PLANE, TEX_NOISE, 21, (0, 0, -0.5), (0, 0, 1), scale=3.0, colour=(120, 130, 110)),
            prim(PRIM_SPHERE, TEX_NOISE, 22, (0.3, 0.1, -0.2), (0.3,), scale=6.0, colour=(150, 110, 110)),
            prim(PRIM_BOX, TEX_NOISE, 23, (-0.3, -0.15, -0.3), (0.2, 0.25, 0.2), scale=6.0, colour=(110, 120, 160)),
        ])

        def pose(i):
            a = np.deg2rad(1.0 * i)
            return look_at((1.2 * np.cos(a), 1.2 * np.sin(a), 0.3), (0, 0, -0.2))
        return Config(2, "cfg2", (n, n, n), r or 2, np.full(3, -ext / 2, np.float32), ext, 3.0 * ext / n, 128,
                      wd, hd, wh, hh, Kd, Kh, _t_depth_rgb(), 100, prims, pose, quad, 0.02)
    if cfg == 3:
        n, ext = 512, 3.0
        g = np.random.default_rng(SEED0 + 3000 - 1)
        plist = [prim(PRIM_PLANE, TEX_NOISE, 31, (0, 0, -0.75), (0, 0, 1), scale=2.5, colour=(125, 125, 115))]
        for k in range(20):
            rad = g.uniform(0.05, 0.4)
            ang, rho = g.uniform(0, 2 * np.pi), 1.1 * np.sqrt(g.uniform(0, 1))
            col = g.uniform(90, 170, size=3)
            if g.uniform() < 0.5:
                plist.append(prim(PRIM_SPHERE, TEX_NOISE, 100 + k, (rho * np.cos(ang), rho * np.sin(ang), -0.75 + rad),
                                  (rad,), scale=g.uniform(4, 10), colour=col))
            else:
                h = rad * g.uniform(0.5, 1.0, size=3)
                plist.append(prim(PRIM_BOX, TEX_NOISE, 100 + k, (rho * np.cos(ang), rho * np.sin(ang), -0.75 + h[2]),
                                  h, scale=g.uniform(4, 10), colour=col))
        prims = np.stack(plist)

        def pose(i):
            a = np.deg2rad(1.2 * i)
            T = look_at((1.6 * np.cos(a), 1.6 * np.sin(a), 0.45), (0, 0, -0.45))
            j = _rng(3, 100000 + i)                        # handheld jitter: 2 mm / 0.3 deg per frame
            T[:3, 3] += j.normal(0, 0.002, size=3)
            ax = j.normal(size=3)
            T[:3, :3] = rot_axis(ax, np.deg2rad(j.normal(0, 0.3))) @ T[:3, :3]
            return T
        return Config(3, "cfg3", (n, n, n), r or 2, np.full(3, -ext / 2, np.float32), ext, 3.0 * ext / n, 128,
                      wd, hd, wh, hh, Kd, Kh, _t_depth_rgb(), 300, prims, pose, quad, 0.02)
    if cfg == 4:
        n, ext = 384, 2.0
        prims = np.stack([
            prim(PRIM_PLANE, TEX_NOISE, 41, (0, 0, -0.5), (0, 0, 1), scale=3.0, colour=(120, 125, 120)),
            prim(PRIM_TORUS, TEX_NOISE, 42, (0, 0, -0.38), (0.38, 0.12), scale=7.0, colour=(160, 120, 100)),
            prim(PRIM_CYLINDER, TEX_NOISE, 43, (0, 0, -0.15), (0.13, 0.35), scale=7.0, colour=(100, 130, 160)),
        ])

        def pose(i):
            a = np.deg2rad(1.8 * i)
            return look_at((1.2 * np.cos(a), 1.2 * np.sin(a), 0.4), (0, 0, -0.25))
        return Config(4, "cfg4", (n, n, n), r or 3, np.full(3, -ext / 2, np.float32), ext, 3.0 * ext / n, 128,
                      wd, hd, wh, hh, Kd, Kh, _t_depth_rgb(), 200, prims, pose, quad, 0.02)
    if cfg == 5:
        n, ext = 512, 0.5
        per = 1.45e-3                                     # stripe period 1.45..2.9 mm = 2..4 HD px at 0.75 m
        prims = np.stack([
            prim(PRIM_BOX, TEX_STRIPES, 51, (0, 0, -0.03), (0.07, 0.05, 0.09), scale=per),
            prim(PRIM_SPHERE, TEX_STRIPES, 52, (0.0, 0.0, 0.105), (0.05,), scale=per),
            prim(PRIM_CYLINDER, TEX_STRIPES, 53, (0.0, 0.0, -0.135), (0.11, 0.015), scale=per),
        ])

        def pose(i):
            a = np.deg2rad(0.9 * i)
            el = np.deg2rad(20.0 + 0.5 * np.sin(2 * np.pi * i / 50.0))
            R = 0.75
            return look_at((R * np.cos(el) * np.cos(a), R * np.cos(el) * np.sin(a), R * np.sin(el)), (0, 0, 0))
        return Config(5, "cfg5", (n, n, n), r or 2, np.full(3, -ext / 2, np.float32), ext, 0.004, 128,
                      wd, hd, wh, hh, Kd, Kh, _t_depth_rgb(), 400, prims, pose, quad, 0.02)
    raise ValueError(f"unknown config {cfg}")


def quantise_depth(z: np.ndarray, rng, sigma_of_z, dropout: float) -> np.ndarray:
    """z-depth (m, 0 = miss) -> uint16 mm with noise before quantisation and dropouts after."""
    hitm = (z > 0) & (z <= MAX_RANGE_M)
    zn = np.where(hitm, z, 0.0).astype(np.float64)
    zn = zn + rng.standard_normal(z.shape) * sigma_of_z(zn)
    d = np.clip(np.rint(1000.0 * zn), 1, 65535)
    d = np.where(hitm, d, 0).astype(np.uint16)
    if dropout > 0:
        d[rng.random(z.shape) < dropout] = 0
    return d


def frame(c: Config, i: int, want_rgb: bool = True):
    """Frame ``i`` of config ``c``: (depth uint16 [hd,wd], rgb uint8 [hh,wh,3] | None, T_world_depth float32 4x4)."""
    T32 = rigid32(c.pose(i))
    Td = T32.astype(np.float64)
    z, _ = render(c.prims, c.K_depth, Td, c.wd, c.hd, True, False)
    depth = quantise_depth(z, _rng(c.cfg, i), c.noise, c.dropout)
    rgb = None
    if want_rgb:
        Trgb = Td @ c.T_depth_rgb.astype(np.float64)
        _, rgb = render(c.prims, c.K_rgb, Trgb, c.wh, c.hh, False, True, c.bg)
    return depth, rgb, T32


# ----------------------------------------------------------------------------------------------
# closed-form test frames (no renderer involved)
# ----------------------------------------------------------------------------------------------

def plane_depth(wd: int, hd: int, d_mm: int) -> np.ndarray:
    """Fronto-parallel plane at z = d_mm."""
    return np.full((hd, wd), d_mm, dtype=np.uint16)


def tilted_plane_depth(wd, hd, K, d0_m: float, theta: float) -> np.ndarray:
    """Plane through (0,0,d0) rotated by theta about the camera y axis: z = d0 / (1 + tan(theta) * (x-cx)/fx)...

    Plane normal n = (sin t, 0, -cos t) (facing the camera), points p with n.(p - (0,0,d0)) = 0.
    Ray p = z * ((x-cx)/fx, (y-cy)/fy, 1)  ->  z = d0 cos t / (cos t - sin t * (x-cx)/fx).
    """
    xs = (np.arange(wd, dtype=np.float64) - float(K[0, 2])) / float(K[0, 0])
    z = d0_m * np.cos(theta) / (np.cos(theta) - np.sin(theta) * xs)
    d = np.clip(np.rint(1000.0 * z), 1, 65535).astype(np.uint16)
    return np.broadcast_to(d[None, :], (hd, wd)).copy()


def const_rgb(wh: int, hh: int, colour) -> np.ndarray:
    img = np.empty((hh, wh, 3), dtype=np.uint8)
    img[...] = np.asarray(colour, dtype=np.uint8)
    return img


def coord_rgb(wh: int, hh: int) -> np.ndarray:
    """RGB whose bytes encode the pixel: R = x mod 256, G = y mod 256, B = (x//256) + 16*(y//256)."""
    x = np.arange(wh)[None, :].repeat(hh, 0)
    y = np.arange(hh)[:, None].repeat(wh, 1)
    return np.stack([x % 256, y % 256, (x // 256) + 16 * (y // 256)], axis=-1).astype(np.uint8)


STRESS_KINDS = ("free_space", "in_band", "colour")


def stress_params(c: "Config", kind: str):
    """(mu, sigma) a volume needs for the saturating frame of this kind: the configuration's own,
    except mu = extent for "in_band" (the wall cuts the cube: every voxel lies inside the truncation band) and
    sigma = extent for "colour" ("sigma raised to cover the cube": every colour voxel passes the gate)."""
    assert kind in STRESS_KINDS
    return (float(c.extent) if kind == "in_band" else c.mu), (float(c.extent) if kind == "colour" else c.sigma)


def stress_frame(c: "Config", seed: int = 0, kind: str = "free_space"):
    """Saturating frame for config ``c``.  The camera is backed off along -x until the whole cube is
    inside the depth frustum and sees a fronto-parallel wall,
      "free_space": behind the cube, further than sigma: EVERY geometry voxel is updated with tsdf = 1, no colour voxel is;
      "in_band":    through the centre of the cube, for a volume with mu = extent (stress_params): every geometry voxel is
                    updated with a tsdf strictly inside (-1, 1), i.e. through the general running average;
      "colour":     the same wall for a volume with sigma = extent: every colour voxel passes the sigma gate as well.
    The wall moves by 3 mm per ``seed`` so that repeated frames differ.  Returns (depth, rgb, T_world_depth)."""
    assert kind in STRESS_KINDS
    ext = float(c.extent)
    centre = np.asarray(c.origin, np.float64) + ext / 2
    fx, fy = float(c.K_depth[0, 0]), float(c.K_depth[1, 1])
    half = ext / 2
    tan_h, tan_v = (c.wd / 2 - 1.0) / fx, (c.hd / 2 - 1.0) / fy
    d = half + 1.05 * half / min(tan_h, tan_v)                 # distance camera -> cube centre
    T = look_at(centre + np.array([-d, 0.0, 0.0]), centre)
    wall_mm = int(np.ceil(1000.0 * (d + half + 0.5 if kind == "free_space" else d))) + 3 * int(seed)
    assert wall_mm < 65535
    depth = np.full((c.hd, c.wd), wall_mm, dtype=np.uint16)
    return depth, random_rgb(c.wh, c.hh, 900 + seed), rigid32(T)


def random_rgb(wh: int, hh: int, seed: int) -> np.ndarray:
    return np.random.default_rng(SEED0 + seed).integers(0, 256, size=(hh, wh, 3), dtype=np.uint8)
