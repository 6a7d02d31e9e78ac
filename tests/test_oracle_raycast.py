"""Pins of the ray-casting oracle (ref_raycast) against closed forms -- no GPU.

The paper names ray casting of the volumes without equations; the definition is readings R1-R6 in
oracle/ref_fusion.c.  Each test binds it to geometry that can be computed by hand: a fronto-parallel plane (the zero
crossing of a linear TSDF ramp), an analytic sphere seen from a rotated and translated camera, front faces only."""
import numpy as np

import oracle
import synth

CFG = synth.config(1)
I4 = np.eye(4, dtype=np.float32)
VS = 1.0 / 64


def plane_volume(d_mm=1500, frames=3, colour=(200, 90, 30)):
    v = oracle.RefVolume(CFG.dims_geo, CFG.r, CFG.origin, CFG.extent, CFG.mu, CFG.w_max)
    for _ in range(frames):
        v.integrate(synth.plane_depth(CFG.wd, CFG.hd, d_mm), synth.const_rgb(CFG.wh, CFG.hh, colour), I4, CFG.K_depth,
                    CFG.K_rgb, CFG.T_depth_rgb)
    return v


def test_empty_volume_and_bad_ranges():
    v = oracle.RefVolume((16, 16, 16), 2, (-0.5, -0.5, 1.0), 1.0, 0.1, 128)
    depth, rgb = v.raycast(40, 30, I4, CFG.K_depth, 0.5, 3.0)
    assert not depth.any() and not rgb.any()                                        # R6
    try:
        v.raycast(40, 30, I4, CFG.K_depth, 2.0, 1.0)
        assert False
    except ValueError:
        pass


def test_plane_zero_crossing_is_the_plane_depth():
    """Linear ramp F = (d - z_c) / mu on voxel centres z_c; samples one voxel apart.  With t_near on a voxel centre the
    interpolated crossing (R4) is d itself (up to the int16 rounding of F: < 1e-4 m); with t_near on a voxel face every
    sample sits half a voxel before its voxel's centre, so the estimate is d - vs / 2."""
    v = plane_volume()
    d = 1.5
    depth, rgb = v.raycast(CFG.wd, CFG.hd, I4, CFG.K_depth, 1.0 + 0.5 * VS, 2.0)
    # pixels whose ray is inside the volume laterally all the way to the plane
    x = (np.arange(CFG.wd) - 79.5) / 131.25 * d
    y = (np.arange(CFG.hd) - 59.5) / 131.25 * d
    inside = (np.abs(x)[None, :] < 0.5 - VS) & (np.abs(y)[:, None] < 0.5 - VS)
    assert inside.sum() > 5000
    assert np.all(depth[inside] > 0)
    assert np.abs(depth[inside] - d).max() < 1e-4
    outside = (np.abs(x)[None, :] > 0.5 + VS) | (np.abs(y)[:, None] > 0.5 + VS)
    assert not depth[outside].any()                                                 # rays that leave the cube before the plane
    depth2, _ = v.raycast(CFG.wd, CFG.hd, I4, CFG.K_depth, 1.0, 2.0)
    assert np.abs(depth2[inside] - (d - 0.5 * VS)).max() < 1e-4
    # R5: the colour volume holds the constant colour around the plane
    assert np.all(rgb[inside] == np.array([200, 90, 30], np.uint8))
    assert not rgb[~(depth > 0)].any()


def test_front_faces_only():
    """Seen from behind (camera beyond the plane, looking back), the ray goes from F < 0 to F > 0: not a hit (R4)."""
    v = plane_volume()
    T = np.array([[-1, 0, 0, 0], [0, 1, 0, 0], [0, 0, -1, 3.0], [0, 0, 0, 1]], np.float32)   # at z = 3 looking towards -z
    depth, _ = v.raycast(CFG.wd, CFG.hd, T, CFG.K_depth, 0.5, 2.5)
    assert not depth.any()


def test_sphere_from_a_rotated_translated_camera():
    """Config 1's sphere (R = 0.3 m at (0, 0, 1.5)) fused from its 5 frames, then viewed from a camera that is neither at
    the origin nor axis-aligned: the ray-cast depth must agree with the analytic ray-sphere depth to about a voxel
    (a transposed rotation, swapped axes or a wrong index order moves the silhouette by many pixels)."""
    v = oracle.RefVolume(CFG.dims_geo, CFG.r, CFG.origin, CFG.extent, CFG.mu, CFG.w_max)
    for fi in range(5):
        depth, rgb, T = synth.frame(CFG, fi)
        v.integrate(depth, rgb, T, CFG.K_depth, CFG.K_rgb, CFG.T_depth_rgb)
    Tc = synth.rigid32(synth.look_at((0.25, -0.15, 0.1), (0.0, 0.0, 1.5), up=(0.0, -1.0, 0.0)))
    got, rgb = v.raycast(CFG.wd, CFG.hd, Tc, CFG.K_depth, 0.3, 3.0)
    want, _ = synth.render(CFG.prims, CFG.K_depth, Tc.astype(np.float64), CFG.wd, CFG.hd, True, False)
    both = (got > 0) & (want > 0)
    assert both.sum() > 2000
    err = np.abs(got[both] - want[both])
    assert np.median(err) < 0.5 * VS and np.percentile(err, 95) < 2.0 * VS
    # silhouettes agree up to a pixel-wide rim
    assert ((got > 0) != (want > 0)).sum() < 0.15 * both.sum()
    # the hit colours come from the textured sphere: not black where the colour volume was filled
    assert (rgb[both].sum(axis=1) > 0).mean() > 0.9


# ---- reading R7: trilinear TSDF sampling (ref_raycast_trilinear) ------------------------------------------------------

def test_trilinear_plane_depth_is_exact_for_any_t_near():
    """A plane inside the truncation band is a TSDF that is linear in space, and trilinear interpolation reproduces a linear
    function exactly: the zero crossing is the plane for ANY phase of the samples (the nearest-voxel reading is off by up to
    half a voxel, previous test), from the integrating camera and from a rotated, translated one."""
    v = plane_volume()
    d = 1.5
    x = (np.arange(CFG.wd) - 79.5) / 131.25 * d
    y = (np.arange(CFG.hd) - 59.5) / 131.25 * d
    inside = (np.abs(x)[None, :] < 0.5 - 2 * VS) & (np.abs(y)[:, None] < 0.5 - 2 * VS)
    for t_near in (1.0, 1.0 + 0.5 * VS, 1.0 + 0.123 * VS, 1.0 + 0.77 * VS):
        depth, rgb = v.raycast_trilinear(CFG.wd, CFG.hd, I4, CFG.K_depth, t_near, 2.0)
        assert np.all(depth[inside] > 0) and np.abs(depth[inside] - d).max() < 2e-5, (t_near, np.abs(depth[inside] - d).max())
        assert np.all(rgb[inside] == np.array([200, 90, 30], np.uint8))
    # another camera: 12 degrees of yaw about the plane's centre, shifted; the exact depth of the plane z_world = d along its rays
    Tc = synth.rigid32(synth.look_at((0.25, -0.1, 0.2), (0.0, 0.0, 1.5), up=(0.0, -1.0, 0.0))).astype(np.float64)
    depth, _ = v.raycast_trilinear(CFG.wd, CFG.hd, Tc.astype(np.float32), CFG.K_depth, 0.3, 3.0)
    xx, yy = np.meshgrid(np.arange(CFG.wd, dtype=np.float64), np.arange(CFG.hd, dtype=np.float64))
    K = np.asarray(CFG.K_depth, np.float64).reshape(3, 3)
    ray = np.stack([(xx - K[0, 2]) / K[0, 0], (yy - K[1, 2]) / K[1, 1], np.ones_like(xx)], -1) @ Tc[:3, :3].T
    want = (d - Tc[2, 3]) / ray[..., 2]
    hit = Tc[:3, 3] + want[..., None] * ray
    ok = (np.abs(hit[..., 0]) < 0.5 - 3 * VS) & (np.abs(hit[..., 1]) < 0.5 - 3 * VS)
    assert ok.sum() > 3000 and np.all(depth[ok] > 0)
    assert np.abs(depth[ok] - want[ok]).max() < 5e-5, np.abs(depth[ok] - want[ok]).max()


def test_trilinear_against_a_float64_loop_and_scipy():
    """Every step of R7 / R4 again in binary64 with explicit Python loops over a handful of rays, the interpolation itself
    also through scipy.ndimage.map_coordinates(order=1): same hit sample, depth within 1e-5 m."""
    from scipy.ndimage import map_coordinates
    v = oracle.RefVolume(CFG.dims_geo, CFG.r, CFG.origin, CFG.extent, CFG.mu, CFG.w_max)
    for fi in range(5):
        depth, rgb, T = synth.frame(CFG, fi)
        v.integrate(depth, rgb, T, CFG.K_depth, CFG.K_rgb, CFG.T_depth_rgb)
    Tc = synth.rigid32(synth.look_at((0.25, -0.15, 0.1), (0.0, 0.0, 1.5), up=(0.0, -1.0, 0.0)))
    got, _ = v.raycast_trilinear(CFG.wd, CFG.hd, Tc, CFG.K_depth, 0.3, 3.0)
    q = oracle.geo_q(v.geo).astype(np.float64).reshape(CFG.dims_geo[::-1])           # [k, j, i]
    wgt = oracle.geo_w(v.geo).reshape(CFG.dims_geo[::-1])
    K = np.asarray(CFG.K_depth, np.float64).reshape(3, 3)
    T64, org = Tc.astype(np.float64), np.asarray(CFG.origin, np.float64)
    rng = np.random.default_rng(5)
    checked = hits = 0
    for _ in range(60):
        x, y = int(rng.integers(0, CFG.wd)), int(rng.integers(0, CFG.hd))
        dirw = T64[:3, :3] @ np.array([(x - K[0, 2]) / K[0, 0], (y - K[1, 2]) / K[1, 1], 1.0])
        want, prev = 0.0, None
        fragile = False
        for k in range(4000):
            t = 0.3 + k * VS
            if t > 3.0:
                break
            g = (T64[:3, 3] + t * dirw - org) / VS - 0.5
            b = np.floor(g).astype(int)
            cur = None
            if np.all(b >= 0) and np.all(b <= np.array(CFG.dims_geo) - 2):
                fr = g - b
                fragile |= bool(np.any(np.minimum(fr, 1 - fr) < 1e-4))                  # a corner set that binary32 may choose differently
                known, F = True, 0.0
                for c in range(8):
                    i, j, kk = b[0] + (c & 1), b[1] + ((c >> 1) & 1), b[2] + (c >> 2)
                    known &= bool(wgt[kk, j, i] != 0)
                    F += (fr[2] if c & 4 else 1 - fr[2]) * (fr[1] if c & 2 else 1 - fr[1]) * (fr[0] if c & 1 else 1 - fr[0]) * q[kk, j, i]
                if known:
                    assert abs(F - map_coordinates(q, [[g[2]], [g[1]], [g[0]]], order=1)[0]) < 1e-6 * 32767
                    cur = (t, F)
                    fragile |= abs(F) < 0.5
            if cur and prev and prev[1] > 0 and not cur[1] > 0:
                want = prev[0] + VS * prev[1] / (prev[1] - cur[1])
                break
            prev = cur
        if fragile:
            continue
        checked += 1
        hits += want > 0
        assert (got[y, x] > 0) == (want > 0) and abs(got[y, x] - want) < 1e-5, (x, y, got[y, x], want)
    assert checked > 30 and hits > 5


def test_trilinear_sphere_is_closer_than_nearest_voxel_and_unknown_corners_block_a_hit():
    """The sphere of config 1 from a rotated camera: the trilinear depth is within a fifth of a voxel of the analytic one in
    the median (nearest voxel: up to half a voxel), its x-differences are free of voxel-sized steps; and a sample with a
    never-observed voxel among its 8 corners is unknown: wiping one voxel layer in front of the surface removes every hit
    that needs it, nothing else."""
    v = oracle.RefVolume(CFG.dims_geo, CFG.r, CFG.origin, CFG.extent, CFG.mu, CFG.w_max)
    for fi in range(5):
        depth, rgb, T = synth.frame(CFG, fi)
        v.integrate(depth, rgb, T, CFG.K_depth, CFG.K_rgb, CFG.T_depth_rgb)
    Tc = synth.rigid32(synth.look_at((0.25, -0.15, 0.1), (0.0, 0.0, 1.5), up=(0.0, -1.0, 0.0)))
    tri, _ = v.raycast_trilinear(CFG.wd, CFG.hd, Tc, CFG.K_depth, 0.3, 3.0)
    near, _ = v.raycast(CFG.wd, CFG.hd, Tc, CFG.K_depth, 0.3, 3.0)
    want, _ = synth.render(CFG.prims, CFG.K_depth, Tc.astype(np.float64), CFG.wd, CFG.hd, True, False)
    both = (tri > 0) & (near > 0) & (want > 0)
    assert both.sum() > 2000
    e_tri, e_near = np.abs(tri[both] - want[both]), np.abs(near[both] - want[both])
    assert np.median(e_tri) < 0.2 * VS and np.median(e_tri) < 0.7 * np.median(e_near), (np.median(e_tri) / VS, np.median(e_near) / VS)
    # smoothness: second differences along x of the depth map (the analytic surface is smooth)
    run = both[:, :-2] & both[:, 1:-1] & both[:, 2:]
    dd = lambda z: np.abs(z[:, :-2] - 2 * z[:, 1:-1] + z[:, 2:])[run]
    assert np.percentile(dd(tri), 90) < 0.5 * np.percentile(dd(near), 90)
    # unknown corners: front faces only, and an unobserved layer
    back = np.array([[-1, 0, 0, 0], [0, 1, 0, 0], [0, 0, -1, 3.0], [0, 0, 0, 1]], np.float32)
    assert not v.raycast_trilinear(CFG.wd, CFG.hd, back, CFG.K_depth, 0.5, 2.5)[0][(np.abs(np.arange(CFG.hd) - 60) < 5)][:, 75:85].any()
    geo = v.geo.reshape(CFG.dims_geo[::-1]).copy()
    kz = int((1.2 - CFG.origin[2]) / VS)                                                # the sphere's front pole is at z = 1.2
    v.geo.reshape(CFG.dims_geo[::-1])[kz - 1:kz + 2] = 0                                 # three layers never observed
    cut, _ = v.raycast_trilinear(CFG.wd, CFG.hd, I4, CFG.K_depth, 0.3, 3.0)
    v.geo.reshape(CFG.dims_geo[::-1])[:] = geo
    full, _ = v.raycast_trilinear(CFG.wd, CFG.hd, I4, CFG.K_depth, 0.3, 3.0)
    lost = (full > 0) & ~(cut > 0)
    assert lost.sum() > 50 and np.all(np.abs(full[lost] - 1.2) < 3 * VS)                # hits near the wiped layers are gone
    kept = (full > 0) & (cut > 0)
    assert kept.sum() > 1000 and np.array_equal(full[kept], cut[kept])                   # the others are untouched
