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
