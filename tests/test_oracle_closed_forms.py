"""Pins of the CPU oracle against closed forms and invariants (no GPU).

Each test binds oracle/ref_fusion.c to something other than itself: a closed form derived from the
paper's equations (cited per test), evaluated here in float64 numpy.
"""
import numpy as np
import pytest

import oracle
import synth

CFG = synth.config(1)
I4 = np.eye(4, dtype=np.float32)


def make(n=32, r=2, mu_vox=3.0, w_max=128, sigma=0.020, extent=1.0, centre=(0, 0, 1.5)):
    origin = (np.asarray(centre) - extent / 2).astype(np.float32)
    return oracle.RefVolume((n, n, n), r, origin, extent, mu_vox * extent / n, w_max, sigma=sigma), origin


def centres(n, s, origin):
    k, j, i = np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij")
    return (origin[0] + (i + 0.5) * s, origin[1] + (j + 0.5) * s, origin[2] + (k + 0.5) * s)


def pixel_of(X, Y, Z, K):
    u = float(K[0, 0]) * X / Z + float(K[0, 2])
    v = float(K[1, 1]) * Y / Z + float(K[1, 2])
    safe = (np.abs(u + 0.5 - np.rint(u + 0.5)) > 1e-3) & (np.abs(v + 0.5 - np.rint(v + 0.5)) > 1e-3)
    return np.floor(u + 0.5), np.floor(v + 0.5), safe


def test_tsdf_column_worked_vector():
    """Config-1 geometry, identity pose, all pixels 1500 mm, one frame: the z-column of SURVEY 8(c)
    (linear ramp, zero crossing between layers 31|32 at 1.5 m, w = 1, behind the band untouched)."""
    v = oracle.RefVolume(CFG.dims_geo, CFG.r, CFG.origin, CFG.extent, CFG.mu, CFG.w_max)
    v.integrate(synth.plane_depth(160, 120, 1500), synth.const_rgb(320, 240, (1, 2, 3)), I4, CFG.K_depth, CFG.K_rgb,
                CFG.T_depth_rgb)
    q, w = oracle.geo_q(v.geo)[:, 32, 32], oracle.geo_w(v.geo)[:, 32, 32]
    # ideal ramp: q = 32767 * (1.5 - z_k) / mu, z_k = 1 + (k + .5)/64, mu = 3/64  -> thirds of 32767 at half-voxel offsets
    ideal = np.clip((1.5 - (1.0 + (np.arange(64) + 0.5) / 64.0)) / (3.0 / 64.0), -np.inf, 1.0) * 32767.0
    upd = ideal >= -32767.0 - 1e-6
    assert np.all(np.abs(q[upd] - ideal[upd]) <= 1.0)             # +-1 q-unit: 0.001f is one ulp above 1e-3 (exact ties)
    assert np.all(q[:29] == 32767) and q[31] > 0 > q[32]          # zero crossing brackets the plane depth
    assert np.all(w[upd] == 1) and np.all(v.geo[35:, 32, 32] == 0)
    assert list(q[29:35]) == [27306, 16384, 5461, -5461, -16383, -27306]


@pytest.mark.parametrize("d_mm,n_frames", [(1500, 3), (1370, 2)])
def test_tsdf_plane_all_voxels(d_mm, n_frames):
    """Fronto-parallel plane, identity pose: every in-frustum voxel with z <= d + mu holds
    rint(32767 * min(1, (d - z)/mu)) (+-1), constant over frames (no drift), weight = n; every other voxel
    keeps its initial bytes (BASELINE closed forms: zero crossing, linear ramp, unchanged outside)."""
    n = 32
    v, origin = make(n)
    for _ in range(n_frames):
        v.integrate(synth.plane_depth(160, 120, d_mm), synth.const_rgb(320, 240, (9, 9, 9)), I4, CFG.K_depth, CFG.K_rgb,
                    CFG.T_depth_rgb)
    X, Y, Z = centres(n, 1.0 / n, origin)
    xf, yf, safe = pixel_of(X, Y, Z, CFG.K_depth)
    inside = (xf >= 0) & (xf < 160) & (yf >= 0) & (yf < 120)
    d, mu = d_mm * 1e-3, 3.0 / n
    band_safe = np.abs(d - Z + mu) > 1e-5
    upd = inside & (d - Z >= -mu)
    ideal = 32767.0 * np.minimum(1.0, (d - Z) / mu)
    q, w = oracle.geo_q(v.geo), oracle.geo_w(v.geo)
    m = safe & band_safe
    assert (m & upd).sum() > 1000 and (m & ~upd).sum() > 1000
    assert np.all(np.abs(q[m & upd] - ideal[m & upd]) <= 1.0)
    assert np.all(w[m & upd] == n_frames)
    assert np.all(v.geo[m & ~upd] == 0)


def test_weight_increments_and_saturates():
    """w_max + 5 frames -> w = w_max (BASELINE: weights increment and saturate at w_max)."""
    v, origin = make(16, r=1, w_max=7)
    ws = []
    for _ in range(12):
        v.integrate(synth.plane_depth(160, 120, 1500), synth.const_rgb(320, 240, (9, 9, 9)), I4, CFG.K_depth, CFG.K_rgb,
                    CFG.T_depth_rgb)
        ws.append(int(oracle.geo_w(v.geo)[2, 8, 8]))
    assert ws == [1, 2, 3, 4, 5, 6, 7, 7, 7, 7, 7, 7]
    assert int(oracle.geo_q(v.geo)[2, 8, 8]) == 32767


def test_zero_depth_is_noop_and_frustum():
    """All-zero depth frame changes nothing (L103 'if non-zero'); a camera looking away changes nothing (L101)."""
    v, _ = make(16)
    z = np.zeros((120, 160), np.uint16)
    cnt = v.integrate(z, synth.random_rgb(320, 240, 1), I4, CFG.K_depth, CFG.K_rgb, CFG.T_depth_rgb)
    assert not v.geo.any() and not v.col.any() and not cnt.any()
    T = I4.copy()
    T[:3, :3] = np.diag([-1, 1, -1]).astype(np.float32)          # rotate 180 deg about y: volume is behind the camera
    cnt = v.integrate(synth.plane_depth(160, 120, 1500), synth.random_rgb(320, 240, 1), T, CFG.K_depth, CFG.K_rgb,
                      CFG.T_depth_rgb)
    assert not v.geo.any() and not v.col.any() and not cnt.any()


def test_sigma_gate_shell_and_view_weight():
    """Plane at d: the colour voxels touched are exactly those with |P_vc - P_vd| <= sigma (L108), and their first
    weight is rint(255 * cos(off-axis angle)) since N || +z for a fronto-parallel plane (eq. 8):
    W(x, y) = 1 / sqrt(1 + ((x-cx)/fx)^2 + ((y-cy)/fy)^2)."""
    n, r = 32, 2
    v, origin = make(n, r)
    d = 1.5
    v.integrate(synth.plane_depth(160, 120, 1500), synth.const_rgb(320, 240, (50, 60, 70)), I4, CFG.K_depth, CFG.K_rgb,
                CFG.T_depth_rgb)
    X, Y, Z = centres(n * r, 1.0 / (n * r), origin)
    xf, yf, safe = pixel_of(X, Y, Z, CFG.K_depth)
    inside = (xf >= 0) & (xf + 1 < 160) & (yf >= 0) & (yf + 1 < 120)
    K = CFG.K_depth.astype(np.float64)
    Xd, Yd = (xf - K[0, 2]) * d / K[0, 0], (yf - K[1, 2]) * d / K[1, 1]
    dist = np.sqrt((X - Xd) ** 2 + (Y - Yd) ** 2 + (Z - d) ** 2)
    m = safe & (np.abs(dist - 0.020) > 1e-5)
    expect = inside & (dist <= 0.020)
    wq = oracle.col_w(v.col)
    assert (m & expect).sum() > 5000
    assert np.array_equal((wq > 0)[m], expect[m])
    W = 1.0 / np.sqrt(1.0 + ((xf - K[0, 2]) / K[0, 0]) ** 2 + ((yf - K[1, 2]) / K[1, 1]) ** 2)
    tie_safe = np.abs(255.0 * W - np.floor(255.0 * W) - 0.5) > 1e-3
    mm = m & expect & tie_safe
    assert np.array_equal(wq[mm], np.rint(255.0 * W[mm]).astype(np.int64))
    # the shell is symmetric about the plane and 2*sigma thick on the axis: layers with |z_k - d| <= sigma
    zc = origin[2] + (np.arange(n * r) + 0.5) / (n * r)
    col = wq[:, n * r // 2, n * r // 2] > 0
    lateral = np.hypot(X[0, n * r // 2, n * r // 2] - Xd[0, n * r // 2, n * r // 2], Y[0, n * r // 2, n * r // 2] - Yd[0, n * r // 2, n * r // 2])
    assert np.array_equal(col, np.sqrt((zc - d) ** 2 + lateral ** 2) <= 0.020)


def test_tilted_plane_weight_is_cos_theta():
    """Plane tilted by theta about the camera y axis, seen near the optical axis: W = cos(theta) (eq. 8 + L110)."""
    K = synth.intrinsics(60.0, 39.5, 29.5)
    for theta in (0.3, 0.6):
        n = 24
        origin = np.array([-0.3, -0.3, 1.7], np.float32)
        v = oracle.RefVolume((n, n, n), 1, origin, 0.6, 0.05, 64, sigma=0.030)
        dep = synth.tilted_plane_depth(80, 60, K, 2.0, theta)
        v.integrate(dep, synth.const_rgb(160, 120, (5, 5, 5)), I4, K, synth.intrinsics(120.0, 79.5, 59.5), CFG.T_depth_rgb)
        wq = oracle.col_w(v.col)
        near_axis = wq[:, 10:14, 10:14]
        got = near_axis[near_axis > 0] / 255.0
        assert got.size > 8
        assert np.all(np.abs(got - np.cos(theta)) < 0.03)
