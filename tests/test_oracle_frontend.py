"""Pins of the front-end / ICP oracle (oracle/frontend.py; readings F1-F7 of DESIGN.md 8f) -- no GPU.
The paper prints nothing for these steps: the pins are closed forms, hand-computed small cases,
invariants and an independent float64 brute force."""
import math

import numpy as np
import pytest

import synth
from oracle import frontend as fe

K = synth.intrinsics(262.5, 159.5, 119.5)             # 320 x 240
W, H = 320, 240


def rays(K_, w, h):
    x, y = np.meshgrid(np.arange(w, dtype=np.float64), np.arange(h, dtype=np.float64))
    return np.stack([(x - K_[0, 2]) / K_[0, 0], (y - K_[1, 2]) / K_[1, 1], np.ones_like(x)], -1)


def plane_depth_exact(K_, w, h, n, c):
    """z-depth of the plane n . P = c seen from the origin (float64)."""
    return c / (rays(K_, w, h) @ np.asarray(n, np.float64))


# ------------------------------------------------------------------------------------------------ F1 bilateral
def test_bilateral_tables():
    ws, wr = fe.bilateral_tables(4.5, 0.030)
    assert ws.shape == (7, 7) and ws[3, 3] == 1.0 and np.array_equal(ws, ws.T) and np.array_equal(ws, ws[::-1, ::-1])
    assert abs(float(ws[0, 0]) - math.exp(-18 / (2 * 4.5 ** 2))) < 1e-7 and abs(float(ws[3, 5]) - math.exp(-4 / 40.5)) < 1e-7
    assert wr.size == 91 and wr[0] == 1.0 and np.all(np.diff(wr) < 0)
    assert abs(float(wr[30]) - math.exp(-0.5)) < 1e-7 and abs(float(wr[90]) - math.exp(-4.5)) < 1e-8


def test_bilateral_two_pixels_by_hand():
    """A 1 x 2 image (1000, 1010) mm: out(0) = (1000 + a 1010) / (1 + a), a = ws(dx = 1) wr(10 mm)."""
    a = math.exp(-1 / 40.5) * math.exp(-100 / 1800.0)
    out = fe.bilateral(np.array([[1000, 1010]], np.uint16))
    assert abs(float(out[0, 0]) - 1e-3 * (1000 + a * 1010) / (1 + a)) < 2e-7
    assert abs(float(out[0, 1]) - 1e-3 * (1010 + a * 1000) / (1 + a)) < 2e-7


def test_bilateral_constant_edges_and_holes():
    d = np.full((40, 60), 1500, np.uint16)
    d[:, 30:] = 1700                                     # a 200 mm step: beyond ceil(3 sigma_r) = 90 mm, the sides do not mix
    d[10, 10] = 0                                        # a hole stays a hole and contributes nothing
    d[20:27, 40:47] = 0
    d[23, 43] = 1650                                     # an island: only itself in reach
    out = fe.bilateral(d)
    assert out[10, 10] == 0 and not out[20:27, 40:47][d[20:27, 40:47] == 0].any()
    left, right = out[:, :30], out[:, 30:]
    # up to 49 binary32 additions per sum: a few 1e-7 relative; mixing across the step would shift by millimetres
    assert np.abs(left[left > 0] - 1.5).max() < 2e-6 and np.abs(right[(right > 0) & (d[:, 30:] == 1700)] - 1.7).max() < 2e-6
    assert abs(float(out[23, 43]) - 1.65) < 2e-7


def test_bilateral_smooths_noise_but_keeps_the_mean():
    rng = np.random.default_rng(1)
    d = np.rint(2000 + rng.normal(0, 4.0, size=(120, 160))).astype(np.uint16)
    out = fe.bilateral(d)[8:-8, 8:-8] * 1000.0
    assert abs(out.mean() - 2000) < 0.2 and out.std() < 4.0 / 4.0        # 49 nearly equal weights: about 1/7 of the noise


# ------------------------------------------------------------------------------------------------ F2 pyramid
def test_half_sample_block_rules():
    D = np.array([[1.0, 1.02, 2.0, 0.0], [1.04, 5.0, 0.0, 2.0], [0.0, 3.0, 1.0, 1.0], [3.0, 3.0, 1.2, 1.0]], np.float32)
    out = fe.half_sample(D, 0.030)
    assert abs(float(out[0, 0]) - (1.0 + 1.02 + 1.04) / 3) < 1e-6     # 5.0 is farther than 3 sigma_r = 0.09 from the block's first pixel
    assert abs(float(out[0, 1]) - 2.0) < 1e-7                          # zeros are skipped
    assert out[1, 0] == 0                                               # first pixel invalid: the block is invalid
    assert abs(float(out[1, 1]) - 1.0) < 1e-7                          # 1.2 rejected


def test_pyramid_levels_are_geometrically_consistent():
    """Fronto-parallel plane: every level's vertices lie on z = D, and vertex x of level l + 1 is the mean of the two level-l
    vertices of its block -- which fixes the principal-point rule c' = (c - 1/2) / 2."""
    pyr = fe.pyramid(np.full((H, W), 1.25, np.float32), K, 3)
    assert [p[0].shape for p in pyr] == [(240, 320), (120, 160), (60, 80)]
    for lv in range(2):
        V0, V1 = pyr[lv][1].astype(np.float64), pyr[lv + 1][1].astype(np.float64)
        assert np.all(V1[..., 2] == 1.25)
        assert np.abs(V1[..., 0] - 0.5 * (V0[0::2, 0::2, 0] + V0[0::2, 1::2, 0])).max() < 1e-6
        assert np.abs(V1[..., 1] - 0.5 * (V0[0::2, 0::2, 1] + V0[1::2, 0::2, 1])).max() < 1e-6
    fx, fy, cx, cy = fe.level_intrinsics(K, 2)
    assert (float(fx), float(fy)) == (65.625, 65.625) and abs(float(cx) - 39.5) < 1e-6 and abs(float(cy) - 29.5) < 1e-6


# ------------------------------------------------------------------------------------------------ F3 / F4 maps
def test_vertex_and_normal_maps_of_a_tilted_plane():
    n = np.array([0.3, -0.2, 0.933], np.float64); n /= np.linalg.norm(n)
    D = plane_depth_exact(K, W, H, n, 1.4).astype(np.float32)
    pyr = fe.pyramid(D, K, 1)
    V, N = pyr[0][1].astype(np.float64), pyr[0][2].astype(np.float64)
    assert np.abs(V - rays(K, W, H) * D[..., None].astype(np.float64)).max() < 2e-7      # eq. 7
    assert np.abs(V @ n - 1.4).max() < 2e-6                                              # the vertices lie on the plane
    inner = N[:-1, :-1]
    assert np.abs(np.linalg.norm(inner, axis=-1) - 1).max() < 1e-6
    assert np.abs(inner - n).max() < 2e-3                      # eq. 8: the plane's normal, pointing away from the camera (n_z > 0);
    assert not N[-1].any() and not N[:, -1].any()              # float32 depth at 1.4 m limits the differences to ~1e-3; no neighbour: invalid


def test_normals_of_a_sphere_are_radial_and_holes_invalidate_neighbours():
    c = synth.config(1)
    T = np.eye(4)
    z, _ = synth.render(c.prims, c.K_depth, T, c.wd, c.hd, True, False)
    pyr = fe.pyramid(z, c.K_depth, 1)
    V, N = pyr[0][1].astype(np.float64), pyr[0][2].astype(np.float64)
    on = (z > 0) & (np.linalg.norm(N, axis=-1) > 0)
    radial = (V - np.array([0, 0, 1.5])) / 0.3
    m = on & (np.abs(np.linalg.norm(radial, axis=-1) - 1) < 1e-3)
    m[:, :-1] &= m[:, 1:]; m[:-1] &= m[1:]                      # both forward neighbours on the sphere too
    facing = m & (-(radial * V).sum(-1) / np.maximum(np.linalg.norm(V, axis=-1), 1e-9) > 0.5)
    assert facing.sum() > 1500
    # forward differences over one pixel (11 mm at 1.5 m on a 300 mm sphere): a few degrees off the radial direction at most,
    # and pointing away from the camera: N = -radial on the visible side
    assert ((N * -radial).sum(-1)[facing] > math.cos(math.radians(6))).all()
    z2 = z.copy(); z2[60, 80] = 0
    N2 = fe.pyramid(z2, c.K_depth, 1)[0][2]
    assert not N2[60, 80].any() and not N2[60, 79].any() and not N2[59, 80].any() and N2[59, 79].any()


# ------------------------------------------------------------------------------------------------ F5 / F6 ICP
def scene_pair(dT, quantised=False):
    """Config 2's scene seen from pose A (the prediction) and from pose B = A dT (the measurement), 320 x 240."""
    c = synth.config(2)
    A = synth.look_at((0.9, -0.6, 0.55), (0.0, 0.0, 0.0))
    B = A @ dT
    za, _ = synth.render(c.prims, K, A, W, H, True, False)
    zb, _ = synth.render(c.prims, K, B, W, H, True, False)
    pred = fe.pyramid(za, K, 3)
    if quantised:
        meas = fe.measure(np.clip(np.rint(zb * 1000.0), 0, 65535).astype(np.uint16), K, 3)
    else:
        meas = fe.pyramid(zb, K, 3)
    return meas, pred


def small_motion(rx, ry, rz, t):
    T = np.eye(4)
    T[:3, :3] = synth.rot_axis((1, 0, 0), rx) @ synth.rot_axis((0, 1, 0), ry) @ synth.rot_axis((0, 0, 1), rz)
    T[:3, 3] = t
    return T


def test_icp_step_at_the_solution_and_symmetry():
    meas, pred = scene_pair(np.eye(4))
    A, b, e, cnt = fe.icp_step(meas, pred, K, 0, np.eye(4))
    valid = int(np.any(meas[0][2] != 0, axis=-1).sum())
    assert cnt == valid and cnt > 30000                     # every pixel with a normal finds itself
    assert e == 0.0 and not b.any()
    assert np.array_equal(A, A.T) and np.all(np.linalg.eigvalsh(A) > 0)


def test_icp_step_against_a_float64_pixel_loop():
    """The vectorised binary32 step against a plain per-pixel loop in float64 written from reading F5, on the coarsest level."""
    dT = small_motion(0.01, -0.015, 0.008, (0.01, -0.006, 0.012))
    meas, pred = scene_pair(dT)
    lv = 2
    T = small_motion(0.002, 0.001, -0.001, (0.002, 0.001, -0.003))
    A, b, e, cnt = fe.icp_step(meas, pred, K, lv, T)
    _, V, N = meas[lv]; _, Vp, Np = pred[lv]
    h, w, _ = V.shape
    fx, fy, cx, cy = [float(v) for v in fe.level_intrinsics(K, lv)]
    T32 = T.astype(np.float32).astype(np.float64)
    A2, b2, e2, c2, fragile = np.zeros((6, 6)), np.zeros(6), 0.0, 0, 0
    for y in range(h):
        for x in range(w):
            n = N[y, x].astype(np.float64)
            if not n.any():
                continue
            p = T32[:3, :3] @ V[y, x].astype(np.float64) + T32[:3, 3]
            m = T32[:3, :3] @ n
            if p[2] <= 0:
                continue
            u, v = fx * p[0] / p[2] + cx, fy * p[1] / p[2] + cy
            xi, yi = math.floor(u + 0.5), math.floor(v + 0.5)
            if abs(u + 0.5 - round(u + 0.5)) < 1e-4 or abs(v + 0.5 - round(v + 0.5)) < 1e-4:
                fragile += 1
            if not (0 <= xi < w and 0 <= yi < h):
                continue
            q, nq = Vp[yi, xi].astype(np.float64), Np[yi, xi].astype(np.float64)
            if not nq.any():
                continue
            d = q - p
            if abs(d @ d - 0.01) < 1e-6 or abs(m @ nq - 0.94) < 1e-5:
                fragile += 1
            if d @ d > 0.10 ** 2 or m @ nq < 0.94:
                continue
            J = np.concatenate([np.cross(p, nq), nq])
            r = nq @ d
            A2 += np.outer(J, J); b2 += J * r; e2 += r * r; c2 += 1
    assert c2 > 1500 and abs(cnt - c2) <= fragile
    if cnt == c2:
        assert np.abs(A - A2).max() <= 1e-5 * np.abs(A2).max() and np.abs(b - b2).max() <= 1e-5 * np.abs(b2).max() + 1e-9
        assert abs(e - e2) <= 1e-5 * e2


def test_se3_update_left_multiplies_a_rodrigues_rotation():
    from scipy.linalg import expm
    A = np.diag([2.0, 3.0, 4.0, 5.0, 6.0, 7.0])
    xi = np.array([0.02, -0.03, 0.05, 0.01, 0.02, -0.04])
    T0 = small_motion(0.3, -0.2, 0.1, (0.5, -0.1, 0.2))
    T1, got = fe.se3_update(T0, A, A @ xi)
    assert np.allclose(got, xi, atol=1e-14)
    Kx = np.array([[0, -xi[2], xi[1]], [xi[2], 0, -xi[0]], [-xi[1], xi[0], 0]])
    Rinc = expm(Kx)
    assert np.allclose(T1[:3, :3], Rinc @ T0[:3, :3], atol=1e-13) and np.allclose(T1[:3, 3], Rinc @ T0[:3, 3] + xi[3:], atol=1e-13)
    assert np.allclose(T1[:3, :3] @ T1[:3, :3].T, np.eye(3), atol=1e-13) and np.array_equal(T1[3], [0, 0, 0, 1])


@pytest.mark.parametrize("quantised", [False, True])
def test_track_recovers_a_known_motion(quantised):
    """Prediction rendered from pose A, measurement from B = A dT (1.3 degrees, 17 mm): coarse-to-fine ICP from the identity
    ends at dT -- current camera -> prediction camera -- to a fraction of a millimetre on exact depth, and to about a
    millimetre on depth quantised to whole millimetres and bilateral-filtered."""
    dT = small_motion(0.012, -0.018, 0.009, (0.012, -0.007, 0.010))
    meas, pred = scene_pair(dT, quantised)
    T, rms, cnt = fe.track(meas, pred, K)
    err = np.linalg.inv(dT) @ T
    ang = math.degrees(math.acos(min(1.0, (np.trace(err[:3, :3]) - 1) / 2)))
    tol_t, tol_a = (1.5e-3, 0.08) if quantised else (5e-4, 0.03)
    assert cnt > 40000 and np.linalg.norm(err[:3, 3]) < tol_t and ang < tol_a, (np.linalg.norm(err[:3, 3]), ang)
    assert rms < 3e-3
    # and the first coarse step already moves the right way: the error to dT shrinks
    A, b, _, _ = fe.icp_step(meas, pred, K, 2, np.eye(4))
    T1, _ = fe.se3_update(np.eye(4), A, b)
    assert np.linalg.norm((np.linalg.inv(dT) @ T1)[:3, 3]) < 0.6 * np.linalg.norm(dT[:3, 3])


def test_conditioning_closed_forms():
    """F6's gate: 1 for a diagonal A; 1 - c^2 / (a b) for one coupled pair (the second pivot is b - c^2 / a); unchanged by a
    rescaling of the parameters; 0 for a singular or indefinite A."""
    assert abs(fe.conditioning(np.diag([2.0, 3.0, 4.0, 5.0, 6.0, 7.0])) - 1.0) < 1e-15
    A = np.diag([2.0, 3.0, 4.0, 5.0, 6.0, 7.0]); A[1, 4] = A[4, 1] = 3.0
    assert abs(fe.conditioning(A) - (1.0 - 9.0 / 18.0)) < 1e-15
    S = np.diag([1.0, 1e3, 1.0, 1e-3, 10.0, 1.0])
    assert abs(fe.conditioning(S @ A @ S) - 0.5) < 1e-12
    J = np.array([1.0, 2.0, 0.5, -1.0, 0.3, 0.7])
    assert fe.conditioning(np.outer(J, J)) == 0.0                               # rank 1
    assert fe.conditioning(np.diag([1.0, 1.0, -1.0, 1.0, 1.0, 1.0])) == 0.0     # indefinite


def test_track_refuses_an_unobservable_motion():
    """A camera facing a wall: sliding along the wall and turning about its normal change nothing, so three of the six
    parameters are unobservable; A is singular up to rounding and F7 reports status 3 instead of solving.  (Exact depth: the
    normals are the plane's to rounding; on a structured scene the same gate stays far from its threshold.)"""
    n = np.array([0.1, -0.2, 0.97], np.float64); n /= np.linalg.norm(n)
    D = plane_depth_exact(K, W, H, n, 1.4)
    pyr = fe.pyramid(D.astype(np.float32), K, 3)
    A, _, _, cnt = fe.icp_step(pyr, pyr, K, 2, np.eye(4))
    assert cnt > 3000 and fe.conditioning(A) < 1e-6
    with pytest.raises(fe.TrackingLost) as e:
        fe.track(pyr, pyr, K)
    assert e.value.status == 3
    meas, pred = scene_pair(np.eye(4))
    A, _, _, _ = fe.icp_step(meas, pred, K, 0, np.eye(4))
    assert fe.conditioning(A) > 1e-3
    empty = [(np.zeros_like(d), np.zeros_like(v), np.zeros_like(nn)) for d, v, nn in pred]
    with pytest.raises(fe.TrackingLost) as e:
        fe.track(meas, empty, K)
    assert e.value.status == 1


def test_filtered_prediction_removes_voxel_steps():
    """F8: a plane with voxel-sized steps (what nearest-voxel ray casting leaves): unfiltered, most forward-difference normals
    miss the plane's normal by more than the ICP gate of 20 degrees; rounded to millimetres and filtered, nearly all agree."""
    n = np.array([0.45, 0.2, 0.87], np.float64); n /= np.linalg.norm(n)
    D = plane_depth_exact(K, W, H, n, 1.3)
    stepped = (np.floor(D / 0.004) * 0.004).astype(np.float32)                       # 4 mm terraces
    raw = fe.pyramid(stepped, K, 1)[0][2].astype(np.float64)[8:-8, 8:-8]
    fil = fe.predict(stepped, K, 1)[0][2].astype(np.float64)[8:-8, 8:-8]
    good = lambda N: float(((N @ n) > 0.94).mean())
    assert good(raw) < 0.6 and good(fil) > 0.99
    q = fe.predict(np.array([[0.0, 1.2344, 70.0, 1.2345]], np.float32), K, 1)[0][0]
    assert q[0, 0] == 0 and abs(float(q[0, 2]) - 65.535) < 1e-5                       # 0 stays invalid; clamp at 65535 mm
