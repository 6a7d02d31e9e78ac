"""More oracle pins (no GPU): eq. 9/10 recursions, the 0.8 gate, HD mapping, fp64 brute force."""
import numpy as np
import pytest

import oracle
import synth
from bruteforce_np import BruteVolume

CFG = synth.config(1)
I4 = np.eye(4, dtype=np.float32)


def plane_vol(n=24, r=2, sigma=0.020, oz=1.0):
    origin = np.array([-0.5, -0.5, oz], np.float32)
    return oracle.RefVolume((n, n, n), r, origin, 1.0, 3.0 / n, 128, sigma=sigma)


def weight_sequence(W, n, gate=0.8):
    """eq. 10 on the u8 scale with the L115 gate, real arithmetic: returns the stored weights after each frame."""
    wq, out = 0, []
    for _ in range(n):
        if 255.0 * W > gate * wq:
            wq = min(255, int(np.rint(wq + W * (255 - wq))))
        out.append(wq)
    return out


def test_weight_sequences_of_the_survey():
    """Sequences listed in SURVEY 8(c) re-derived from eq. 10 + L115 (not from the oracle)."""
    assert weight_sequence(1.0, 3) == [255, 255, 255]
    assert weight_sequence(0.9, 4) == [230, 252, 255, 255]
    assert weight_sequence(0.8, 6)[:4] == [204, 245, 253, 255] and weight_sequence(0.8, 6)[4:] == [255, 255]
    assert weight_sequence(0.75, 5) == [191, 239, 251, 251, 251]
    assert weight_sequence(0.7, 4) == [178, 232, 232, 232]
    assert weight_sequence(0.3, 4) == [76, 130, 130, 130]


def test_weight_recursion_and_gate_on_a_plane():
    """Same plane for 6 frames: every colour voxel's stored weight follows eq. 10 (W_n = 1-(1-W)^n up to u8
    rounding) until the 0.8 gate of L115 closes; W is the closed-form off-axis cosine of its depth pixel."""
    n, r = 24, 2
    v = plane_vol(n, r, oz=0.3)
    K = synth.intrinsics(70.0, 79.5, 59.5)              # wide field of view: W spans ~0.62 .. 1
    Kh = synth.intrinsics(140.0, 159.5, 119.5)
    hist = []
    for _ in range(6):
        v.integrate(synth.plane_depth(160, 120, 500), synth.const_rgb(320, 240, (200, 100, 50)), I4, K, Kh, CFG.T_depth_rgb)
        hist.append(oracle.col_w(v.col).copy())
    N = n * r
    k, j, i = np.meshgrid(np.arange(N), np.arange(N), np.arange(N), indexing="ij")
    X, Y, Z = -0.5 + (i + 0.5) / N, -0.5 + (j + 0.5) / N, 0.3 + (k + 0.5) / N
    u, vv = 70.0 * X / Z + 79.5, 70.0 * Y / Z + 59.5
    safe = (np.abs(u + 0.5 - np.rint(u + 0.5)) > 1e-3) & (np.abs(vv + 0.5 - np.rint(vv + 0.5)) > 1e-3)
    xf, yf = np.floor(u + 0.5), np.floor(vv + 0.5)
    W = 1.0 / np.sqrt(1.0 + ((xf - 79.5) / 70.0) ** 2 + ((yf - 59.5) / 70.0) ** 2)
    touched = hist[0] > 0
    sel = np.flatnonzero(touched & safe)[::3]
    assert sel.size > 500
    Wmin, Wmax = W.reshape(-1)[sel].min(), W.reshape(-1)[sel].max()
    assert Wmin < 0.72 and Wmax > 0.99                   # covers gate-closing and never-closing voxels
    bad = 0
    for idx in sel:
        w = float(W.reshape(-1)[idx])
        got = [int(h.reshape(-1)[idx]) for h in hist]
        # skip voxels within rounding distance of a gate / tie decision (A16)
        wq, fragile = 0, False
        for _ in range(6):
            if abs(255.0 * w - 0.8 * wq) < 1e-2 or abs((wq + w * (255 - wq)) % 1.0 - 0.5) < 1e-2:
                fragile = True
            if 255.0 * w > 0.8 * wq:
                wq = min(255, int(np.rint(wq + w * (255 - wq))))
        if fragile:
            continue
        bad += got != weight_sequence(w, 6)
        if w >= 0.81:                                     # gate never closes: unquantised closed form within u8 rounding
            assert all(abs(g / 255.0 - (1 - (1 - w) ** (t + 1))) < 4.0 / 255 for t, g in enumerate(got))
    assert bad == 0


def test_constant_colour_frame_gives_constant_colour_volume():
    """eq. 9 with HD == c everywhere: every voxel with weight > 0 holds exactly c, all others stay 0 (BASELINE)."""
    c = synth.config(1)
    v = oracle.RefVolume((32, 32, 32), 2, c.origin, c.extent, 3.0 / 32, 128)
    col = (37, 201, 114)
    for i in range(5):
        depth, _, T = synth.frame(c, i, want_rgb=False)
        v.integrate(depth, synth.const_rgb(c.wh, c.hh, col), T, c.K_depth, c.K_rgb, c.T_depth_rgb)
    wq, rgb = oracle.col_w(v.col), oracle.col_rgb(v.col)
    assert (wq > 0).sum() > 2000
    assert np.all(rgb[wq > 0] == np.array(col))
    assert not v.col[wq == 0].any()


def test_two_alternating_colours():
    """Frame 1 colour c1, frame 2 colour c2, same W: C1 = c1, C2 = rint((c1*wq1 + 255 W c2)/(wq1 + 255 W)) (eq. 9)."""
    v = plane_vol(16, 2)
    c1, c2 = np.array([250, 10, 100]), np.array([20, 240, 101])
    dep = synth.plane_depth(160, 120, 1500)
    v.integrate(dep, synth.const_rgb(320, 240, c1), I4, CFG.K_depth, CFG.K_rgb, CFG.T_depth_rgb)
    wq1 = oracle.col_w(v.col).copy()
    assert np.all(oracle.col_rgb(v.col)[wq1 > 0] == c1)
    v.integrate(dep, synth.const_rgb(320, 240, c2), I4, CFG.K_depth, CFG.K_rgb, CFG.T_depth_rgb)
    rgb2 = oracle.col_rgb(v.col)
    N = 32
    k, j, i = np.meshgrid(np.arange(N), np.arange(N), np.arange(N), indexing="ij")
    X, Y, Z = -0.5 + (i + 0.5) / N, -0.5 + (j + 0.5) / N, 1.0 + (k + 0.5) / N
    xf, yf = np.floor(131.25 * X / Z + 79.5 + 0.5), np.floor(131.25 * Y / Z + 59.5 + 0.5)
    W = 1.0 / np.sqrt(1.0 + ((xf - 79.5) / 131.25) ** 2 + ((yf - 59.5) / 131.25) ** 2)
    m = wq1 > 0
    expect = (c1[None, :] * wq1[m][:, None] + 255.0 * W[m][:, None] * c2[None, :]) / (wq1[m] + 255.0 * W[m])[:, None]
    assert m.sum() > 500
    assert np.all(np.abs(rgb2[m] - expect) <= 0.5 + 1e-3)


def test_r1_colour_voxels_pick_the_geometry_voxels_pixel():
    """r = 1 (PCL's symmetric scheme, L85): colour voxel (i,j,k) has the same centre as geometry voxel (i,j,k), so every
    colour-updated voxel was also TSDF-updated and |sdf| <= sigma there (|Z - D| <= |P_vc - P_vd| <= sigma)."""
    c = synth.config(1)
    n = 48
    v = oracle.RefVolume((n, n, n), 1, c.origin, c.extent, 3.0 / n, 128)       # mu = 62.5 mm > sigma
    depth, rgb, T = synth.frame(c, 2)
    v.integrate(depth, rgb, T, c.K_depth, c.K_rgb, c.T_depth_rgb)
    wq, gw, q = oracle.col_w(v.col), oracle.geo_w(v.geo), oracle.geo_q(v.geo)
    assert (wq > 0).sum() > 500
    assert np.all(gw[wq > 0] == 1)
    assert np.all(np.abs(q[wq > 0]) <= 32767 * 0.020 / (3.0 / n) + 1)


def test_hd_mapping_coordinate_coded():
    """Coordinate-coded RGB (R = x mod 256, G = y mod 256, B = tile id): after one frame each updated colour voxel reveals
    the HD pixel it sampled; it must be the nearest pixel of K_hd (R_calib P_vc + t_calib) (eq. 3-4, A10/A11), with the RGB
    camera 25 mm to the right of the depth camera."""
    c = synth.config(1)
    n, r = 24, 2
    v = oracle.RefVolume((n, n, n), r, c.origin, c.extent, 3.0 / n, 128)
    T = synth.rigid32(c.pose(1))
    depth, _, _ = synth.frame(c, 1, want_rgb=False)
    v.integrate(depth, synth.coord_rgb(c.wh, c.hh), T, c.K_depth, c.K_rgb, c.T_depth_rgb)
    wq, rgb = oracle.col_w(v.col), oracle.col_rgb(v.col)
    N = n * r
    k, j, i = np.meshgrid(np.arange(N), np.arange(N), np.arange(N), indexing="ij")
    Pw = np.stack([c.origin[0] + (i + 0.5) / N, c.origin[1] + (j + 0.5) / N, c.origin[2] + (k + 0.5) / N, np.ones_like(i)], -1)
    Pc = Pw @ np.linalg.inv(T.astype(np.float64)).T
    Ph = Pc @ np.linalg.inv(c.T_depth_rgb.astype(np.float64)).T
    assert np.allclose(Ph[..., 0], Pc[..., 0] - 0.025)                      # t_calib = (-25 mm, 0, 0)
    u = 262.5 * Ph[..., 0] / Ph[..., 2] + 159.5
    w_ = 262.5 * Ph[..., 1] / Ph[..., 2] + 119.5
    safe = (np.abs(u + 0.5 - np.rint(u + 0.5)) > 2e-3) & (np.abs(w_ + 0.5 - np.rint(w_ + 0.5)) > 2e-3)
    m = (wq > 0) & safe
    assert m.sum() > 600
    xh, yh = np.floor(u + 0.5).astype(int)[m], np.floor(w_ + 0.5).astype(int)[m]
    assert np.array_equal(rgb[m][:, 0], xh % 256) and np.array_equal(rgb[m][:, 1], yh % 256)
    assert np.array_equal(rgb[m][:, 2], xh // 256 + 16 * (yh // 256))


def test_rigid_inverse_constants():
    """S0: (R_n, t_n) = inverse(T_world_depth) and (R_calib, t_calib) = inverse(T_depth_rgb) vs numpy.linalg.inv."""
    c = synth.config(3)
    v = oracle.RefVolume((4, 4, 4), 1, c.origin, c.extent, 0.1, 8)
    for i in (0, 17, 250):
        T = synth.rigid32(c.pose(i))
        R, t, Rc, tc = v.frame_constants(T, c.T_depth_rgb)
        inv = np.linalg.inv(T.astype(np.float64))
        assert np.abs(R - inv[:3, :3]).max() < 2e-7 and np.abs(t - inv[:3, 3]).max() < 5e-7
        assert np.allclose(Rc, np.eye(3)) and np.allclose(tc, [-0.025, 0, 0])


@pytest.mark.parametrize("cfgn,r,n,frames", [(1, 2, 20, (0, 2, 4)), (1, 3, 12, (1, 3)), (2, 3, 20, (5, 40, 80)), (2, 1, 40, (7,)), (3, 2, 32, (10, 11))])
def test_bruteforce_fp64_whole_pipeline(cfgn, r, n, frames):
    """Oracle (binary32, fixed order) vs the independent float64 numpy brute force on tiny volumes, general poses,
    noisy depth with dropouts, textured RGB: identical integer state on every non-fragile voxel (A16)."""
    c = synth.config(cfgn).scaled(n, r)
    v = oracle.RefVolume(c.dims_geo, c.r, c.origin, c.extent, c.mu, c.w_max)
    b = BruteVolume(c.dims_geo, c.r, c.origin, c.extent, c.mu, c.w_max)
    for fi in frames:
        depth, rgb, T = synth.frame(c, fi)
        cnt = v.integrate(depth, rgb, T, c.K_depth, c.K_rgb, c.T_depth_rgb)
        b.integrate(depth, rgb, T, c.K_depth, c.K_rgb, c.T_depth_rgb)
        okc = ~b.frag_col
        # counters: read / updated sets agree wherever not fragile
        assert abs(int(cnt[2]) - int(b.read_col.sum())) <= int(b.frag_col.sum())
    okg = ~b.frag_geo
    q, w = oracle.geo_q(v.geo), oracle.geo_w(v.geo)
    assert okg.mean() > 0.95 and okc.mean() > 0.95
    assert (w > 0).sum() > 200 and (b.wq > 0).sum() > 20
    assert np.array_equal(w[okg], b.w[okg])
    assert np.abs(q[okg] - b.q[okg]).max() <= 1 and (q[okg] == b.q[okg]).mean() > 0.995
    assert np.array_equal(oracle.col_w(v.col)[okc], b.wq[okc])
    dC = np.abs(oracle.col_rgb(v.col)[okc] - b.C[okc])
    assert dC.max() <= 1 and (dC == 0).mean() > 0.995


def test_subset_equals_dense():
    c = synth.config(1).scaled(24, 2)
    v = oracle.RefVolume(c.dims_geo, c.r, c.origin, c.extent, c.mu, c.w_max)
    s = oracle.RefVolume(c.dims_geo, c.r, c.origin, c.extent, c.mu, c.w_max, allocate=False)
    rng = np.random.default_rng(5)
    gi = np.sort(rng.choice(24 ** 3, 3000, replace=False)).astype(np.int64)
    ci = np.sort(rng.choice(48 ** 3, 20000, replace=False)).astype(np.int64)
    gw, cw = np.zeros(gi.size, np.uint32), np.zeros(ci.size, np.uint32)
    for fi in range(4):
        depth, rgb, T = synth.frame(c, fi)
        v.integrate(depth, rgb, T, c.K_depth, c.K_rgb, c.T_depth_rgb)
        s.integrate_subset(gi, gw, ci, cw, depth, rgb, T, c.K_depth, c.K_rgb, c.T_depth_rgb)
    assert np.array_equal(v.geo.reshape(-1)[gi], gw) and np.array_equal(v.col.reshape(-1)[ci], cw)
    assert gw.any() and cw.any()
