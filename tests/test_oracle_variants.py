"""Pins of the oracle's alternative readings, no GPU: each switch against
a closed form, an invariant that separates it from the default reading, and the independent float64 brute force."""
import numpy as np
import pytest

import oracle
import synth
from bruteforce_np import BruteVolume

CFG = synth.config(1)
I4 = np.eye(4, dtype=np.float32)
HD_POINT, RAY, ADD = oracle.VAR_HD_FROM_DEPTH_POINT, oracle.VAR_TSDF_ALONG_RAY, oracle.VAR_ADDITIVE_WEIGHT


def skewed_hd(c):
    """An HD camera whose intrinsics are NOT an exact multiple of the depth camera's.  (With the configs' K_hd = 2 K_c and no
    vertical offset, the point of a depth pixel projects exactly onto the boundary between two HD rows, v_hd = 2 y + 1/2: the
    literal reading then samples a row that rounding decides -- fine for bit-exact parity, useless for a float64 pin.)"""
    K = np.array(c.K_rgb, np.float32).reshape(3, 3).copy()
    K[0, 0] *= 1.013; K[1, 1] *= 1.013; K[0, 2] += 0.37; K[1, 2] += 0.21
    return K


def test_variant_argument_is_checked():
    c = synth.config(1).scaled(8, 1)
    depth, rgb, T = synth.frame(c, 0)
    for bad in (3, 5, 7, 8, -1):
        v = oracle.RefVolume(c.dims_geo, c.r, c.origin, c.extent, c.mu, c.w_max, variant=bad)
        with pytest.raises(ValueError):
            v.integrate(depth, rgb, T, c.K_depth, c.K_rgb, c.T_depth_rgb)


# ---------------------------------------------------------------- (c) signed distance along the viewing ray
def test_ray_tsdf_closed_form_on_a_plane():
    """Plane z = D seen from the origin: the distance from voxel P to the plane ALONG the ray through P is
    (D - Z) |P| / Z = (D - Z) / cos(theta).  One frame: q = rint(32767 min(1, that / mu)) where the voxel is updated."""
    n, D = 32, 1.5
    origin = np.array([-0.5, -0.5, 1.0], np.float32)
    mu = 0.115
    v = oracle.RefVolume((n, n, n), 1, origin, 1.0, mu, 64, variant=RAY)
    d = oracle.RefVolume((n, n, n), 1, origin, 1.0, mu, 64)
    K = synth.intrinsics(70.0, 79.5, 59.5)                                   # wide: 1 / cos(theta) up to ~1.14 in the volume
    for vol in (v, d):
        vol.integrate(synth.plane_depth(160, 120, 1500), synth.const_rgb(320, 240, (9, 9, 9)), I4, K, CFG.K_rgb, CFG.T_depth_rgb)
    k, j, i = np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij")
    X, Y, Z = -0.5 + (i + 0.5) / n, -0.5 + (j + 0.5) / n, 1.0 + (k + 0.5) / n
    lam = np.sqrt(X * X + Y * Y + Z * Z) / Z
    sdf = (D - Z) * lam
    w, q = oracle.geo_w(v.geo), oracle.geo_q(v.geo)
    mu32 = float(np.float32(mu))
    clear = np.abs(sdf + mu32) > 1e-5
    assert np.array_equal((w == 1)[clear], (sdf >= -mu32)[clear])
    m = (w == 1) & clear
    assert m.sum() > 15000 and lam[m].max() > 1.1
    expect = 32767.0 * np.minimum(1.0, sdf[m] / mu32)
    # binary32 D - Z near 1.5 m carries up to ~3e-7 m of rounding: 3e-7 / mu * 32767 < 0.1 code
    assert np.abs(q[m] - expect).max() <= 0.5 + 0.1
    # against the default reading: |sdf| grows by 1 / cos(theta) >= 1, so fewer voxels behind the surface are updated and
    # the ramp is steeper everywhere else; on the optical axis (X = Y ~ 0) the two coincide up to rounding
    wd_, qd = oracle.geo_w(d.geo), oracle.geo_q(d.geo)
    assert np.all(wd_[w == 1] == 1) and (wd_ == 1).sum() > (w == 1).sum()
    both = (w == 1) & (wd_ == 1)
    assert np.all(np.abs(q[both]) >= np.abs(qd[both]) - 1)
    steeper = both & (np.abs(qd) < 30000) & (np.abs(qd) > 2000) & (lam > 1.05)
    assert steeper.sum() > 500 and np.all(np.abs(q[steeper]) > np.abs(qd[steeper]))
    axis = both & (np.abs(X) < 0.02) & (np.abs(Y) < 0.02)
    assert axis.sum() >= 30 and np.abs(q[axis] - qd[axis]).max() <= 32767 * 0.0012 * 0.5 / mu32 + 1   # lam - 1 <= 4e-4 there


# ---------------------------------------------------------------- (b) HD pixel from the depth pixel's point
def test_hd_from_depth_point_coordinate_coded():
    """Coordinate-coded RGB: each updated colour voxel reveals the HD pixel it sampled.  Under the literal reading it is the
    nearest pixel of K_hd (R_calib P_vd + t_calib), P_vd = K_c^-1 (x, y, D(x, y)) of the voxel's depth pixel (eq. 7, eq. 3-4)
    -- so every voxel behind one depth pixel carries the same colour, which the default reading (A11) avoids."""
    c = synth.config(1)
    n, r = 24, 2
    T = synth.rigid32(c.pose(1))
    depth, _, _ = synth.frame(c, 1, want_rgb=False)
    vols = {}
    for var in (0, HD_POINT):
        vols[var] = oracle.RefVolume((n, n, n), r, c.origin, c.extent, 3.0 / n, 128, variant=var)
        vols[var].integrate(depth, synth.coord_rgb(c.wh, c.hh), T, c.K_depth, skewed_hd(c), c.T_depth_rgb)
    v = vols[HD_POINT]
    wq, rgb = oracle.col_w(v.col), oracle.col_rgb(v.col)
    N = n * r
    k, j, i = np.meshgrid(np.arange(N), np.arange(N), np.arange(N), indexing="ij")
    Pw = np.stack([c.origin[0] + (i + 0.5) / N, c.origin[1] + (j + 0.5) / N, c.origin[2] + (k + 0.5) / N, np.ones_like(i)], -1)
    Pc = Pw @ np.linalg.inv(T.astype(np.float64)).T
    Kd = np.asarray(c.K_depth, np.float64)
    u = Kd[0, 0] * Pc[..., 0] / Pc[..., 2] + Kd[0, 2]
    w_ = Kd[1, 1] * Pc[..., 1] / Pc[..., 2] + Kd[1, 2]
    safe = (np.abs(u + 0.5 - np.rint(u + 0.5)) > 2e-3) & (np.abs(w_ + 0.5 - np.rint(w_ + 0.5)) > 2e-3)
    m = (wq > 0) & safe
    assert m.sum() > 600
    x, y = np.floor(u + 0.5).astype(int)[m], np.floor(w_ + 0.5).astype(int)[m]
    D = depth[y, x].astype(np.float64) * 1e-3
    Pd = np.stack([(x - Kd[0, 2]) * D / Kd[0, 0], (y - Kd[1, 2]) * D / Kd[1, 1], D, np.ones_like(D)], -1)
    Ph = Pd @ np.linalg.inv(c.T_depth_rgb.astype(np.float64)).T
    Kh = skewed_hd(c).astype(np.float64)
    uh = Kh[0, 0] * Ph[:, 0] / Ph[:, 2] + Kh[0, 2]
    vh = Kh[1, 1] * Ph[:, 1] / Ph[:, 2] + Kh[1, 2]
    ok = (np.abs(uh + 0.5 - np.rint(uh + 0.5)) > 2e-3) & (np.abs(vh + 0.5 - np.rint(vh + 0.5)) > 2e-3)
    xh, yh = np.floor(uh + 0.5).astype(int), np.floor(vh + 0.5).astype(int)
    got = rgb[m]
    assert ok.sum() > 500
    assert np.array_equal(got[ok, 0], xh[ok] % 256) and np.array_equal(got[ok, 1], yh[ok] % 256)
    assert np.array_equal(got[ok, 2], xh[ok] // 256 + 16 * (yh[ok] // 256))
    # one colour per depth pixel; the default reading gives the voxels of one depth pixel several HD pixels
    pix = y * c.wd + x
    words = (v.col & np.uint32(0xffffff))[m]
    words0 = (vols[0].col & np.uint32(0xffffff))[m]
    order = np.argsort(pix, kind="stable")
    ps, ws, w0 = pix[order], words[order], words0[order]
    same_pix = ps[1:] == ps[:-1]
    assert same_pix.sum() > 200
    assert np.all(ws[1:][same_pix] == ws[:-1][same_pix])
    assert (w0[1:][same_pix] != w0[:-1][same_pix]).mean() > 0.3
    # which voxels are updated, and their weights, do not depend on the reading (only A13 could differ: not in this frame)
    assert np.array_equal(oracle.col_w(vols[0].col), wq) and np.array_equal(vols[0].geo, v.geo)


# ---------------------------------------------------------------- (d) additive colour weight
def weight_sequence_additive(W, n, gate=0.8):
    """W_new = min(W_pre + W, 1) on the u8 scale with the L115 gate, real arithmetic."""
    wq, out = 0, []
    for _ in range(n):
        if 255.0 * W > gate * wq:
            wq = min(255, int(np.rint(wq + 255.0 * W)))
        out.append(wq)
    return out


def test_additive_weight_sequences():
    """Same plane for 5 frames: the stored weight of every colour voxel follows W_pre + W until it saturates or the 0.8
    gate closes; W = the closed-form off-axis cosine of the voxel's depth pixel.  Differs from eq. 10 from frame 2 on."""
    assert weight_sequence_additive(0.9, 3) == [230, 255, 255]                 # eq. 10 gives 230, 252, 255
    assert weight_sequence_additive(0.7, 4) == [178, 255, 255, 255]            # eq. 10: 178, 232, 232, 232
    assert weight_sequence_additive(0.3, 4) == [76, 152, 152, 152]             # eq. 10: 76, 130, 130, 130
    n, r = 24, 2
    origin = np.array([-0.5, -0.5, 0.3], np.float32)
    v = oracle.RefVolume((n, n, n), r, origin, 1.0, 3.0 / n, 128, variant=ADD)
    K = synth.intrinsics(70.0, 79.5, 59.5)
    Kh = synth.intrinsics(140.0, 159.5, 119.5)
    hist = []
    for _ in range(5):
        v.integrate(synth.plane_depth(160, 120, 500), synth.const_rgb(320, 240, (200, 100, 50)), I4, K, Kh, CFG.T_depth_rgb)
        hist.append(oracle.col_w(v.col).copy())
    N = n * r
    k, j, i = np.meshgrid(np.arange(N), np.arange(N), np.arange(N), indexing="ij")
    X, Y, Z = -0.5 + (i + 0.5) / N, -0.5 + (j + 0.5) / N, 0.3 + (k + 0.5) / N
    u, vv = 70.0 * X / Z + 79.5, 70.0 * Y / Z + 59.5
    safe = (np.abs(u + 0.5 - np.rint(u + 0.5)) > 1e-3) & (np.abs(vv + 0.5 - np.rint(vv + 0.5)) > 1e-3)
    xf, yf = np.floor(u + 0.5), np.floor(vv + 0.5)
    W = 1.0 / np.sqrt(1.0 + ((xf - 79.5) / 70.0) ** 2 + ((yf - 59.5) / 70.0) ** 2)
    sel = np.flatnonzero((hist[0] > 0) & safe)[::3]
    assert sel.size > 500
    checked = 0
    for idx in sel:
        w = float(W.reshape(-1)[idx])
        wq, fragile = 0, False
        for _ in range(5):
            if abs(255.0 * w - 0.8 * wq) < 1e-2 or abs((wq + 255.0 * w) % 1.0 - 0.5) < 1e-2:
                fragile = True
            if 255.0 * w > 0.8 * wq:
                wq = min(255, int(np.rint(wq + 255.0 * w)))
        if fragile:
            continue
        assert [int(h.reshape(-1)[idx]) for h in hist] == weight_sequence_additive(w, 5)
        checked += 1
    assert checked > 400
    # colours are untouched by the switch in the first frame (eq. 9 uses W_pre = 0 either way)
    assert np.all(oracle.col_rgb(v.col)[hist[0] > 0] == np.array((200, 100, 50)))


# ---------------------------------------------------------------- all three against the float64 brute force
@pytest.mark.parametrize("variant", [HD_POINT, RAY, ADD])
@pytest.mark.parametrize("cfgn,r,n,frames", [(1, 2, 20, (0, 2, 4)), (2, 3, 16, (5, 40, 80)), (3, 2, 24, (10, 11))])
def test_bruteforce_fp64_variants(variant, cfgn, r, n, frames):
    c = synth.config(cfgn).scaled(n, r)
    v = oracle.RefVolume(c.dims_geo, c.r, c.origin, c.extent, c.mu, c.w_max, variant=variant)
    b = BruteVolume(c.dims_geo, c.r, c.origin, c.extent, c.mu, c.w_max, variant=variant)
    d = oracle.RefVolume(c.dims_geo, c.r, c.origin, c.extent, c.mu, c.w_max)
    Kh = skewed_hd(c)
    for fi in frames:
        depth, rgb, T = synth.frame(c, fi)
        v.integrate(depth, rgb, T, c.K_depth, Kh, c.T_depth_rgb)
        b.integrate(depth, rgb, T, c.K_depth, Kh, c.T_depth_rgb)
        d.integrate(depth, rgb, T, c.K_depth, Kh, c.T_depth_rgb)
    okg, okc = ~b.frag_geo, ~b.frag_col
    q, w = oracle.geo_q(v.geo), oracle.geo_w(v.geo)
    assert okg.mean() > 0.95 and okc.mean() > 0.95
    assert (w > 0).sum() > 200 and (b.wq > 0).sum() > 20
    assert np.array_equal(w[okg], b.w[okg])
    assert np.abs(q[okg] - b.q[okg]).max() <= 1 and (q[okg] == b.q[okg]).mean() > 0.995
    assert np.array_equal(oracle.col_w(v.col)[okc], b.wq[okc])
    dC = np.abs(oracle.col_rgb(v.col)[okc] - b.C[okc])
    assert dC.max() <= 1 and (dC == 0).mean() > 0.995
    # the switch is live: the state differs from the default reading's, and only in the volume it concerns
    if variant == RAY:
        assert not np.array_equal(v.geo, d.geo) and np.array_equal(v.col, d.col)
    else:
        assert np.array_equal(v.geo, d.geo) and not np.array_equal(v.col, d.col)
