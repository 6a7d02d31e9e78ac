"""GPU parity of vol_raycast against the oracle's ref_raycast: depth bit for bit, colours byte for byte."""
import numpy as np
import pytest

import synth
from parity_util import integrate_both, make_pair

pytestmark = pytest.mark.gpu


def cast_both(g, o, w, h, T, K, t_near, t_far, with_rgb=True, trilinear=False):
    import torch
    dd = torch.full((h * w,), -1.0, dtype=torch.float32, device="cuda")
    dr = torch.full((h * w * 3,), 7, dtype=torch.uint8, device="cuda") if with_rgb else None
    (g.raycast_trilinear if trilinear else g.raycast)(w, h, T, K, t_near, t_far, dd, dr)
    torch.cuda.synchronize()
    od, orgb = (o.raycast_trilinear if trilinear else o.raycast)(w, h, T, K, t_near, t_far)
    gd = dd.cpu().numpy().reshape(h, w)
    assert np.array_equal(gd.view(np.uint32), od.view(np.uint32)), f"{int((gd.view(np.uint32) != od.view(np.uint32)).sum())} depths differ"
    if with_rgb:
        assert np.array_equal(dr.cpu().numpy().reshape(h, w, 3), orgb)
    return od, orgb


def fused_pair(c, frames):
    g, o = make_pair(c)
    for fi in frames:
        depth, rgb, T = synth.frame(c, fi)
        integrate_both(g, o, c, depth, rgb, T, counting=False)
    return g, o


@pytest.mark.parametrize("tri", [False, True])
def test_raycast_cfg1_views(tri):
    """Config 1 after its 5 frames: the scan's own camera, an oblique camera, a camera inside the volume, a ragged image
    size (not a multiple of the 8 x 8 pixel CTA), t_near on and off the voxel grid.  Both readings of the TSDF sample:
    nearest voxel (R3) and trilinear (R7)."""
    c = synth.config(1)
    g, o = fused_pair(c, range(5))
    d, rgb = cast_both(g, o, c.wd, c.hd, synth.frame(c, 2)[2], c.K_depth, 0.4, 3.0, trilinear=tri)
    assert (d > 0).sum() > 2000 and (rgb.sum(axis=2) > 0).sum() > 2000
    T = synth.rigid32(synth.look_at((0.25, -0.15, 0.1), (0.0, 0.0, 1.5), up=(0.0, -1.0, 0.0)))
    d, _ = cast_both(g, o, 157, 93, T, c.K_depth, 0.3125, 2.75, trilinear=tri)
    assert (d > 0).sum() > 2000
    T = synth.rigid32(synth.look_at((0.1, 0.3, 1.15), (0.0, 0.0, 1.5), up=(0.0, -1.0, 0.0)))     # inside the cube
    cast_both(g, o, c.wd, c.hd, T, c.K_depth, 0.0, 1.0, trilinear=tri)
    cast_both(g, o, c.wd, c.hd, T, c.K_depth, 0.05, 0.05, trilinear=tri)                           # a single sample: no pair, no hit
    cast_both(g, o, 64, 48, T, c.K_rgb, 0.0, 2.0, with_rgb=False, trilinear=tri)                   # depth only


def test_raycast_cfg2_r3_and_empty_volume():
    c = synth.config(2).scaled(96, 3)
    g, o = make_pair(c)
    T0 = synth.frame(c, 0)[2]
    d, rgb = cast_both(g, o, 80, 60, T0, c.K_depth / np.array([[8, 1, 8], [1, 8, 8], [1, 1, 1]], np.float32), 0.2, 4.0)
    assert not d.any() and not rgb.any()                                                           # nothing observed yet
    for fi in (0, 10, 20, 30):
        depth, rgb_in, T = synth.frame(c, fi)
        integrate_both(g, o, c, depth, rgb_in, T, counting=False)
    d, rgb = cast_both(g, o, c.wd, c.hd, synth.frame(c, 15)[2], c.K_depth, 0.2, 4.0)
    assert (d > 0).mean() > 0.2
    want = synth.frame(c, 15)[0].astype(np.float32) * 1e-3
    both = (d > 0) & (want > 0)
    assert np.median(np.abs(d[both] - want[both])) < 2.0 * c.extent / 96                          # it is the scene that was fused
    dt, _ = cast_both(g, o, c.wd, c.hd, synth.frame(c, 15)[2], c.K_depth, 0.2, 4.0, trilinear=True)
    both = (dt > 0) & (want > 0)
    assert (dt > 0).mean() > 0.2 and np.median(np.abs(dt[both] - want[both])) < 1.0 * c.extent / 96
    cast_both(g, o, 301, 203, synth.frame(c, 33)[2], c.K_depth / np.array([[2, 1, 2], [1, 2, 2], [1, 1, 1]], np.float32), 0.37, 3.1, trilinear=True)


def test_raycast_skip_flags_follow_the_volume():
    """The casters' skip flags are rebuilt whenever the geometry volume has changed -- by vol_integrate, by vol_upload (content
    the integration never saw: every tile must be looked at) and by vol_reset (nothing left to hit) -- and not otherwise: casts
    between changes, from different cameras, both readings, always equal the oracle's."""
    import paper_1602_06645_b200 as vf
    c = synth.config(2).scaled(96, 2)
    g, o = fused_pair(c, (0, 10))
    Ta, Tb = synth.frame(c, 5)[2], synth.frame(c, 40)[2]
    for tri in (False, True):
        cast_both(g, o, c.wd, c.hd, Ta, c.K_depth, 0.2, 4.0, trilinear=tri)
        cast_both(g, o, c.wd, c.hd, Tb, c.K_depth, 0.2, 4.0, trilinear=tri)            # flags reused
    depth, rgb, T = synth.frame(c, 20)
    integrate_both(g, o, c, depth, rgb, T, counting=False)                          # the volume changes: rebuilt
    for tri in (True, False):
        d, _ = cast_both(g, o, c.wd, c.hd, Tb, c.K_depth, 0.2, 4.0, trilinear=tri)
        assert (d > 0).mean() > 0.1
    # a second volume receives the state through vol_upload: no integration has flagged anything there
    h = vf.Volume(c.dims_geo, c.r, c.origin, c.extent, c.mu, c.w_max)
    cast_both(h, type(o)(c.dims_geo, c.r, c.origin, c.extent, c.mu, c.w_max), 80, 60, Ta, c.K_depth / np.array([[8, 1, 8], [1, 8, 8], [1, 1, 1]], np.float32), 0.2, 4.0)
    h.upload(o.geo, o.col)
    for tri in (False, True):
        d, _ = cast_both(h, o, c.wd, c.hd, Ta, c.K_depth, 0.2, 4.0, trilinear=tri)
        assert (d > 0).mean() > 0.1
    h.reset()
    import torch
    dd = torch.full((c.wd * c.hd,), -1.0, dtype=torch.float32, device="cuda")
    for fn in (h.raycast, h.raycast_trilinear):
        fn(c.wd, c.hd, Ta, c.K_depth, 0.2, 4.0, dd)
        assert float(dd.abs().max()) == 0.0                                         # empty again
    h.close(); g.close()


def test_raycast_rejects_bad_arguments():
    import torch
    import paper_1602_06645_b200 as vf
    c = synth.config(1).scaled(32, 2)
    g, o = make_pair(c)
    dd = torch.zeros(c.wd * c.hd, dtype=torch.float32, device="cuda")
    I4 = np.eye(4, dtype=np.float32)
    Tbad = I4.copy(); Tbad[0, 0] = 2.0
    for args in ((Tbad, c.K_depth, 0.1, 2.0), (I4, c.K_depth, 2.0, 1.0), (I4, c.K_depth, -1.0, 1.0)):
        with pytest.raises(vf.VolError) as e:
            g.raycast(c.wd, c.hd, args[0], args[1], args[2], args[3], dd)
        assert e.value.code == vf.VOL_E_ARG
        with pytest.raises(vf.VolError) as e:
            g.raycast_trilinear(c.wd, c.hd, args[0], args[1], args[2], args[3], dd)
        assert e.value.code == vf.VOL_E_ARG
    shard = vf.Volume(c.dims_geo, c.r, c.origin, c.extent, c.mu, c.w_max, shard_rank=0, shard_world=2)
    with pytest.raises(vf.VolError):
        shard.raycast(c.wd, c.hd, I4, c.K_depth, 0.1, 2.0, dd)


def test_raycast_cfg3_full_size():
    """BASELINE config 3 at full size (512^3 / 1024^3): two frames fused on both sides, the oracle over the WHOLE volumes --
    every one of the 1.2 G words and the eight per-frame counters (voxels and 32-byte sectors read / changed) are compared
    (the every-voxel comparison at the headline size) -- then a 640 x 480 ray cast from a third pose of the
    trajectory compared bit for bit."""
    from parity_util import check_counters, compare_states
    c = synth.config(3)
    g, o = make_pair(c)
    for fi in (0, 6):
        depth, rgb, T = synth.frame(c, fi)
        st, cnt = integrate_both(g, o, c, depth, rgb, T, counting=True)
        check_counters(st, cnt, f"cfg3 full size, frame {fi}")
    compare_states(g, o, "cfg3 full size, every voxel")
    d, rgb = cast_both(g, o, c.wd, c.hd, synth.frame(c, 3)[2], c.K_depth, 0.3, 5.0)
    assert (d > 0).mean() > 0.5 and (rgb.sum(axis=2) > 0).mean() > 0.3
    d, rgb = cast_both(g, o, c.wd, c.hd, synth.frame(c, 3)[2], c.K_depth, 0.3, 5.0, trilinear=True)
    assert (d > 0).mean() > 0.5 and (rgb.sum(axis=2) > 0).mean() > 0.3
    g.close()


def test_sample_colour_and_polygon_texture_map():
    """vol_sample_colour against the oracle, word for word: random points inside and outside config 1's
    fused colour volume, and the texture map of a polygon laid on the sphere's surface by eq. 11-14."""
    import torch
    c = synth.config(1)
    g, o = fused_pair(c, range(5))
    rng = np.random.default_rng(9)
    pts = rng.uniform(-0.7, 0.7, size=(200000, 3)).astype(np.float32) + np.array([0, 0, 1.5], np.float32)
    # a triangle tangent to the sphere (centre (0,0,1.5), R = 0.3) on its camera-facing side
    Va, Vb, Vc = np.array([-0.1, -0.08, 1.225]), np.array([0.12, -0.08, 1.228]), np.array([-0.1, 0.1, 1.23])
    size_pixel = 0.001
    w, h = int(np.linalg.norm(Vb - Va) / size_pixel), int(np.linalg.norm(Vc - Va) / size_pixel)      # eq. 11, 12
    green, blue = (Vb - Va) / (w - 1), (Vc - Va) / (h - 1)                                            # eq. 13, 14
    jj, ii = np.meshgrid(np.arange(h), np.arange(w), indexing="ij")
    tex_pts = (Va + ii[..., None] * green + jj[..., None] * blue).reshape(-1, 3).astype(np.float32)
    allp = np.concatenate([pts, tex_pts])
    dp = torch.from_numpy(allp).cuda()
    dw = torch.full((allp.shape[0],), -1, dtype=torch.int32, device="cuda")
    g.sample_colour(dp, allp.shape[0], dw)
    torch.cuda.synchronize()
    got = dw.cpu().numpy().view(np.uint32)
    want = o.sample_colour(allp)
    assert np.array_equal(got, want)
    assert (want[: pts.shape[0]] >> 24 > 0).sum() > 500 and (want[pts.shape[0]:] >> 24 > 0).mean() > 0.3   # both hit filled voxels
    g.sample_colour(dp, 0, dw)                                                                         # n = 0 is a no-op


def test_sample_colour_trilinear():
    """vol_sample_colour_trilinear (reading S2) against the oracle, word for word: 300 000 random points in and around
    config 1's fused colour volume (most footprints are partly unobserved), points on the volume's faces and corners,
    non-finite points, and a dense polygon map on the sphere."""
    import torch
    c = synth.config(1)
    g, o = fused_pair(c, range(5))
    rng = np.random.default_rng(19)
    pts = rng.uniform(-0.8, 0.8, size=(300000, 3)).astype(np.float32) + np.array([0, 0, 1.5], np.float32)
    surf = rng.normal(size=(200000, 3))
    surf = (0.3 * surf / np.linalg.norm(surf, axis=1, keepdims=True) * rng.uniform(0.97, 1.03, size=(200000, 1))
            + np.array([0, 0, 1.5])).astype(np.float32)                                                  # a shell around the sphere
    lo, hi = np.asarray(c.origin, np.float64), np.asarray(c.origin, np.float64) + c.extent
    t = rng.uniform(0, 1, size=(2000, 3))
    face = lo + t * (hi - lo)
    face[np.arange(2000), rng.integers(0, 3, 2000)] = np.where(rng.random(2000) < 0.5, lo[0], hi[0])    # cubic volume: on a face
    odd = np.array([[np.nan, 0, 1.5], [0, np.inf, 1.5], [0, 0, -np.inf], [1e30, 0, 1.5], lo, hi, lo - 1e-4, hi + 1e-4], np.float32)
    allp = np.concatenate([pts, surf, face.astype(np.float32), odd])
    dp = torch.from_numpy(allp).cuda()
    dw = torch.full((allp.shape[0],), -1, dtype=torch.int32, device="cuda")
    g.sample_colour_trilinear(dp, allp.shape[0], dw)
    torch.cuda.synchronize()
    got = dw.cpu().numpy().view(np.uint32)
    want = o.sample_colour_trilinear(allp)
    assert np.array_equal(got, want), f"{int((got != want).sum())} words differ"
    s = want[300000:500000]
    assert (s != 0).mean() > 0.3 and ((s >> 24) < 250).sum() > 1000 and ((s >> 24) > 250).sum() > 1000   # full and partial footprints
    assert not got[-8:-4].any()                                                                          # non-finite points
    g.sample_colour_trilinear(dp, 0, dw)                                                                 # n = 0 is a no-op
