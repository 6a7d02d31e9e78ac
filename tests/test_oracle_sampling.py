"""Pins of the colour-volume sampler (ref_sample_colour; PAPER.md L164 and eq. 11-14) -- no GPU."""
import numpy as np

import oracle


def coded_volume(n=12, r=2, origin=(-0.3, 0.1, 0.5), extent=0.6):
    v = oracle.RefVolume((n, n, n), r, origin, extent, 0.1, 128)
    nc = n * r
    k, j, i = np.meshgrid(np.arange(nc), np.arange(nc), np.arange(nc), indexing="ij")
    v.col[...] = (i | (j << 8) | (k << 16) | (0xff << 24)).astype(np.uint32)          # the word encodes its own voxel index
    return v, nc, extent / nc


def test_sampler_returns_the_voxel_that_contains_the_point():
    v, nc, vc = coded_volume()
    rng = np.random.default_rng(5)
    idx = rng.integers(0, nc, size=(5000, 3))
    frac = rng.uniform(0.05, 0.95, size=(5000, 3))                                   # stay off the cell faces
    pts = np.asarray(v.desc.origin[:], np.float64) + (idx + frac) * vc
    w = v.sample_colour(pts.astype(np.float32))
    assert np.array_equal(w & 0xff, idx[:, 0]) and np.array_equal((w >> 8) & 0xff, idx[:, 1]) and np.array_equal((w >> 16) & 0xff, idx[:, 2])
    assert np.all(w >> 24 == 0xff)
    out = np.array([[-0.31, 0.2, 0.6], [0.31, 0.2, 0.6], [0.0, 0.05, 0.6], [0.0, 0.2, 1.11], [np.nan, 0.2, 0.6]], np.float32)
    assert not v.sample_colour(out).any()                                            # outside (or NaN): 0


def test_texture_map_of_a_polygon_eq_11_to_14():
    """Eq. 11-14 (L150-162) on a triangle lying in a plane of constant z inside a volume whose colour depends on (x, y) only:
    pixel (i, j) of the w x h map sits at V_a + i * V_aV_green + j * V_aV_blue and must show the colour of that place."""
    v, nc, vc = coded_volume()
    o = np.asarray(v.desc.origin[:], np.float64)
    Va, Vb, Vc = o + np.array([0.11, 0.07, 0.3]), o + np.array([0.47, 0.07, 0.3]), o + np.array([0.11, 0.52, 0.3])
    size_pixel = 0.004
    w = int(np.linalg.norm(Vb - Va) / size_pixel)                                    # eq. 11
    h = int(np.linalg.norm(Vc - Va) / size_pixel)                                    # eq. 12
    green, blue = (Vb - Va) / (w - 1), (Vc - Va) / (h - 1)                           # eq. 13, 14
    jj, ii = np.meshgrid(np.arange(h), np.arange(w), indexing="ij")
    pos = Va + ii[..., None] * green + jj[..., None] * blue
    tex = v.sample_colour(pos.reshape(-1, 3).astype(np.float32)).reshape(h, w)
    assert (w, h) == (90, 112)
    gx = (pos[..., 0] - o[0]) / vc
    gy = (pos[..., 1] - o[1]) / vc
    safe = (np.abs(gx - np.rint(gx)) > 1e-3) & (np.abs(gy - np.rint(gy)) > 1e-3)
    assert safe.mean() > 0.9
    assert np.array_equal((tex & 0xff)[safe], np.floor(gx)[safe].astype(np.uint32))
    assert np.array_equal(((tex >> 8) & 0xff)[safe], np.floor(gy)[safe].astype(np.uint32))
    assert np.all(((tex >> 16) & 0xff) == int(np.floor(0.3 / vc)))
    # V_a, V_b, V_c map to the three corners of the upper-left triangle (L146)
    assert (tex[0, 0] & 0xff, tex[0, w - 1] & 0xff) == (int((Va[0] - o[0]) / vc), int((Vb[0] - o[0]) / vc))
    assert (tex[h - 1, 0] >> 8) & 0xff == int((Vc[1] - o[1]) / vc)


# ---------------------------------------------------------------- trilinear sampling (reading S2)
def trilinear_fp64(col, origin, vc, pts):
    """Independent float64 restatement of reading S2, vectorised over the points (not the oracle's loop)."""
    nc = np.array(col.shape[::-1])                                                   # (nx, ny, nz)
    g = (np.asarray(pts, np.float64) - np.asarray(origin, np.float64)) / vc - 0.5
    b = np.floor(g).astype(np.int64)
    f = g - b
    sw = np.zeros(len(g)); sa = np.zeros(len(g)); sc = np.zeros((len(g), 3))
    for dz in (0, 1):
        for dy in (0, 1):
            for dx in (0, 1):
                idx = b + np.array([dx, dy, dz])
                inside = np.all((idx >= 0) & (idx < nc), axis=1)
                ic = np.clip(idx, 0, nc - 1)
                cw = col[ic[:, 2], ic[:, 1], ic[:, 0]].astype(np.int64)
                w = np.where(dx, f[:, 0], 1 - f[:, 0]) * np.where(dy, f[:, 1], 1 - f[:, 1]) * np.where(dz, f[:, 2], 1 - f[:, 2])
                w = np.where(inside & ((cw >> 24) > 0), w, 0.0)
                sw += w; sa += w * (cw >> 24)
                for ch in range(3):
                    sc[:, ch] += w * ((cw >> (8 * ch)) & 0xff)
    return sw, sa, sc


def test_trilinear_constant_and_voxel_centres():
    """A fully observed volume of one colour returns that colour and weight everywhere inside; at a voxel centre the
    interpolation returns that voxel's own word; far outside (or NaN) it returns 0."""
    v, nc, vc = coded_volume()
    o = np.asarray(v.desc.origin[:], np.float64)
    coded = v.col.copy()
    v.col[...] = np.uint32(37 | (201 << 8) | (114 << 16) | (180 << 24))
    rng = np.random.default_rng(2)
    pts = o + rng.uniform(0.6, nc - 0.6, size=(4000, 3)) * vc
    assert np.all(v.sample_colour_trilinear(pts.astype(np.float32)) == v.col[0, 0, 0])
    v.col[...] = coded
    idx = rng.integers(0, nc, size=(3000, 3))
    centres = (o + (idx + 0.5) * vc).astype(np.float32)
    got = v.sample_colour_trilinear(centres)
    # a binary32 centre is within ~1e-5 voxel of the true centre: the other seven weights are below 1e-4 and vanish in the rounding
    assert np.array_equal(got, v.sample_colour(centres))
    out = np.array([[-0.35, 0.2, 0.6], [0.35, 0.2, 0.6], [0.0, 0.2, 1.2], [np.nan, 0.2, 0.6], [np.inf, 0.2, 0.6]], np.float32)
    assert not v.sample_colour_trilinear(out).any()


def test_trilinear_reproduces_a_linear_ramp():
    """Trilinear interpolation is exact for colours that are linear in position: with R = i, G = j, B = k (voxel indices) the
    sample at grid coordinate g is (g_x, g_y, g_z) itself, rounded to the nearest integer."""
    v, nc, vc = coded_volume()
    o = np.asarray(v.desc.origin[:], np.float64)
    rng = np.random.default_rng(3)
    g = rng.uniform(0.0, nc - 1.0, size=(6000, 3))                                   # between the first and last centres
    pts = (o + (g + 0.5) * vc).astype(np.float32)
    g32 = (pts.astype(np.float64) - o) / vc - 0.5
    safe = np.all(np.abs(g32 - np.floor(g32) - 0.5) > 2e-3, axis=1)                  # off the rounding ties
    w = v.sample_colour_trilinear(pts)
    assert safe.sum() > 5500
    for ch in range(3):
        assert np.array_equal(((w >> (8 * ch)) & 0xff)[safe], np.rint(g32[:, ch])[safe].astype(np.uint32))
    assert np.all(w >> 24 == 255)


def test_trilinear_skips_unobserved_voxels_and_reports_coverage():
    """Half of the volume (i >= 12) never observed: next to the boundary the colour comes from the observed side alone
    (normalised), and the weight byte falls linearly to 0 across the last observed half voxel."""
    v, nc, vc = coded_volume()
    o = np.asarray(v.desc.origin[:], np.float64)
    v.col[...] = np.uint32(50 | (60 << 8) | (70 << 16) | (200 << 24))
    v.col[:, :, 12:] = np.uint32(255 | (255 << 8) | (255 << 16))                     # colour bytes set, weight 0: must be ignored
    for fx, expect_a in ((0.0, 200), (0.25, 150), (0.5, 100), (0.9, 20)):
        p = (o + np.array([11.5 + fx, 7.5 + 0.3, 9.5 + 0.6]) * vc).astype(np.float32)
        w = int(v.sample_colour_trilinear(p[None])[0])
        assert (w & 0xff, (w >> 8) & 0xff, (w >> 16) & 0xff) == (50, 60, 70)
        assert abs((w >> 24) - expect_a) <= 1
    p = (o + np.array([12.5 + 0.2, 7.8, 9.9]) * vc).astype(np.float32)               # footprint wholly unobserved
    assert int(v.sample_colour_trilinear(p[None])[0]) == 0
    # at the border of the volume the footprint sticks out: the missing voxels count like unobserved ones
    p = (o + np.array([0.25, 0.25, 0.25]) * vc).astype(np.float32)
    w = int(v.sample_colour_trilinear(p[None])[0])
    assert (w & 0xffffff) == (50 | (60 << 8) | (70 << 16)) and abs((w >> 24) - 200 * 0.75 ** 3) <= 1


def test_trilinear_against_float64_on_a_random_volume():
    """Random colours, random weights with 30 % unobserved voxels, points everywhere including a margin outside: the
    binary32 oracle agrees with the float64 restatement to the rounding of the last step."""
    n, r = 10, 2
    origin, extent = (-0.3, 0.1, 0.5), 0.6
    v = oracle.RefVolume((n, n, n), r, origin, extent, 0.1, 128)
    rng = np.random.default_rng(11)
    nc, vc = n * r, extent / (n * r)
    v.col[...] = rng.integers(0, 2 ** 32, size=v.col.shape, dtype=np.uint32)
    v.col[rng.random(v.col.shape) < 0.3] &= np.uint32(0x00ffffff)
    pts = (np.asarray(origin) + rng.uniform(-1.5, nc + 1.5, size=(20000, 3)) * vc).astype(np.float32)
    got = v.sample_colour_trilinear(pts)
    o32 = np.asarray(v.desc.origin[:], np.float64)
    vc32 = float(np.float32(np.float32(extent) / np.float32(n)) / np.float32(r))
    sw, sa, sc = trilinear_fp64(v.col, o32, vc32, pts)
    g = (pts.astype(np.float64) - o32) / vc32 - 0.5
    edge = np.any(np.abs(g - np.rint(g)) < 1e-3, axis=1)                             # floor() may differ there
    has = sw > 1e-6
    assert np.array_equal((got != 0)[~edge & (sw > 1e-3)], np.ones((~edge & (sw > 1e-3)).sum(), bool))
    assert not got[~edge & (sw == 0)].any()
    m = ~edge & (sw > 1e-3)
    assert m.sum() > 10000
    for ch in range(3):
        d = np.abs(((got >> (8 * ch)) & 0xff)[m] - sc[m, ch] / sw[m])
        assert d.max() <= 0.5 + 2e-2
    assert np.abs((got >> 24)[m] - np.minimum(255, sa[m])).max() <= 0.5 + 2e-2
