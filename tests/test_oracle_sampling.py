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
