"""The oracle against the hand-derived fixtures of tests/golden/ (see its README for the derivations)."""
import os

import numpy as np

import oracle
import synth

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
I4 = np.eye(4, dtype=np.float32)


def rows(name):
    for line in open(os.path.join(GOLD, name)):
        line = line.split("#")[0].strip()
        if line:
            k, v = line.split(":")
            yield k.strip(), [int(x) for x in v.split()]


def test_weight_sequences_fixture():
    """One colour voxel, synthetic frames whose only eligible pixel has exactly the view weight W: drive the oracle's
    per-voxel update through ref_integrate_subset with a tilted plane is overkill -- instead the plane of
    test_weight_recursion_and_gate_on_a_plane is used: every voxel's sequence must be the fixture row of ITS W when W is
    one of the fixture values; here the fixture itself is checked against eq. 10 evaluated in exact rational arithmetic."""
    from fractions import Fraction
    for W, seq in rows("weight_sequences.txt"):
        Wf = Fraction(W)
        wq, out = 0, []
        for _ in seq:
            if 255 * Wf > Fraction(8, 10) * wq:
                x = wq + Wf * (255 - wq)                      # eq. 10 scaled by 255
                f = x.numerator // x.denominator
                rem = x - f
                wq = min(255, f + (1 if rem > Fraction(1, 2) or (rem == Fraction(1, 2) and f % 2 == 1) else 0))
            out.append(wq)
        assert out == seq, (W, out, seq)


def test_oracle_follows_weight_sequences():
    """Fronto-parallel plane: the on-axis colour voxels see W = 0.99998 (-> the W = 1.0 row); voxels whose pixel has
    W within 1e-4 of another fixture value must follow that row frame by frame."""
    c = synth.config(1)
    v = oracle.RefVolume(c.dims_geo, c.r, c.origin, c.extent, c.mu, c.w_max)
    depth, rgb = synth.plane_depth(c.wd, c.hd, 1500), synth.const_rgb(c.wh, c.hh, (10, 20, 30))
    hist = []
    for _ in range(6):
        v.integrate(depth, rgb, I4, c.K_depth, c.K_rgb, c.T_depth_rgb)
        hist.append(oracle.col_w(v.col).copy())
    fixture = {float(W): seq for W, seq in rows("weight_sequences.txt")}
    n = v.col.shape[0]
    s = c.extent / n
    k, j, i = np.nonzero(hist[0])
    X = c.origin[0] + (i + 0.5) * s; Y = c.origin[1] + (j + 0.5) * s; Z = c.origin[2] + (k + 0.5) * s
    x = np.floor(131.25 * X / Z + 79.5 + 0.5); y = np.floor(131.25 * Y / Z + 59.5 + 0.5)
    Wpix = 1.0 / np.sqrt(1.0 + ((x - 79.5) / 131.25) ** 2 + ((y - 59.5) / 131.25) ** 2)     # cosine of the off-axis angle
    checked = 0
    for W, seq in fixture.items():
        sel = np.abs(Wpix - W) < (2e-5 if W == 1.0 else 1e-4)
        if W == 1.0:
            sel = Wpix > 0.99995
        # stay away from the rounding boundaries of rint(255 W): only voxels whose first weight equals the row's
        sel &= hist[0][k, j, i] == seq[0]
        for f in range(min(6, len(seq))):
            assert np.all(hist[f][k[sel], j[sel], i[sel]] == seq[f]), (W, f)
        checked += int(sel.sum())
    assert checked >= 20


def test_tsdf_column_fixture():
    c = synth.config(1)
    v = oracle.RefVolume(c.dims_geo, c.r, c.origin, c.extent, c.mu, c.w_max)
    v.integrate(synth.plane_depth(c.wd, c.hd, 1500), synth.const_rgb(c.wh, c.hh, (1, 2, 3)), I4, c.K_depth, c.K_rgb, c.T_depth_rgb)
    q = oracle.geo_q(v.geo)[:, 32, 32]
    for k, (val,) in rows("tsdf_column_cfg1.txt"):
        assert q[int(k)] == val, (k, q[int(k)], val)
    assert v.geo[35, 32, 32] == 0 and np.all(q[:29] == 32767)


def test_tsdf_column_fixture_is_the_closed_form():
    """The fixture itself, against reading A5 evaluated in float64: q = 32767 * (d - z_k) / mu with d = 1.5 m,
    z_k = 1 + (k + 0.5) / 64, mu = 3 / 64 -- thirds and halves of 32767.  Every stored value is within half a unit of it
    (the two exact ties, k = 30 and k = 33, resolve upwards because D = 1500 * 0.001f is one ulp above 1.5)."""
    for k, (val,) in rows("tsdf_column_cfg1.txt"):
        k = int(k)
        ideal = 32767.0 * (1.5 - (1.0 + (k + 0.5) / 64.0)) / (3.0 / 64.0)
        if ideal > 32767.0:
            assert val == 32767
        elif ideal < -32767.0:
            assert val == 0                                  # behind the band: the untouched word
        else:
            assert abs(val - ideal) <= 0.5 + 1e-6, (k, val, ideal)
