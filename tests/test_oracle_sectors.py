"""The oracle's sector counters ("DRAM sectors are 32 B = 8 x-adjacent voxels; report both voxel-exact and
sector-exact counts") pinned to the state arrays themselves: the set of changed words is visible as the difference between
the arrays before and after a frame, and a sector is 8 consecutive words of the linear layout."""
import numpy as np

import oracle
import synth


def _sectors(mask):
    return np.unique(np.flatnonzero(mask.reshape(-1)) >> 3).size


def test_sector_counters_equal_the_sectors_of_the_changed_words():
    c = synth.config(1).scaled(40, 3)
    c.dims_geo = (44, 38, 27)                       # rows of 44 and 132 words: sectors straddle rows and layers
    o = oracle.RefVolume(c.dims_geo, c.r, c.origin, c.extent, c.mu, c.w_max)
    plain = oracle.RefVolume(c.dims_geo, c.r, c.origin, c.extent, c.mu, c.w_max)
    for n, fi in enumerate((0, 2, 4)):
        depth, rgb, T = synth.frame(c, fi)
        g0, c0 = o.geo.copy(), o.col.copy()
        cnt = o.integrate_sectors(depth, rgb, T, c.K_depth, c.K_rgb, c.T_depth_rgb)
        ref = plain.integrate(depth, rgb, T, c.K_depth, c.K_rgb, c.T_depth_rgb)
        assert np.array_equal(cnt[:4], ref) and np.array_equal(o.geo, plain.geo) and np.array_equal(o.col, plain.col)
        gch, cch = o.geo != g0, o.col != c0
        assert int(gch.sum()) == cnt[1] and int(cch.sum()) == cnt[3]
        assert _sectors(gch) == cnt[5] and _sectors(cch) == cnt[7]
        # every changed voxel was read; on the first frame (empty volumes, every HD pixel inside the image) read = changed
        assert cnt[4] >= cnt[5] and cnt[6] >= cnt[7] and cnt[0] >= cnt[4] and cnt[2] >= cnt[6]
        if n == 0:
            assert cnt[0] == cnt[1] and cnt[4] == cnt[5] and cnt[2] == cnt[3] and cnt[6] == cnt[7]
        # between one word per sector and eight
        assert cnt[1] <= 8 * cnt[5] and cnt[3] <= 8 * cnt[7]


def test_a_plane_fills_whole_sectors_of_the_geometry_volume():
    """Fronto-parallel plane, identity pose: every in-frustum voxel in front of the band is read, so away from the frustum's
    edge whole rows are -- the sector count approaches a eighth of the voxel count."""
    c = synth.config(1)
    o = oracle.RefVolume(c.dims_geo, c.r, c.origin, c.extent, c.mu, c.w_max)
    cnt = o.integrate_sectors(synth.plane_depth(c.wd, c.hd, 1500), synth.const_rgb(c.wh, c.hh, (9, 99, 199)),
                              np.eye(4, dtype=np.float32), c.K_depth, c.K_rgb, c.T_depth_rgb)
    assert cnt[0] > 50000 and cnt[0] / 8 <= cnt[4] <= cnt[0] / 8 * 1.25


def test_thread_count_is_reported():
    assert 1 <= oracle.threads() <= 1024
