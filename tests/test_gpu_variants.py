"""GPU parity of the alternative readings (vol_opts_t.variant): the CUDA path with one step read
differently against the oracle with the same switch, byte for byte, on the same seeded inputs."""
import numpy as np
import pytest

import synth
from parity_util import check_counters, compare_states, integrate_both, make_pair, run_sequence, sampled_full_size

pytestmark = pytest.mark.gpu
VARIANTS = [1, 2, 4]          # HD pixel from the depth point, TSDF along the viewing ray, additive colour weight


@pytest.mark.parametrize("variant", VARIANTS)
def test_variant_small_configs_every_voxel(variant):
    """Every word and the per-frame counters: config 1 (r = 2 and r = 3, ragged dims), config 3's noisy jittered frames,
    config 5 (mu << sigma)."""
    run_sequence(synth.config(1).scaled(48, 2), [0, 2, 4], variant=variant)
    c = synth.config(1).scaled(40, 3)
    c.dims_geo = (44, 38, 27)
    run_sequence(c, [0, 1, 3], variant=variant)
    run_sequence(synth.config(3).scaled(128, 2), [0, 1, 150, 299], variant=variant)
    run_sequence(synth.config(5).scaled(96, 2), [0, 200], variant=variant)


@pytest.mark.parametrize("variant", VARIANTS)
def test_variant_camera_inside_volume(variant):
    """Tiles that straddle the camera plane take the plain per-voxel routines: the switches live there too."""
    c = synth.config(2).scaled(64, 2)
    g, o = make_pair(c, variant=variant)
    T = synth.rigid32(synth.look_at((0.75, 0.6, 0.35), (0, 0, -0.2)))
    depth, _ = synth.render(c.prims, c.K_depth, T.astype(np.float64), c.wd, c.hd, True, False)
    depth = synth.quantise_depth(depth, np.random.default_rng(1), c.noise, 0.02)
    rgb = synth.random_rgb(c.wh, c.hh, 3)
    for _ in range(2):
        st, cnt = integrate_both(g, o, c, depth, rgb, T)
        check_counters(st, cnt)
    assert cnt[0] > 1000
    compare_states(g, o, f"inside, variant {variant}")


@pytest.mark.parametrize("variant", VARIANTS)
def test_variant_repeated_frame_saturation(variant):
    """The same frame 8 times: weights saturate and the 0.8 gate closes (the additive weight closes it after two frames)."""
    c = synth.config(1).scaled(32, 2)
    c.w_max = 5
    g, o = make_pair(c, variant=variant)
    depth, rgb, T = synth.frame(c, 2)
    for n in range(8):
        st, cnt = integrate_both(g, o, c, depth, rgb, T)
        check_counters(st, cnt, f"repeat {n}")
    compare_states(g, o, f"saturation, variant {variant}")


@pytest.mark.parametrize("variant", VARIANTS)
def test_variant_cfg3_full_size_sampled(variant):
    """BASELINE config 3 at full size (512^3 / 1024^3), 24 frames spread over the orbit, device and host entry points
    alternating, in the launch configuration bench.py times; compared on the seeded sample of columns."""
    ng, nc = sampled_full_size(synth.config(3), range(0, 300, 13), 40, 31, alternate_host=True, variant=variant)
    assert ng > 100000 and nc > 50000


def test_variant_is_live_and_reported():
    """Each switch changes the state of the volume it concerns (and only that one), and vol_info reports it."""
    import paper_1602_06645_b200 as vf
    c = synth.config(1).scaled(48, 2)
    states = {}
    for variant in [0] + VARIANTS:
        g, _ = make_pair(c, variant=variant)
        assert g.info.variant == variant
        for fi in (0, 2, 4):
            depth, rgb, T = synth.frame(c, fi)
            g.integrate_host(depth, rgb, T, c.K_depth, c.K_rgb, c.T_depth_rgb)
        states[variant] = g.download()
        g.close()
    geo0, col0 = states[0]
    assert np.array_equal(states[1][0], geo0) and not np.array_equal(states[1][1], col0)
    assert not np.array_equal(states[2][0], geo0) and np.array_equal(states[2][1], col0)
    assert np.array_equal(states[4][0], geo0) and not np.array_equal(states[4][1], col0)
    for bad in (3, 5, 6, 7, 8, -1):                       # combinations and unknown values are rejected
        with pytest.raises(vf.VolError):
            vf.Volume(c.dims_geo, c.r, c.origin, c.extent, c.mu, c.w_max, variant=bad)


@pytest.mark.parametrize("variant", VARIANTS)
def test_variant_shards_reassemble(variant):
    """The switches under z-slab sharding: three shards hold exactly the slabs of the unsharded volume of the same variant
    (which is byte-identical to the oracle's)."""
    import paper_1602_06645_b200 as vf
    from parity_util import to_dev
    c = synth.config(1).scaled(40, 2)
    c.dims_geo = (40, 40, 44)                          # 6 slabs, the last one partial
    g, o = make_pair(c, variant=variant)
    shards = [vf.Volume(c.dims_geo, c.r, c.origin, c.extent, c.mu, c.w_max, shard_rank=k, shard_world=3, variant=variant) for k in range(3)]
    for fi in (0, 3):
        depth, rgb, T = synth.frame(c, fi)
        integrate_both(g, o, c, depth, rgb, T)
        dd, dr = to_dev(depth), to_dev(rgb)
        for s in shards:
            s.integrate(dd, c.wd, c.hd, dr, c.wh, c.hh, T, c.K_depth, c.K_rgb, c.T_depth_rgb)
    geo, col = compare_states(g, o, f"unsharded, variant {variant}")
    nz, r, S = 44, c.r, vf.VOL_SLAB
    for k, s in enumerate(shards):
        sg, sc = s.download()
        layers = [z for z in range(nz) if (z // S) % 3 == k]
        assert np.array_equal(sg, geo[layers])
        assert np.array_equal(sc, col[[z for z in range(nz * r) if (z // (S * r)) % 3 == k]])
        s.close()
