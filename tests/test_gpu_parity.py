"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, same seeded inputs."""
import numpy as np
import pytest

import synth
from parity_util import check_counters, compare_states, integrate_both, make_pair, run_sequence, to_dev
from parity_util import sampled_full_size as _sampled_full_size

pytestmark = pytest.mark.gpu
I4 = np.eye(4, dtype=np.float32)


def test_cfg1_full_sequence():
    """Config 1 as specified: 64^3 / 128^3, 5 frames, state and counters checked after every frame."""
    run_sequence(synth.config(1), range(5))


@pytest.mark.parametrize("r", [1, 2, 3, 4])
def test_cfg1_all_ratios(r):
    run_sequence(synth.config(1, r=r).scaled(48, r), [0, 2, 4])


def test_ragged_dims_and_tail_tiles():
    """Dims that are not multiples of the tile (32 x 4 x 8) or of the micro-block: ragged tails on every axis."""
    c = synth.config(1).scaled(40, 3)
    c.dims_geo = (44, 38, 27)
    run_sequence(c, [0, 1, 3])


def test_odd_x_dimension():
    """dims_geo[0] that is not a multiple of 4 or 8: rows are not aligned to 32-byte sectors (SURVEY 8(b) has no such rule)."""
    c = synth.config(1).scaled(40, 2)
    c.dims_geo = (45, 39, 29)
    run_sequence(c, [0, 2, 4])
    c = synth.config(2).scaled(64, 3)
    c.dims_geo = (61, 66, 50)
    run_sequence(c, [0, 50])


def test_cfg2_scaled_orbit():
    """Config 2's scene, cameras, noise and 2 % dropouts on a 96^3 / 192^3 grid; 6 frames spread over the orbit."""
    run_sequence(synth.config(2).scaled(96, 2), [0, 17, 34, 51, 68, 99])


def test_cfg3_scaled_jittered():
    run_sequence(synth.config(3).scaled(128, 2), [0, 1, 2, 150, 299])


def test_cfg4_scaled_r3():
    run_sequence(synth.config(4).scaled(64, 3), [0, 50, 100])


def test_cfg5_scaled_small_object():
    """Config 5: 0.5 m cube, mu = 4 mm << sigma = 20 mm, no background: the colour shell dominates."""
    run_sequence(synth.config(5).scaled(96, 2), [0, 100, 200, 399])


def test_weight_saturation_and_gate_many_frames():
    """Same frame 12 times with w_max = 5: weights saturate, the 0.8 gate closes, stores get skipped."""
    c = synth.config(1).scaled(32, 2)
    c.w_max = 5
    g, o = make_pair(c)
    depth, rgb, T = synth.frame(c, 2)
    for n in range(12):
        st, cnt = integrate_both(g, o, c, depth, rgb, T)
        check_counters(st, cnt, f"repeat {n}")
    compare_states(g, o, "saturation")


def test_saturated_free_space_is_left_out_exactly():
    """Steady state of a long scan: sub-boxes that hold nothing but saturated free space (tsdf_q = 32767, w = w_max) and
    stay in free space are not visited by the plain kernel.  w_max = 3 so that it happens within a few frames; frames of a
    moving camera, counters off (the launch configuration of bench.py), every word compared with the oracle after every
    frame; then one counted frame: the counters are still the method's, and they say how much was left out."""
    c = synth.config(2).scaled(96, 2)
    c.w_max = 3
    g, o = make_pair(c)
    for n, fi in enumerate([0, 0, 0, 0, 1, 2, 3, 4, 5, 6, 30, 31]):
        depth, rgb, T = synth.frame(c, fi)
        integrate_both(g, o, c, depth, rgb, T, counting=False)
        compare_states(g, o, f"frame {fi} (#{n})")
    depth, rgb, T = synth.frame(c, 32)
    st, cnt = integrate_both(g, o, c, depth, rgb, T, counting=True)
    check_counters(st, cnt, "counted frame")
    compare_states(g, o, "after the counted frame")
    assert 5000 < st.geo_skippable < st.geo_read, (st.geo_skippable, st.geo_read)    # a part of the free space is left out by now
    assert st.geo_changed <= st.geo_read - st.geo_skippable and 0 < st.geo_sectors_skippable <= st.geo_sectors_read


def test_degenerate_frames():
    """All-zero depth is a no-op; a camera looking away touches nothing; both leave a seeded state untouched."""
    c = synth.config(1).scaled(32, 2)
    g, o = make_pair(c)
    depth, rgb, T = synth.frame(c, 0)
    integrate_both(g, o, c, depth, rgb, T)
    before, _ = g.download()
    st, cnt = integrate_both(g, o, c, np.zeros_like(depth), rgb, T)
    check_counters(st, cnt)
    assert st.tiles_geo == 0 and st.items_col == 0
    Tb = I4.copy()
    Tb[:3, :3] = np.diag([-1, 1, -1]).astype(np.float32)
    st, cnt = integrate_both(g, o, c, depth, rgb, Tb)
    check_counters(st, cnt)
    geo, _ = compare_states(g, o, "degenerate")
    assert np.array_equal(geo, before)


def test_camera_inside_volume_and_near_plane():
    """Camera inside the volume: tiles straddle the camera plane (Z <= 0 voxels, huge projected rectangles)."""
    c = synth.config(2).scaled(64, 2)
    g, o = make_pair(c)
    T = synth.rigid32(synth.look_at((0.75, 0.6, 0.35), (0, 0, -0.2)))
    depth, _ = synth.render(c.prims, c.K_depth, T.astype(np.float64), c.wd, c.hd, True, False)
    depth = synth.quantise_depth(depth, np.random.default_rng(1), c.noise, 0.02)
    rgb = synth.random_rgb(c.wh, c.hh, 3)
    st, cnt = integrate_both(g, o, c, depth, rgb, T)
    check_counters(st, cnt)
    assert cnt[0] > 1000
    compare_states(g, o, "inside")


def test_host_entry_point_and_upload_roundtrip():
    """vol_integrate_host (host buffers, copies inside) gives the same state; vol_upload / vol_reset round-trip."""
    c = synth.config(1).scaled(32, 2)
    g, o = make_pair(c)
    for fi in (0, 4):
        depth, rgb, T = synth.frame(c, fi)
        g.integrate_host(depth, rgb, T, c.K_depth, c.K_rgb, c.T_depth_rgb)
        o.integrate(depth, rgb, T, c.K_depth, c.K_rgb, c.T_depth_rgb)
    geo, col = compare_states(g, o, "host entry")
    g.reset()
    z, zc = g.download()
    assert not z.any() and not zc.any()
    g.upload(geo, col)
    compare_states(g, o, "after upload")
    gi = np.array([0, 5, 32 * 32 * 16 + 77, 32 ** 3 - 1], np.int64)
    ci = np.array([1, 64 * 64 * 30 + 64 * 31 + 29, 64 ** 3 - 1], np.int64)
    gw, cw = g.download_voxels(gi, ci)
    assert np.array_equal(gw, geo.reshape(-1)[gi]) and np.array_equal(cw, col.reshape(-1)[ci])


def test_host_frames_enqueued_back_to_back():
    """vol_integrate_host without any synchronisation between frames: the copies of frame n + 1 (pinned host memory, the
    library's copy stream, two staging sets) overlap the kernels of frame n.  16 frames of config 3's noisy orbit on a
    non-default stream, statistics read back with vol_frame_stats_async; the final state and every frame's record must
    equal the one-frame-at-a-time run's, and the oracle's."""
    import torch
    c = synth.config(3).scaled(160, 2)
    frames = [synth.frame(c, fi) for fi in range(0, 160, 10)]
    pinned = [(torch.from_numpy(d.copy()).pin_memory(), torch.from_numpy(rgb.copy()).pin_memory(), T) for d, rgb, T in frames]
    g, o = make_pair(c)
    g.set_counting(True)
    serial = []
    for d, rgb, T in frames:
        g.integrate_host(d, rgb, T, c.K_depth, c.K_rgb, c.T_depth_rgb)
        st = g.frame_stats()
        serial.append((st.geo_read, st.geo_changed, st.col_read, st.col_changed, st.tiles_geo, st.items_col, st.cells_col))
        cnt = o.integrate(d, rgb, T, c.K_depth, c.K_rgb, c.T_depth_rgb)
        check_counters(st, cnt)
    compare_states(g, o, "one frame at a time")
    stream = torch.cuda.Stream()
    raw = torch.zeros((len(frames), 16), dtype=torch.int64).pin_memory()
    for rep in range(3):                                            # three times: whichever way the copies and kernels interleave
        g.reset(stream)
        for n, (d, rgb, T) in enumerate(pinned):
            g.integrate_host(d, rgb, T, c.K_depth, c.K_rgb, c.T_depth_rgb, stream=stream)
            g.frame_stats_async(raw[n], stream)
        stream.synchronize()
        got = []
        for n in range(len(frames)):
            st = g.decode_stats(raw[n])
            got.append((st.geo_read, st.geo_changed, st.col_read, st.col_changed, st.tiles_geo, st.items_col, st.cells_col))
        assert got == serial, f"repeat {rep}"
        compare_states(g, o, f"back to back, repeat {rep}")


def test_device_frames_pipelined_back_to_back():
    """vol_integrate with device-resident frames enqueued directly one after the other: the pre-pass of frame n + 1 is a
    programmatic dependent launch and runs under the tail of frame n's fused kernel (two scratch sets, three control
    blocks).  24 frames of config 3's noisy orbit (the volume large enough for the fused kernel to run for tens of
    microseconds), no counters, nothing between the calls, on a stream of its own, repeated.  The state must equal the oracle's, byte for byte, every time; and the
    statistics record read back asynchronously after a frame must be that frame's even when two more frames follow it."""
    import torch
    c = synth.config(3).scaled(192, 2)
    frames = [synth.frame(c, fi) for fi in range(0, 240, 10)]
    g, o = make_pair(c)
    for d, rgb, T in frames:
        o.integrate(d, rgb, T, c.K_depth, c.K_rgb, c.T_depth_rgb)
    dev = [(to_dev(d), to_dev(rgb), T) for d, rgb, T in frames]
    stream = torch.cuda.Stream()
    torch.cuda.synchronize()
    for rep in range(4):
        g.reset(stream)
        for dd, dr, T in dev:
            g.integrate(dd, c.wd, c.hd, dr, c.wh, c.hh, T, c.K_depth, c.K_rgb, c.T_depth_rgb, stream=stream)
        stream.synchronize()
        compare_states(g, o, f"pipelined, repeat {rep}")
    # statistics of frame n, read in stream order, while frames n + 1 and n + 2 are already enqueued behind it
    g.reset(stream)
    raw = torch.zeros((len(dev), 16), dtype=torch.int64).pin_memory()
    for n, (dd, dr, T) in enumerate(dev):
        g.integrate(dd, c.wd, c.hd, dr, c.wh, c.hh, T, c.K_depth, c.K_rgb, c.T_depth_rgb, stream=stream)
        g.frame_stats_async(raw[n], stream)
    stream.synchronize()
    tiles = [g.decode_stats(raw[n]).tiles_geo for n in range(len(dev))]
    g.reset(stream)
    for n, (dd, dr, T) in enumerate(dev):
        g.integrate(dd, c.wd, c.hd, dr, c.wh, c.hh, T, c.K_depth, c.K_rgb, c.T_depth_rgb, stream=stream)
        assert g.frame_stats(stream).tiles_geo == tiles[n] > 0, n
    compare_states(g, o, "with statistics")
    g.close()


def test_shards_reassemble_to_the_unsharded_volume():
    """z-slab sharding (VOL_SLAB layers dealt round-robin): two shards run one after the other on this GPU hold exactly
    the slabs of the unsharded result; no voxel is owned twice or dropped."""
    import paper_1602_06645_b200 as vf
    c = synth.config(1).scaled(40, 2)
    c.dims_geo = (40, 40, 44)                          # 6 slabs, the last one partial
    g, o = make_pair(c)
    shards = [vf.Volume(c.dims_geo, c.r, c.origin, c.extent, c.mu, c.w_max, shard_rank=k, shard_world=2) for k in range(2)]
    for fi in (0, 3):
        depth, rgb, T = synth.frame(c, fi)
        integrate_both(g, o, c, depth, rgb, T)
        dd, dr = to_dev(depth), to_dev(rgb)
        for s in shards:
            s.integrate(dd, c.wd, c.hd, dr, c.wh, c.hh, T, c.K_depth, c.K_rgb, c.T_depth_rgb)
    geo, col = compare_states(g, o, "unsharded")
    nz, r, S = 44, c.r, vf.VOL_SLAB
    for k, s in enumerate(shards):
        sg, sc = s.download()
        layers = [z for z in range(nz) if (z // S) % 2 == k]
        assert sg.shape[0] == len(layers)
        assert np.array_equal(sg, geo[layers])
        clayers = [z for z in range(nz * r) if (z // (S * r)) % 2 == k]
        assert np.array_equal(sc, col[clayers])


def test_bad_arguments_leave_state_untouched():
    import paper_1602_06645_b200 as vf
    c = synth.config(1).scaled(32, 2)
    g, o = make_pair(c)
    depth, rgb, T = synth.frame(c, 0)
    integrate_both(g, o, c, depth, rgb, T)
    dd, dr = to_dev(depth), to_dev(rgb)
    Tbad = T.copy(); Tbad[0, 0] = 2.0
    Kbad = c.K_depth.copy(); Kbad[0, 1] = 0.5
    for args in ((Tbad, c.K_depth), (T, Kbad)):
        with pytest.raises(vf.VolError) as e:
            g.integrate(dd, c.wd, c.hd, dr, c.wh, c.hh, args[0], args[1], c.K_rgb, c.T_depth_rgb)
        assert e.value.code == vf.VOL_E_ARG
    compare_states(g, o, "after rejected calls")


def test_exact_arithmetic_selftest():
    """The branch-free reciprocal / quotient of the hot path equal __frcp_rn / __fdiv_rn bit for bit: every binary32
    in the reciprocal's operand range, a 1/257 stride of the TSDF quotient's numerators x all 513 denominators, and a
    1/1021 stride of the colour quotient's new-sample weights x stored weights x colour / HD byte pairs, with both weight
    roundings (the exhaustive sweep is `vf.selftest(exhaustive=True)`, ~1e12 quotients)."""
    import paper_1602_06645_b200 as vf
    assert vf.selftest(False) == (0, 0, 0)


def test_cfg3_full_size_whole_sequence_sampled():
    """BASELINE config 3 as specified: 512^3 / 1024^3 (the benchmark workload), all 300 frames of the jittered orbit,
    alternating between the device and the host entry point; geometry weights reach w_max = 128 on the way."""
    ng, nc = _sampled_full_size(synth.config(3), range(300), 40, 31, alternate_host=True)
    assert ng > 100000 and nc > 100000


def test_cfg3_full_size_pipelined_sampled():
    """The benchmark workload the way bench.py's timed region runs it: device-resident frames, 16 at a time, enqueued with
    nothing between the calls (the pre-pass of frame n + 1 under the tail of frame n's fused kernel), 64 frames."""
    ng, nc = _sampled_full_size(synth.config(3), range(64), 40, 33, burst=16)
    assert ng > 100000 and nc > 30000


def test_cfg2_cfg4_cfg5_full_size_whole_sequences_sampled():
    """BASELINE configs 2 (100 frames), 4 (r = 3, 200 frames) and 5 (400 frames) at full size, every frame."""
    for cfg, n_cols, seed in ((2, 48, 21), (4, 32, 42), (5, 32, 52)):
        c = synth.config(cfg)
        ng, nc = _sampled_full_size(c, range(c.n_frames), n_cols, seed, alternate_host=True)
        assert ng > 50000 and nc > 50000, (cfg, ng, nc)


def test_cfg4_r4_full_size_sampled():
    """The largest configuration: 384^3 geometry, 1536^3 colour (14.5 GB, word offsets beyond 2^32 bytes), 24 frames spread
    over the orbit, device and host entry points alternating."""
    ng, nc = _sampled_full_size(synth.config(4, r=4), list(range(0, 200, 9)) + [199, 199], 32, 41, alternate_host=True)
    assert ng > 50000 and nc > 50000


@pytest.mark.parametrize("kind", synth.STRESS_KINDS)
def test_stress_frames_full_size_sampled(kind):
    """The saturating frames bench.py times on the benchmark volumes, 512^3 / 1024^3, in bench.py's
    launch configuration: the wall behind the cube (every geometry voxel updated in free space), the wall through the cube
    with mu = extent (every geometry voxel through the general running average) and the same with sigma = extent (every
    colour voxel updated as well).  Six frames each -- the wall moves, the RGB image is random, weights grow and the 0.8 gate
    starts to act -- against the oracle on a seeded sample of columns."""
    c = synth.config(3)
    mu, sigma = synth.stress_params(c, kind)
    ng, nc = _sampled_full_size(c, range(6), 24, 77, frame_fn=lambda cc, i: synth.stress_frame(cc, i, kind), mu=mu, sigma=sigma,
                                expect_colour=kind == "colour")
    col = 64 * 512                                               # voxels of one sampled 8 x 8 column
    if kind == "colour":
        assert 8 * col <= ng <= 16 * col                         # (mu is the configuration's: the voxels behind the wall's band are not)
    else:
        assert ng >= 20 * col and ng % col == 0                  # every geometry voxel of the sample was updated
    assert (nc >= 20 * col * 8 * 0.99) if kind == "colour" else nc == 0


def test_stress_frames_every_voxel_small():
    """The same three frames on a 64^3 / 128^3 grid, every voxel and the counters: a saturating frame reads every voxel."""
    import paper_1602_06645_b200 as vf
    import oracle
    c = synth.config(3).scaled(64, 2)
    for kind in synth.STRESS_KINDS:
        mu, sigma = synth.stress_params(c, kind)
        g = vf.Volume(c.dims_geo, c.r, c.origin, c.extent, mu, c.w_max, sigma=sigma)
        o = oracle.RefVolume(c.dims_geo, c.r, c.origin, c.extent, mu, c.w_max, sigma=sigma)
        for i in range(3):
            depth, rgb, T = synth.stress_frame(c, i, kind)
            st, cnt = integrate_both(g, o, c, depth, rgb, T)
            check_counters(st, cnt, f"{kind} frame {i}")
            assert (st.geo_read == 64 ** 3) == (kind != "colour") and (st.col_read > 0.9 * 128 ** 3) == (kind == "colour"), (kind, st.geo_read, st.col_read)
        compare_states(g, o, kind)
        g.close()


def test_cfg2_full_size_every_voxel():
    """BASELINE config 2 at full size (256^3 / 512^3): the oracle runs over both whole volumes; every word and the four
    per-frame counters are compared after each of 3 frames spread over the orbit."""
    run_sequence(synth.config(2), [0, 33, 66])


def test_run_to_run_determinism_and_noop_repeat():
    """T4 invariants on the GPU alone: two independent runs of the same sequence give identical bytes (no dependence on
    the work-queue order), and a frame that changes nothing (zero depth) leaves every byte and the counters at zero."""
    import paper_1602_06645_b200 as vf
    c = synth.config(3).scaled(128, 2)
    states = []
    for _ in range(2):
        g = vf.Volume(c.dims_geo, c.r, c.origin, c.extent, c.mu, c.w_max)
        for fi in (0, 7, 150):
            depth, rgb, T = synth.frame(c, fi)
            g.integrate(to_dev(depth), c.wd, c.hd, to_dev(rgb), c.wh, c.hh, T, c.K_depth, c.K_rgb, c.T_depth_rgb)
        states.append(g.download())
        if len(states) == 2:
            g.set_counting(True)
            g.integrate(to_dev(np.zeros_like(depth)), c.wd, c.hd, to_dev(rgb), c.wh, c.hh, T, c.K_depth, c.K_rgb, c.T_depth_rgb)
            st = g.frame_stats()
            assert (st.geo_read, st.geo_changed, st.col_read, st.col_changed, st.tiles_geo, st.items_col) == (0, 0, 0, 0, 0, 0)
            again = g.download()
            assert np.array_equal(again[0], states[1][0]) and np.array_equal(again[1], states[1][1])
        g.close()
    assert np.array_equal(states[0][0], states[1][0]) and np.array_equal(states[0][1], states[1][1])


def test_large_sigma_and_odd_parameters():
    """sigma = 150 mm on a coarse grid: every mark box exceeds MARK_FINE_MAX or spans many tiles (tile-granular marks), the
    colour shell is thicker than the objects; plus w_max = 1, a non-default gate, and a truncation band of half a voxel."""
    c = synth.config(2).scaled(48, 3)
    c.w_max = 1
    c.mu = 0.5 * c.extent / 48
    g, o = make_pair(c, sigma=0.150, gate=0.5)
    for fi in (0, 40):
        depth, rgb, T = synth.frame(c, fi)
        st, cnt = integrate_both(g, o, c, depth, rgb, T)
        check_counters(st, cnt, f"large sigma frame {fi}")
    compare_states(g, o, "large sigma")


def test_minimal_volume_frame_size_change_and_streams():
    """A 4 x 1 x 1 volume; the frame size changes between calls (scratch is reallocated); two volumes alive at once; a
    non-default stream."""
    import torch
    import oracle
    import paper_1602_06645_b200 as vf
    c1 = synth.config(1).scaled(32, 2)
    c2 = synth.config(2).scaled(32, 2)
    tiny = vf.Volume((4, 1, 1), 2, (-0.1, 0.0, 1.4), 0.4, 0.3, 128)
    otiny = oracle.RefVolume((4, 1, 1), 2, (-0.1, 0.0, 1.4), 0.4, 0.3, 128)
    g1, o1 = make_pair(c1)
    s = torch.cuda.Stream()
    for c, fi in ((c1, 0), (c2, 10), (c1, 3)):                       # 160x120 -> 640x480 -> 160x120 frames into the SAME volumes
        depth, rgb, T = synth.frame(c, fi)
        dd, dr = to_dev(depth), to_dev(rgb)
        torch.cuda.synchronize()
        with torch.cuda.stream(s):
            for vol in (g1, tiny):
                vol.integrate(dd, c.wd, c.hd, dr, c.wh, c.hh, T, c.K_depth, c.K_rgb, c.T_depth_rgb, stream=s)
        s.synchronize()
        for ov in (o1, otiny):
            ov.integrate(depth, rgb, T, c.K_depth, c.K_rgb, c.T_depth_rgb)
    compare_states(g1, o1, "frame size change")
    compare_states(tiny, otiny, "4x1x1 volume")
    assert (oracle.geo_w(o1.geo) > 0).sum() > 1000
    assert np.all(oracle.geo_w(otiny.geo) == 2) and (otiny.col > 0).sum() >= 1      # the tiny volume is really in view
    tiny.close()
