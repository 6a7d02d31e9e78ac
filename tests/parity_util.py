"""Shared helpers of the GPU parity tests: drive the CUDA path (through the C ABI) and the CPU oracle with the same
seeded frames and compare their states element by element."""
import numpy as np

import oracle
import synth


def to_dev(a):
    import torch
    t = torch.from_numpy(np.ascontiguousarray(a).view(np.uint8).reshape(-1).copy())
    return t.cuda()


def make_pair(c, **kw):
    import paper_1602_06645_b200 as vf
    g = vf.Volume(c.dims_geo, c.r, c.origin, c.extent, c.mu, c.w_max, sigma=kw.get("sigma", 0.0), gate=kw.get("gate", 0.0))
    o = oracle.RefVolume(c.dims_geo, c.r, c.origin, c.extent, c.mu, c.w_max, sigma=kw.get("sigma", 0.020), gate=kw.get("gate", 0.8))
    return g, o


def integrate_both(g, o, c, depth, rgb, T, counting=True):
    """One frame on both sides; returns (gpu stats, oracle counters)."""
    dd, dr = to_dev(depth), to_dev(rgb)
    g.set_counting(counting)
    g.integrate(dd, depth.shape[1], depth.shape[0], dr, rgb.shape[1], rgb.shape[0], T, c.K_depth, c.K_rgb, c.T_depth_rgb)
    st = g.frame_stats()
    cnt = o.integrate(depth, rgb, T, c.K_depth, c.K_rgb, c.T_depth_rgb)
    return st, cnt


def compare_states(g, o, where=""):
    """Parity bar (BASELINE.json north_star): geometry weight and colour weight bit-exact, TSDF within 1e-5 after
    dequantisation (one q step is 3.05e-5, so this means identical q), colour channels within 1 LSB.  Under the
    canonical arithmetic the words are in fact byte-identical, which is what is asserted; the looser bar is evaluated
    first so that a failure reports which part broke."""
    geo, col = g.download()
    og, oc = o.geo, o.col
    assert geo.shape == og.shape and col.shape == oc.shape
    dq = np.abs(oracle.geo_q(geo) - oracle.geo_q(og))
    assert np.array_equal(oracle.geo_w(geo), oracle.geo_w(og)), f"{where}: geometry weights differ"
    assert dq.max() / 32767.0 <= 1e-5, f"{where}: TSDF differs, max |dq| = {dq.max()} at {int((dq > 0).sum())} voxels"
    assert np.array_equal(oracle.col_w(col), oracle.col_w(oc)), f"{where}: colour weights differ at {int((oracle.col_w(col) != oracle.col_w(oc)).sum())} voxels"
    dc = np.abs(oracle.col_rgb(col) - oracle.col_rgb(oc))
    assert dc.max() <= 1, f"{where}: colour differs by {dc.max()}"
    n_bad = int((geo != og).sum()) + int((col != oc).sum())
    assert n_bad == 0, f"{where}: {n_bad} words not byte-identical"
    return geo, col


def check_counters(st, cnt, where=""):
    got = [st.geo_read, st.geo_changed, st.col_read, st.col_changed]
    assert got == [int(x) for x in cnt], f"{where}: counters {got} != oracle {list(cnt)}"


def run_sequence(c, frames, counting=True, check_every=1):
    g, o = make_pair(c)
    for n, fi in enumerate(frames):
        depth, rgb, T = synth.frame(c, fi)
        st, cnt = integrate_both(g, o, c, depth, rgb, T, counting)
        if counting:
            check_counters(st, cnt, f"{c.name} frame {fi}")
        if (n + 1) % check_every == 0 or n == len(frames) - 1:
            compare_states(g, o, f"{c.name} frame {fi}")
    return g, o
