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
    g = vf.Volume(c.dims_geo, c.r, c.origin, c.extent, c.mu, c.w_max, sigma=kw.get("sigma", 0.0), gate=kw.get("gate", 0.0),
                  variant=kw.get("variant", 0))
    o = oracle.RefVolume(c.dims_geo, c.r, c.origin, c.extent, c.mu, c.w_max, sigma=kw.get("sigma", 0.020), gate=kw.get("gate", 0.8),
                         variant=kw.get("variant", 0))
    return g, o


def integrate_both(g, o, c, depth, rgb, T, counting=True):
    """One frame on both sides; returns (gpu stats, oracle counters -- with the four sector counters when counting)."""
    dd, dr = to_dev(depth), to_dev(rgb)
    g.set_counting(counting)
    g.integrate(dd, depth.shape[1], depth.shape[0], dr, rgb.shape[1], rgb.shape[0], T, c.K_depth, c.K_rgb, c.T_depth_rgb)
    st = g.frame_stats()
    if counting:
        cnt = o.integrate_sectors(depth, rgb, T, c.K_depth, c.K_rgb, c.T_depth_rgb)
    else:
        cnt = o.integrate(depth, rgb, T, c.K_depth, c.K_rgb, c.T_depth_rgb)
    return st, cnt


def describe_mismatches(geo, og, col, oc, o, frame=None, limit=4):
    """Text for a failing comparison: the first differing voxels of each volume with their indices and the fields
    of both words; with frame = (c, depth, T_world_depth) also, in binary64, where the voxel projects in that depth frame and
    how far it is from the decisions that gate its update: geometry (u, v), sdf + mu; colour (u, v), d^2 - sigma^2."""
    lines = []
    ctx = None
    if frame is not None:
        c, depth, T = frame
        Ti = np.linalg.inv(np.asarray(T, np.float64).reshape(4, 4))
        K = np.asarray(c.K_depth, np.float64).reshape(3, 3)
        ctx = (c, np.asarray(depth), Ti, K)

    def project(idx, dims, vs):
        nx, ny, _ = dims
        i, j, k = int(idx % nx), int((idx // nx) % ny), int(idx // (nx * ny))
        txt = f"({i}, {j}, {k})"
        if ctx is None:
            return txt, None
        c, depth, Ti, K = ctx
        pw = np.asarray(o.desc.origin, np.float64) + (np.array([i, j, k]) + 0.5) * vs
        pc = Ti[:3, :3] @ pw + Ti[:3, 3]
        if pc[2] <= 0:
            return txt + " behind the camera", None
        u, v = K[0, 0] * pc[0] / pc[2] + K[0, 2], K[1, 1] * pc[1] / pc[2] + K[1, 2]
        ui, vi = int(np.floor(u + 0.5)), int(np.floor(v + 0.5))
        inside = 0 <= ui < depth.shape[1] and 0 <= vi < depth.shape[0]
        d = float(depth[vi, ui]) * 1e-3 if inside else 0.0
        return txt + f" -> (u, v) = ({u:.4f}, {v:.4f}), Z = {pc[2]:.6f}, D = {d:.3f}", (pc, ui, vi, d, K)

    vs = float(o.desc.extent) / int(o.desc.nx)
    for name, a, b, dims, size, fields in (("geometry", geo, og, (int(o.desc.nx), int(o.desc.ny), int(o.desc.nz)), vs,
                                            lambda w: f"q = {int(np.int16(w & 0xffff))}, w = {int(w >> 16)}"),
                                           ("colour", col, oc, tuple(int(x) * int(o.desc.r) for x in (o.desc.nx, o.desc.ny, o.desc.nz)), vs / int(o.desc.r),
                                            lambda w: f"rgb = ({int(w & 255)}, {int((w >> 8) & 255)}, {int((w >> 16) & 255)}), wq = {int(w >> 24)}")):
        bad = np.flatnonzero(a.reshape(-1) != b.reshape(-1))
        if bad.size == 0:
            continue
        lines.append(f"{name}: {bad.size} words differ")
        for idx in bad[:limit]:
            where, pr = project(int(idx), dims, size)
            extra = ""
            if pr is not None and pr[3] > 0:
                pc, ui, vi, d, K = pr
                if name == "geometry":
                    extra = f", sdf + mu = {d - pc[2] + float(o.desc.mu):.6f}"
                else:
                    pvd = np.array([(ui - K[0, 2]) * d / K[0, 0], (vi - K[1, 2]) * d / K[1, 1], d])
                    extra = f", d^2 - sigma^2 = {float(((pc - pvd) ** 2).sum()) - float(o.desc.sigma) ** 2:.3e}"
            lines.append(f"  voxel {where}{extra}: CUDA {fields(int(a.reshape(-1)[idx]))} | oracle {fields(int(b.reshape(-1)[idx]))}")
    return "\n".join(lines)


def compare_states(g, o, where="", frame=None):
    """Parity bar (BASELINE.json north_star): geometry weight and colour weight bit-exact, TSDF within 1e-5 after
    dequantisation (one q step is 3.05e-5, so this means identical q), colour channels within 1 LSB.  Under the
    canonical arithmetic the words are in fact byte-identical, which is what is asserted; the looser bar is evaluated
    first so that a failure reports which part broke."""
    geo, col = g.download()
    og, oc = o.geo, o.col
    assert geo.shape == og.shape and col.shape == oc.shape
    dq = np.abs(oracle.geo_q(geo) - oracle.geo_q(og))
    if not (np.array_equal(geo, og) and np.array_equal(col, oc)):
        print(describe_mismatches(geo, og, col, oc, o, frame))          # shown by pytest with the failing assertion below
    assert np.array_equal(oracle.geo_w(geo), oracle.geo_w(og)), f"{where}: geometry weights differ"
    assert dq.max() / 32767.0 <= 1e-5, f"{where}: TSDF differs, max |dq| = {dq.max()} at {int((dq > 0).sum())} voxels"
    assert np.array_equal(oracle.col_w(col), oracle.col_w(oc)), f"{where}: colour weights differ at {int((oracle.col_w(col) != oracle.col_w(oc)).sum())} voxels"
    dc = np.abs(oracle.col_rgb(col) - oracle.col_rgb(oc))
    assert dc.max() <= 1, f"{where}: colour differs by {dc.max()}"
    n_bad = int((geo != og).sum()) + int((col != oc).sum())
    assert n_bad == 0, f"{where}: {n_bad} words not byte-identical\n" + describe_mismatches(geo, og, col, oc, o, frame)
    return geo, col


def check_counters(st, cnt, where=""):
    """The four voxel counters of the frame -- and, when the oracle counted them, the four sector counters -- are the oracle's."""
    got = [st.geo_read, st.geo_changed, st.col_read, st.col_changed,
           st.geo_sectors_read, st.geo_sectors_written, st.col_sectors_read, st.col_sectors_written][:len(cnt)]
    assert got == [int(x) for x in cnt], f"{where}: counters {got} != oracle {list(cnt)}"
    assert st.geo_visited >= st.geo_read and st.col_gated >= st.col_read


def run_sequence(c, frames, counting=True, check_every=1, **kw):
    g, o = make_pair(c, **kw)
    for n, fi in enumerate(frames):
        depth, rgb, T = synth.frame(c, fi)
        st, cnt = integrate_both(g, o, c, depth, rgb, T, counting)
        if counting:
            check_counters(st, cnt, f"{c.name} frame {fi}")
        if (n + 1) % check_every == 0 or n == len(frames) - 1:
            compare_states(g, o, f"{c.name} frame {fi}", frame=(c, depth, T))
    return g, o


def sampled_full_size(c, frames, n_cols, seed, alternate_host=False, variant=0, frame_fn=None, mu=None, sigma=None, expect_colour=True,
                      burst=0):
    """Full-size volumes in the launch configuration bench.py times (device-resident frames, counters off), compared on a
    seeded sample: every voxel of n_cols random 8 x 8 (x, y) geometry columns and all their colour children.  Voxels never
    interact, so the oracle run on the sample alone gives their exact state (ref_integrate_subset).
    frame_fn(c, i) supplies frame i (default: the configuration's scan); mu / sigma override the configuration's.
    burst > 0: the frames are made resident `burst` at a time and then enqueued with nothing between the calls, as in
    bench.py's timed region (the next frame's pre-pass then runs under the tail of the fused kernel)."""
    import paper_1602_06645_b200 as vf
    frame_fn = frame_fn or synth.frame
    mu = c.mu if mu is None else mu
    sigma = c.sigma if sigma is None else sigma
    nx, ny, nz = c.dims_geo
    r = c.r
    rng = np.random.default_rng(seed)
    bx, by = rng.integers(0, nx // 8, n_cols), rng.integers(0, ny // 8, n_cols)
    k = np.arange(nz, dtype=np.int64)[:, None, None, None]
    j = (by[None, :, None, None] * 8 + np.arange(8)[None, None, :, None]).astype(np.int64)
    i = (bx[None, :, None, None] * 8 + np.arange(8)[None, None, None, :]).astype(np.int64)
    geo_idx = np.unique(((k * ny + j) * nx + i).reshape(-1))
    kc = np.arange(nz * r, dtype=np.int64)[:, None, None, None]
    jc = (by[None, :, None, None] * 8 * r + np.arange(8 * r)[None, None, :, None]).astype(np.int64)
    ic = (bx[None, :, None, None] * 8 * r + np.arange(8 * r)[None, None, None, :]).astype(np.int64)
    col_idx = np.unique(((kc * (ny * r) + jc) * (nx * r) + ic).reshape(-1))
    gw, cw = np.zeros(geo_idx.size, np.uint32), np.zeros(col_idx.size, np.uint32)
    o = oracle.RefVolume(c.dims_geo, r, c.origin, c.extent, mu, c.w_max, sigma=sigma, allocate=False, variant=variant)
    g = vf.Volume(c.dims_geo, r, c.origin, c.extent, mu, c.w_max, sigma=sigma, variant=variant)
    try:
        pending = []
        for n, fi in enumerate(frames):
            depth, rgb, T = frame_fn(c, fi)
            if burst:
                pending.append((to_dev(depth), to_dev(rgb), T))
                if len(pending) == burst or n == len(frames) - 1:
                    import torch
                    torch.cuda.synchronize()
                    for dd, dr, Tp in pending:
                        g.integrate(dd, c.wd, c.hd, dr, c.wh, c.hh, Tp, c.K_depth, c.K_rgb, c.T_depth_rgb)
                    torch.cuda.synchronize()
                    pending = []
            elif alternate_host and n % 2:                          # every other frame through vol_integrate_host
                g.integrate_host(depth, rgb, T, c.K_depth, c.K_rgb, c.T_depth_rgb)
            else:
                g.integrate(to_dev(depth), c.wd, c.hd, to_dev(rgb), c.wh, c.hh, T, c.K_depth, c.K_rgb, c.T_depth_rgb)
            o.integrate_subset(geo_idx, gw, col_idx, cw, depth, rgb, T, c.K_depth, c.K_rgb, c.T_depth_rgb)
            if n % 64 == 63:                                      # intermediate states too
                ggw, gcw = g.download_voxels(geo_idx, col_idx)
                assert int((ggw != gw).sum()) == 0 and int((gcw != cw).sum()) == 0, f"{c.name}: differs after frame {fi}"
        ggw, gcw = g.download_voxels(geo_idx, col_idx)
    finally:
        g.close()
    assert (gw >> 16).max() == min(len(frames), c.w_max) and ((cw >> 24).max() > 0) == expect_colour   # the sample does see the surface
    assert int((ggw != gw).sum()) == 0, f"{c.name}: {int((ggw != gw).sum())} geometry words differ on the sample"
    assert int((gcw != cw).sum()) == 0, f"{c.name}: {int((gcw != cw).sum())} colour words differ on the sample"
    return int((gw != 0).sum()), int((cw != 0).sum())
