"""vol_icp_step_static (include/volfrontend.h): the F5 step that allocates nothing -- its scratch is a static device array --
against the existing path, vol_frontend_icp_step, on the same maps.  Collected last on purpose (pytest -x)."""
import numpy as np
import pytest

import synth
from oracle import frontend as ofe
from parity_util import to_dev

pytestmark = pytest.mark.gpu


def small_motion(rx, ry, rz, t):
    T = np.eye(4)
    T[:3, :3] = synth.rot_axis((1, 0, 0), rx) @ synth.rot_axis((0, 1, 0), ry) @ synth.rot_axis((0, 0, 1), rz)
    T[:3, 3] = t
    return T


def padded(m):
    """[h, w, 3] float32 host map -> CUDA tensor of h*w*4 floats (x, y, z, 0): the layout the front end keeps on the device"""
    import torch
    out = np.zeros(m.shape[:2] + (4,), np.float32)
    out[..., :3] = m
    return torch.from_numpy(out.reshape(-1)).cuda()


def test_static_scratch_step_equals_the_allocating_path():
    """Two calls in a row on different levels (the larger first, so the second runs over stale slots of the first), then
    more with other estimates: the same correspondences (count identical) and A, b, sum r^2 equal to binary64 summation
    order -- the tolerance of tests/test_gpu_frontend.py -- and the same bits when a call is repeated.  Oversized maps are
    refused with VOL_E_TOOBIG and a message that names the limit; nothing is launched for them."""
    import torch
    import paper_1602_06645_b200 as vf
    c = synth.config(2)
    dT = small_motion(0.012, -0.018, 0.009, (0.012, -0.007, 0.010))
    A = synth.look_at((0.9, -0.6, 0.55), (0.0, 0.0, 0.0))
    za, _ = synth.render(c.prims, c.K_depth, A, c.wd, c.hd, True, False)
    zb, _ = synth.render(c.prims, c.K_depth, A @ dT, c.wd, c.hd, True, False)
    db = synth.quantise_depth(zb, np.random.default_rng(3), c.noise, 0.02)
    fe = vf.Frontend(c.wd, c.hd, 3)
    fe.measure(to_dev(db), c.K_depth)
    fe.predict_depth(torch.from_numpy(za).cuda(), c.K_depth)
    maps, Ks = {}, {}
    for lv in range(3):
        _, V, N = fe.maps(0, lv)
        _, Vp, Np = fe.maps(1, lv)
        maps[lv] = tuple(padded(m) for m in (V, N, Vp, Np))
        fx, fy, cx, cy = ofe.level_intrinsics(c.K_depth, lv)
        Ks[lv] = np.array([fx, 0, cx, 0, fy, cy, 0, 0, 1], np.float32)
    out = torch.zeros(vf.ICP_SUMS, dtype=torch.float64, device="cuda")

    def static_step(lv, T):
        out.fill_(-1.0)
        vf.icp_step_static(*maps[lv], c.wd >> lv, c.hd >> lv, Ks[lv], T.astype(np.float32), out)
        return out.cpu().numpy().copy()

    calls = [(0, np.eye(4)), (2, np.eye(4)), (1, dT), (0, dT), (2, small_motion(0.03, 0.02, -0.01, (0.03, 0.0, -0.02))), (0, np.eye(4))]
    for n, (lv, T) in enumerate(calls):
        s = static_step(lv, T)
        A0, b0, e0, cnt0 = fe.icp_step(lv, T.astype(np.float32))
        A1 = np.zeros((6, 6)); A1[np.triu_indices(6)] = s[:21]; A1 = A1 + np.triu(A1, 1).T
        assert int(s[28]) == cnt0 and cnt0 > 5000, (n, lv, s[28], cnt0)
        scale = np.abs(A0).max()
        assert np.abs(A1 - A0).max() <= 1e-11 * scale and np.abs(s[21:27] - b0).max() <= 1e-11 * scale, (n, lv)
        assert abs(s[27] - e0) <= 1e-11 * e0, (n, lv)
        assert static_step(lv, T).tobytes() == s.tobytes(), (n, lv)              # fixed summation order: bit-reproducible
    # a stream of the caller's own
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        out.fill_(-1.0)
    vf.icp_step_static(*maps[1], c.wd >> 1, c.hd >> 1, Ks[1], dT.astype(np.float32), out, stream=stream)
    stream.synchronize()
    assert int(out[28].item()) == fe.icp_step(1, dT.astype(np.float32))[3]
    # beyond the static array: 4096 x 4096 needs 65536 blocks; 2048 x 1024 = 8192 is the last size that fits
    big = torch.zeros(4, dtype=torch.float32, device="cuda")                    # never read: the call is refused before any launch
    out.fill_(-1.0)
    with pytest.raises(vf.VolError) as e:
        vf.icp_step_static(big, big, big, big, 4096, 4096, Ks[0], np.eye(4, dtype=np.float32), out)
    assert e.value.code == vf.VOL_E_TOOBIG and "8192" in str(e.value) and "4096 x 4096" in str(e.value)
    with pytest.raises(vf.VolError) as e:
        vf.icp_step_static(big, big, big, big, 2048, 1032, Ks[0], np.eye(4, dtype=np.float32), out)
    assert e.value.code == vf.VOL_E_TOOBIG
    torch.cuda.synchronize()
    assert float(out[0].item()) == -1.0
    with pytest.raises(vf.VolError) as e:                                       # bad arguments are still VOL_E_ARG
        vf.icp_step_static(*maps[0], 0, c.hd, Ks[0], np.eye(4, dtype=np.float32), out)
    assert e.value.code == vf.VOL_E_ARG
    fe.close()


def test_static_scratch_largest_size_that_fits():
    """2048 x 1024 pixels = exactly VOL_ICP_STATIC_MAX_BLOCKS blocks: a plane seen head-on against itself; every valid pixel
    is its own correspondence, so count = valid pixels, r = 0 and A equals the sum of J J^T computed on the host."""
    import torch
    import paper_1602_06645_b200 as vf
    w, h = 2048, 1024
    assert ((w + 31) // 32) * ((h + 7) // 8) == vf.ICP_STATIC_MAX_BLOCKS
    K = synth.intrinsics(900.0, (w - 1) / 2.0, (h - 1) / 2.0)
    D = np.full((h, w), np.float32(1.5))
    (_, V, N), = ofe.pyramid(D, K, 1)
    tv, tn = padded(V), padded(N)
    out = torch.zeros(vf.ICP_SUMS, dtype=torch.float64, device="cuda")
    for _ in range(2):
        out.fill_(-1.0)
        vf.icp_step_static(tv, tn, tv, tn, w, h, K, np.eye(4, dtype=np.float32), out)
        s = out.cpu().numpy()
        ok = np.any(N != 0, axis=-1)
        assert int(s[28]) == int(ok.sum()) > 2000000 and s[27] == 0.0 and not s[21:27].any()
        p, n = V[ok].astype(np.float64), N[ok].astype(np.float64)
        J = np.concatenate([np.cross(p.astype(np.float32), n.astype(np.float32)).astype(np.float64), n], axis=1)
        A0 = J.T @ J
        A1 = np.zeros((6, 6)); A1[np.triu_indices(6)] = s[:21]; A1 = A1 + np.triu(A1, 1).T
        assert np.abs(A1 - A0).max() <= 1e-6 * np.abs(A0).max()
