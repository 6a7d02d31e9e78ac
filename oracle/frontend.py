"""CPU ORACLE of the depth front end and the ICP tracking step (TEST INFRASTRUCTURE).

PAPER.md L33 (section III): "A vertex map and normal map pyramid based on input depth map is calculated; the value is then
used to estimate the camera motion using iterative closest point (ICP) algorithm [3] in conjunction with a predicted surface
vertex map ... obtained by ray tracing the geometry volume" (L35).  The paper gives no equations for any of this (it defers
to KinectFusion / PCL): the definitions are readings F1-F8 of DESIGN.md section 8f, written out below step by step --
** parity unpinned by the paper **; pinned by closed forms in tests/test_oracle_frontend.py.

Plain numpy, vectorised over the image, one array operation per arithmetic operation.  Arithmetic is binary32 with one
rounding per operation and NO fused multiply-add (numpy has none), in the order written; the sums of the ICP normal
equations are binary64.  Nothing here is shared with, or imported by, the CUDA path.
"""
from __future__ import annotations

import numpy as np

F32 = np.float32
RADIUS = 3                      # F1: 7 x 7 window


def level_intrinsics(K, level):
    """F2: halving the resolution maps pixel block (2x, 2x+1) to pixel x: f' = f / 2, c' = (c - 1/2) / 2 (pixel centres at integers)."""
    fx, fy, cx, cy = F32(K[0][0]), F32(K[1][1]), F32(K[0][2]), F32(K[1][2])
    for _ in range(level):
        fx, fy = F32(fx * F32(0.5)), F32(fy * F32(0.5))
        cx, cy = F32(F32(cx - F32(0.5)) * F32(0.5)), F32(F32(cy - F32(0.5)) * F32(0.5))
    return fx, fy, cx, cy


def bilateral_tables(sigma_s_px, sigma_r_m):
    """F1: the two weight tables, evaluated in binary64 and rounded once to binary32.  Range differences are whole
    millimetres (the depth map is uint16 mm), so the range kernel is a table over |delta| = 0 .. ceil(3 sigma_r)."""
    ss, sr = float(F32(sigma_s_px)), float(F32(sigma_r_m)) * 1000.0
    d = np.arange(-RADIUS, RADIUS + 1, dtype=np.float64)
    ws = np.exp(-(d[:, None] ** 2 + d[None, :] ** 2) / (2.0 * ss * ss)).astype(F32)           # [dy + R][dx + R]
    kmax = int(np.ceil(3.0 * sr))
    k = np.arange(kmax + 1, dtype=np.float64)
    wr = np.exp(-(k * k) / (2.0 * sr * sr)).astype(F32)
    return ws, wr


def bilateral(depth_u16, sigma_s_px=4.5, sigma_r_m=0.030):
    """F1: bilateral filter of the raw depth map -> float32 metres (0 = invalid).
    out(u) = sum_q ws(q - u) wr(|d(q) - d(u)|) d(q) / sum_q ws wr  over the valid pixels q of the 7 x 7 window inside the
    image with |d(q) - d(u)| <= ceil(3 sigma_r) mm, accumulated row by row; then mm -> m (x 0.001)."""
    d = np.asarray(depth_u16, dtype=np.int32)
    h, w = d.shape
    ws, wr = bilateral_tables(sigma_s_px, sigma_r_m)
    kmax = wr.size - 1
    sw = np.zeros((h, w), F32)
    sd = np.zeros((h, w), F32)
    pad = np.zeros((h + 2 * RADIUS, w + 2 * RADIUS), np.int32)
    pad[RADIUS:RADIUS + h, RADIUS:RADIUS + w] = d
    for dy in range(-RADIUS, RADIUS + 1):
        for dx in range(-RADIUS, RADIUS + 1):
            q = pad[RADIUS + dy:RADIUS + dy + h, RADIUS + dx:RADIUS + dx + w]
            delta = np.abs(q - d)
            use = (q > 0) & (delta <= kmax)
            wgt = (ws[dy + RADIUS, dx + RADIUS] * wr[np.minimum(delta, kmax)]).astype(F32)
            wgt = np.where(use, wgt, F32(0.0))
            sw = (sw + wgt).astype(F32)
            sd = (sd + (wgt * q.astype(F32)).astype(F32)).astype(F32)
    valid = d > 0
    out = np.zeros((h, w), F32)
    out[valid] = ((sd[valid] / sw[valid]).astype(F32) * F32(0.001)).astype(F32)
    return out


def half_sample(D, sigma_r_m=0.030):
    """F2: next pyramid level: the mean of the valid values of the 2 x 2 block that lie within 3 sigma_r of the block's
    first pixel D(2x, 2y), summed in the order (0,0), (1,0), (0,1), (1,1); 0 where D(2x, 2y) is invalid."""
    D = np.asarray(D, F32)
    h, w = D.shape
    assert h % 2 == 0 and w % 2 == 0
    thr = F32(F32(3.0) * F32(sigma_r_m))
    c = D[0::2, 0::2]
    s = np.zeros_like(c)
    n = np.zeros(c.shape, F32)
    for oy, ox in ((0, 0), (0, 1), (1, 0), (1, 1)):
        v = D[oy::2, ox::2]
        use = (v > 0) & (np.abs((v - c).astype(F32)) <= thr)
        s = np.where(use, (s + v).astype(F32), s)
        n = np.where(use, (n + F32(1.0)).astype(F32), n)
    out = np.zeros_like(c)
    ok = c > 0
    out[ok] = (s[ok] / n[ok]).astype(F32)
    return out


def vertex_map(D, fx, fy, cx, cy):
    """F3 = eq. 7: V(x, y) = D (x - cx) / fx, D (y - cy) / fy, D -- as ((x - cx) * D) / fx; 0 where invalid."""
    D = np.asarray(D, F32)
    h, w = D.shape
    x = np.arange(w, dtype=F32)[None, :]
    y = np.arange(h, dtype=F32)[:, None]
    V = np.zeros((h, w, 3), F32)
    V[..., 0] = (((x - F32(cx)).astype(F32) * D).astype(F32) / F32(fx)).astype(F32)
    V[..., 1] = (((y - F32(cy)).astype(F32) * D).astype(F32) / F32(fy)).astype(F32)
    V[..., 2] = D
    V[~(D > 0)] = 0
    return V


def normal_map(V):
    """F4 = eq. 8 (L110-113): N = (V(x+1, y) - V) x (V(x, y+1) - V), normalised; it points AWAY from the camera on a surface
    facing it (the paper's weight is N . viewing direction).  (0, 0, 0) where a neighbour is missing or invalid."""
    V = np.asarray(V, F32)
    h, w, _ = V.shape
    N = np.zeros_like(V)
    v0, v1, v2 = V[:-1, :-1], V[:-1, 1:], V[1:, :-1]
    ok = (v0[..., 2] > 0) & (v1[..., 2] > 0) & (v2[..., 2] > 0)
    a = (v1 - v0).astype(F32)
    b = (v2 - v0).astype(F32)
    nx = ((a[..., 1] * b[..., 2]).astype(F32) - (a[..., 2] * b[..., 1]).astype(F32)).astype(F32)
    ny = ((a[..., 2] * b[..., 0]).astype(F32) - (a[..., 0] * b[..., 2]).astype(F32)).astype(F32)
    nz = ((a[..., 0] * b[..., 1]).astype(F32) - (a[..., 1] * b[..., 0]).astype(F32)).astype(F32)
    ln = np.sqrt((((nx * nx).astype(F32) + (ny * ny).astype(F32)).astype(F32) + (nz * nz).astype(F32)).astype(F32)).astype(F32)
    ok = ok & (ln > 0)
    lns = np.where(ok, ln, F32(1.0))
    n = np.stack([(nx / lns).astype(F32), (ny / lns).astype(F32), (nz / lns).astype(F32)], axis=-1)
    N[:-1, :-1] = np.where(ok[..., None], n, F32(0.0))
    return N


def pyramid(D0, K, levels, sigma_r_m=0.030):
    """F2-F4: depth, vertex and normal maps of `levels` levels from a level-0 float32 depth map (metres)."""
    out = []
    D = np.asarray(D0, F32)
    for lv in range(levels):
        if lv > 0:
            D = half_sample(D, sigma_r_m)
        fx, fy, cx, cy = level_intrinsics(K, lv)
        V = vertex_map(D, fx, fy, cx, cy)
        out.append((D, V, normal_map(V)))
    return out


def measure(depth_u16, K, levels=3, sigma_s_px=4.5, sigma_r_m=0.030):
    """The measured side of the tracker: F1, then F2-F4."""
    return pyramid(bilateral(depth_u16, sigma_s_px, sigma_r_m), K, levels, sigma_r_m)


def predict(depth_m, K, levels=3, sigma_s_px=4.5, sigma_r_m=0.030):
    """F8: the predicted side of the tracker from a ray-cast depth map (float32 metres, 0 = no surface).  The ray caster
    samples the nearest voxel (reading R3), which leaves voxel-sized steps in the depth map and makes forward-difference
    normals useless; the map is therefore rounded to whole millimetres (half-even, clamped to 65535) and passed through the
    same filter as the measurement (F1) before F2-F4."""
    q = np.minimum(np.rint((np.asarray(depth_m, F32) * F32(1000.0)).astype(F32)), F32(65535.0)).astype(np.uint16)
    return pyramid(bilateral(q, sigma_s_px, sigma_r_m), K, levels, sigma_r_m)


def _mat3(R, v, t=None):
    """R v (+ t) in the order ((R0 vx + R1 vy) + R2 vz) (+ t), one rounding per operation."""
    out = []
    for i in range(3):
        s = ((R[i, 0] * v[..., 0]).astype(F32) + (R[i, 1] * v[..., 1]).astype(F32)).astype(F32)
        s = (s + (R[i, 2] * v[..., 2]).astype(F32)).astype(F32)
        if t is not None:
            s = (s + t[i]).astype(F32)
        out.append(s)
    return out


def icp_step(meas, pred, K, level, T_pred_cur, dist_m=0.10, cos_min=0.94):
    """F5: one linearised point-to-plane step with projective data association (KinectFusion).
    meas / pred: pyramids (lists of (D, V, N)); V, N of `meas` are in the current camera's frame, those of `pred` in the
    frame of the camera the prediction was ray-cast from.  T_pred_cur: 4 x 4, current camera -> prediction camera (the estimate).
    Per measured pixel with a valid normal: p = R v + t, m = R n; (xh, yh) = nearest pixel of K_l p; reject unless the
    prediction is valid there, |q - p| <= dist_m and m . nq >= cos_min;  r = nq . (q - p),  J = [p x nq ; nq].
    Returns (A [6,6], b [6], sum r^2, count) with A = sum J J^T, b = sum J r accumulated in binary64 from the binary32 J, r."""
    _, V, N = meas[level]
    _, Vp, Np = pred[level]
    h, w, _ = V.shape
    fx, fy, cx, cy = level_intrinsics(K, level)
    T = np.asarray(T_pred_cur, F32).reshape(4, 4)
    R, t = T[:3, :3], T[:3, 3]
    has = np.any(N != 0, axis=-1)
    p = _mat3(R, V, t)
    m = _mat3(R, N)
    ok = has & (p[2] > 0)
    pzs = np.where(ok, p[2], F32(1.0))
    u = ((fx * (p[0] / pzs).astype(F32)).astype(F32) + cx).astype(F32)
    v = ((fy * (p[1] / pzs).astype(F32)).astype(F32) + cy).astype(F32)
    xf = np.floor((u + F32(0.5)).astype(F32))
    yf = np.floor((v + F32(0.5)).astype(F32))
    ok = ok & (xf >= 0) & (xf < F32(w)) & (yf >= 0) & (yf < F32(h))
    xi = np.where(ok, xf, 0).astype(np.int64)
    yi = np.where(ok, yf, 0).astype(np.int64)
    q = Vp[yi, xi]
    nq = Np[yi, xi]
    ok = ok & np.any(nq != 0, axis=-1)
    d = [(q[..., i] - p[i]).astype(F32) for i in range(3)]
    dist2 = (((d[0] * d[0]).astype(F32) + (d[1] * d[1]).astype(F32)).astype(F32) + (d[2] * d[2]).astype(F32)).astype(F32)
    ok = ok & ~(dist2 > F32(F32(dist_m) * F32(dist_m)))
    cosang = (((m[0] * nq[..., 0]).astype(F32) + (m[1] * nq[..., 1]).astype(F32)).astype(F32) + (m[2] * nq[..., 2]).astype(F32)).astype(F32)
    ok = ok & ~(cosang < F32(cos_min))
    r = (((nq[..., 0] * d[0]).astype(F32) + (nq[..., 1] * d[1]).astype(F32)).astype(F32) + (nq[..., 2] * d[2]).astype(F32)).astype(F32)
    J = np.stack([
        ((p[1] * nq[..., 2]).astype(F32) - (p[2] * nq[..., 1]).astype(F32)).astype(F32),
        ((p[2] * nq[..., 0]).astype(F32) - (p[0] * nq[..., 2]).astype(F32)).astype(F32),
        ((p[0] * nq[..., 1]).astype(F32) - (p[1] * nq[..., 0]).astype(F32)).astype(F32),
        nq[..., 0], nq[..., 1], nq[..., 2]], axis=-1)
    Jd = J[ok].astype(np.float64)
    rd = r[ok].astype(np.float64)
    return Jd.T @ Jd, Jd.T @ rd, float(rd @ rd), int(ok.sum())


def se3_update(T, A, b):
    """F6: solve A xi = b (binary64), xi = (omega, v); T <- [exp(omega) R, exp(omega) t + v] (Rodrigues; left-multiplied: the
    increment acts on points already in the prediction camera's frame)."""
    xi = np.linalg.solve(np.asarray(A, np.float64), np.asarray(b, np.float64))
    om, v = xi[:3], xi[3:]
    th = float(np.linalg.norm(om))
    Kx = np.array([[0, -om[2], om[1]], [om[2], 0, -om[0]], [-om[1], om[0], 0]], np.float64)
    if th < 1e-12:
        Rinc = np.eye(3) + Kx
    else:
        Rinc = np.eye(3) + (np.sin(th) / th) * Kx + ((1.0 - np.cos(th)) / (th * th)) * (Kx @ Kx)
    T = np.asarray(T, np.float64).reshape(4, 4)
    out = np.eye(4)
    out[:3, :3] = Rinc @ T[:3, :3]
    out[:3, 3] = Rinc @ T[:3, 3] + v
    return out, xi


class TrackingLost(ValueError):
    """F7: the pose could not be estimated; .status = 1 too few correspondences, 2 A not positive definite, 3 A too close to singular."""

    def __init__(self, status, what):
        super().__init__("tracking lost: " + what)
        self.status = status


COND_MIN = float(F32(1e-3))     # F6: the default gate on conditioning(A)


def conditioning(A):
    """F6: min_j d_j / A_jj, d_j = L_jj^2 the j-th pivot of the Cholesky factorisation A = L L^T in the order of the
    parameters (omega, v): the share of parameter j's information that parameters 0 .. j-1 do not already explain.  1 for
    a diagonal A, -> 0 as A becomes singular, unchanged when a parameter is rescaled (A -> S A S, S diagonal), so radians
    against metres does not matter.  0 if A is not positive definite."""
    A = np.asarray(A, np.float64)
    try:
        L = np.linalg.cholesky(A)
    except np.linalg.LinAlgError:
        return 0.0
    return float(np.min(np.diag(L) ** 2 / np.diag(A)))


def track(meas, pred, K, T_init=None, iterations=(10, 5, 4), dist_m=0.10, cos_min=0.94, min_count=100, cond_min=COND_MIN):
    """F7: coarse to fine -- iterations[l] steps at level l, from the coarsest level down; the estimate is kept in binary64
    and rounded to binary32 for each step.  A step with fewer than min_count correspondences, or whose A fails the
    conditioning gate, raises TrackingLost.  Returns (T_pred_cur [4,4] float64, rms residual of the last step, its count)."""
    T = np.eye(4) if T_init is None else np.asarray(T_init, np.float64).reshape(4, 4).copy()
    rms, cnt = 0.0, 0
    for level in range(len(iterations) - 1, -1, -1):
        for _ in range(iterations[level]):
            A, b, e, cnt = icp_step(meas, pred, K, level, T.astype(F32), dist_m, cos_min)
            if cnt < min_count:
                raise TrackingLost(1, "too few correspondences")
            rms = float(np.sqrt(e / cnt))
            cond = conditioning(A)
            if cond == 0.0:
                raise TrackingLost(2, "normal equations not positive definite")
            if cond < cond_min:
                raise TrackingLost(3, "motion unobservable (conditioning %.3g)" % cond)
            T, _ = se3_update(T, A, b)
    return T, rms, cnt
