"""Independent float64 brute force of the fusion step (numpy, vectorised over ALL voxels).

Written directly from PAPER.md eq. 5-10 (L91-124) and the TSDF definition (readings A5/A6) in real
(float64) arithmetic -- not from oracle/ref_fusion.c.  It is the "brute force on tiny inputs" pin of the
oracle: the oracle works in binary32 with a fixed operation order, this works in binary64 with matrix
algebra, so the two agree exactly except at *fragile* voxels whose decisions sit within rounding
distance of a boundary.  Those are reported in a mask and excluded (and counted) by the tests.
"""
import numpy as np

EPS_PX = 1e-3      # distance of a projected coordinate from a pixel-rounding boundary
EPS_M = 2e-5       # metres: sdf + mu, dist - sigma
EPS_W = 2e-3       # on the 0..255 weight scale


def grid_centres(dims, s, origin):
    nx, ny, nz = dims
    k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    return np.stack([origin[0] + (i + 0.5) * s, origin[1] + (j + 0.5) * s, origin[2] + (k + 0.5) * s], axis=-1)


def project(P, K, w, h):
    """Pinhole projection of camera-space points (..,3): nearest pixel, inside flag, fragile flag."""
    Z = P[..., 2]
    ok = Z > 0
    Zs = np.where(ok, Z, 1.0)
    u = K[0, 0] * P[..., 0] / Zs + K[0, 2]
    v = K[1, 1] * P[..., 1] / Zs + K[1, 2]
    xf, yf = np.floor(u + 0.5), np.floor(v + 0.5)
    inside = ok & (xf >= 0) & (xf < w) & (yf >= 0) & (yf < h)
    frag = (np.abs(u + 0.5 - np.rint(u + 0.5)) < EPS_PX) | (np.abs(v + 0.5 - np.rint(v + 0.5)) < EPS_PX) | (np.abs(Z) < 1e-6)
    # only boundaries that matter: anywhere near the image (a flip far outside changes nothing)
    near = (u > -2) & (u < w + 1) & (v > -2) & (v < h + 1)
    x = np.clip(xf, 0, w - 1).astype(np.int64)
    y = np.clip(yf, 0, h - 1).astype(np.int64)
    return x, y, inside, frag & near


def backproject(x, y, D, K):
    return np.stack([(x - K[0, 2]) * D / K[0, 0], (y - K[1, 2]) * D / K[1, 1], D], axis=-1)


class BruteVolume:
    def __init__(self, dims_geo, r, origin, extent, mu, w_max, sigma=0.020, gate=0.8, variant=0):
        # variant: 0, or one alternative reading: 1 = HD pixel from the depth pixel's 3D point,
        # 2 = signed distance along the voxel's viewing ray, 4 = additive colour weight
        self.variant = int(variant)
        self.dims_geo, self.r = tuple(dims_geo), int(r)
        self.dims_col = tuple(d * r for d in dims_geo)
        self.origin = np.asarray(origin, np.float64)
        self.vs = float(np.float32(extent)) / dims_geo[0]
        self.vc = self.vs / r
        self.mu, self.w_max, self.sigma, self.gate = float(np.float32(mu)), int(w_max), float(np.float32(sigma)), float(np.float32(gate))
        nx, ny, nz = self.dims_geo
        self.q = np.zeros((nz, ny, nx), np.int64)
        self.w = np.zeros((nz, ny, nx), np.int64)
        self.C = np.zeros((nz * r, ny * r, nx * r, 3), np.int64)
        self.wq = np.zeros((nz * r, ny * r, nx * r), np.int64)
        self.frag_geo = np.zeros_like(self.q, dtype=bool)       # sticky
        self.frag_col = np.zeros_like(self.wq, dtype=bool)
        self.Pg = grid_centres(self.dims_geo, self.vs, self.origin)
        self.Pc = grid_centres(self.dims_col, self.vc, self.origin)

    def integrate(self, depth, rgb, T_world_depth, K_depth, K_rgb, T_depth_rgb):
        depth = np.asarray(depth)
        hd, wd = depth.shape
        hh, wh = rgb.shape[:2]
        Kd, Kh = np.asarray(K_depth, np.float64), np.asarray(K_rgb, np.float64)
        Tcw = np.linalg.inv(np.asarray(T_world_depth, np.float64))      # (R_n, t_n) of eq. 5
        Thd = np.linalg.inv(np.asarray(T_depth_rgb, np.float64))        # (R_calib, t_calib) of eq. 3
        Dm = depth.astype(np.float64) * 1e-3

        # ---- geometry: projective TSDF (A5/A6)
        Pc = self.Pg @ Tcw[:3, :3].T + Tcw[:3, 3]
        x, y, inside, frag = project(Pc, Kd, wd, hd)
        D = Dm[y, x]
        sdf = D - Pc[..., 2]
        if self.variant == 2:                                            # metric distance along the ray through the voxel
            sdf = sdf * np.linalg.norm(Pc, axis=-1) / np.where(Pc[..., 2] > 0, Pc[..., 2], 1.0)
        upd = inside & (D > 0) & (sdf >= -self.mu)
        frag = frag | (inside & (D > 0) & (np.abs(sdf + self.mu) < EPS_M))
        tsdf = np.minimum(1.0, sdf / self.mu)
        qn = np.rint((self.q * self.w + tsdf * 32767.0) / (self.w + 1.0)).astype(np.int64)
        self.q = np.where(upd, qn, self.q)
        self.w = np.where(upd, np.minimum(self.w + 1, self.w_max), self.w)
        self.frag_geo |= frag
        self.upd_geo = upd

        # ---- colour: eq. 5-10
        P = self.Pc @ Tcw[:3, :3].T + Tcw[:3, 3]                          # eq. 5
        x, y, inside, frag = project(P, Kd, wd, hd)                      # eq. 6
        x1, y1 = np.minimum(x + 1, wd - 1), np.minimum(y + 1, hd - 1)
        D0, D1, D2 = Dm[y, x], Dm[y, x1], Dm[y1, x]
        valid = inside & (D0 > 0) & (x + 1 < wd) & (y + 1 < hd) & (D1 > 0) & (D2 > 0)      # L103, A7
        Pd = backproject(x, y, D0, Kd)                                   # eq. 7
        P1 = backproject(x + 1, y, D1, Kd)
        P2 = backproject(x, y + 1, D2, Kd)
        dist = np.linalg.norm(P - Pd, axis=-1)
        near = valid & (dist <= self.sigma)                              # L108
        frag = frag | (valid & (np.abs(dist - self.sigma) < EPS_M))
        N = np.cross(P1 - Pd, P2 - Pd)                                   # eq. 8
        den = np.linalg.norm(N, axis=-1) * np.linalg.norm(Pd, axis=-1)
        W = np.where(den > 0, np.minimum(1.0, np.einsum("...i,...i", N, Pd) / np.where(den > 0, den, 1.0)), 0.0)
        read = near & (den > 0) & (W > 0)                                # L110, A8
        frag = frag | (near & (np.abs(W) < 1e-5))
        W255 = W * 255.0
        passg = read & (W255 > self.gate * self.wq)                      # L115, A9
        frag = frag | (read & (np.abs(W255 - self.gate * self.wq) < EPS_W))
        Ph = (Pd if self.variant == 1 else P) @ Thd[:3, :3].T + Thd[:3, 3]    # eq. 3 (A11: the voxel's own position; variant 1: eq. 7's point)
        xh, yh, inside_h, frag_h = project(Ph, Kh, wh, hh)               # eq. 4
        upd = passg & inside_h                                           # A13
        frag = frag | (passg & frag_h)
        HD = rgb[yh, xh].astype(np.float64)                              # A14
        wqf = self.wq.astype(np.float64)
        Cn = (self.C * wqf[..., None] + W255[..., None] * HD) / np.where(upd, wqf + W255, 1.0)[..., None]   # eq. 9
        Cn = np.clip(np.rint(Cn), 0, 255).astype(np.int64)
        wn_real = wqf + W * (255.0 - wqf)                                # eq. 10 on the 0..255 scale (A12)
        if self.variant == 4:
            wn_real = wqf + W255                                         # W_pre + W
        frag = frag | (upd & (np.abs(wn_real - np.floor(wn_real) - 0.5) < EPS_W))
        wn = np.minimum(255, np.rint(wn_real)).astype(np.int64)
        self.C = np.where(upd[..., None], Cn, self.C)
        self.wq = np.where(upd, wn, self.wq)
        self.frag_col |= frag
        self.read_col, self.upd_col, self.W = read, upd, W
        self.xh, self.yh = xh, yh
