// fused.cuh -- K2: the fused per-tile integration kernel (S2-S8).
//
// Persistent CTAs pop tiles from the work list.  A CTA that owns a geometry tile updates its TILE_VOX TSDF voxels
// (one 16-byte vector of 4 x-adjacent voxels per thread) and then the tile's r^3 * TILE_VOX colour children: a
// second-level cull keeps only the 16x4x2 colour micro-blocks that can intersect the sigma shell, and each surviving
// micro-block is processed by one warp (one 16-byte vector per lane).
#pragma once
#include "params.cuh"

namespace vf {

// O-G for one geometry voxel (readings A5/A6).
// (X, Y, Z) = voxel centre in the depth camera (eq. 5).  Returns true if the voxel reached its read.
__device__ __forceinline__ bool geo_voxel(const Params &p, float X, float Y, float Z, uint32_t &word)
{
    int x, y;
    if (!project_px(p.fx, p.fy, p.cx, p.cy, p.wd_f, p.hd_f, X, Y, Z, x, y)) return false;
    const uint32_t d = __ldg(p.depth + y * p.wd + x);
    if (d == 0u) return false;                                            // "if non-zero" (L103)
    const float D = __fmul_rn((float)d, 0.001f);
    const float sdf = __fsub_rn(D, Z);
    if (sdf < p.neg_mu) return false;                                     // behind the truncation band: unchanged
    const float tsdf = fminf(1.0f, __fmul_rn(sdf, p.inv_mu));
    const int q = (int)(short)(word & 0xffffu);
    const int w = (int)(short)(word >> 16);
    const float num = __fmaf_rn((float)q, (float)w, __fmul_rn(tsdf, 32767.0f));
    const int qn = __float2int_rn(__fdiv_rn(num, __fadd_rn((float)w, 1.0f)));
    const int wn = min(w + 1, p.w_max);
    word = ((uint32_t)qn & 0xffffu) | ((uint32_t)wn << 16);
    return true;
}

// eq. 9-10 for one colour voxel that passed the sigma gate with view weight W.
// (X, Y, Z) = voxel centre in the depth camera.  Updates `word` in place.
__device__ __forceinline__ void col_voxel_update(const Params &p, float X, float Y, float Z, float W, uint32_t &word)
{
    const int wq = (int)(word >> 24);
    const float W255 = __fmul_rn(W, 255.0f);
    if (!(W255 > __fmul_rn(p.gate, (float)wq))) return;                   // L115, A9
    // HD pixel of the voxel's own position (eq. 3-4; A10, A11)
    const float Xh = __fmaf_rn(p.Rc[2], Z, __fmaf_rn(p.Rc[1], Y, __fmaf_rn(p.Rc[0], X, p.tc[0])));
    const float Yh = __fmaf_rn(p.Rc[5], Z, __fmaf_rn(p.Rc[4], Y, __fmaf_rn(p.Rc[3], X, p.tc[1])));
    const float Zh = __fmaf_rn(p.Rc[8], Z, __fmaf_rn(p.Rc[7], Y, __fmaf_rn(p.Rc[6], X, p.tc[2])));
    int xh, yh;
    if (!project_px(p.fxh, p.fyh, p.cxh, p.cyh, p.wh_f, p.hh_f, Xh, Yh, Zh, xh, yh)) return;   // A13
    const uint8_t *hd = p.rgb + (size_t)(yh * p.wh + xh) * 3;             // A14: nearest pixel
    const float den = __fadd_rn((float)wq, W255);
    uint32_t nw = 0;
#pragma unroll
    for (int ch = 0; ch < 3; ++ch) {                                      // eq. 9
        const int C = (int)((word >> (8 * ch)) & 0xffu);
        const float num = __fmaf_rn(W255, (float)__ldg(hd + ch), (float)(C * wq));
        const float cn = rintf(__fdiv_rn(num, den));
        const int ci = cn < 0.0f ? 0 : (cn > 255.0f ? 255 : (int)cn);
        nw |= (uint32_t)ci << (8 * ch);
    }
    int wn = __float2int_rn(__fmaf_rn(W, (float)(255 - wq), (float)wq)); // eq. 10, A12
    wn = min(wn, 255);
    word = nw | ((uint32_t)wn << 24);
}

template <bool COUNT>
__global__ void __launch_bounds__(CTA) k_fused(const __grid_constant__ Params p)
{
    __shared__ uint32_t s_item;
    __shared__ uint32_t s_nmb;
    __shared__ uint16_t s_mb[MAX_MB];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t n_front = p.ctrl[CTRL_FRONT], n_back = p.ctrl[CTRL_BACK];
    const uint32_t n_items = n_front + n_back;
    unsigned long long c_gr = 0, c_gc = 0, c_cr = 0, c_cc = 0;
    const int r = p.r;

    for (;;) {
        if (tid == 0) { s_item = atomicAdd(&p.ctrl[CTRL_CURSOR], 1u); s_nmb = 0; }
        __syncthreads();
        const uint32_t it = s_item;
        if (it >= n_items) break;
        const uint32_t item = p.work[it < n_front ? it : (uint32_t)p.n_tiles - 1u - (it - n_front)];
        const int tile = (int)(item & ITEM_ID);
        const int ttx = tile % p.tiles_x, tty = (tile / p.tiles_x) % p.tiles_y, ttz = tile / (p.tiles_x * p.tiles_y);
        const int gx0 = ttx * TX, gy0 = tty * TY;
        const int gz0 = local_to_global_tz(p, ttz) * TZ;      // global layer of the tile's first z layer
        const int lz0 = ttz * TZ;                             // local (stored) layer

        // ---------------- second-level cull of the colour micro-blocks (threads), overlapped with nothing yet
        if (item & ITEM_COL) {
            const int mbx = r * TX / MBX, mby = r * TY / MBY, mbz = r * TZ / MBZ;
            const int nmb = mbx * mby * mbz;
            for (int m = tid; m < nmb; m += CTA) {
                const int bx = m % mbx, by = (m / mbx) % mby, bz = m / (mbx * mby);
                const int ic0 = r * gx0 + bx * MBX, jc0 = r * gy0 + by * MBY, kc0 = r * gz0 + bz * MBZ;
                bool keep = false;
                if (ic0 < p.cnx && jc0 < p.cny && kc0 < r * p.nz) {
                    const float wx = p.ox + ((float)ic0 + 0.5f * (float)MBX) * p.vc;
                    const float wy = p.oy + ((float)jc0 + 0.5f * (float)MBY) * p.vc;
                    const float wz = p.oz + ((float)kc0 + 0.5f * (float)MBZ) * p.vc;
                    const float cX = p.R[0] * wx + p.R[1] * wy + p.R[2] * wz + p.t[0];
                    const float cY = p.R[3] * wx + p.R[4] * wy + p.R[5] * wz + p.t[1];
                    const float cZ = p.R[6] * wx + p.R[7] * wy + p.R[8] * wz + p.t[2];
                    int x0, x1, y0, y1; float zmin, zmax;
                    if (box_rect(p, cX, cY, cZ, p.mb_ex, p.mb_ey, p.mb_ez, x0, x1, y0, y1, zmin, zmax)) {
                        uint32_t mn, mx;
                        depth_range(p, x0, x1, y0, y1, mn, mx);
                        if (mx != 0u) {
                            const float dmin = (float)mn * 0.001f - 1e-4f, dmax = (float)mx * 0.001f + 1e-4f;
                            keep = (zmin <= dmax + p.sigma) && (zmax >= dmin - p.sigma);
                        }
                    }
                }
                if (keep) s_mb[atomicAdd(&s_nmb, 1u)] = (uint16_t)m;
            }
        }

        // ---------------- geometry: S2 + S3, one uint4 (4 x-adjacent voxels) per thread
        if (item & ITEM_GEO) {
            const int vx = tid % (TX / 4), y = (tid / (TX / 4)) % TY, z = tid / ((TX / 4) * TY);
            const int i0 = gx0 + 4 * vx, j = gy0 + y, kg = gz0 + z, kl = lz0 + z;
            if (i0 < p.nx && j < p.ny && kg < p.nz) {
                uint4 *ptr = reinterpret_cast<uint4 *>(p.geo + ((size_t)kl * p.ny + j) * p.nx + i0);
                uint4 v = *ptr;
                const uint4 old = v;
                const float py = __fmaf_rn((float)j + 0.5f, p.vs, p.oy);
                const float pz = __fmaf_rn((float)kg + 0.5f, p.vs, p.oz);
                uint32_t *w4 = reinterpret_cast<uint32_t *>(&v);
                const uint32_t *o4 = reinterpret_cast<const uint32_t *>(&old);
                bool any = false;
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const float px = __fmaf_rn((float)(i0 + e) + 0.5f, p.vs, p.ox);
                    const float X = __fmaf_rn(p.R[2], pz, __fmaf_rn(p.R[1], py, __fmaf_rn(p.R[0], px, p.t[0])));
                    const float Y = __fmaf_rn(p.R[5], pz, __fmaf_rn(p.R[4], py, __fmaf_rn(p.R[3], px, p.t[1])));
                    const float Z = __fmaf_rn(p.R[8], pz, __fmaf_rn(p.R[7], py, __fmaf_rn(p.R[6], px, p.t[2])));
                    const bool rd = geo_voxel(p, X, Y, Z, w4[e]);
                    const bool ch = w4[e] != o4[e];
                    any |= ch;
                    if (COUNT) { c_gr += rd; c_gc += ch; }
                }
                if (any) *ptr = v;                                // skip the store when nothing changed
            }
        }
        __syncthreads();

        // ---------------- colour: S4-S8, one warp per surviving micro-block, one uint4 (4 colour voxels) per lane
        if (item & ITEM_COL) {
            const uint32_t nkeep = s_nmb;
            if (tid == 0) atomicAdd(&p.ctrl[CTRL_BLOCKS_COL], nkeep);
            const int mbx = r * TX / MBX, mby = r * TY / MBY;
            const size_t cnx = (size_t)p.cnx, cny = (size_t)p.cny;
            for (uint32_t q = warp; q < nkeep; q += CTA / 32) {
                const int m = s_mb[q];
                const int bx = m % mbx, by = (m / mbx) % mby, bz = m / (mbx * mby);
                const int ic0 = r * gx0 + bx * MBX + 4 * (lane & 3);
                const int jc = r * gy0 + by * MBY + ((lane >> 2) & 3);
                const int kz = bz * MBZ + (lane >> 4);
                const int kcg = r * gz0 + kz, kcl = r * lz0 + kz;
                if (!(ic0 < p.cnx && jc < p.cny && kcg < r * p.nz)) continue;
                const float py = __fmaf_rn((float)jc + 0.5f, p.vc, p.oy);
                const float pz = __fmaf_rn((float)kcg + 0.5f, p.vc, p.oz);
                float X[4], Y[4], Z[4], W[4];
                unsigned pass = 0;
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const float px = __fmaf_rn((float)(ic0 + e) + 0.5f, p.vc, p.ox);
                    X[e] = __fmaf_rn(p.R[2], pz, __fmaf_rn(p.R[1], py, __fmaf_rn(p.R[0], px, p.t[0])));    // eq. 5
                    Y[e] = __fmaf_rn(p.R[5], pz, __fmaf_rn(p.R[4], py, __fmaf_rn(p.R[3], px, p.t[1])));
                    Z[e] = __fmaf_rn(p.R[8], pz, __fmaf_rn(p.R[7], py, __fmaf_rn(p.R[6], px, p.t[2])));
                    int x, y;
                    W[e] = 0.0f;
                    if (project_px(p.fx, p.fy, p.cx, p.cy, p.wd_f, p.hd_f, X[e], Y[e], Z[e], x, y)) {      // eq. 6
                        const float4 pm = __ldg(p.pixmap + y * p.wd + x);                               // eq. 7-8 per pixel (S1)
                        if (pm.w > 0.0f) {
                            const float dx = __fsub_rn(X[e], pm.x), dy = __fsub_rn(Y[e], pm.y), dz = __fsub_rn(Z[e], pm.z);
                            const float d2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
                            if (!(d2 > p.sig2)) { pass |= 1u << e; W[e] = pm.w; }                          // sigma gate, L108
                        }
                    }
                }
                if (pass) {
                    uint4 *ptr = reinterpret_cast<uint4 *>(p.col + ((size_t)kcl * cny + (size_t)jc) * cnx + (size_t)ic0);
                    uint4 v = *ptr;                                   // first HBM touch of these colour voxels (S6)
                    const uint4 old = v;
                    uint32_t *w4 = reinterpret_cast<uint32_t *>(&v);
                    const uint32_t *o4 = reinterpret_cast<const uint32_t *>(&old);
                    bool any = false;
#pragma unroll
                    for (int e = 0; e < 4; ++e) {
                        if (pass & (1u << e)) {
                            col_voxel_update(p, X[e], Y[e], Z[e], W[e], w4[e]);
                            const bool ch = w4[e] != o4[e];
                            any |= ch;
                            if (COUNT) { c_cr += 1; c_cc += ch; }
                        }
                    }
                    if (any) *ptr = v;
                }
            }
        }
        __syncthreads();      // s_item / s_mb are rewritten by the next iteration
    }

    if (COUNT) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            c_gr += __shfl_xor_sync(0xffffffffu, c_gr, o); c_gc += __shfl_xor_sync(0xffffffffu, c_gc, o);
            c_cr += __shfl_xor_sync(0xffffffffu, c_cr, o); c_cc += __shfl_xor_sync(0xffffffffu, c_cc, o);
        }
        if (lane == 0) {
            if (c_gr) atomicAdd(&p.counters[0], c_gr);
            if (c_gc) atomicAdd(&p.counters[1], c_gc);
            if (c_cr) atomicAdd(&p.counters[2], c_cr);
            if (c_cc) atomicAdd(&p.counters[3], c_cc);
        }
    }
}

}  // namespace vf
