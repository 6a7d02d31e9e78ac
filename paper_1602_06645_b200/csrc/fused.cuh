// fused.cuh -- K2: the fused integration kernel (S2-S8), warp-centric and persistent.
//
// Every warp pops work items from one queue until it is empty -- first the colour items (one non-zero shell-mark word
// = up to 32 colour cells of 8x4x4 voxels of one tile), then the geometry items (one tile of 32x4x8 TSDF voxels, marched
// along z with per-column bases hoisted).  A lane always owns one 16-byte vector of 4 x-adjacent voxels, so a warp
// reads/writes whole 32-byte sectors (colour rows) or 128-byte lines (geometry rows).  No block-level barriers.
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

struct Counts { unsigned long long gr, gc, cr, cc; };

// one geometry tile, one warp: lane = (vx = lane & 7, y = lane >> 3) owns voxels (gx0 + 4 vx .. + 3, gy0 + y) of every layer
template <bool COUNT>
__device__ __forceinline__ void geometry_tile(const Params &p, int tile, int lane, Counts &c)
{
    const int ttx = tile % p.tiles_x, t2 = tile / p.tiles_x, tty = t2 % p.tiles_y, ttz = t2 / p.tiles_y;
    const int i0 = ttx * TX + 4 * (lane & 7), j = tty * TY + (lane >> 3);
    const int gz0 = local_to_global_tz(p, ttz) * TZ, lz0 = ttz * TZ;
    if (!(i0 < p.nx && j < p.ny)) return;
    const int nl = min(TZ, p.nz - gz0);
    // per-column bases of eq. 5: fma(R_1, py, fma(R_0, px, t)) -- the z term is added per layer with one fma each
    const float py = __fmaf_rn((float)j + 0.5f, p.vs, p.oy);
    float bX[4], bY[4], bZ[4];
#pragma unroll
    for (int e = 0; e < 4; ++e) {
        const float px = __fmaf_rn((float)(i0 + e) + 0.5f, p.vs, p.ox);
        bX[e] = __fmaf_rn(p.R[1], py, __fmaf_rn(p.R[0], px, p.t[0]));
        bY[e] = __fmaf_rn(p.R[4], py, __fmaf_rn(p.R[3], px, p.t[1]));
        bZ[e] = __fmaf_rn(p.R[7], py, __fmaf_rn(p.R[6], px, p.t[2]));
    }
    const size_t layer = (size_t)p.ny * p.nx;
    uint4 *ptr = reinterpret_cast<uint4 *>(p.geo + ((size_t)lz0 * p.ny + j) * p.nx + i0);
    uint4 cur = *ptr;
    for (int z = 0; z < nl; ++z) {
        uint4 nxt = cur;
        uint4 *pn = reinterpret_cast<uint4 *>(reinterpret_cast<uint32_t *>(ptr) + layer);
        if (z + 1 < nl) nxt = *pn;                                // prefetch the next layer while this one is computed
        const float pz = __fmaf_rn((float)(gz0 + z) + 0.5f, p.vs, p.oz);
        uint4 v = cur;
        uint32_t *w4 = reinterpret_cast<uint32_t *>(&v);
        const uint32_t *o4 = reinterpret_cast<const uint32_t *>(&cur);
        bool any = false;
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const float X = __fmaf_rn(p.R[2], pz, bX[e]);
            const float Y = __fmaf_rn(p.R[5], pz, bY[e]);
            const float Z = __fmaf_rn(p.R[8], pz, bZ[e]);
            const bool rd = geo_voxel(p, X, Y, Z, w4[e]);
            const bool ch = w4[e] != o4[e];
            any |= ch;
            if (COUNT) { c.gr += rd; c.gc += ch; }
        }
        if (any) *ptr = v;                                        // skip the store when nothing changed
        ptr = pn; cur = nxt;
    }
}

// one colour work item, one warp: the set bits of one shell-mark word are colour cells of 8 x 4 x 4 voxels;
// lane = (vx = lane & 1, y = (lane >> 1) & 3, z = lane >> 3) owns 4 x-adjacent voxels of each cell
template <int R, bool COUNT>
__device__ __forceinline__ void colour_item(const Params &p, uint32_t wi, int lane, Counts &c)
{
    constexpr int CX = cells_x(R), CY = cells_y(R), WPT = words_per_tile(R);
    uint32_t bits = 0;
    if (lane == 0) { bits = __ldcg(p.marks + wi); p.marks[wi] = 0u; }     // consume the marks (self-cleaning)
    bits = __shfl_sync(0xffffffffu, bits, 0);
    const int tile = (int)(wi / WPT), word = (int)(wi % WPT);
    const int ttx = tile % p.tiles_x, t2 = tile / p.tiles_x, tty = t2 % p.tiles_y, ttz = t2 / p.tiles_y;
    const int cgx0 = ttx * TX * R, cgy0 = tty * TY * R;
    const int cgz0 = local_to_global_tz(p, ttz) * TZ * R, clz0 = ttz * TZ * R;
    const size_t cnx = (size_t)p.cnx, cny = (size_t)p.cny;
    if (COUNT && lane == 0) atomicAdd(&p.ctrl[CTRL_CELLS], (uint32_t)__popc(bits));
    while (bits) {
        const int b = word * 32 + (__ffs(bits) - 1);
        bits &= bits - 1;
        const int cx = b % CX, cy = (b / CX) % CY, cz = b / (CX * CY);
        const int ic0 = cgx0 + cx * CLX + 4 * (lane & 1);
        const int jc = cgy0 + cy * CLY + ((lane >> 1) & 3);
        const int kz = cz * CLZ + (lane >> 3);
        const int kcg = cgz0 + kz, kcl = clz0 + kz;
        if (!(ic0 < p.cnx && jc < p.cny && kcg < p.cnz)) continue;
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
            uint4 v = *ptr;                                       // first HBM touch of these colour voxels (S6)
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
                    if (COUNT) { c.cr += 1; c.cc += ch; }
                }
            }
            if (any) *ptr = v;
        }
    }
}

template <int R, bool COUNT>
__global__ void __launch_bounds__(CTA) k_fused(const __grid_constant__ Params p)
{
    const int lane = threadIdx.x & 31;
    const uint32_t n_col = __ldcg(&p.ctrl[CTRL_NCOL]), n_items = n_col + __ldcg(&p.ctrl[CTRL_NGEO]);
    Counts c = {0, 0, 0, 0};
    for (;;) {
        uint32_t it = 0;
        if (lane == 0) it = atomicAdd(&p.ctrl[CTRL_CURSOR], 1u);
        it = __shfl_sync(0xffffffffu, it, 0);
        if (it >= n_items) break;
        if (it < n_col) colour_item<R, COUNT>(p, __ldcg(p.work_col + it), lane, c);
        else            geometry_tile<COUNT>(p, (int)__ldcg(p.work_geo + (it - n_col)), lane, c);
    }
    if (COUNT) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            c.gr += __shfl_xor_sync(0xffffffffu, c.gr, o); c.gc += __shfl_xor_sync(0xffffffffu, c.gc, o);
            c.cr += __shfl_xor_sync(0xffffffffu, c.cr, o); c.cc += __shfl_xor_sync(0xffffffffu, c.cc, o);
        }
        if (lane == 0) {
            if (c.gr) atomicAdd(&p.counters[0], c.gr);
            if (c.gc) atomicAdd(&p.counters[1], c.gc);
            if (c.cr) atomicAdd(&p.counters[2], c.cr);
            if (c.cc) atomicAdd(&p.counters[3], c.cc);
        }
    }
}

}  // namespace vf
