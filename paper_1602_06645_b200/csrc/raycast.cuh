// raycast.cuh -- NEXT row: ray casting of the geometry + colour volumes into a depth map and an RGB
// image of a virtual camera (ICP prediction and live preview; the paper gives no equations -- the
// definition is readings R1-R6 of DESIGN.md "Ray casting", same canonical arithmetic as the integration).
#pragma once
#include "params.cuh"

namespace vf {

struct RayParams {
    int   w, h;
    float fx, fy, cx, cy;
    float T[12];                 // rows 0..2 of T_world_cam (row-major 3 x 4)
    float t_near, t_far;
    float *depth;                // w * h, metres along the camera z axis, 0 = no surface
    uint8_t *rgb;                // w * h * 3 or nullptr
};

// One thread per pixel; a CTA covers 8 x 8 pixels (two warps of 8 x 4), so the rays of a warp stay close together and
// their gathers share sectors.  Two exact shortcuts:
//  * samples outside the volume are "unknown" and cannot produce a hit, so only the samples between the ray's entry into
//    and exit from the volume's box (one sample of slack on both sides) are visited;
//  * a hit needs a sample with tsdf <= 0 in an observed voxel (R4), and p.tile_neg lists (conservatively) the geometry
//    tiles that may hold one.  A sample in any other tile cannot complete a hit, so its voxel is not read, and the ray
//    jumps to the last sample that is safely inside that tile.  Such a sample may still be the F_prev of the next one:
//    it is then evaluated lazily, only if the next sample turns out to be a candidate.
struct RaySample { float t, f; bool known; int i, j, k; };        // (i, j, k) = the voxel that contains the sample, if inside

// R2-R3 for sample k: canonical arithmetic, identical to the oracle's
__device__ __forceinline__ RaySample ray_sample(const Params &p, const float (&dw)[3], const float (&ow)[3], float vs, float inv_vs,
                                                float t_near, int k, bool &inside, int &tile)
{
    RaySample s;
    s.t = __fmaf_rn((float)k, vs, t_near); s.f = 0.0f; s.known = false;
    const float fi = floorf(__fmul_rn(__fsub_rn(__fmaf_rn(s.t, dw[0], ow[0]), p.ox), inv_vs));
    const float fj = floorf(__fmul_rn(__fsub_rn(__fmaf_rn(s.t, dw[1], ow[1]), p.oy), inv_vs));
    const float fk = floorf(__fmul_rn(__fsub_rn(__fmaf_rn(s.t, dw[2], ow[2]), p.oz), inv_vs));
    inside = fi >= 0.0f && fi < (float)p.nx && fj >= 0.0f && fj < (float)p.ny && fk >= 0.0f && fk < (float)p.nz;
    tile = -1; s.i = s.j = s.k = 0;
    if (inside) {
        s.i = (int)fi; s.j = (int)fj; s.k = (int)fk;
        // (indices are non-negative here: unsigned shifts instead of signed divisions -- the kernel is issue-bound)
        tile = (int)((((unsigned)s.k / TZ) * (unsigned)p.tiles_y + (unsigned)s.j / TY) * (unsigned)p.tiles_x + (unsigned)s.i / TX);   // the voxel itself is read by ray_voxel() when needed
    }
    return s;
}

__device__ __forceinline__ void ray_voxel(const Params &p, RaySample &s)
{
    const uint32_t word = __ldg(p.geo + ((size_t)s.k * (size_t)p.ny + (size_t)s.j) * (size_t)p.nx + (size_t)s.i);
    s.known = (word >> 16) != 0u;                                                         // R3
    s.f = s.known ? (float)(int)(short)(word & 0xffffu) : 0.0f;
}

__global__ void __launch_bounds__(64) k_raycast(const __grid_constant__ Params p, const __grid_constant__ RayParams q)
{
    const int x = blockIdx.x * 8 + (threadIdx.x & 7), y = blockIdx.y * 8 + (threadIdx.x >> 3);
    if (x >= q.w || y >= q.h) return;
    const float dx = __fdiv_rn(__fsub_rn((float)x, q.cx), q.fx), dy = __fdiv_rn(__fsub_rn((float)y, q.cy), q.fy);   // R1
    float dw[3], ow[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        dw[a] = __fmaf_rn(q.T[4 * a + 1], dy, __fmaf_rn(q.T[4 * a + 0], dx, q.T[4 * a + 2]));
        ow[a] = q.T[4 * a + 3];
    }
    const float vs = p.vs, inv_vs = __frcp_rn(p.vs);
    const float org[3] = {p.ox, p.oy, p.oz};
    // culling only: parameter interval in which the ray can be inside the box (slab test, grown by one voxel)
    float ta = q.t_near, tb = q.t_far;
    {
        const float lo[3] = {p.ox - vs, p.oy - vs, p.oz - vs};
        const float hi[3] = {p.ox + vs * (float)(p.nx + 1), p.oy + vs * (float)(p.ny + 1), p.oz + vs * (float)(p.nz + 1)};
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            if (fabsf(dw[a]) > 1e-12f) {
                const float t0 = (lo[a] - ow[a]) / dw[a], t1 = (hi[a] - ow[a]) / dw[a];
                ta = fmaxf(ta, fminf(t0, t1)); tb = fminf(tb, fmaxf(t0, t1));
            } else if (ow[a] < lo[a] || ow[a] > hi[a]) tb = -1.0f;
        }
    }
    // culling only: the ray in grid coordinates, g(t) = go + t * gd, for the tile-exit computation
    // (1 / gd is taken once per ray: the exit parameter only has to be right to a few hundredths of a voxel)
    float go[3], gd[3], rgd[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) { go[a] = (ow[a] - org[a]) * inv_vs; gd[a] = dw[a] * inv_vs; rgd[a] = fabsf(gd[a]) > 1e-9f ? 1.0f / gd[a] : 0.0f; }
    const int tdim[3] = {TX, TY, TZ};
    float depth = 0.0f;
    if (ta <= tb) {
        int k = max(0, (int)floorf((ta - q.t_near) * inv_vs) - 1);
        const int k1 = (int)fminf(ceilf((tb - q.t_near) * inv_vs) + 1.0f, 2.0e9f);
        RaySample prev; prev.t = 0.0f; prev.f = 0.0f; prev.known = false;
        bool prev_pending = false;                          // sample k - 1 was skipped: evaluate it when it is needed
        while (k <= k1) {
            bool inside; int tile;
            RaySample cur = ray_sample(p, dw, ow, vs, inv_vs, q.t_near, k, inside, tile);   // R2
            if (cur.t > q.t_far) break;
            if (!inside) { prev = cur; prev_pending = false; ++k; continue; }             // unknown sample
            // coarse level first: a brick of BRICK^3 voxels (1 x 8 x 4 tiles) without such a voxel is crossed in one jump
            const unsigned brick = (((unsigned)cur.k / BRICK) * (unsigned)p.bricks_y + (unsigned)cur.j / BRICK) * (unsigned)p.bricks_x + (unsigned)cur.i / BRICK;
            const bool brick_free = __ldg(p.brick_neg + brick) == 0;
            if (brick_free || __ldg(p.tile_neg + (unsigned)tile) == 0) {
                // no observed voxel with tsdf <= 0 in this brick / tile: jump to the last sample safely inside it
                // (the tile's box comes from the sample's canonical voxel indices, the exit from free-form arithmetic: if
                // the two disagree at a tile boundary the exit lies behind the sample and nothing is skipped)
                const int vox[3] = {cur.i, cur.j, cur.k};
                float t_exit = 3.0e38f;
#pragma unroll
                for (int a = 0; a < 3; ++a) {
                    const int bd = brick_free ? BRICK : tdim[a];
                    const float lo = (float)(vox[a] & ~(bd - 1));                           // box sizes are powers of two
                    if (gd[a] > 1e-9f) t_exit = fminf(t_exit, (lo + (float)bd - 0.05f - go[a]) * rgd[a]);
                    else if (gd[a] < -1e-9f) t_exit = fminf(t_exit, (lo + 0.05f - go[a]) * rgd[a]);
                }
                const int kk = (int)fminf(floorf((t_exit - q.t_near) * inv_vs) - 1.0f, (float)k1);
                k = max(k, kk) + 1;
                prev_pending = true;
                continue;
            }
            ray_voxel(p, cur);
            if (cur.known && !(cur.f > 0.0f)) {                                            // candidate: needs F_prev
                if (prev_pending) {
                    bool in2; int tile2;
                    prev = ray_sample(p, dw, ow, vs, inv_vs, q.t_near, k - 1, in2, tile2);
                    if (in2) ray_voxel(p, prev);
                }
                if (prev.known && prev.f > 0.0f) {                                         // R4
                    depth = __fmaf_rn(vs, __fdiv_rn(prev.f, __fsub_rn(prev.f, cur.f)), prev.t);
                    break;
                }
            }
            prev = cur; prev_pending = false; ++k;
        }
    }
    uint32_t c = 0u;
    if (depth > 0.0f && q.rgb) {                                                                // R5
        const float hx = floorf(__fmul_rn(__fsub_rn(__fmaf_rn(depth, dw[0], ow[0]), org[0]), p.inv_vc));
        const float hy = floorf(__fmul_rn(__fsub_rn(__fmaf_rn(depth, dw[1], ow[1]), org[1]), p.inv_vc));
        const float hz = floorf(__fmul_rn(__fsub_rn(__fmaf_rn(depth, dw[2], ow[2]), org[2]), p.inv_vc));
        if (hx >= 0.0f && hx < (float)p.cnx && hy >= 0.0f && hy < (float)p.cny && hz >= 0.0f && hz < (float)p.cnz) {
            const uint32_t cw = __ldg(p.col + ((size_t)(int)hz * (size_t)p.cny + (size_t)(int)hy) * (size_t)p.cnx + (size_t)(int)hx);
            if ((cw >> 24) != 0u) c = cw;
        }
    }
    const size_t o = (size_t)y * (size_t)q.w + (size_t)x;
    q.depth[o] = depth;
    if (q.rgb) { q.rgb[3 * o] = (uint8_t)c; q.rgb[3 * o + 1] = (uint8_t)(c >> 8); q.rgb[3 * o + 2] = (uint8_t)(c >> 16); }
}

// NEXT row: colour-volume lookup at world points -- the primitive under the paper's per-polygon
// texture maps (the positions come from eq. 11-14).  Reading S1: the colour voxel whose cell contains the
// point, nearest voxel; the packed word {R, G, B, wq}, or 0 outside the volume.  One thread per point.
__global__ void __launch_bounds__(256) k_sample_colour(const __grid_constant__ Params p, const float *__restrict__ pts, long long n,
                                                       uint32_t *__restrict__ words)
{
    const long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= n) return;
    const float hx = floorf(__fmul_rn(__fsub_rn(__ldg(pts + 3 * m + 0), p.ox), p.inv_vc));
    const float hy = floorf(__fmul_rn(__fsub_rn(__ldg(pts + 3 * m + 1), p.oy), p.inv_vc));
    const float hz = floorf(__fmul_rn(__fsub_rn(__ldg(pts + 3 * m + 2), p.oz), p.inv_vc));
    uint32_t w = 0u;
    if (hx >= 0.0f && hx < (float)p.cnx && hy >= 0.0f && hy < (float)p.cny && hz >= 0.0f && hz < (float)p.cnz)
        w = __ldg(p.col + ((size_t)(int)hz * (size_t)p.cny + (size_t)(int)hy) * (size_t)p.cnx + (size_t)(int)hx);
    words[m] = w;
}

// The same lookup with trilinear interpolation (reading S2): grid coordinate g = (p - origin) / vc - 1/2,
// b = floor(g), f = g - b; the 8 voxels b + {0,1}^3 with weights (wz * wy) * wx; voxels outside the volume or never
// observed (wq = 0) are left out and the colour is normalised over the rest, C = rint(sum w C / sum w); the weight byte
// is rint(sum w wq) -- how much of the footprint has been seen.  The 8 words are requested first, then accumulated in
// the canonical order (z-major, then y, then x).  One thread per point.
__global__ void __launch_bounds__(256) k_sample_colour_trilinear(const __grid_constant__ Params p, const float *__restrict__ pts, long long n,
                                                                 uint32_t *__restrict__ words)
{
    const long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= n) return;
    const float o[3] = {p.ox, p.oy, p.oz};
    const int cn[3] = {p.cnx, p.cny, p.cnz};
    float b[3], f[3];
    bool ok = true;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const float g = __fsub_rn(__fmul_rn(__fsub_rn(__ldg(pts + 3 * m + a), o[a]), p.inv_vc), 0.5f);
        b[a] = floorf(g);
        f[a] = __fsub_rn(g, b[a]);
        ok = ok && (b[a] >= -1.0f) && (b[a] <= (float)(cn[a] - 1));      // the footprint touches the volume; false for NaN / inf
    }
    uint32_t word = 0u;
    if (ok) {
        const int i0 = (int)b[0], j0 = (int)b[1], k0 = (int)b[2];
        uint32_t cw[8];
#pragma unroll
        for (int c = 0; c < 8; ++c) {
            const int i = i0 + (c & 1), j = j0 + ((c >> 1) & 1), k = k0 + (c >> 2);
            const bool in = i >= 0 && i < cn[0] && j >= 0 && j < cn[1] && k >= 0 && k < cn[2];
            cw[c] = in ? __ldg(p.col + ((size_t)k * (size_t)cn[1] + (size_t)j) * (size_t)cn[0] + (size_t)i) : 0u;
        }
        float sw = 0.0f, sa = 0.0f, sc[3] = {0.0f, 0.0f, 0.0f};
#pragma unroll
        for (int c = 0; c < 8; ++c) {
            if ((cw[c] >> 24) == 0u) continue;
            const float wx = (c & 1) ? f[0] : __fsub_rn(1.0f, f[0]);
            const float wy = (c & 2) ? f[1] : __fsub_rn(1.0f, f[1]);
            const float wz = (c & 4) ? f[2] : __fsub_rn(1.0f, f[2]);
            const float w = __fmul_rn(__fmul_rn(wz, wy), wx);
            sw = __fadd_rn(sw, w);
            sa = __fmaf_rn(w, (float)(cw[c] >> 24), sa);
#pragma unroll
            for (int ch = 0; ch < 3; ++ch) sc[ch] = __fmaf_rn(w, (float)((cw[c] >> (8 * ch)) & 0xffu), sc[ch]);
        }
        if (sw > 0.0f) {
#pragma unroll
            for (int ch = 0; ch < 3; ++ch) {
                const float cq = rintf(__fdiv_rn(sc[ch], sw));
                const int ci = cq < 0.0f ? 0 : (cq > 255.0f ? 255 : (int)cq);
                word |= (uint32_t)ci << (8 * ch);
            }
            const float aq = rintf(sa);
            const int ai = aq < 0.0f ? 0 : (aq > 255.0f ? 255 : (int)aq);
            word |= (uint32_t)ai << 24;
        }
    }
    words[m] = word;
}

}  // namespace vf
