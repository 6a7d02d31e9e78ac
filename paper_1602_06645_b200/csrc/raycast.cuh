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
    const uint8_t *sub_neg;      // per 8 x 4 x 4 sub-box of the geometry volume: 1 = it holds an observed voxel with tsdf <= 0 (k_sub_neg)
    int sbx, sby;                // sub-boxes along x and y
    const uint8_t *tile_any, *brick_any;   // the same per tile and per brick, exact as well (k_sub_neg); indexed like tile_neg / brick_neg
    const uint8_t *sub_dil, *tile_dil, *brick_dil;   // the three again, each box OR-ed with its 7 neighbours at +1 (k_dilate): for R7
};

// dst(x, y, z) = OR of src over (x, y, z) + {0, 1}^3 (inside the grid).  A trilinear sample whose BASE corner lies in a box
// has its 8 corners in that box and its neighbours at +1 only, so one look-up of dst answers for all of them.
struct DilateJob { const uint8_t *src; uint8_t *dst; int nx, ny, nz; unsigned first_block; };
__global__ void __launch_bounds__(256) k_dilate(const __grid_constant__ DilateJob j0, const __grid_constant__ DilateJob j1, const __grid_constant__ DilateJob j2)
{
    const DilateJob &job = blockIdx.x >= j2.first_block ? j2 : (blockIdx.x >= j1.first_block ? j1 : j0);     // three grids, one launch
    const int nx = job.nx, ny = job.ny, nz = job.nz;
    const long long n = (long long)nx * ny * nz, m = (long long)(blockIdx.x - job.first_block) * blockDim.x + threadIdx.x;
    if (m >= n) return;
    const int x = (int)(m % nx), y = (int)((m / nx) % ny), z = (int)(m / ((long long)nx * ny));
    uint8_t a = 0;
#pragma unroll
    for (int c = 0; c < 8; ++c) {
        const int xx = x + (c & 1), yy = y + ((c >> 1) & 1), zz = z + (c >> 2);
        if (xx < nx && yy < ny && zz < nz) a |= __ldg(job.src + ((size_t)zz * ny + yy) * nx + xx);
    }
    job.dst[m] = a ? 1 : 0;
}

// The finest level of the ray casters' skip hierarchy, rebuilt (when the volume has changed) just before a ray cast: for
// every tile that the integration flagged (tile_neg: "may hold an observed voxel with tsdf <= 0" -- a loose, one-sided test
// against the depth range of the tile's footprint, accumulated since the last rebuild) the tile's voxels are read once and each of
// its 8 sub-boxes gets the exact answer.  One warp per tile, lane = (x, y) column of a sub-box.  A ray then reads voxels
// only in the shell of sub-boxes around the zero crossing (and behind it) instead of in every flagged tile it crosses.
__global__ void __launch_bounds__(256) k_sub_neg(const __grid_constant__ Params p, uint8_t *__restrict__ sub_neg, int sbx_n, int sby_n, int sbz_n,
                                                 uint8_t *__restrict__ tile_any, uint8_t *__restrict__ brick_any)
{
    const int tile = blockIdx.x * 8 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (tile >= p.n_tiles) return;
    const int ttx = tile % p.tiles_x, tty = (tile / p.tiles_x) % p.tiles_y, ttz = tile / (p.tiles_x * p.tiles_y);
    const bool flagged = __ldg(p.tile_neg + tile) != 0;
    const int j = tty * TY + (lane >> 3);
    bool tile_has = false;
    if (!flagged) {                                            // nothing to read: 8 zero bytes
        if (lane < SUBX * SUBZ) sub_neg[((size_t)(ttz * SUBZ + lane % SUBZ) * sby_n + tty) * sbx_n + ttx * SUBX + lane / SUBZ] = 0;
    } else if ((p.nx & 3) == 0 && ttx * TX + TX <= p.nx && tty * TY + TY <= p.ny && ttz * TZ + TZ <= p.nz) {
        // a whole tile with 16-byte aligned rows: one 16-byte load per lane and layer covers the layer (32 x 4 voxels); lanes
        // 2 bx and 2 bx + 1 of every row hold sub-box bx
        unsigned any_z[SUBZ];
#pragma unroll
        for (int bz = 0; bz < SUBZ; ++bz) {
            bool any = false;
#pragma unroll
            for (int e = 0; e < TZ / SUBZ; ++e) {
                const uint4 w = __ldcg(reinterpret_cast<const uint4 *>(p.geo + ((size_t)(ttz * TZ + bz * (TZ / SUBZ) + e) * (size_t)p.ny + (size_t)j) * (size_t)p.nx + (size_t)(ttx * TX)) + (lane & 7));
                const uint32_t ww[4] = {w.x, w.y, w.z, w.w};
#pragma unroll
                for (int u = 0; u < 4; ++u) any = any || ((ww[u] >> 16) != 0u && (int)(short)(ww[u] & 0xffffu) <= 0);
            }
            any_z[bz] = __ballot_sync(0xffffffffu, any);
        }
#pragma unroll
        for (int sb = 0; sb < SUBX * SUBZ; ++sb) {
            const int bx = sb / SUBZ, bz = sb % SUBZ;
            const bool box_any = (any_z[bz] & (0x03030303u << (2 * bx))) != 0u;
            if (lane == 0) sub_neg[((size_t)(ttz * SUBZ + bz) * sby_n + tty) * sbx_n + ttx * SUBX + bx] = box_any ? 1 : 0;
            tile_has = tile_has || box_any;
        }
    } else {
#pragma unroll
        for (int sb = 0; sb < SUBX * SUBZ; ++sb) {
            const int bx = sb / SUBZ, bz = sb % SUBZ;
            bool any = false;
            const int i = ttx * TX + bx * (TX / SUBX) + (lane & 7), k0 = ttz * TZ + bz * (TZ / SUBZ);
            if (i < p.nx && j < p.ny) {
#pragma unroll
                for (int e = 0; e < TZ / SUBZ; ++e) {
                    if (k0 + e < p.nz) {
                        const uint32_t w = __ldcg(p.geo + ((size_t)(k0 + e) * (size_t)p.ny + (size_t)j) * (size_t)p.nx + (size_t)i);
                        any = any || ((w >> 16) != 0u && (int)(short)(w & 0xffffu) <= 0);
                    }
                }
            }
            const bool box_any = __any_sync(0xffffffffu, any);
            if (lane == 0) sub_neg[((size_t)(ttz * SUBZ + bz) * sby_n + tty) * sbx_n + ttx * SUBX + bx] = box_any ? 1 : 0;
            tile_has = tile_has || box_any;
        }
    }
    if (lane == 0) {
        tile_any[tile] = tile_has ? 1 : 0;
        if (tile_has) brick_any[((ttz / 4) * p.bricks_y + tty / 8) * p.bricks_x + ttx] = 1;     // (zeroed before the launch)
        // The exact answer also replaces the integration's loose flag, so that the next rebuild reads only the tiles that hold
        // such a voxel now or were flagged since.  Safe: a tile can only receive a tsdf <= 0 in a frame whose classification
        // flags it again (prepass.cuh sets the flag every time its condition holds, not only the first time).
        if (flagged && !tile_has) p.tile_neg[tile] = 0;
    }
}

// One thread per pixel; a CTA covers 8 x 8 pixels (two warps of 8 x 4), so the rays of a warp stay close together and
// their gathers share sectors.  Two exact shortcuts:
//  * samples outside the volume are "unknown" and cannot produce a hit, so only the samples between the ray's entry into
//    and exit from the volume's box (one sample of slack on both sides) are visited;
//  * a hit needs a sample with tsdf <= 0 in an observed voxel (R4); q.brick_any / tile_any / sub_neg say exactly which
//    bricks, tiles and sub-boxes hold one (k_sub_neg, from the integration's conservative p.tile_neg).  A sample in any other tile cannot complete a hit, so its voxel is not read, and the ray
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
            // coarse level first: a brick of BRICK^3 voxels (1 x 8 x 4 tiles) without such a voxel is crossed in one jump;
            const unsigned brick = (((unsigned)cur.k / BRICK) * (unsigned)p.bricks_y + (unsigned)cur.j / BRICK) * (unsigned)p.bricks_x + (unsigned)cur.i / BRICK;
            // then the tile, then the sub-box of 8 x 4 x 4 voxels (exact: k_sub_neg)
            int level = 3;
            if (__ldg(q.brick_any + brick) == 0) level = 0;
            else if (__ldg(q.tile_any + (unsigned)tile) == 0) level = 1;
            else if (__ldg(q.sub_neg + (((unsigned)cur.k / (TZ / SUBZ)) * (unsigned)q.sby + (unsigned)cur.j / TY) * (unsigned)q.sbx + (unsigned)cur.i / (TX / SUBX)) == 0) level = 2;
            if (level < 3) {
                // no observed voxel with tsdf <= 0 in this brick / tile / sub-box: jump to the last sample safely inside it
                // (the box comes from the sample's canonical voxel indices, the exit from free-form arithmetic: if
                // the two disagree at a box boundary the exit lies behind the sample and nothing is skipped)
                const int vox[3] = {cur.i, cur.j, cur.k};
                const int bdim[3][3] = {{BRICK, BRICK, BRICK}, {TX, TY, TZ}, {TX / SUBX, TY, TZ / SUBZ}};
                float t_exit = 3.0e38f;
#pragma unroll
                for (int a = 0; a < 3; ++a) {
                    const int bd = level == 0 ? bdim[0][a] : (level == 1 ? bdim[1][a] : bdim[2][a]);
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

// ---- reading R7: the TSDF of a sample is interpolated trilinearly from the 8 voxels around it (oracle: ref_raycast_trilinear).
// A TSDF that is linear in space is reproduced exactly, so the depth map has no voxel-sized terraces and the tracker can
// use it without F8.  Same marching (R2), hit rule (R4) and colour (R5); the two shortcuts carry over with one change:
// a sample can only complete a hit if its F <= 0, F is a blend with non-negative weights of 8 observed voxels, so at least
// one of those voxels has tsdf <= 0.  The corners are the base corner floor(g) and its neighbours at +1, so the flags of the
// three levels are dilated by one box towards +x, +y, +z (k_dilate) and looked up once, for the base corner's box; a jump ends
// at the last sample whose base corner is still inside that box.
struct TriSample { float t, f; bool known, in; int i0, j0, k0; float fx, fy, fz; };

// R2 + the index part of R7 for sample k: canonical arithmetic, identical to the oracle's
__device__ __forceinline__ TriSample tri_sample(const Params &p, const float (&dw)[3], const float (&ow)[3], float vs, float inv_vs, float t_near, int k)
{
    TriSample s;
    s.t = __fmaf_rn((float)k, vs, t_near); s.f = 0.0f; s.known = false;
    const float gx = __fsub_rn(__fmul_rn(__fsub_rn(__fmaf_rn(s.t, dw[0], ow[0]), p.ox), inv_vs), 0.5f);
    const float gy = __fsub_rn(__fmul_rn(__fsub_rn(__fmaf_rn(s.t, dw[1], ow[1]), p.oy), inv_vs), 0.5f);
    const float gz = __fsub_rn(__fmul_rn(__fsub_rn(__fmaf_rn(s.t, dw[2], ow[2]), p.oz), inv_vs), 0.5f);
    const float bx = floorf(gx), by = floorf(gy), bz = floorf(gz);
    s.fx = __fsub_rn(gx, bx); s.fy = __fsub_rn(gy, by); s.fz = __fsub_rn(gz, bz);
    s.in = bx >= 0.0f && bx <= (float)(p.nx - 2) && by >= 0.0f && by <= (float)(p.ny - 2) && bz >= 0.0f && bz <= (float)(p.nz - 2);
    s.i0 = s.j0 = s.k0 = 0;
    if (s.in) { s.i0 = (int)bx; s.j0 = (int)by; s.k0 = (int)bz; }
    return s;
}

// the value part of R7: 8 loads first; if none of the 8 stored values is <= 0 the blend is positive (or the sample unknown) and
// the sample cannot complete a hit: false is returned and nothing is computed (the caller evaluates the sample again, with
// force, should it turn out to be the F_prev of a candidate).  Otherwise the blend in the canonical order (corner
// c = x + 2 y + 4 z, weight (wz * wy) * wx).
__device__ __forceinline__ bool tri_value(const Params &p, TriSample &s, bool force)
{
    if (!s.in) return true;
    const uint32_t *base = p.geo + ((size_t)s.k0 * (size_t)p.ny + (size_t)s.j0) * (size_t)p.nx + (size_t)s.i0;
    const size_t sy = (size_t)p.nx, sz = (size_t)p.nx * (size_t)p.ny;
    uint32_t w[8];
#pragma unroll
    for (int c = 0; c < 8; ++c) w[c] = __ldg(base + (c & 1) + ((c >> 1) & 1) * sy + (c >> 2) * sz);
    if (!force) {
        bool any = false;
#pragma unroll
        for (int c = 0; c < 8; ++c) any = any || (int)(short)(w[c] & 0xffffu) <= 0;
        if (!any) return false;
    }
    bool known = true;
    float f = 0.0f;
#pragma unroll
    for (int c = 0; c < 8; ++c) {
        known = known && (w[c] >> 16) != 0u;
        const float wx = (c & 1) ? s.fx : __fsub_rn(1.0f, s.fx);
        const float wy = (c & 2) ? s.fy : __fsub_rn(1.0f, s.fy);
        const float wz = (c & 4) ? s.fz : __fsub_rn(1.0f, s.fz);
        f = __fmaf_rn(__fmul_rn(__fmul_rn(wz, wy), wx), (float)(int)(short)(w[c] & 0xffffu), f);
    }
    s.known = known; s.f = known ? f : 0.0f;
    return true;
}

__global__ void __launch_bounds__(64) k_raycast_trilinear(const __grid_constant__ Params p, const __grid_constant__ RayParams q)
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
    // culling only: the ray in CELL coordinates u(t) = go + t * gd (voxel v covers [v, v + 1)); the corners of a sample are
    // floor(u - 1/2) and that + 1, so they all lie in the box [lo, lo + n) iff lo + 1/2 <= u < lo + n - 1/2 on every axis
    float go[3], gd[3], rgd[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) { go[a] = (ow[a] - org[a]) * inv_vs; gd[a] = dw[a] * inv_vs; rgd[a] = fabsf(gd[a]) > 1e-9f ? 1.0f / gd[a] : 0.0f; }
    float depth = 0.0f;
    if (ta <= tb) {
        int k = max(0, (int)floorf((ta - q.t_near) * inv_vs) - 1);
        const int k1 = (int)fminf(ceilf((tb - q.t_near) * inv_vs) + 1.0f, 2.0e9f);
        TriSample prev; prev.t = 0.0f; prev.f = 0.0f; prev.known = false;
        bool prev_pending = false;                          // sample k - 1 was skipped: evaluate it when it is needed
        while (k <= k1) {
            TriSample cur = tri_sample(p, dw, ow, vs, inv_vs, q.t_near, k);               // R2
            if (cur.t > q.t_far) break;
            if (!cur.in) { prev = cur; prev_pending = false; ++k; continue; }             // unknown sample
            // can any corner hold an observed tsdf <= 0?  One look-up per level, in the dilated flags, for the box of the BASE
            // corner: brick, then tile, then sub-box
            const unsigned ax0 = (unsigned)cur.i0, ay0 = (unsigned)cur.j0, az0 = (unsigned)cur.k0;
            int level = 3;
            if (__ldg(q.brick_dil + ((az0 / BRICK) * (unsigned)p.bricks_y + ay0 / BRICK) * (unsigned)p.bricks_x + ax0 / BRICK) == 0) level = 0;
            else if (__ldg(q.tile_dil + ((az0 / TZ) * (unsigned)p.tiles_y + ay0 / TY) * (unsigned)p.tiles_x + ax0 / TX) == 0) level = 1;
            else if (__ldg(q.sub_dil + ((az0 / (TZ / SUBZ)) * (unsigned)q.sby + ay0 / TY) * (unsigned)q.sbx + ax0 / (TX / SUBX)) == 0) level = 2;
            if (level < 3) {
                // this sample cannot complete a hit, and neither can any later sample whose base corner lies in that box: jump
                // to the last of them.  The base corner is floor(u - 1/2), so it is in [lo, lo + n) while lo + 1/2 <= u <
                // lo + n + 1/2 (free-form arithmetic with 0.05 cells of slack; if it disagrees with the canonical indices the
                // exit lies behind the sample: no jump)
                const int vox[3] = {cur.i0, cur.j0, cur.k0};
                const int bdim[3][3] = {{BRICK, BRICK, BRICK}, {TX, TY, TZ}, {TX / SUBX, TY, TZ / SUBZ}};
                float t_exit = 3.0e38f;
#pragma unroll
                for (int a = 0; a < 3; ++a) {
                    const int bd = level == 0 ? bdim[0][a] : (level == 1 ? bdim[1][a] : bdim[2][a]);
                    const float lo = (float)(vox[a] & ~(bd - 1));                           // box sizes are powers of two
                    if (gd[a] > 1e-9f) t_exit = fminf(t_exit, (lo + (float)bd + 0.45f - go[a]) * rgd[a]);
                    else if (gd[a] < -1e-9f) t_exit = fminf(t_exit, (lo + 0.55f - go[a]) * rgd[a]);
                }
                const int kn = (int)fminf(floorf((t_exit - q.t_near) * inv_vs) - 1.0f, (float)k1);
                k = max(k, kn) + 1;
                prev_pending = true;
                continue;
            }
            if (!tri_value(p, cur, false)) { prev_pending = true; ++k; continue; }         // all 8 values > 0: not a candidate
            if (cur.known && !(cur.f > 0.0f)) {                                            // candidate: needs F_prev
                if (prev_pending) {
                    prev = tri_sample(p, dw, ow, vs, inv_vs, q.t_near, k - 1);
                    tri_value(p, prev, true);
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
