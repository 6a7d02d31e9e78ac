// prepass.cuh -- S1 (per-pixel map) and S9 (tile classification) kernels.
#pragma once
#include "params.cuh"

namespace vf {

// eq. 7: back-projection of depth pixel (x, y, D) with K_c^-1, canonical order
__device__ __forceinline__ float3 backproject(const Params &p, int x, int y, float D)
{
    float3 P;
    P.x = __fdiv_rn(__fmul_rn(__fsub_rn((float)x, p.cx), D), p.fx);
    P.y = __fdiv_rn(__fmul_rn(__fsub_rn((float)y, p.cy), D), p.fy);
    P.z = D;
    return P;
}

// K0 -- one CTA per 32 x 32 pixel region (256 threads x 4 rows).
//  (a) pixel map: everything of eq. 7-8 and the view weight (L110) depends only on the depth pixel, so it is computed
//      once per pixel instead of once per colour voxel: {X_vd, Y_vd, Z_vd, W}; W = 0 encodes "no colour update possible"
//      (invalid depth, missing forward neighbour (A7), degenerate normal, W <= 0 (A8)).
//  (b) min/max valid depth per 8x8, 16x16, 32x32 block (pyramid levels 0-2); the last CTA to finish builds the coarser
//      levels.  Thread 0 of CTA 0 also resets the per-frame work-list counters.
__global__ void __launch_bounds__(256) k_prepass(const __grid_constant__ Params p)
{
    __shared__ uint32_t s_mn[16], s_mx[16];
    __shared__ bool s_last;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    if (threadIdx.x < 16) { s_mn[threadIdx.x] = 0xffffu; s_mx[threadIdx.x] = 0u; }
    if (blockIdx.x == 0 && blockIdx.y == 0 && threadIdx.x == 0) {
        p.ctrl[CTRL_FRONT] = 0; p.ctrl[CTRL_BACK] = 0; p.ctrl[CTRL_CURSOR] = 0; p.ctrl[CTRL_BLOCKS_COL] = 0;
    }
    __syncthreads();
    const int x = blockIdx.x * 32 + tx;
#pragma unroll
    for (int m = 0; m < 4; ++m) {
        const int y = blockIdx.y * 32 + m * 8 + ty;
        uint32_t d0 = 0;
        if (x < p.wd && y < p.hd) {
            d0 = __ldg(p.depth + (size_t)y * p.wd + x);
            float4 out = make_float4(0.f, 0.f, 0.f, 0.f);
            if (d0 != 0) {
                const float D = __fmul_rn((float)d0, 0.001f);                      // mm -> m (A4)
                const float3 Pd = backproject(p, x, y, D);
                out.x = Pd.x; out.y = Pd.y; out.z = Pd.z;
                if (x + 1 < p.wd && y + 1 < p.hd) {
                    const uint32_t d1 = __ldg(p.depth + (size_t)y * p.wd + x + 1);
                    const uint32_t d2 = __ldg(p.depth + (size_t)(y + 1) * p.wd + x);
                    if (d1 != 0 && d2 != 0) {
                        const float3 P1 = backproject(p, x + 1, y, __fmul_rn((float)d1, 0.001f));
                        const float3 P2 = backproject(p, x, y + 1, __fmul_rn((float)d2, 0.001f));
                        const float ax = __fsub_rn(P1.x, Pd.x), ay = __fsub_rn(P1.y, Pd.y), az = __fsub_rn(P1.z, Pd.z);
                        const float bx = __fsub_rn(P2.x, Pd.x), by = __fsub_rn(P2.y, Pd.y), bz = __fsub_rn(P2.z, Pd.z);
                        const float nx = __fmaf_rn(ay, bz, -__fmul_rn(az, by));       // eq. 8
                        const float ny = __fmaf_rn(az, bx, -__fmul_rn(ax, bz));
                        const float nz = __fmaf_rn(ax, by, -__fmul_rn(ay, bx));
                        const float dot = __fmaf_rn(nz, Pd.z, __fmaf_rn(ny, Pd.y, __fmul_rn(nx, Pd.x)));
                        const float nn = __fmaf_rn(nz, nz, __fmaf_rn(ny, ny, __fmul_rn(nx, nx)));
                        const float pp = __fmaf_rn(Pd.z, Pd.z, __fmaf_rn(Pd.y, Pd.y, __fmul_rn(Pd.x, Pd.x)));
                        const float den = __fsqrt_rn(__fmul_rn(nn, pp));
                        if (den > 0.0f) {
                            const float W = fminf(1.0f, __fdiv_rn(dot, den));         // L110, A8
                            if (W > 0.0f) out.w = W;
                        }
                    }
                }
            }
            p.pixmap[(size_t)y * p.wd + x] = out;
        }
        // min / max over the 8-pixel run of this row that lies in one level-0 block, then one shared atomic per run
        uint32_t mn = d0 ? d0 : 0xffffu, mx = d0;
#pragma unroll
        for (int o = 1; o < 8; o <<= 1) {
            mn = min(mn, __shfl_xor_sync(0xffffffffu, mn, o));
            mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, o));
        }
        if ((tx & 7) == 0) { atomicMin(&s_mn[m * 4 + (tx >> 3)], mn); atomicMax(&s_mx[m * 4 + (tx >> 3)], mx); }
    }
    __syncthreads();
    // level 0: 4 x 4 entries, level 1: 2 x 2, level 2: 1
    const int t = threadIdx.x;
    if (t < 16) {
        const int bx = blockIdx.x * 4 + (t & 3), by = blockIdx.y * 4 + (t >> 2);
        if (bx < p.pyr_w[0] && by < p.pyr_h[0]) p.pyr[p.pyr_off[0] + by * p.pyr_w[0] + bx] = s_mn[t] | (s_mx[t] << 16);
    } else if (t < 20 && p.pyr_levels > 1) {
        const int q = t - 16, qx = q & 1, qy = q >> 1;
        uint32_t mn = 0xffffu, mx = 0u;
        for (int a = 0; a < 2; ++a) for (int b = 0; b < 2; ++b) {
            mn = min(mn, s_mn[(qy * 2 + a) * 4 + qx * 2 + b]); mx = max(mx, s_mx[(qy * 2 + a) * 4 + qx * 2 + b]);
        }
        const int bx = blockIdx.x * 2 + qx, by = blockIdx.y * 2 + qy;
        if (bx < p.pyr_w[1] && by < p.pyr_h[1]) p.pyr[p.pyr_off[1] + by * p.pyr_w[1] + bx] = mn | (mx << 16);
    } else if (t == 20 && p.pyr_levels > 2) {
        uint32_t mn = 0xffffu, mx = 0u;
        for (int a = 0; a < 16; ++a) { mn = min(mn, s_mn[a]); mx = max(mx, s_mx[a]); }
        p.pyr[p.pyr_off[2] + blockIdx.y * p.pyr_w[2] + blockIdx.x] = mn | (mx << 16);
    }
    if (p.pyr_levels <= 3) return;
    // the last CTA to arrive reduces level 2 into levels 3.. (each level halves both dimensions)
    __threadfence();
    __syncthreads();
    if (t == 0) {
        const uint32_t n = gridDim.x * gridDim.y;
        s_last = (atomicAdd(&p.ctrl[CTRL_TICKET], 1u) == n - 1u);
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    for (int l = 3; l < p.pyr_levels; ++l) {
        const int w = p.pyr_w[l], h = p.pyr_h[l], pw = p.pyr_w[l - 1], ph = p.pyr_h[l - 1];
        const uint32_t *src = p.pyr + p.pyr_off[l - 1];
        for (int e = t; e < w * h; e += blockDim.x) {
            const int ex = e % w, ey = e / w;
            uint32_t mn = 0xffffu, mx = 0u;
            for (int a = 0; a < 2; ++a) for (int b = 0; b < 2; ++b) {
                const int sx = ex * 2 + b, sy = ey * 2 + a;
                if (sx < pw && sy < ph) { const uint32_t v = __ldcg(src + sy * pw + sx); mn = min(mn, v & 0xffffu); mx = max(mx, v >> 16); }
            }
            p.pyr[p.pyr_off[l] + e] = mn | (mx << 16);
        }
        __threadfence();
        __syncthreads();
    }
    if (t == 0) p.ctrl[CTRL_TICKET] = 0;
}

// K1 -- S9: one thread per geometry tile of this shard.  Conservative test against the depth pyramid; surviving tiles go
// to the work list: tiles whose colour children may pass the sigma gate (heavier) from the front, geometry-only tiles
// from the back, so the fused kernel pops the heavy items first.
__global__ void __launch_bounds__(256) k_classify(const __grid_constant__ Params p)
{
    const int tile = blockIdx.x * blockDim.x + threadIdx.x;
    uint32_t flags = 0;
    if (tile < p.n_tiles) {
        const int ttx = tile % p.tiles_x, tty = (tile / p.tiles_x) % p.tiles_y, ttz = tile / (p.tiles_x * p.tiles_y);
        const int gz = local_to_global_tz(p, ttz);
        // tile box centre in world, then camera space (culling only: plain arithmetic with slack in tile_e*)
        const float wx = p.ox + ((float)(ttx * TX) + 0.5f * (float)TX) * p.vs;
        const float wy = p.oy + ((float)(tty * TY) + 0.5f * (float)TY) * p.vs;
        const float wz = p.oz + ((float)(gz * TZ) + 0.5f * (float)TZ) * p.vs;
        const float cX = p.R[0] * wx + p.R[1] * wy + p.R[2] * wz + p.t[0];
        const float cY = p.R[3] * wx + p.R[4] * wy + p.R[5] * wz + p.t[1];
        const float cZ = p.R[6] * wx + p.R[7] * wy + p.R[8] * wz + p.t[2];
        int x0, x1, y0, y1; float zmin, zmax;
        if (box_rect(p, cX, cY, cZ, p.tile_ex, p.tile_ey, p.tile_ez, x0, x1, y0, y1, zmin, zmax)) {
            uint32_t mn, mx;
            depth_range(p, x0, x1, y0, y1, mn, mx);
            if (mx != 0u) {
                const float dmin = (float)mn * 0.001f - 1e-4f, dmax = (float)mx * 0.001f + 1e-4f;
                if (zmin <= dmax + p.mu) flags |= ITEM_GEO;                          // sdf >= -mu possible
                if (zmin <= dmax + p.sigma && zmax >= dmin - p.sigma) flags |= ITEM_COL;   // |Z - Z_vd| <= sigma possible
            }
        }
    }
    // warp-aggregated append
    const unsigned lane = threadIdx.x & 31;
    const unsigned mcol = __ballot_sync(0xffffffffu, (flags & ITEM_COL) != 0u);
    const unsigned mgeo = __ballot_sync(0xffffffffu, flags != 0u && (flags & ITEM_COL) == 0u);
    uint32_t bf = 0, bb = 0;
    if (lane == 0) {
        if (mcol) bf = atomicAdd(&p.ctrl[CTRL_FRONT], (uint32_t)__popc(mcol));
        if (mgeo) bb = atomicAdd(&p.ctrl[CTRL_BACK], (uint32_t)__popc(mgeo));
    }
    bf = __shfl_sync(0xffffffffu, bf, 0); bb = __shfl_sync(0xffffffffu, bb, 0);
    const unsigned lt = (1u << lane) - 1u;
    if (flags & ITEM_COL) p.work[bf + __popc(mcol & lt)] = (uint32_t)tile | flags;
    else if (flags) p.work[(uint32_t)p.n_tiles - 1u - (bb + __popc(mgeo & lt))] = (uint32_t)tile | flags;
}

}  // namespace vf
