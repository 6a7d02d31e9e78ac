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
// their gathers share sectors.  Samples outside the volume are "unknown" and cannot produce a hit, so only the samples
// between the ray's entry into and exit from the volume's box (one sample of slack on both sides) are visited.
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
    float depth = 0.0f;
    if (ta <= tb) {
        const int k0 = max(0, (int)floorf((ta - q.t_near) * inv_vs) - 1);
        const int k1 = (int)fminf(ceilf((tb - q.t_near) * inv_vs) + 1.0f, 2.0e9f);
        float t_prev = 0.0f, f_prev = 0.0f;
        bool known_prev = false;
        for (int k = k0; k <= k1; ++k) {
            const float t = __fmaf_rn((float)k, vs, q.t_near);                                  // R2
            if (t > q.t_far) break;
            const float fi = floorf(__fmul_rn(__fsub_rn(__fmaf_rn(t, dw[0], ow[0]), org[0]), inv_vs));
            const float fj = floorf(__fmul_rn(__fsub_rn(__fmaf_rn(t, dw[1], ow[1]), org[1]), inv_vs));
            const float fk = floorf(__fmul_rn(__fsub_rn(__fmaf_rn(t, dw[2], ow[2]), org[2]), inv_vs));
            bool known = false; float f = 0.0f;
            if (fi >= 0.0f && fi < (float)p.nx && fj >= 0.0f && fj < (float)p.ny && fk >= 0.0f && fk < (float)p.nz) {
                const uint32_t word = __ldg(p.geo + ((size_t)(int)fk * (size_t)p.ny + (size_t)(int)fj) * (size_t)p.nx + (size_t)(int)fi);
                if ((word >> 16) != 0u) { known = true; f = (float)(int)(short)(word & 0xffffu); }  // R3
            }
            if (known && known_prev && f_prev > 0.0f && !(f > 0.0f)) {                          // R4
                depth = __fmaf_rn(vs, __fdiv_rn(f_prev, __fsub_rn(f_prev, f)), t_prev);
                break;
            }
            known_prev = known; t_prev = t; f_prev = f;
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

}  // namespace vf
