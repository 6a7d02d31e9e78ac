// prepass.cuh -- S1 (per-pixel map, depth pyramid, shell-mark jobs: kernel k_prepass) and the producer roles of the fused
// kernel: S9 for geometry (classification of tiles and their sub-boxes), the shell marks (S1 continued) and S9 for colour
// (work items from the marks).
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

// culling only: set the mark bits of every colour cell that intersects the colour-voxel index box
// [i0,i1] x [j0,j1] x [k0,k1] (inclusive, already clamped to the colour grid).  The cell layers (cz) of the box are dealt
// round-robin to `nsub` cooperating lanes; this lane is number `sub`.  Per (cell layer, tile) the rows of the box form
// one contiguous run of at most 4 r^2 <= 64 mark bits, which never spans more than two words: one or two
// fire-and-forget reductions (no return value, so a lane never waits on the L2 round trip).
// (Testing every cell of the box against the piece itself marks 16 % fewer cells on config 3 but costs the marking more
// than it saves the fused kernel: measured, not used.)
// A box of more than MARK_FINE_MAX cells is marked tile by tile instead (all cells of every tile it meets): bounded work
// for pathological frames, at the price of looser marks.
constexpr int MARK_FINE_MAX = 8192;

template <int R>
__device__ __forceinline__ void mark_box(const Params &p, int i0, int i1, int j0, int j1, int k0, int k1, int sub, int nsub)
{
    constexpr int CX = cells_x(R), CY = cells_y(R), CZ = cells_z(R), NC = cells_per_tile(R), WPT = words_per_tile(R);
    const int cx0 = i0 / CLX, cx1 = i1 / CLX, cy0 = j0 / CLY, cy1 = j1 / CLY, cz0 = k0 / CLZ, cz1 = k1 / CLZ;
    const int tx0 = cx0 / CX, tx1 = cx1 / CX, ty0 = cy0 / CY, ty1 = cy1 / CY;
    if ((cx1 - cx0 + 1) * (cy1 - cy0 + 1) * (cz1 - cz0 + 1) > MARK_FINE_MAX) {
        for (int gz = cz0 / CZ + sub; gz <= cz1 / CZ; gz += nsub) {
            if (gz % p.shard_world != p.shard_rank) continue;
            const int tzl = gz / p.shard_world;
            for (int tty = ty0; tty <= ty1; ++tty)
                for (int ttx = tx0; ttx <= tx1; ++ttx) {
                    uint32_t *w = p.marks + (size_t)((tzl * p.tiles_y + tty) * p.tiles_x + ttx) * WPT;
#pragma unroll
                    for (int k = 0; k < WPT; ++k) atomicOr(w + k, (k + 1) * 32 <= NC ? 0xffffffffu : (1u << (NC & 31)) - 1u);
                }
        }
        return;
    }
    for (int cz = cz0 + sub; cz <= cz1; cz += nsub) {
        const int gz = cz / CZ, czin = cz - gz * CZ;
        if (gz % p.shard_world != p.shard_rank) continue;
        const int tzl = gz / p.shard_world;
        for (int tty = ty0; tty <= ty1; ++tty) {
            const int la = max(cy0, tty * CY) - tty * CY, lb = min(cy1, tty * CY + CY - 1) - tty * CY;
            for (int ttx = tx0; ttx <= tx1; ++ttx) {
                const int a = max(cx0, ttx * CX) - ttx * CX, b = min(cx1, ttx * CX + CX - 1) - ttx * CX;
                const unsigned long long row = (1ull << (b - a + 1)) - 1ull;
                const int bit0 = (czin * CY + la) * CX + a;
                unsigned long long m = 0ull;
                for (int cy = la; cy <= lb; ++cy) m |= row << ((bit0 & 31) + (cy - la) * CX);
                uint32_t *w = p.marks + (size_t)((tzl * p.tiles_y + tty) * p.tiles_x + ttx) * WPT + (bit0 >> 5);
                const uint32_t lo = (uint32_t)m, hi = (uint32_t)(m >> 32);
                if (lo) atomicOr(w, lo);
                if (hi) atomicOr(w + 1, hi);
            }
        }
    }
}

// culling only: world interval [lo, hi] grown by g -> inclusive colour-voxel index range of the voxel CENTRES inside it.
__device__ __forceinline__ bool index_box(const Params &p, float lo, float hi, float g, float o, int n, int &a, int &b)
{
    const float fa = fmaxf(((lo - g) - o) * p.inv_vc - 0.5f, -1.0f);
    const float fb = fminf(((hi + g) - o) * p.inv_vc - 0.5f, (float)n);
    a = max(0, (int)floorf(fa)); b = min(n - 1, (int)ceilf(fb));
    return a <= b;
}

// culling only: a colour voxel passes the sigma gate (L108) of pixel (x, y) only if (i) it projects onto that pixel,
// i.e. X/Z and Y/Z lie inside the pixel's footprint, and (ii) it is within sigma of the pixel's depth point, hence
// |Z - Z_vd| <= sigma.  For a rectangle of pixels [xa, xb] x [ya, yb] whose eligible depths span [zmin, zmax] that set is
// inside the frustum piece {(a Z, b Z, Z)}: a, b over the footprint (grown by 0.01 px against fp32 rounding of eq. 6),
// Z in [zmin - sigma, zmax + sigma].  The piece is convex, so its world-space bounding box is that of its 8 corners.
// Returns the inclusive colour-voxel index box of the centres inside it (false if empty).
__device__ __forceinline__ bool shell_box(const Params &p, float xa, float xb, float ya, float yb, float zmin, float zmax,
                                          int &i0, int &i1, int &j0, int &j1, int &k0, int &k1)
{
    const float a0 = ((xa - 0.51f) - p.cx) / p.fx, a1 = ((xb + 0.51f) - p.cx) / p.fx;
    const float b0 = ((ya - 0.51f) - p.cy) / p.fy, b1 = ((yb + 0.51f) - p.cy) / p.fy;
    const float z0 = fmaxf(zmin - p.sigma_g, 1e-6f), z1 = zmax + p.sigma_g;
    float lo[3], hi[3];
#pragma unroll
    for (int ax = 0; ax < 3; ++ax) {
        const float ra = p.Rw[3 * ax], rb = p.Rw[3 * ax + 1], rc = p.Rw[3 * ax + 2];
        // direction of the four edge rays; world coordinate = tw + Z * d
        const float d00 = ra * a0 + rb * b0 + rc, d10 = ra * a1 + rb * b0 + rc, d01 = ra * a0 + rb * b1 + rc, d11 = ra * a1 + rb * b1 + rc;
        const float dmin = fminf(fminf(d00, d10), fminf(d01, d11)), dmax = fmaxf(fmaxf(d00, d10), fmaxf(d01, d11));
        lo[ax] = p.tw[ax] + fminf(dmin * z0, dmin * z1);
        hi[ax] = p.tw[ax] + fmaxf(dmax * z0, dmax * z1);
    }
    const float s = p.slack * (1.0f + z1);
    return index_box(p, lo[0], hi[0], s, p.ox, p.cnx, i0, i1) && index_box(p, lo[1], hi[1], s, p.oy, p.cny, j0, j1) &&
           index_box(p, lo[2], hi[2], s, p.oz, p.cnz, k0, k1);
}

// K0 -- one CTA per 32 x 32 pixel region; thread (tx, tq) owns pixels (x = tx, y = 4 tq + m), m = 0..3.
//  (a) pixel map: everything of eq. 7-8 and the view weight (L110) depends only on the depth pixel, so it is computed
//      once per pixel instead of once per colour voxel: {X_vd, Y_vd, Z_vd, W}; W = 0 encodes "no colour update possible"
//      (invalid depth, missing forward neighbour (A7), degenerate normal, W <= 0 (A8)).
//      Beside it the depth in metres as a float map (what the TSDF update gathers).
//  (b) min/max valid depth per 8x8, 16x16, 32x32 block (pyramid levels 0-2) and of the whole frame (two atomics per CTA).
//      Used to cull geometry tiles.
//  (c) shell-mark jobs: a colour voxel can pass the sigma gate (L108) only inside the frustum piece of shell_box().  Every
//      4 x 4 pixel patch queues the world-space bounding box of its piece as ONE job if that box is at most PATCH_SPREAD_MAX x
//      larger than a compact piece's (a smooth surface seen head-on).  Otherwise the patch is cut into its 4 rows or its 4
//      columns, whichever have the smaller depth ranges (a surface seen at a grazing angle: the pieces of the strips are
//      staggered along the view direction, and their boxes follow the shear that one box for the patch would fill in) --
//      or, if even those ranges exceed STRIP_RANGE_MAX (a depth edge), into its pixels.  (With a sigma so large that even a compact
//      patch's box spans more than MARK_FINE_MAX cells, the patches of a CTA's 32 x 32 region are merged into one job.)
//      The fused kernel's warps turn the jobs into marks: bits of the colour cells that meet a job's box.  Marks are
//      consumed (and cleared) by the fused kernel.
constexpr float PATCH_SPREAD_MAX = 2.4f, STRIP_RANGE_MAX = 0.02f;
enum { JOB_PATCH = 0, JOB_ROW = 1, JOB_COLUMN = 2, JOB_PIXEL = 3 };      // bits 31:30 of a job's first word: the pixels it covers

template <int R>
__global__ void __launch_bounds__(256) k_prepass(const __grid_constant__ Params p)
{
    __shared__ uint32_t s_mn[16], s_mx[16];
    __shared__ uint32_t s_njobs, s_base, s_rlo, s_rhi;      // s_rlo / s_rhi: depth range (float bits) of the region job, see (c)
    __shared__ uint4 s_jobs[1024];      // mark jobs: {x | y << 15 | JOB_* << 30 of the first pixel, depth range of its eligible pixels}
    const int t = threadIdx.x, tx = t & 31, tq = t >> 5;
    pdl_launch_dependents();
    if (t < 16) { s_mn[t] = 0xffffu; s_mx[t] = 0u; }
    if (t == 0) { s_njobs = 0u; s_rlo = 0x7f800000u; s_rhi = 0u; }
    // the control block of the NEXT frame starts at zero ("no valid depth yet" for the minimum); this frame's was cleared by the
    // pre-pass before it (params.cuh, CTRL_SETS)
    if (blockIdx.x == 0 && blockIdx.y == 0)
        for (int i = t; i < CTRL_N; i += 256) p.ctrl_next[i] = i == Q_DMIN ? 0xffffu : 0u;
    __syncthreads();
    const int x = blockIdx.x * 32 + tx;
    uint32_t mn = 0xffffu, mx = 0u;
    float zpx[4];                             // depths of this thread's colour-eligible pixels (0 = not eligible)
    // all twelve depth loads of the thread are issued first (the frame has just arrived: they come from DRAM); a missing
    // forward neighbour reads as 0 = invalid, which is what reading A7 makes of it
    uint32_t dd0[4], dd1[4], dd2[4];
#pragma unroll
    for (int m = 0; m < 4; ++m) {
        const int y = blockIdx.y * 32 + tq * 4 + m;
        const bool in = x < p.wd && y < p.hd;
        dd0[m] = in ? __ldg(p.depth + (size_t)y * p.wd + x) : 0u;
        dd1[m] = in && x + 1 < p.wd && y + 1 < p.hd ? __ldg(p.depth + (size_t)y * p.wd + x + 1) : 0u;
        dd2[m] = in && x + 1 < p.wd && y + 1 < p.hd ? __ldg(p.depth + (size_t)(y + 1) * p.wd + x) : 0u;
    }
#pragma unroll
    for (int m = 0; m < 4; ++m) {
        const int y = blockIdx.y * 32 + tq * 4 + m;
        zpx[m] = 0.0f;
        if (x < p.wd && y < p.hd) {
            const uint32_t d0 = dd0[m];
            float4 out = make_float4(0.f, 0.f, 0.f, 0.f);
            if (d0 != 0) {
                mn = min(mn, d0); mx = max(mx, d0);
                const float D = __fmul_rn((float)d0, 0.001f);                      // mm -> m (A4)
                const float3 Pd = backproject(p, x, y, D);
                out.x = Pd.x; out.y = Pd.y; out.z = Pd.z;
                {
                    const uint32_t d1 = dd1[m], d2 = dd2[m];
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
                if (out.w > 0.0f) zpx[m] = D;
            }
            p.pixmap[(size_t)y * p.wd + x] = out;
            p.depthf[(size_t)y * p.wd + x] = out.z;                              // D, or 0 = invalid
        }
    }
    {   // (c) every 4 x 4 patch = 4 lanes x the thread's 4 rows.  All shuffles are executed by the whole warp.
        float zlo = 1e30f, zhi = -1e30f;
#pragma unroll
        for (int m = 0; m < 4; ++m) if (zpx[m] > 0.0f) { zlo = fminf(zlo, zpx[m]); zhi = fmaxf(zhi, zpx[m]); }
#pragma unroll
        for (int o = 1; o < 4; o <<= 1) {
            zlo = fminf(zlo, __shfl_xor_sync(0xffffffffu, zlo, o));
            zhi = fmaxf(zhi, __shfl_xor_sync(0xffffffffu, zhi, o));
        }
        // depth ranges of the patch's rows (over the 4 lanes) and of its columns (this lane's 4 pixels)
        float rlo[4], rhi[4], clo = 1e30f, chi = -1e30f;
#pragma unroll
        for (int m = 0; m < 4; ++m) {
            rlo[m] = zpx[m] > 0.0f ? zpx[m] : 1e30f; rhi[m] = zpx[m] > 0.0f ? zpx[m] : -1e30f;
            clo = fminf(clo, rlo[m]); chi = fmaxf(chi, rhi[m]);
#pragma unroll
            for (int o = 1; o < 4; o <<= 1) {
                rlo[m] = fminf(rlo[m], __shfl_xor_sync(0xffffffffu, rlo[m], o));
                rhi[m] = fmaxf(rhi[m], __shfl_xor_sync(0xffffffffu, rhi[m], o));
            }
        }
        float rmax = 0.0f, cmax = chi >= clo ? chi - clo : 0.0f;
#pragma unroll
        for (int m = 0; m < 4; ++m) if (rhi[m] >= rlo[m]) rmax = fmaxf(rmax, rhi[m] - rlo[m]);
#pragma unroll
        for (int o = 1; o < 4; o <<= 1) cmax = fmaxf(cmax, __shfl_xor_sync(0xffffffffu, cmax, o));
        if (zlo <= zhi) {
            const int xp = blockIdx.x * 32 + (tx & ~3), yp = blockIdx.y * 32 + tq * 4;
            int i0, i1, j0, j1, k0, k1;
            if (shell_box(p, (float)xp, (float)(xp + 3), (float)yp, (float)(yp + 3), zlo, zhi, i0, i1, j0, j1, k0, k1)) {
                const int ncell = (i1 / CLX - i0 / CLX + 1) * (j1 / CLY - j0 / CLY + 1) * (k1 / CLZ - k0 / CLZ + 1);
                // a compact piece (smooth surface seen head-on) spans about n0 cells: 2 sigma deep, the patch's footprint wide
                const float c = (float)CLY * p.vc, wfoot = 4.0f * zhi / p.fx;
                const float n0 = (2.0f * p.sigma / c + 2.0f) * (wfoot / c + 2.0f) * (0.5f * wfoot / c + 2.0f);
                const uint32_t xy = (uint32_t)xp | ((uint32_t)yp << 15);
                if (n0 > (float)MARK_FINE_MAX) {
                    // sigma is so large that even a compact patch's box spans thousands of cells (mark_box then works tile
                    // by tile): the boxes of neighbouring patches are nearly the same, and the CTA's whole 32 x 32 region
                    // becomes ONE job with the union of their depth ranges (positive floats order like their bit patterns)
                    if ((tx & 3) == 0) { atomicMin(&s_rlo, __float_as_uint(zlo)); atomicMax(&s_rhi, __float_as_uint(zhi)); }
                } else if ((float)ncell <= PATCH_SPREAD_MAX * n0) {
                    if ((tx & 3) == 0) s_jobs[atomicAdd(&s_njobs, 1u)] = make_uint4(xy | ((uint32_t)JOB_PATCH << 30), __float_as_uint(zlo), __float_as_uint(zhi), 0u);
                } else if (fminf(rmax, cmax) <= STRIP_RANGE_MAX) {
                    if (rmax <= cmax) {                               // rows: lane m of the patch queues row m
                        const int m = tx & 3;
                        const float lo = m == 0 ? rlo[0] : m == 1 ? rlo[1] : m == 2 ? rlo[2] : rlo[3];
                        const float hi = m == 0 ? rhi[0] : m == 1 ? rhi[1] : m == 2 ? rhi[2] : rhi[3];
                        if (lo <= hi)
                            s_jobs[atomicAdd(&s_njobs, 1u)] = make_uint4((uint32_t)xp | ((uint32_t)(yp + m) << 15) | ((uint32_t)JOB_ROW << 30), __float_as_uint(lo), __float_as_uint(hi), 0u);
                    } else if (clo <= chi) {                          // columns: every lane queues its own
                        s_jobs[atomicAdd(&s_njobs, 1u)] = make_uint4((uint32_t)x | ((uint32_t)yp << 15) | ((uint32_t)JOB_COLUMN << 30), __float_as_uint(clo), __float_as_uint(chi), 0u);
                    }
                } else {
#pragma unroll
                    for (int m = 0; m < 4; ++m)
                        if (zpx[m] > 0.0f)
                            s_jobs[atomicAdd(&s_njobs, 1u)] = make_uint4((uint32_t)x | ((uint32_t)(yp + m) << 15) | ((uint32_t)JOB_PIXEL << 30), __float_as_uint(zpx[m]), __float_as_uint(zpx[m]), 0u);
                }
            }
        }
    }
    __syncthreads();
    if (t == 0 && s_rhi >= s_rlo && s_rhi != 0u)             // the region job: fourth word = 1
        s_jobs[s_njobs++] = make_uint4((uint32_t)(blockIdx.x * 32) | ((uint32_t)(blockIdx.y * 32) << 15) | ((uint32_t)JOB_PATCH << 30), s_rlo, s_rhi, 1u);
    __syncthreads();
    {   // append this CTA's jobs to the frame's queue (one reservation per CTA)
        const uint32_t njobs = s_njobs;
        if (t == 0) s_base = njobs ? atomicAdd(&p.ctrl[Q_NJOBS], njobs) : 0u;
        __syncthreads();
        for (uint32_t j = (uint32_t)t; j < njobs; j += 256u)
            if (s_base + j < p.jobs_cap) p.jobs[s_base + j] = s_jobs[j];       // (always true: at most one job per pixel)
    }
    // (b) level-0 block = 8 lanes x 2 threads-rows (tq pair)
#pragma unroll
    for (int o = 1; o < 8; o <<= 1) {
        mn = min(mn, __shfl_xor_sync(0xffffffffu, mn, o));
        mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    }
    if ((tx & 7) == 0) { atomicMin(&s_mn[(tq >> 1) * 4 + (tx >> 3)], mn); atomicMax(&s_mx[(tq >> 1) * 4 + (tx >> 3)], mx); }
    __syncthreads();
    // level 0: 4 x 4 entries, level 1: 2 x 2, level 2: 1
    if (t < 16) {
        const int bx = blockIdx.x * 4 + (t & 3), by = blockIdx.y * 4 + (t >> 2);
        if (bx < p.pyr_w[0] && by < p.pyr_h[0]) p.pyr[p.pyr_off[0] + by * p.pyr_w[0] + bx] = s_mn[t] | (s_mx[t] << 16);
    } else if (t < 20 && p.pyr_levels > 1) {
        const int q = t - 16, qx = q & 1, qy = q >> 1;
        uint32_t a_mn = 0xffffu, a_mx = 0u;
        for (int a = 0; a < 2; ++a) for (int b = 0; b < 2; ++b) {
            a_mn = min(a_mn, s_mn[(qy * 2 + a) * 4 + qx * 2 + b]); a_mx = max(a_mx, s_mx[(qy * 2 + a) * 4 + qx * 2 + b]);
        }
        const int bx = blockIdx.x * 2 + qx, by = blockIdx.y * 2 + qy;
        if (bx < p.pyr_w[1] && by < p.pyr_h[1]) p.pyr[p.pyr_off[1] + by * p.pyr_w[1] + bx] = a_mn | (a_mx << 16);
    } else if (t == 20) {
        uint32_t a_mn = 0xffffu, a_mx = 0u;
        for (int a = 0; a < 16; ++a) { a_mn = min(a_mn, s_mn[a]); a_mx = max(a_mx, s_mx[a]); }
        if (p.pyr_levels > 2) p.pyr[p.pyr_off[2] + blockIdx.y * p.pyr_w[2] + blockIdx.x] = a_mn | (a_mx << 16);
        if (a_mx != 0u) { atomicMin(&p.ctrl[Q_DMIN], a_mn); atomicMax(&p.ctrl[Q_DMAX], a_mx); }
    }
    // This kernel is itself a programmatic dependent launch: it reads only the frame and writes only this frame's scratch set
    // and control block, so its CTAs may run beside the last warps of the previous frame's fused kernel.  It must not
    // COMPLETE before that kernel has, though: this frame's fused kernel waits for this grid alone, and it works on the
    // volumes and the work lists the previous one is still using.
    pdl_wait();
}

// camera-space centre of geometry tile (ttx, tty, ttz local) -- culling only
__device__ __forceinline__ void tile_centre(const Params &p, int ttx, int tty, int ttz, float &cX, float &cY, float &cZ)
{
    const int gz = local_to_global_tz(p, ttz);
    const float wx = p.ox + ((float)(ttx * TX) + 0.5f * (float)TX) * p.vs;
    const float wy = p.oy + ((float)(tty * TY) + 0.5f * (float)TY) * p.vs;
    const float wz = p.oz + ((float)(gz * TZ) + 0.5f * (float)TZ) * p.vs;
    cX = p.R[0] * wx + p.R[1] * wy + p.R[2] * wz + p.t[0];
    cY = p.R[3] * wx + p.R[4] * wy + p.R[5] * wz + p.t[1];
    cZ = p.R[6] * wx + p.R[7] * wy + p.R[8] * wz + p.t[2];
}

// is this geometry tile NEAR: does its box come within 2 mm of the camera plane (or behind it)?  Its voxels may then have
// Z <= 0 or Z outside the range of the branch-free reciprocal, and the fused kernel takes the plain per-voxel routines.
// Evaluated identically by the classification and by the consumers of geometry and colour items.
__device__ __forceinline__ bool tile_is_near(const Params &p, int ttx, int tty, int ttz)
{
    float cX, cY, cZ;
    tile_centre(p, ttx, tty, ttz, cX, cY, cZ);
    return !(cZ - p.tile_ez > 2e-3f);
}

// culling only: can any voxel of the camera-space box (centre c, half extents e) pass the TSDF tests (frustum, valid
// depth, sdf >= -mu)?  Conservative: max valid depth over the box's pixel rectangle against the box's nearest Z.
// Returns 0 = no, 1 = maybe, 2 = maybe and the whole box lies in front of every valid depth of its rectangle (free space:
// a finer look at the box would find the same), 3 = ... by more than mu: every voxel of the box that is updated at all gets
// tsdf = 1 exactly (sdf >= mu + 0.1 mm, against the slack of this fp32 evaluation and the rounding of sdf / mu).
__device__ __forceinline__ int box_may_update(const Params &p, float cX, float cY, float cZ, float eX, float eY, float eZ)
{
    int x0, x1, y0, y1; float zmin, zmax;
    if (!box_rect(p, cX, cY, cZ, eX, eY, eZ, x0, x1, y0, y1, zmin, zmax)) return 0;
    uint32_t mn, mx;
    depth_range(p, x0, x1, y0, y1, mn, mx);
    if (mx == 0u || !(zmin <= ((float)mx * 0.001f + 1e-4f) + p.mu)) return 0;
    const float dmin = (float)mn * 0.001f - 1e-4f;
    return zmax <= dmin ? (zmax + p.mu * 1.0001f + 1e-4f <= dmin ? 3 : 2) : 1;
}

// The three producer roles of the fused kernel.  Each is one CHUNK of work for one warp; chunks are claimed from counters
// in ctrl[], so every warp of the grid helps and nobody ever waits for work that has not been claimed.

// S9 for geometry, 32 tiles of this shard, one lane per tile: conservative test of the tile's
// camera-space box against the depth pyramid (any voxel with sdf >= -mu?).  Tiles that pass are refined on their
// SUBX x 1 x SUBZ sub-boxes, 8 lanes per tile, and appended to the geometry work list together with the mask of the sub-boxes
// that passed (warp-aggregated reservation).  The item is published by the store itself: a consumer polls its slot.
__device__ __forceinline__ void classify_chunk(const Params &p, uint32_t chunk, int lane)
{
    // lane l takes tile chunk + l * n_chunks: a sample spread over the whole volume, so that the tiles near the surface
    // (whose sub-boxes have to be looked at) are dealt evenly to the chunks
    const int tile = (int)chunk + lane * ((p.n_tiles + CLS_CHUNK - 1) / CLS_CHUNK);
    int ttx = 0, tty = 0, ttz = 0, coarse = 0;
    float cX = 0.f, cY = 0.f, cZ = 0.f;
    bool near = false;
    if (tile < p.n_tiles) {
        ttx = tile % p.tiles_x; tty = (tile / p.tiles_x) % p.tiles_y; ttz = tile / (p.tiles_x * p.tiles_y);
        tile_centre(p, ttx, tty, ttz, cX, cY, cZ);
        near = !(cZ - p.tile_ez > 2e-3f);
        coarse = box_may_update(p, cX, cY, cZ, p.tile_ex, p.tile_ey, p.tile_ez);
    }
    unsigned surv = __ballot_sync(0xffffffffu, coarse != 0);
    uint32_t mask = 0u, free3 = 0u;                  // sub-boxes to visit; sub-boxes in free space by more than mu
    const float sx = (float)(TX / SUBX) * p.vs, sz = (float)(TZ / SUBZ) * p.vs;
    const int sb = lane & 7, bx = sb / SUBZ, bz = sb % SUBZ;        // item mask bit = bx * SUBZ + bz
    const float dx = ((float)bx - 0.5f * (float)(SUBX - 1)) * sx, dz = ((float)bz - 0.5f * (float)(SUBZ - 1)) * sz;
    while (surv) {                                   // four survivors at a time: lane = (survivor, sub-box)
        int src[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) { src[k] = surv ? __ffs(surv) - 1 : -1; surv &= surv - 1u; }
        const int mine = src[lane >> 3];
        const float sX = __shfl_sync(0xffffffffu, cX, mine & 31), sY = __shfl_sync(0xffffffffu, cY, mine & 31), sZ = __shfl_sync(0xffffffffu, cZ, mine & 31);
        const int cls = mine < 0 ? 0 : box_may_update(p, sX + p.R[0] * dx + p.R[2] * dz, sY + p.R[3] * dx + p.R[5] * dz,
                                                      sZ + p.R[6] * dx + p.R[8] * dz, p.sub_ex, p.sub_ey, p.sub_ez);
        const unsigned b = __ballot_sync(0xffffffffu, cls != 0), b3 = __ballot_sync(0xffffffffu, cls == 3);
#pragma unroll
        for (int k = 0; k < 4; ++k) if (lane == src[k]) { mask = (b >> (8 * k)) & 0xffu; free3 = (b3 >> (8 * k)) & 0xffu; }
    }
    // a partial last slab: sub-boxes whose first layer lies beyond the volume are not queued at all
    if (local_to_global_tz(p, ttz) * TZ + TZ / SUBZ >= p.nz) mask &= 0x55u;
    if (near && mask) mask = 0xffu;                  // NEAR tiles are processed whole, by the plain routines
    else if (mask) {
        // saturated free space stays what it is: (32767 w_max + 32767) / (w_max + 1) = 32767 exactly, w = min(w_max + 1, w_max)
        const uint32_t skip = mask & free3 & (uint32_t)p.tile_sat[tile];
        if (p.counting) p.tile_skip[tile] = (uint8_t)skip; else mask &= ~skip;
    }
    // For the ray caster (raycast.cuh): a voxel can only receive tsdf <= 0 in a visited tile that is NOT wholly in front of
    // every depth it can see (in front by >= 0.1 mm, mu <= 1 m: every new sample is >= 3 q-units, so the running average of
    // positive values stays >= 1).  Flag those tiles and their bricks; flags are only ever set (vol_reset clears them,
    // vol_upload sets all): a conservative superset.
    const bool behind = coarse == 1 || (coarse == 2 && !(p.mu <= 1.0f));
    if (mask && behind) {
        p.tile_neg[tile] = 1; p.brick_neg[((ttz / 4) * p.bricks_y + tty / 8) * p.bricks_x + ttx] = 1;
    }
    const unsigned mg = __ballot_sync(0xffffffffu, mask != 0u), lt = (1u << lane) - 1u;
    uint32_t bg = 0;
    if (lane == 0 && mg) bg = atomicAdd(&p.ctrl[ST_NGEO], (uint32_t)__popc(mg));
    bg = __shfl_sync(0xffffffffu, bg, 0);
    if (mask) __stcg(p.work_geo + bg + __popc(mg & lt), item_pack(ttx, tty, ttz, (int)mask));
}

// S1 (c) continued: mark jobs [8 chunk, 8 chunk + 8), 4 lanes per job; the 4 lanes share the job's cell layers.
template <int R>
__device__ __forceinline__ void mark_chunk(const Params &p, uint32_t chunk, uint32_t njobs, int lane)
{
    const uint32_t j = chunk * MARK_CHUNK + ((uint32_t)lane >> 2);
    if (j >= njobs) return;
    const uint4 job = __ldcg(p.jobs + j);
    const float xa = (float)(job.x & 0x7fffu), ya = (float)((job.x >> 15) & 0x7fffu);
    const uint32_t shape = job.x >> 30;
    float ex = shape == JOB_PATCH || shape == JOB_ROW ? 3.0f : 0.0f, ey = shape == JOB_PATCH || shape == JOB_COLUMN ? 3.0f : 0.0f;
    if (job.w != 0u) { ex = fminf(31.0f, p.wd_f - 1.0f - xa); ey = fminf(31.0f, p.hd_f - 1.0f - ya); }      // a CTA's 32 x 32 region (k_prepass)
    int i0, i1, j0, j1, k0, k1;
    if (shell_box(p, xa, xa + ex, ya, ya + ey, __uint_as_float(job.y), __uint_as_float(job.z), i0, i1, j0, j1, k0, k1))
        mark_box<R>(p, i0, i1, j0, j1, k0, k1, lane & 3, 4);
}

// S9 for colour, tiles [128 chunk, 128 chunk + 128), four consecutive tiles per lane, once every mark has been set: one work
// item per non-zero NIBBLE of a tile's shell-mark words, i.e. up to 4 colour cells; the item carries the nibble's bits, and the
// mark words are cleared here.  (A colour item is several times longer
// than a geometry sub-box; with 8 cells per item the longest ones left a tail.)
template <int R>
__device__ __forceinline__ void scan_chunk(const Params &p, uint32_t chunk, int lane)
{
    constexpr int WPT = words_per_tile(R), TPL = SCAN_CHUNK / 32;
    const int tile0 = (int)chunk * SCAN_CHUNK + lane * TPL;
    uint32_t mk[TPL][WPT];                              // the mark words
    int nbig = 0, nsmall = 0;                           // nibbles with 3-4 / 1-2 bits set
#pragma unroll
    for (int k = 0; k < TPL; ++k)
#pragma unroll
        for (int w = 0; w < WPT; ++w) {
            uint32_t m = 0u;
            if (tile0 + k < p.n_tiles) {
                m = __ldcg(p.marks + (size_t)(tile0 + k) * WPT + w);
                if (m) p.marks[(size_t)(tile0 + k) * WPT + w] = 0u;      // consumed: the marks are all zero again for the next frame
            }
            mk[k][w] = m;
            // per nibble: number of bits, 0..4, in place (SWAR)
            uint32_t c2 = (m & 0x55555555u) + ((m >> 1) & 0x55555555u);
            c2 = (c2 & 0x33333333u) + ((c2 >> 2) & 0x33333333u);
            const uint32_t ge3 = ((c2 + 0x11111111u) >> 2) & 0x11111111u & ~(c2 >> 2 & 0x11111111u) | ((c2 >> 2) & 0x11111111u);   // count >= 3
            const uint32_t nzn = (c2 | (c2 >> 1) | (c2 >> 2)) & 0x11111111u;                                                       // count >= 1
            nbig += __popc(ge3); nsmall += __popc(nzn & ~ge3);
        }
    // the long items (3 or 4 cells) go to the front of the list, the short ones to its back: the consumers take the front
    // first, so that the kernel ends on short items
    int preb = nbig, pres = nsmall;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int vb = __shfl_up_sync(0xffffffffu, preb, o), vs = __shfl_up_sync(0xffffffffu, pres, o);
        if (lane >= o) { preb += vb; pres += vs; }
    }
    const int totb = __shfl_sync(0xffffffffu, preb, 31), tots = __shfl_sync(0xffffffffu, pres, 31);
    if (totb + tots == 0) return;
    uint32_t bb = 0, bs = 0;
    if (lane == 0 && totb) bb = atomicAdd(&p.ctrl[ST_NCOL], (uint32_t)totb);
    if (lane == 0 && tots) bs = atomicAdd(&p.ctrl[ST_NCOL_SMALL], (uint32_t)tots);
    bb = __shfl_sync(0xffffffffu, bb, 0); bs = __shfl_sync(0xffffffffu, bs, 0);
    if (nbig + nsmall) {
        uint32_t posb = bb + (uint32_t)(preb - nbig), poss = p.work_col_cap - 1u - (bs + (uint32_t)(pres - nsmall));
#pragma unroll
        for (int k = 0; k < TPL; ++k) {
            const int tile = tile0 + k;
            const int ttx = tile % p.tiles_x, tty = (tile / p.tiles_x) % p.tiles_y, ttz = tile / (p.tiles_x * p.tiles_y);
#pragma unroll
            for (int w = 0; w < WPT; ++w) {
                const uint32_t m = mk[k][w];
#pragma unroll 1
                for (int n = 0; n < 8 && (m >> (4 * n)) != 0u; ++n) {
                    const uint32_t bits = m & (0xfu << (4 * n));
                    if (bits == 0u) continue;
                    const uint2 item = make_uint2(item_pack(ttx, tty, ttz, 8 * w + n), bits);
                    if (__popc(bits) >= 3) p.work_col[posb++] = item; else p.work_col[poss--] = item;
                }
            }
        }
    }
}

}  // namespace vf
