// params.cuh -- per-frame constants (S0), work-list layout and shared device helpers of the integration kernels.
//
// Canonical arithmetic: every per-voxel decision is taken in IEEE binary32
// with an explicit operation order -- __fmaf_rn where the method fuses, __fmul_rn/__fadd_rn elsewhere (never
// contracted by the compiler), correctly rounded __frcp_rn/__fdiv_rn/__fsqrt_rn, floorf for the pixel rounding
// (reading A2).  The file is compiled with --fmad=false as a second line of defence.  Code marked "culling only"
// is free-form arithmetic with explicit slack: it may only decide that work is skipped when no voxel can pass.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace vf {

// geometry tile (culling / work unit, one warp): TX x TY x TZ geometry voxels = 32 lanes x uint4 x TZ layers
constexpr int TX = 32, TY = 4, TZ = 8;
// colour cell (shell-mark / work unit, one warp pass): 8 x 4 x 4 colour voxels = 32 lanes x uint4
constexpr int CLX = 8, CLY = 4, CLZ = 4;
// tile classification refines a tile that passes the coarse test on SUBX x 1 x SUBZ sub-boxes of 8 x 4 x 4 voxels; the
// fused kernel visits only the sub-boxes that pass (one warp pass each: lane = (x, y) column of 4 voxels along z)
constexpr int SUBX = 4, SUBZ = 2;
constexpr int BRICK = 32;                                   // ray-casting skip brick: BRICK^3 geometry voxels = 1 x 8 x 4 tiles
constexpr int WARPS_PER_CTA = 8;
constexpr int CTA = 32 * WARPS_PER_CTA;

// alternative readings of the method (volfusion.h VOL_VARIANT_*), one at a time: a template
// parameter of the fused kernel, so the default reading's code is unchanged
enum { VAR_PAPER = 0, VAR_HD_FROM_DEPTH_POINT = 1, VAR_TSDF_ALONG_RAY = 2, VAR_ADDITIVE_WEIGHT = 4 };

// cells of one tile's colour children per axis, and 32-bit mark words per tile, for ratio r
__host__ __device__ constexpr int cells_x(int r) { return TX * r / CLX; }   // 4r
__host__ __device__ constexpr int cells_y(int r) { return TY * r / CLY; }   // r
__host__ __device__ constexpr int cells_z(int r) { return TZ * r / CLZ; }   // 2r
__host__ __device__ constexpr int cells_per_tile(int r) { return cells_x(r) * cells_y(r) * cells_z(r); }   // 8 r^3
__host__ __device__ constexpr int words_per_tile(int r) { return (cells_per_tile(r) + 31) / 32; }          // 1, 2, 7, 16

struct Params {
    // volume (fixed at vol_create)
    int   nx, ny, nz;            // full geometry dims
    int   r;
    int   cnx, cny, cnz;         // full colour dims
    int   local_nz;              // geometry layers stored by this shard
    int   tiles_x, tiles_y, tiles_z_local, n_tiles;
    int   shard_rank, shard_world;
    float ox, oy, oz;            // volume corner (world)
    float vs, vc;                // geometry / colour voxel size
    float mu, neg_mu, inv_mu, sig2, sigma, gate;
    int   w_max;
    int   variant;               // VAR_*
    // frame (S0: computed on the host in fp64, rounded once)
    float R[9], t[3];            // (R_n, t_n) of eq. 5: world -> depth camera
    float Rc[9], tc[3];          // (R_calib, t_calib) of eq. 3: depth camera -> HD camera
    float fx, fy, cx, cy;        // K_c
    float fxh, fyh, cxh, cyh;    // K_hd
    int   wd, hd, wh, hh;
    float wd_f, hd_f, wh_f, hh_f;
    // culling only
    float Rw[9], tw[3];          // depth camera -> world (the caller's T_world_depth)
    float tile_ex, tile_ey, tile_ez;   // conservative camera-axis half extents of a geometry tile
    float sub_ex, sub_ey, sub_ez;      // ... of one of its SUBX x 1 x SUBZ sub-boxes
    float sigma_g;                     // sigma grown by the fp32 slack
    float inv_vc, slack;         // 1 / colour voxel size; metres of slack for fp32 evaluation of culling geometry
    // device buffers
    const uint16_t *depth;
    const uint8_t  *rgb;
    uint32_t *geo;               // this shard's geometry words
    uint32_t *col;               // this shard's colour words
    float    *depthf;            // S1 output: D = depth_mm * 0.001f per depth pixel (0 = invalid), what the TSDF update gathers
    float4   *pixmap;            // S1 output: {X_vd, Y_vd, Z_vd, W} per depth pixel; W = 0 when no colour update is possible
    uint32_t *pyr;               // min/max valid-depth pyramid: entry = min_mm | max_mm << 16 (0xffff / 0 = empty)
    int       pyr_off[3], pyr_w[3], pyr_h[3], pyr_levels;   // levels: blocks of 8, 16, 32 pixels (fewer for tiny images)
    uint4    *jobs;              // shell-mark jobs of the frame (per 4 x 4 pixel patch: one, or one per strip, or one per pixel), jobs_cap entries
    uint32_t  jobs_cap;
    int       parity;            // frame parity: which of the two sets of per-frame scratch (pixmap, depthf, pyr, jobs) this frame uses
    uint32_t *work_geo;          // geometry work list (n_tiles entries, all zero between frames: a slot is cleared by the warp that takes it)
    uint32_t *marks;             // shell marks: words_per_tile(r) words per tile, bit = colour cell that may hold sigma-shell voxels
    uint2    *work_col;          // colour work list: one item per non-zero mark NIBBLE (up to 4 colour cells): {tile | nibble index, the nibble's
                                 // bits}; items of 3 or 4 cells from the front (ST_NCOL of them), items of 1 or 2 cells from the back
    uint32_t  work_col_cap;      // its capacity
    uint8_t  *tile_sat;          // per geometry tile: bit bx * SUBZ + bz = every voxel of that sub-box holds the saturated free-space word
                                 // (tsdf_q = 32767, w = w_max).  Kept by the fused kernel for the sub-boxes it visits; a sub-box
                                 // with its bit set that lies in front of every depth it can see by more than mu cannot change
                                 // this frame and is not queued (vol_reset / vol_upload clear the bits)
    uint8_t  *tile_skip;         // counting variant only: the sub-boxes of the tile that would not have been queued for that reason
    int       counting;          // the counting variant visits them all the same: its counters are the method's, not the kernel's
    uint32_t *sec_map[4];        // counting variant only: one bit per 32-byte sector of the geometry (read, written) and the colour
                                 // volume (read, written), zeroed before every frame: a sector is counted when its bit is first set
    uint8_t  *tile_neg;          // per geometry tile: 1 = the tile may hold an observed voxel with tsdf <= 0.  Set by the tile
                                 // classification (k_mark_classify), never cleared except by vol_reset (vol_upload sets
                                 // all): a conservative superset, used by the ray caster to skip free space
    uint8_t  *brick_neg;         // the same per brick of BRICK^3 geometry voxels (1 x 8 x 4 tiles): the ray caster's coarse level
    int       bricks_x, bricks_y, bricks_z;
    uint32_t *ctrl;              // statistics record and queue control words of this frame, see ST_* / Q_* below
    uint32_t *ctrl_next;         // the next frame's block, cleared by this frame's pre-pass
    unsigned long long *counters;// voxel and sector counters (counting variant only), see CNT_*
};

// work items (32 bits): [6:0] ttx | [15:7] tty | [23:16] ttz (local slab) = tile coordinates, and
//   geometry items: [31:24] = mask of the tile's SUBX x 1 x SUBZ sub-boxes (bit bx * SUBZ + bz) that may hold a voxel this frame
//                   updates (never 0, so a non-zero slot of the geometry work list is a published item);
//   colour items:   [30:24] = index of the mark NIBBLE within the tile.
// Whether a tile is NEAR (its box comes within 2 mm of the camera plane, or behind it: voxels may have Z <= 0 or Z outside
// the range of the branch-free reciprocal) is recomputed by the consumer from the tile's coordinates (tile_is_near).
// vol_create rejects volumes with more than 128 x 512 x 256 tiles per shard.
constexpr int ITEM_Y_SHIFT = 7, ITEM_Z_SHIFT = 16, ITEM_SUB_SHIFT = 24;
constexpr int ITEM_MAX_TX = 128, ITEM_MAX_TY = 512, ITEM_MAX_TZ = 256;
__device__ __forceinline__ uint32_t item_pack(int ttx, int tty, int ttz, int sub)
{
    return (uint32_t)ttx | ((uint32_t)tty << ITEM_Y_SHIFT) | ((uint32_t)ttz << ITEM_Z_SHIFT) | ((uint32_t)sub << ITEM_SUB_SHIFT);
}
__device__ __forceinline__ void item_unpack(uint32_t item, int &ttx, int &tty, int &ttz, int &sub)
{
    ttx = (int)(item & 127u); tty = (int)((item >> ITEM_Y_SHIFT) & 511u); ttz = (int)((item >> ITEM_Z_SHIFT) & 255u);
    sub = (int)(item >> ITEM_SUB_SHIFT);
}

// ctrl[]: the first VOL_STATS_RAW_BYTES (128) are the statistics record vol_frame_stats* copies out: 8 words ST_*, then 12
// 64-bit counters CNT_* (p.counters).  The queue control words Q_* follow; all of them are zeroed by k_prepass (the two job
// counters alternately, see Params::parity).
enum { ST_NGEO = 0, ST_NCOL = 1, ST_CELLS = 2, ST_SUBS = 3, ST_NJOBS = 4, ST_NCOL_SMALL = 5, ST_N = 8 };
enum { CNT_GEO_READ = 0, CNT_GEO_CHANGED, CNT_COL_READ, CNT_COL_CHANGED, CNT_GEO_SEC_READ, CNT_GEO_SEC_WRITTEN, CNT_COL_SEC_READ,
       CNT_COL_SEC_WRITTEN, CNT_GEO_VISITED, CNT_COL_GATED, CNT_GEO_SKIPPABLE, CNT_GEO_SEC_SKIPPABLE, CNT_N = 12 };
constexpr int CTRL_Q0 = 32;                                  // first queue-control word (byte 128)
// every queue-control word has a 128-byte line (and so, by the address hash, most likely an L2 slice) of its own: thousands
// of warps draw tickets from and poll these words, and requests to one line are served one after the other
constexpr int QS = 32;
enum { Q_CLS_CLAIM = CTRL_Q0, Q_CLS_DONE = CTRL_Q0 + QS, Q_MARK_CLAIM = CTRL_Q0 + 2 * QS, Q_MARK_DONE = CTRL_Q0 + 3 * QS,
       Q_SCAN_CLAIM = CTRL_Q0 + 4 * QS, Q_SCAN_DONE = CTRL_Q0 + 5 * QS, Q_GEO_CURSOR = CTRL_Q0 + 6 * QS, Q_COL_CURSOR = CTRL_Q0 + 7 * QS,
       Q_NJOBS = CTRL_Q0 + 8 * QS,
       // min / max valid depth (mm) of the whole frame
       Q_DMIN = CTRL_Q0 + 9 * QS, Q_DMAX, CTRL_N = CTRL_Q0 + 10 * QS };
// There are CTRL_SETS such blocks, used in turn by successive frames.  The pre-pass of frame n accumulates into block
// n % 3 (job counter, depth range) and cannot zero it first (its CTAs run in no particular order), so every pre-pass clears
// the block of the frame AFTER it instead: (n + 1) % 3, last used by frame n - 2, which has completed -- frame n - 1 may
// still be running when the pre-pass of frame n starts (see k_prepass), hence three blocks and not two.
constexpr int CTRL_SETS = 3;
constexpr int CLS_CHUNK = 32;                                // tiles per classification chunk (one lane each)
constexpr int SCAN_CHUNK = 128;                              // tiles per scan chunk (four per lane)
constexpr int MARK_CHUNK = 8;                                // mark jobs per chunk (4 lanes each)

// programmatic dependent launch: wait for the previous kernel of the stream (completion + memory flush) / allow the next
// kernel's CTAs to be scheduled as this one drains
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// local slab index -> global slab index; slabs of TZ = VOL_SLAB geometry layers are dealt round-robin to ranks
__device__ __forceinline__ int local_to_global_tz(const Params &p, int tz_local) { return tz_local * p.shard_world + p.shard_rank; }

// eq. 1 / eq. 6: pinhole projection + nearest pixel (A2) + frustum test (A3) in the canonical order.
__device__ __forceinline__ bool project_px(float fx, float fy, float cx, float cy, float wf, float hf,
                                           float X, float Y, float Z, int &x, int &y)
{
    if (!(Z > 0.0f)) return false;
    const float iz = __frcp_rn(Z);
    const float u = __fmaf_rn(fx, __fmul_rn(X, iz), cx);
    const float v = __fmaf_rn(fy, __fmul_rn(Y, iz), cy);
    const float uf = floorf(__fadd_rn(u, 0.5f));
    const float vf = floorf(__fadd_rn(v, 0.5f));
    if (!(uf >= 0.0f && uf < wf && vf >= 0.0f && vf < hf)) return false;
    x = (int)uf; y = (int)vf;
    return true;
}

// culling only: min/max valid depth (mm) over the inclusive pixel rectangle [x0,x1] x [y0,y1] (already clamped to the
// image), from the coarsest-needed pyramid level (blocks of 8, 16 or 32 pixels): at most 3 x 3 entries are read.  A rectangle
// larger than 3 x 3 blocks of the top level gets the range of the whole frame.
__device__ __forceinline__ void depth_range(const Params &p, int x0, int x1, int y0, int y1, uint32_t &mn, uint32_t &mx)
{
    int l = 0;
    while (l + 1 < p.pyr_levels && (((x1 >> (3 + l)) - (x0 >> (3 + l))) > 2 || ((y1 >> (3 + l)) - (y0 >> (3 + l))) > 2)) ++l;
    const int bx0 = x0 >> (3 + l), bx1 = x1 >> (3 + l), by0 = y0 >> (3 + l), by1 = y1 >> (3 + l);
    if (bx1 - bx0 > 2 || by1 - by0 > 2) { mn = __ldcg(&p.ctrl[Q_DMIN]); mx = __ldcg(&p.ctrl[Q_DMAX]); return; }
    mn = 0xffffu; mx = 0u;
    const uint32_t *lev = p.pyr + p.pyr_off[l];
    const int lw = p.pyr_w[l];
    for (int by = by0; by <= by1; ++by)
        for (int bx = bx0; bx <= bx1; ++bx) {
            const uint32_t e = __ldg(lev + by * lw + bx);
            mn = min(mn, e & 0xffffu); mx = max(mx, e >> 16);
        }
}

// culling only: conservative pixel rectangle of a camera-space box (centre c, half extents e).  Returns false if the
// box cannot project into the image: first the four side planes of the view frustum (through the camera centre, grown
// by one pixel; valid for any Z > 0, so also for boxes that straddle the camera plane), then the projected rectangle.
// A box that comes within 2 cm of the camera plane gets the whole image.
__device__ __forceinline__ bool box_rect(const Params &p, float cX, float cY, float cZ, float eX, float eY, float eZ,
                                         int &x0, int &x1, int &y0, int &y1, float &zmin, float &zmax)
{
    zmin = cZ - eZ; zmax = cZ + eZ;
    if (!(zmax > 0.0f)) return false;
    {   // u >= -1.5  <=>  fx X + (cx + 1.5) Z >= 0;   u <= wd + 0.5  <=>  -fx X + (wd + 0.5 - cx) Z >= 0   (Z > 0); same in v
        const float kl = p.cx + 1.5f, kr = p.wd_f + 0.5f - p.cx, kt = p.cy + 1.5f, kb = p.hd_f + 0.5f - p.cy;
        const float fxe = p.fx * eX, fye = p.fy * eY;
        if (p.fx * cX + kl * cZ + fxe + fabsf(kl) * eZ < 0.0f) return false;
        if (-p.fx * cX + kr * cZ + fxe + fabsf(kr) * eZ < 0.0f) return false;
        if (p.fy * cY + kt * cZ + fye + fabsf(kt) * eZ < 0.0f) return false;
        if (-p.fy * cY + kb * cZ + fye + fabsf(kb) * eZ < 0.0f) return false;
    }
    if (zmin > 0.02f) {
        const float i0 = 1.0f / zmin, i1 = 1.0f / zmax;
        const float xa = cX - eX, xb = cX + eX, ya = cY - eY, yb = cY + eY;
        const float umin = p.cx + p.fx * (xa >= 0.0f ? xa * i1 : xa * i0);
        const float umax = p.cx + p.fx * (xb >= 0.0f ? xb * i0 : xb * i1);
        const float vmin = p.cy + p.fy * (ya >= 0.0f ? ya * i1 : ya * i0);
        const float vmax = p.cy + p.fy * (yb >= 0.0f ? yb * i0 : yb * i1);
        if (!(umax >= -2.0f && umin <= p.wd_f + 1.0f && vmax >= -2.0f && vmin <= p.hd_f + 1.0f)) return false;
        x0 = max(0, (int)floorf(fmaxf(umin, -4.0f)) - 1); x1 = min(p.wd - 1, (int)ceilf(fminf(umax, p.wd_f + 4.0f)) + 1);
        y0 = max(0, (int)floorf(fmaxf(vmin, -4.0f)) - 1); y1 = min(p.hd - 1, (int)ceilf(fminf(vmax, p.hd_f + 4.0f)) + 1);
        if (x0 > x1 || y0 > y1) return false;
    } else {
        x0 = 0; x1 = p.wd - 1; y0 = 0; y1 = p.hd - 1;
    }
    return true;
}

}  // namespace vf
