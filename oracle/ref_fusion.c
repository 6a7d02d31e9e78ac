/*
 * oracle/ref_fusion.c -- CPU ORACLE for the per-frame volumetric fusion of arXiv 1602.06645.
 *
 * TEST INFRASTRUCTURE ONLY.  Plain, slow, obviously-correct per-voxel loops written from the
 * paper's equations; no pre-pass, no culling, no tiling, no code shared with the CUDA path
 * (paper_1602_06645_b200/).  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may call it.
 *
 * What it computes (citations are PAPER.md lines; readings A1..A17 are SURVEY.md 8(c), restated in
 * DESIGN.md "Readings"):
 *   geometry volume  -- projective TSDF integration.  The paper gives NO equations for it
 *                       (L33-35 defer to KinectFusion/PCL); the definition is reading A5/A6 and is
 *                       pinned by BASELINE.json's closed forms.  ** paper: parity unpinned **
 *   colour volume    -- eq. 5-10, on an asymmetrical colour volume (L87) with r x more
 *                       voxels per axis.  Readings A11 (which point maps to the HD image) and A12
 *                       (u8 weight encoding of eq. 10) are conventions ** parity unpinned ** by the paper.
 *
 *   ray casting (ref_raycast, readings R1-R6), colour sampling (ref_sample_colour*, readings S1-S2) and the alternative
 *                       readings selected by ref_vol_t.variant: the paper gives no definition for any of them
 *                       ** parity unpinned ** by the paper; pinned by closed forms (tests/test_oracle_*.py).
 *
 * Canonical arithmetic: IEEE binary32, round-to-nearest-even, no implicit contraction
 * (-ffp-contract=off); fmaf() where the spec says fma; / and sqrtf correctly rounded; rintf = half-even.
 *
 * Layout (little-endian, x fastest: index ((k*Ny + j)*Nx + i)):
 *   geometry word = int16 tsdf_q (bytes 0-1) | int16 w (bytes 2-3), F = tsdf_q / 32767
 *   colour word   = u8 R | u8 G | u8 B | u8 wq,                  W = wq / 255
 *
 * Build: gcc -O2 -fopenmp -ffp-contract=off -mfma -shared -fPIC ref_fusion.c -lm
 */
#include <math.h>
#ifdef _OPENMP
#include <omp.h>
#endif
#include <stdint.h>
#include <stddef.h>
#include <string.h>

typedef struct {
    int32_t nx, ny, nz;      /* geometry dims */
    int32_t r;               /* colour dims = r * geometry dims (L87) */
    float   origin[3];       /* world position of the volume's corner (A1) */
    float   extent;          /* side length along x, metres; cubic voxels vs = extent / nx */
    float   mu;              /* truncation distance, metres (A5) */
    int32_t w_max;           /* geometry weight cap (A5) */
    float   sigma;           /* colour distance gate, metres; 0.020 in the paper (L108) */
    float   gate;            /* weight gate factor; 0.8 in the paper (L115) */
    int32_t variant;         /* 0 = the readings of DESIGN.md; or ONE of the alternative readings below */
} ref_vol_t;

/* Alternative readings, one at a time:
 *   VAR_HD_FROM_DEPTH_POINT  A11 read literally: the HD pixel is located from the depth pixel's 3D point (X_vd, Y_vd, Z_vd)
 *                            of eq. 7 through eq. 3-4 (L71-81, L115), not from the voxel's own position
 *   VAR_TSDF_ALONG_RAY       A5: the signed distance is measured along the voxel's viewing ray, (D - Z_vc) * |P_vc| / Z_vc
 *                            (KinectFusion's metric distance), not along the optical axis
 *   VAR_ADDITIVE_WEIGHT      A12: W_new = min(W_pre + W, 1) instead of eq. 10 (L122) */
enum { VAR_HD_FROM_DEPTH_POINT = 1, VAR_TSDF_ALONG_RAY = 2, VAR_ADDITIVE_WEIGHT = 4 };

typedef struct {
    const uint16_t *depth; int32_t wd, hd;      /* depth map D_n, mm, 0 = invalid (L101-103) */
    const uint8_t  *rgb;   int32_t wh, hh;      /* HD RGB image, interleaved R,G,B (L115) */
    float T_world_depth[16];                    /* row-major rigid 4x4, depth-camera -> world */
    float K_depth[9], K_rgb[9];                 /* row-major [fx 0 cx; 0 fy cy; 0 0 1] */
    float T_depth_rgb[16];                      /* row-major rigid 4x4, RGB-camera -> depth-camera */
} ref_frame_t;

/* per-frame counters: a voxel is *read* when it reaches the load of its stored
 * word and *changed* when the stored word differs after the store */
enum { CNT_GEO_READ = 0, CNT_GEO_CHANGED = 1, CNT_COL_READ = 2, CNT_COL_CHANGED = 3, CNT_N = 4 };

/* S0: per-frame constants, computed in fp64 and rounded once to fp32 */
typedef struct {
    float R[9], t[3];        /* (R_n, t_n) of eq. 5: world -> current depth camera = inverse(T_world_depth) */
    float Rc[9], tc[3];      /* (R_calib, t_calib) of eq. 3: depth camera -> HD camera = inverse(T_depth_rgb) */
    float fx, fy, cx, cy;    /* K_c  */
    float fxh, fyh, cxh, cyh;/* K_hd */
    float vs, vc;            /* geometry / colour voxel size */
    float inv_mu, sig2;
} consts_t;

/* rigid inverse: R' = R^T, t' = -(R^T t), fp64 with left-to-right sums, one rounding to fp32 */
static void rigid_inverse(const float T[16], float Rout[9], float tout[3])
{
    for (int i = 0; i < 3; ++i) {
        for (int j = 0; j < 3; ++j) Rout[3 * i + j] = T[4 * j + i];
        double s = (double)T[4 * 0 + i] * (double)T[4 * 0 + 3];
        s = s + (double)T[4 * 1 + i] * (double)T[4 * 1 + 3];
        s = s + (double)T[4 * 2 + i] * (double)T[4 * 2 + 3];
        tout[i] = (float)(-s);
    }
}

static void frame_consts(const ref_vol_t *v, const ref_frame_t *f, consts_t *c)
{
    rigid_inverse(f->T_world_depth, c->R, c->t);
    rigid_inverse(f->T_depth_rgb, c->Rc, c->tc);
    c->fx = f->K_depth[0]; c->fy = f->K_depth[4]; c->cx = f->K_depth[2]; c->cy = f->K_depth[5];
    c->fxh = f->K_rgb[0]; c->fyh = f->K_rgb[4]; c->cxh = f->K_rgb[2]; c->cyh = f->K_rgb[5];
    c->vs = v->extent / (float)v->nx;
    c->vc = c->vs / (float)v->r;
    c->inv_mu = 1.0f / v->mu;
    c->sig2 = v->sigma * v->sigma;
}

/* eq. 5 (L91-94), voxel centre convention A1: centre of voxel idx in a grid of voxel size s */
static void voxel_to_camera(const ref_vol_t *v, const consts_t *c, float s, int i, int j, int k,
                            float *X, float *Y, float *Z)
{
    float px = fmaf((float)i + 0.5f, s, v->origin[0]);
    float py = fmaf((float)j + 0.5f, s, v->origin[1]);
    float pz = fmaf((float)k + 0.5f, s, v->origin[2]);
    *X = fmaf(c->R[2], pz, fmaf(c->R[1], py, fmaf(c->R[0], px, c->t[0])));
    *Y = fmaf(c->R[5], pz, fmaf(c->R[4], py, fmaf(c->R[3], px, c->t[1])));
    *Z = fmaf(c->R[8], pz, fmaf(c->R[7], py, fmaf(c->R[6], px, c->t[2])));
}

/* eq. 1 / eq. 6 (L64-67, L96-99): pinhole projection, divide by z, nearest pixel (A2), frustum =
 * Z > 0 and rounded pixel inside the w x h image (A3).  Returns 1 and the pixel if inside. */
static int project(float fx, float fy, float cx, float cy, int w, int h,
                   float X, float Y, float Z, int *x, int *y)
{
    if (!(Z > 0.0f)) return 0;
    float iz = 1.0f / Z;
    float u = fmaf(fx, X * iz, cx);
    float vv = fmaf(fy, Y * iz, cy);
    float uf = floorf(u + 0.5f);
    float vf = floorf(vv + 0.5f);
    if (!(uf >= 0.0f && uf < (float)w && vf >= 0.0f && vf < (float)h)) return 0;
    *x = (int)uf; *y = (int)vf;
    return 1;
}

/* O-G: one geometry voxel (L33-35; definition = readings A5, A6).  Returns bit0 = read, bit1 = changed. */
static int update_geo_voxel(const ref_vol_t *v, const ref_frame_t *f, const consts_t *c,
                            int i, int j, int k, uint32_t *word)
{
    float X, Y, Z; int x, y;
    voxel_to_camera(v, c, c->vs, i, j, k, &X, &Y, &Z);
    if (!project(c->fx, c->fy, c->cx, c->cy, f->wd, f->hd, X, Y, Z, &x, &y)) return 0;
    uint16_t d = f->depth[(size_t)y * (size_t)f->wd + (size_t)x];
    if (d == 0) return 0;                                   /* "if non-zero" (L103) */
    float D = (float)d * 0.001f;                            /* mm -> m (A4) */
    float sdf = D - Z;                                      /* projective signed distance (A5) */
    if (v->variant == VAR_TSDF_ALONG_RAY) {                 /* ... measured along the viewing ray of the voxel */
        float nrm = sqrtf(fmaf(Z, Z, fmaf(Y, Y, X * X)));
        sdf = sdf * (nrm * (1.0f / Z));
    }
    if (sdf < -v->mu) return 0;                             /* behind the truncation band: unchanged */
    float tsdf = fminf(1.0f, sdf * c->inv_mu);
    int q = (int16_t)(*word & 0xffffu);
    int w = (int16_t)(*word >> 16);
    float num = fmaf((float)q, (float)w, tsdf * 32767.0f);  /* running average, per-frame weight 1 */
    int qn = (int)rintf(num / ((float)w + 1.0f));
    int wn = w + 1 < v->w_max ? w + 1 : v->w_max;           /* increment and saturate */
    uint32_t nw = ((uint32_t)(uint16_t)(int16_t)qn) | ((uint32_t)(uint16_t)(int16_t)wn << 16);
    int changed = nw != *word;
    *word = nw;
    return 1 | (changed << 1);
}

/* eq. 7 (L103-106): back-projection of depth pixel (x, y, D) with K_c^-1 */
static void backproject(const consts_t *c, int x, int y, float D, float P[3])
{
    P[0] = (((float)x - c->cx) * D) / c->fx;
    P[1] = (((float)y - c->cy) * D) / c->fy;
    P[2] = D;
}

/* O-C: one colour voxel, eq. 5-10 (L91-124).  Returns bit0 = read, bit1 = changed. */
static int update_col_voxel(const ref_vol_t *v, const ref_frame_t *f, const consts_t *c,
                            int i, int j, int k, uint32_t *word)
{
    float X, Y, Z; int x, y;
    voxel_to_camera(v, c, c->vc, i, j, k, &X, &Y, &Z);                                 /* eq. 5 */
    if (!project(c->fx, c->fy, c->cx, c->cy, f->wd, f->hd, X, Y, Z, &x, &y)) return 0; /* eq. 6 */
    uint16_t d0 = f->depth[(size_t)y * (size_t)f->wd + (size_t)x];
    if (d0 == 0) return 0;                                                             /* L103 */
    if (!(x + 1 < f->wd && y + 1 < f->hd)) return 0;                                   /* A7: no neighbour */
    uint16_t d1 = f->depth[(size_t)y * (size_t)f->wd + (size_t)(x + 1)];
    uint16_t d2 = f->depth[(size_t)(y + 1) * (size_t)f->wd + (size_t)x];
    if (d1 == 0 || d2 == 0) return 0;                                                  /* A7 */
    float Pd[3], P1[3], P2[3];
    backproject(c, x, y, (float)d0 * 0.001f, Pd);                                      /* eq. 7 */
    backproject(c, x + 1, y, (float)d1 * 0.001f, P1);
    backproject(c, x, y + 1, (float)d2 * 0.001f, P2);
    /* sigma gate (L108): Euclidean distance between voxel and depth point */
    float dx = X - Pd[0], dy = Y - Pd[1], dz = Z - Pd[2];
    float dist2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
    if (dist2 > c->sig2) return 0;
    /* eq. 8 (L110-113): normal from forward differences */
    float ax = P1[0] - Pd[0], ay = P1[1] - Pd[1], az = P1[2] - Pd[2];
    float bx = P2[0] - Pd[0], by = P2[1] - Pd[1], bz = P2[2] - Pd[2];
    float nx = fmaf(ay, bz, -(az * by));
    float ny = fmaf(az, bx, -(ax * bz));
    float nz = fmaf(ax, by, -(ay * bx));
    /* weight (L110, A8): cosine between the normal and the viewing ray camera -> point */
    float dot = fmaf(nz, Pd[2], fmaf(ny, Pd[1], nx * Pd[0]));
    float nn = fmaf(nz, nz, fmaf(ny, ny, nx * nx));
    float pp = fmaf(Pd[2], Pd[2], fmaf(Pd[1], Pd[1], Pd[0] * Pd[0]));
    float den = sqrtf(nn * pp);
    if (!(den > 0.0f)) return 0;
    float W = fminf(1.0f, dot / den);
    if (!(W > 0.0f)) return 0;
    /* read C_pre, W_pre */
    uint32_t old = *word;
    int C[3] = { (int)(old & 0xffu), (int)((old >> 8) & 0xffu), (int)((old >> 16) & 0xffu) };
    int wq = (int)(old >> 24);
    float W255 = W * 255.0f;
    if (!(W255 > v->gate * (float)wq)) return 1;                                       /* L115, A9 */
    /* HD pixel of the voxel's own position (eq. 3-4; A10, A11) */
    if (v->variant == VAR_HD_FROM_DEPTH_POINT) { X = Pd[0]; Y = Pd[1]; Z = Pd[2]; }   /* ... or of its depth pixel's point */
    float Xh = fmaf(c->Rc[2], Z, fmaf(c->Rc[1], Y, fmaf(c->Rc[0], X, c->tc[0])));
    float Yh = fmaf(c->Rc[5], Z, fmaf(c->Rc[4], Y, fmaf(c->Rc[3], X, c->tc[1])));
    float Zh = fmaf(c->Rc[8], Z, fmaf(c->Rc[7], Y, fmaf(c->Rc[6], X, c->tc[2])));
    int xh, yh;
    if (!project(c->fxh, c->fyh, c->cxh, c->cyh, f->wh, f->hh, Xh, Yh, Zh, &xh, &yh)) return 1;  /* A13 */
    const uint8_t *hd = f->rgb + ((size_t)yh * (size_t)f->wh + (size_t)xh) * 3;        /* A14: nearest */
    uint32_t nw = 0;
    for (int ch = 0; ch < 3; ++ch) {                                                   /* eq. 9 (L117) */
        float num = fmaf(W255, (float)hd[ch], (float)(C[ch] * wq));
        float cn = rintf(num / ((float)wq + W255));
        int ci = cn < 0.0f ? 0 : (cn > 255.0f ? 255 : (int)cn);
        nw |= (uint32_t)ci << (8 * ch);
    }
    int wn = (int)rintf(fmaf(W, (float)(255 - wq), (float)wq));                        /* eq. 10 (L122), A12 */
    if (v->variant == VAR_ADDITIVE_WEIGHT) wn = (int)rintf((float)wq + W255);          /* ... or W_pre + W */
    if (wn > 255) wn = 255;
    nw |= (uint32_t)wn << 24;
    *word = nw;                                                                        /* L124 */
    return 1 | ((nw != old) << 1);
}

/* ------------------------------------------------------------------------------------------ */
/* exported entry points (host pointers only)                                                  */
/* ------------------------------------------------------------------------------------------ */

/* ref_integrate: one frame over the WHOLE of both volumes -- a plain triple loop over the
 * geometry voxels, then a plain triple loop over the colour voxels.  geo / col are the packed
 * state arrays (layout above), updated in place.  counters[4] (nullable) receives this frame's
 * CNT_* counts.  OpenMP only splits the outermost z loop; voxels are independent (A15).
 * sec (nullable): four byte maps, one byte per 32-byte SECTOR (8 consecutive words of the linear
 * layout) of the geometry / colour array, set to 1 where a voxel of the sector was read / changed
 * (sec[0] geometry read, sec[1] geometry changed, sec[2] colour read, sec[3] colour changed): the
 * DRAM granularity of the same sets (SURVEY 8(d) "report both voxel-exact and sector-exact"). */
static int integrate_all(const ref_vol_t *v, const ref_frame_t *f, uint32_t *geo, uint32_t *col, uint64_t *counters, uint8_t *const sec[4])
{
    if (!v || !f || !geo || !col || !f->depth || !f->rgb) return -1;
    if (v->nx <= 0 || v->ny <= 0 || v->nz <= 0 || v->r < 1 || !(v->mu > 0.0f) || v->w_max < 1 || v->w_max > 512) return -1;
    if (v->variant != 0 && v->variant != VAR_HD_FROM_DEPTH_POINT && v->variant != VAR_TSDF_ALONG_RAY && v->variant != VAR_ADDITIVE_WEIGHT) return -1;
    consts_t c; frame_consts(v, f, &c);
    uint64_t gr = 0, gc = 0, cr = 0, cc = 0;
#pragma omp parallel for schedule(static) reduction(+ : gr, gc)
    for (int k = 0; k < v->nz; ++k)
        for (int j = 0; j < v->ny; ++j)
            for (int i = 0; i < v->nx; ++i) {
                size_t idx = ((size_t)k * (size_t)v->ny + (size_t)j) * (size_t)v->nx + (size_t)i;
                int s = update_geo_voxel(v, f, &c, i, j, k, &geo[idx]);
                gr += (uint64_t)(s & 1); gc += (uint64_t)(s >> 1);
                if (sec) {                      /* (a sector can straddle two layers, i.e. two threads: same value, atomic store) */
                    if (s & 1) {
#pragma omp atomic write
                        sec[0][idx >> 3] = 1;
                    }
                    if (s >> 1) {
#pragma omp atomic write
                        sec[1][idx >> 3] = 1;
                    }
                }
            }
    const int cx = v->nx * v->r, cy = v->ny * v->r, cz = v->nz * v->r;
#pragma omp parallel for schedule(static) reduction(+ : cr, cc)
    for (int k = 0; k < cz; ++k)
        for (int j = 0; j < cy; ++j)
            for (int i = 0; i < cx; ++i) {
                size_t idx = ((size_t)k * (size_t)cy + (size_t)j) * (size_t)cx + (size_t)i;
                int s = update_col_voxel(v, f, &c, i, j, k, &col[idx]);
                cr += (uint64_t)(s & 1); cc += (uint64_t)(s >> 1);
                if (sec) {
                    if (s & 1) {
#pragma omp atomic write
                        sec[2][idx >> 3] = 1;
                    }
                    if (s >> 1) {
#pragma omp atomic write
                        sec[3][idx >> 3] = 1;
                    }
                }
            }
    if (counters) { counters[CNT_GEO_READ] = gr; counters[CNT_GEO_CHANGED] = gc; counters[CNT_COL_READ] = cr; counters[CNT_COL_CHANGED] = cc; }
    return 0;
}

int ref_integrate(const ref_vol_t *v, const ref_frame_t *f, uint32_t *geo, uint32_t *col, uint64_t *counters)
{
    return integrate_all(v, f, geo, col, counters, NULL);
}

/* the same, with the sector maps (caller-zeroed; sizes ceil(N / 8) bytes each) */
int ref_integrate_sectors(const ref_vol_t *v, const ref_frame_t *f, uint32_t *geo, uint32_t *col, uint64_t *counters,
                          uint8_t *geo_read, uint8_t *geo_changed, uint8_t *col_read, uint8_t *col_changed)
{
    uint8_t *const sec[4] = {geo_read, geo_changed, col_read, col_changed};
    if (!geo_read || !geo_changed || !col_read || !col_changed) return -1;
    return integrate_all(v, f, geo, col, counters, sec);
}

/* how many threads the loops above use (reported beside the timed CPU baseline) */
int ref_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ref_integrate_subset: the same per-voxel updates applied to a LIST of voxels only (voxels never
 * interact, so the state of any subset after any number of frames is exact -- SURVEY 8(c) "making
 * the oracle affordable").  geo_idx / col_idx are linear voxel indices into the full grids;
 * geo_words / col_words hold the state of just those voxels and are updated in place. */
int ref_integrate_subset(const ref_vol_t *v, const ref_frame_t *f,
                         const int64_t *geo_idx, int64_t n_geo, uint32_t *geo_words,
                         const int64_t *col_idx, int64_t n_col, uint32_t *col_words)
{
    if (!v || !f || !f->depth || !f->rgb) return -1;
    if (v->nx <= 0 || v->ny <= 0 || v->nz <= 0 || v->r < 1 || !(v->mu > 0.0f) || v->w_max < 1 || v->w_max > 512) return -1;
    if (v->variant != 0 && v->variant != VAR_HD_FROM_DEPTH_POINT && v->variant != VAR_TSDF_ALONG_RAY && v->variant != VAR_ADDITIVE_WEIGHT) return -1;
    consts_t c; frame_consts(v, f, &c);
#pragma omp parallel for schedule(static)
    for (int64_t n = 0; n < n_geo; ++n) {
        int64_t idx = geo_idx[n];
        int i = (int)(idx % v->nx), j = (int)((idx / v->nx) % v->ny), k = (int)(idx / ((int64_t)v->nx * v->ny));
        update_geo_voxel(v, f, &c, i, j, k, &geo_words[n]);
    }
    const int64_t cx = (int64_t)v->nx * v->r, cy = (int64_t)v->ny * v->r;
#pragma omp parallel for schedule(static)
    for (int64_t n = 0; n < n_col; ++n) {
        int64_t idx = col_idx[n];
        int i = (int)(idx % cx), j = (int)((idx / cx) % cy), k = (int)(idx / (cx * cy));
        update_col_voxel(v, f, &c, i, j, k, &col_words[n]);
    }
    return 0;
}

/* ref_frame_constants: expose S0 (for the tests that pin the rigid inverse). out = R[9] t[3] Rc[9] tc[3] */
int ref_frame_constants(const ref_vol_t *v, const ref_frame_t *f, float out[24])
{
    consts_t c; frame_consts(v, f, &c);
    memcpy(out, c.R, 9 * sizeof(float)); memcpy(out + 9, c.t, 3 * sizeof(float));
    memcpy(out + 12, c.Rc, 9 * sizeof(float)); memcpy(out + 21, c.tc, 3 * sizeof(float));
    return 0;
}

/* ------------------------------------------------------------------------------------------ */
/* ref_raycast -- NEXT row: ray casting of the geometry + colour volumes  */
/* ------------------------------------------------------------------------------------------ */
/* The paper names the operation only ("ray casting" of the volumes for the ICP prediction and the
 * live preview) and gives no equations: ** parity unpinned by the paper **.  The
 * definition below is this build's reading R1-R6, written out step by step:
 *   R1  pixel (x, y) of a virtual pinhole camera K, pose T_world_cam: camera-space ray ((x-cx)/fx, (y-cy)/fy, 1),
 *       so the ray parameter t IS the camera-space depth z (eq. 1, inverted as in eq. 7);
 *   R2  samples at t_k = t_near + k * vs (one geometry voxel of depth per step), k = 0, 1, ... while t_k <= t_far;
 *   R3  the TSDF at a sample is the value of the voxel whose cell contains the point (nearest voxel, no
 *       interpolation); voxels never observed (w = 0) and points outside the volume are "unknown";
 *   R4  a hit is the first pair of consecutive known samples with F_prev > 0 >= F_cur (front face only);
 *       its depth is t_prev + vs * F_prev / (F_prev - F_cur) (linear zero crossing);
 *   R5  the colour of a hit is the colour voxel that contains the hit point (nearest, weight > 0), else black;
 *   R6  no hit: depth 0, colour black.
 * Canonical arithmetic as above (binary32, explicit fmaf, correctly rounded division, floorf).
 * depth_out: w*h float32 metres; rgb_out: w*h*3 bytes (nullable).  T_world_cam: row-major rigid 4x4. */
int ref_raycast(const ref_vol_t *v, const uint32_t *geo, const uint32_t *col, int32_t w, int32_t h,
                const float T_world_cam[16], const float K[9], float t_near, float t_far,
                float *depth_out, uint8_t *rgb_out)
{
    if (!v || !geo || !col || !T_world_cam || !K || !depth_out || w <= 0 || h <= 0) return -1;
    if (!(t_near >= 0.0f) || !(t_far >= t_near)) return -1;
    const float fx = K[0], fy = K[4], cx = K[2], cy = K[5];
    const float vs = v->extent / (float)v->nx, vc = vs / (float)v->r;
    const float inv_vs = 1.0f / vs, inv_vc = 1.0f / vc;
    const int cnx = v->nx * v->r, cny = v->ny * v->r, cnz = v->nz * v->r;
#pragma omp parallel for schedule(dynamic, 4)
    for (int y = 0; y < h; ++y)
        for (int x = 0; x < w; ++x) {
            const float dx = ((float)x - cx) / fx, dy = ((float)y - cy) / fy;                     /* R1 */
            float dw[3], ow[3];
            for (int a = 0; a < 3; ++a) {
                dw[a] = fmaf(T_world_cam[4 * a + 1], dy, fmaf(T_world_cam[4 * a + 0], dx, T_world_cam[4 * a + 2]));
                ow[a] = T_world_cam[4 * a + 3];
            }
            float depth = 0.0f, t_prev = 0.0f, f_prev = 0.0f;
            int known_prev = 0;
            uint8_t rgb[3] = {0, 0, 0};
            for (int k = 0;; ++k) {
                const float t = fmaf((float)k, vs, t_near);                                       /* R2 */
                if (t > t_far) break;
                const float gx = (fmaf(t, dw[0], ow[0]) - v->origin[0]) * inv_vs;
                const float gy = (fmaf(t, dw[1], ow[1]) - v->origin[1]) * inv_vs;
                const float gz = (fmaf(t, dw[2], ow[2]) - v->origin[2]) * inv_vs;
                const float fi = floorf(gx), fj = floorf(gy), fk = floorf(gz);
                int known = 0; float f = 0.0f;
                if (fi >= 0.0f && fi < (float)v->nx && fj >= 0.0f && fj < (float)v->ny && fk >= 0.0f && fk < (float)v->nz) {
                    const uint32_t word = geo[((size_t)(int)fk * (size_t)v->ny + (size_t)(int)fj) * (size_t)v->nx + (size_t)(int)fi];
                    if ((int16_t)(word >> 16) != 0) { known = 1; f = (float)(int16_t)(word & 0xffffu); }   /* R3 */
                }
                if (known && known_prev && f_prev > 0.0f && !(f > 0.0f)) {                        /* R4 */
                    depth = fmaf(vs, f_prev / (f_prev - f), t_prev);
                    break;
                }
                known_prev = known; t_prev = t; f_prev = f;
            }
            if (depth > 0.0f) {                                                                   /* R5 */
                const float hx = floorf((fmaf(depth, dw[0], ow[0]) - v->origin[0]) * inv_vc);
                const float hy = floorf((fmaf(depth, dw[1], ow[1]) - v->origin[1]) * inv_vc);
                const float hz = floorf((fmaf(depth, dw[2], ow[2]) - v->origin[2]) * inv_vc);
                if (hx >= 0.0f && hx < (float)cnx && hy >= 0.0f && hy < (float)cny && hz >= 0.0f && hz < (float)cnz) {
                    const uint32_t cw = col[((size_t)(int)hz * (size_t)cny + (size_t)(int)hy) * (size_t)cnx + (size_t)(int)hx];
                    if ((cw >> 24) != 0) { rgb[0] = (uint8_t)cw; rgb[1] = (uint8_t)(cw >> 8); rgb[2] = (uint8_t)(cw >> 16); }
                }
            }
            depth_out[(size_t)y * (size_t)w + (size_t)x] = depth;
            if (rgb_out) { uint8_t *o = rgb_out + ((size_t)y * (size_t)w + (size_t)x) * 3; o[0] = rgb[0]; o[1] = rgb[1]; o[2] = rgb[2]; }
        }
    return 0;
}

/* ref_raycast_trilinear -- the same ray caster with reading R3 replaced by R7 (round 2):
 *   R7  the TSDF at a sample is the TRILINEAR interpolation of the 8 voxels whose centres surround the point: grid coordinate
 *       g = (p - origin) / vs - 1/2 per axis (voxel centres at integers, A1), b = floor(g), f = g - b; corner c = 0..7 is voxel
 *       b + (c & 1, (c >> 1) & 1, c >> 2) with weight (wz * wy) * wx, w = f on the far side and 1 - f on the near side;
 *       F = sum over c, in that order, of weight * q (fmaf).  If any of the 8 voxels lies outside the volume or was never
 *       observed (w = 0) the sample is "unknown".
 * R1, R2, R4 (on these F), R5 and R6 are unchanged.  A TSDF that is linear in space (a plane inside the truncation band) is
 * reproduced exactly by the interpolation, so the zero crossing of R4 is the plane itself for any t_near -- no voxel-sized
 * terraces, which is what the tracker's prediction needs (F8 is not applied to these maps).  ** parity unpinned by the paper ** */
int ref_raycast_trilinear(const ref_vol_t *v, const uint32_t *geo, const uint32_t *col, int32_t w, int32_t h,
                          const float T_world_cam[16], const float K[9], float t_near, float t_far,
                          float *depth_out, uint8_t *rgb_out)
{
    if (!v || !geo || !col || !T_world_cam || !K || !depth_out || w <= 0 || h <= 0) return -1;
    if (!(t_near >= 0.0f) || !(t_far >= t_near)) return -1;
    const float fx = K[0], fy = K[4], cx = K[2], cy = K[5];
    const float vs = v->extent / (float)v->nx, vc = vs / (float)v->r;
    const float inv_vs = 1.0f / vs, inv_vc = 1.0f / vc;
    const int cnx = v->nx * v->r, cny = v->ny * v->r, cnz = v->nz * v->r;
    const int n[3] = {v->nx, v->ny, v->nz};
#pragma omp parallel for schedule(dynamic, 4)
    for (int y = 0; y < h; ++y)
        for (int x = 0; x < w; ++x) {
            const float dx = ((float)x - cx) / fx, dy = ((float)y - cy) / fy;                     /* R1 */
            float dw[3], ow[3];
            for (int a = 0; a < 3; ++a) {
                dw[a] = fmaf(T_world_cam[4 * a + 1], dy, fmaf(T_world_cam[4 * a + 0], dx, T_world_cam[4 * a + 2]));
                ow[a] = T_world_cam[4 * a + 3];
            }
            float depth = 0.0f, t_prev = 0.0f, f_prev = 0.0f;
            int known_prev = 0;
            uint8_t rgb[3] = {0, 0, 0};
            for (int k = 0;; ++k) {
                const float t = fmaf((float)k, vs, t_near);                                       /* R2 */
                if (t > t_far) break;
                float b[3], fr[3];
                int in = 1;
                for (int a = 0; a < 3; ++a) {                                                     /* R7 */
                    const float g = (fmaf(t, dw[a], ow[a]) - v->origin[a]) * inv_vs - 0.5f;
                    b[a] = floorf(g);
                    fr[a] = g - b[a];
                    in = in && b[a] >= 0.0f && b[a] <= (float)(n[a] - 2);                         /* false for NaN / inf as well */
                }
                int known = in; float f = 0.0f;
                if (in) {
                    const int i0 = (int)b[0], j0 = (int)b[1], k0 = (int)b[2];
                    for (int c = 0; c < 8; ++c) {
                        const uint32_t word = geo[((size_t)(k0 + (c >> 2)) * (size_t)v->ny + (size_t)(j0 + ((c >> 1) & 1))) * (size_t)v->nx + (size_t)(i0 + (c & 1))];
                        if ((int16_t)(word >> 16) == 0) known = 0;
                        const float wx = (c & 1) ? fr[0] : 1.0f - fr[0];
                        const float wy = (c & 2) ? fr[1] : 1.0f - fr[1];
                        const float wz = (c & 4) ? fr[2] : 1.0f - fr[2];
                        f = fmaf((wz * wy) * wx, (float)(int16_t)(word & 0xffffu), f);
                    }
                    if (!known) f = 0.0f;
                }
                if (known && known_prev && f_prev > 0.0f && !(f > 0.0f)) {                        /* R4 */
                    depth = fmaf(vs, f_prev / (f_prev - f), t_prev);
                    break;
                }
                known_prev = known; t_prev = t; f_prev = f;
            }
            if (depth > 0.0f) {                                                                   /* R5 */
                const float hx = floorf((fmaf(depth, dw[0], ow[0]) - v->origin[0]) * inv_vc);
                const float hy = floorf((fmaf(depth, dw[1], ow[1]) - v->origin[1]) * inv_vc);
                const float hz = floorf((fmaf(depth, dw[2], ow[2]) - v->origin[2]) * inv_vc);
                if (hx >= 0.0f && hx < (float)cnx && hy >= 0.0f && hy < (float)cny && hz >= 0.0f && hz < (float)cnz) {
                    const uint32_t cw = col[((size_t)(int)hz * (size_t)cny + (size_t)(int)hy) * (size_t)cnx + (size_t)(int)hx];
                    if ((cw >> 24) != 0) { rgb[0] = (uint8_t)cw; rgb[1] = (uint8_t)(cw >> 8); rgb[2] = (uint8_t)(cw >> 16); }
                }
            }
            depth_out[(size_t)y * (size_t)w + (size_t)x] = depth;
            if (rgb_out) { uint8_t *o = rgb_out + ((size_t)y * (size_t)w + (size_t)x) * 3; o[0] = rgb[0]; o[1] = rgb[1]; o[2] = rgb[2]; }
        }
    return 0;
}

/* ------------------------------------------------------------------------------------------ */
/* ref_sample_colour -- NEXT row: colour-volume lookup at world points     */
/* ------------------------------------------------------------------------------------------ */
/* The primitive under the paper's per-polygon texture maps: "Given the 3D world positions, the RGB value of any pixel
 * can be found by accessing the colour volume" (the positions are V_a + i * V_aV_green + j * V_aV_blue of
 * eq. 11-14, computed by the caller).  Reading S1 (the paper does not say how the volume is accessed): the
 * colour voxel whose cell contains the point -- index floor((p - origin) / vc) per axis, evaluated in binary32 as
 * (p - origin) * (1 / vc) -- nearest voxel, no interpolation; the packed word {R, G, B, wq} of that voxel, or 0 for a
 * point outside the volume.  pts: n x 3 floats (world); words_out: n uint32. */
int ref_sample_colour(const ref_vol_t *v, const uint32_t *col, const float *pts, int64_t n, uint32_t *words_out)
{
    if (!v || !col || (n > 0 && (!pts || !words_out)) || n < 0) return -1;
    const float vc = (v->extent / (float)v->nx) / (float)v->r, inv_vc = 1.0f / vc;
    const int cnx = v->nx * v->r, cny = v->ny * v->r, cnz = v->nz * v->r;
#pragma omp parallel for schedule(static)
    for (int64_t m = 0; m < n; ++m) {
        const float hx = floorf((pts[3 * m + 0] - v->origin[0]) * inv_vc);
        const float hy = floorf((pts[3 * m + 1] - v->origin[1]) * inv_vc);
        const float hz = floorf((pts[3 * m + 2] - v->origin[2]) * inv_vc);
        uint32_t w = 0;
        if (hx >= 0.0f && hx < (float)cnx && hy >= 0.0f && hy < (float)cny && hz >= 0.0f && hz < (float)cnz)
            w = col[((size_t)(int)hz * (size_t)cny + (size_t)(int)hy) * (size_t)cnx + (size_t)(int)hx];
        words_out[m] = w;
    }
    return 0;
}

/* ref_sample_colour_trilinear -- the same lookup with trilinear interpolation (second half).
 * Reading S2 (the paper does not say how the volume is accessed; nearest voxel = S1 above): voxel centres sit at
 * (idx + 0.5) * vc (A1), so the continuous grid coordinate of a point is g = (p - origin) / vc - 0.5 per axis; with
 * b = floor(g) and f = g - b, the 8 voxels b + {0,1}^3 carry the weights (1-f or f) per axis, multiplied as (wz * wy) * wx.
 * A voxel outside the volume or never observed (wq = 0) holds no colour: it contributes nothing, and the colour is
 * normalised over the voxels that do --  C = rint(sum w C / sum w)  per channel (half-even).  The weight byte is the plain
 * trilinear interpolation of the stored weights with unobserved voxels counted as 0:  A = rint(sum w wq)  -- so A tells how
 * much of the footprint has been seen.  No observed voxel in the footprint (or a non-finite point): word 0.
 * Canonical binary32, neighbours accumulated in the order z-major, then y, then x (dz, dy, dx = 0,0,0; 0,0,1; 0,1,0; ...),
 * each sum as fmaf(w, value, sum). */
int ref_sample_colour_trilinear(const ref_vol_t *v, const uint32_t *col, const float *pts, int64_t n, uint32_t *words_out)
{
    if (!v || !col || (n > 0 && (!pts || !words_out)) || n < 0) return -1;
    const float vc = (v->extent / (float)v->nx) / (float)v->r, inv_vc = 1.0f / vc;
    const int cn[3] = { v->nx * v->r, v->ny * v->r, v->nz * v->r };
#pragma omp parallel for schedule(static)
    for (int64_t m = 0; m < n; ++m) {
        float b[3], f[3];
        int ok = 1;
        for (int a = 0; a < 3; ++a) {
            const float g = (pts[3 * m + a] - v->origin[a]) * inv_vc - 0.5f;
            b[a] = floorf(g);
            f[a] = g - b[a];
            /* the footprint must touch the volume: b in [-1, cn - 1]; also rejects NaN and infinities */
            if (!(b[a] >= -1.0f && b[a] <= (float)(cn[a] - 1))) ok = 0;
        }
        uint32_t word = 0;
        if (ok) {
            float sw = 0.0f, sa = 0.0f, sc[3] = { 0.0f, 0.0f, 0.0f };
            for (int dz = 0; dz < 2; ++dz)
                for (int dy = 0; dy < 2; ++dy)
                    for (int dx = 0; dx < 2; ++dx) {
                        const int i = (int)b[0] + dx, j = (int)b[1] + dy, k = (int)b[2] + dz;
                        if (i < 0 || i >= cn[0] || j < 0 || j >= cn[1] || k < 0 || k >= cn[2]) continue;
                        const uint32_t cw = col[((size_t)k * (size_t)cn[1] + (size_t)j) * (size_t)cn[0] + (size_t)i];
                        if ((cw >> 24) == 0) continue;
                        const float wx = dx ? f[0] : 1.0f - f[0], wy = dy ? f[1] : 1.0f - f[1], wz = dz ? f[2] : 1.0f - f[2];
                        const float w = (wz * wy) * wx;
                        sw = sw + w;
                        sa = fmaf(w, (float)(cw >> 24), sa);
                        for (int ch = 0; ch < 3; ++ch) sc[ch] = fmaf(w, (float)((cw >> (8 * ch)) & 0xffu), sc[ch]);
                    }
            if (sw > 0.0f) {
                for (int ch = 0; ch < 3; ++ch) {
                    float cq = rintf(sc[ch] / sw);
                    int ci = cq < 0.0f ? 0 : (cq > 255.0f ? 255 : (int)cq);
                    word |= (uint32_t)ci << (8 * ch);
                }
                float aq = rintf(sa);
                int ai = aq < 0.0f ? 0 : (aq > 255.0f ? 255 : (int)aq);
                word |= (uint32_t)ai << 24;
            }
        }
        words_out[m] = word;
    }
    return 0;
}
