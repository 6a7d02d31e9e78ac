/*
 * volfrontend.h -- C ABI of the depth front end and the ICP tracking step, B200 (sm_100a).
 *
 * PAPER.md L33 (section III, KinectFusion background): "A vertex map and normal map pyramid based on input depth map is
 * calculated; the value is then used to estimate the camera motion using iterative closest point (ICP) algorithm [3] in
 * conjunction with a predicted surface vertex map", L35: "The predicted surface vertex map used for camera tracking is
 * obtained by ray tracing the geometry volume."  With these calls the poses that vol_integrate takes as inputs can be
 * estimated from the depth frames themselves.  The paper gives no equations for these steps; the definitions are readings
 * F1-F7 of DESIGN.md section 8f (oracle: oracle/frontend.py):
 *   F1  bilateral filter of the raw depth (7 x 7 window; spatial Gaussian sigma_s px; range Gaussian sigma_r over whole
 *       millimetres, cut at ceil(3 sigma_r) mm; invalid pixels neither filtered nor used) -> float32 metres
 *   F2  pyramid: level l + 1 = mean of the valid pixels of each 2 x 2 block within 3 sigma_r of the block's first pixel;
 *       intrinsics f / 2, (c - 1/2) / 2
 *   F3  vertex map  V = K^-1 (x, y, 1) D                                  (eq. 7)
 *   F4  normal map  N = normalise((V(x+1,y) - V) x (V(x,y+1) - V))        (eq. 8; points away from the camera)
 *   F5  ICP step: per measured pixel p = R v + t, m = R n; nearest pixel of K_l p in the predicted maps; kept if the
 *       prediction is valid, |q - p| <= dist_m and m . n_q >= cos_min; r = n_q . (q - p), J = [p x n_q ; n_q];
 *       A = sum J J^T, b = sum J r in binary64
 *   F6  A xi = b, xi = (omega, v); T <- [exp(omega) R, exp(omega) t + v]
 *   F7  coarse to fine, iterations[l] steps at level l
 *   F8  the ray-cast prediction (nearest-voxel sampling leaves voxel-sized steps) is rounded to whole millimetres and passed
 *       through F1 before F2-F4
 * All map arithmetic is binary32 without fused multiply-add in a fixed order, so the maps are bit-identical to the oracle's.
 *
 * Conventions as in volfusion.h: pointers are marked HOST or DEVICE; K is row-major [fx 0 cx; 0 fy cy; 0 0 1] of level 0;
 * 4 x 4 matrices are row-major rigid transforms; `stream` is a cudaStream_t passed as void*; every function returns VOL_OK
 * or a negative VOL_E_* code (volfusion.h) and validates before any launch.  A front end belongs to one image size.
 */
#ifndef VOLFRONTEND_H
#define VOLFRONTEND_H

#include <stdint.h>
#include "volfusion.h"

#ifdef __cplusplus
extern "C" {
#endif

typedef struct vol_frontend vol_frontend_t;   /* opaque; owns the measured and the predicted map pyramids (device) */

typedef struct {
    float   sigma_s_px;     /* F1 spatial sigma, pixels; <= 0 selects 4.5 */
    float   sigma_r_m;      /* F1 / F2 range sigma, metres; <= 0 selects 0.030 */
    float   dist_m;         /* F5 distance gate; <= 0 selects 0.10 */
    float   cos_min;        /* F5 normal gate (cosine); <= 0 selects 0.94 */
    int32_t device;         /* CUDA device ordinal; < 0 = current device */
    float   cond_min;       /* F6 conditioning gate, see vol_frontend_track; <= 0 selects VOL_ICP_COND_MIN; must be < 1 */
    int32_t trilinear_prediction;   /* != 0: vol_frontend_predict casts its rays with vol_raycast_trilinear (reading R7) and builds the
                                       maps from that depth map directly, without F8 (which exists to smooth the voxel-sized terraces
                                       of the nearest-voxel ray caster) */
} vol_frontend_opts_t;

#define VOL_ICP_COND_MIN 1e-3f
#define VOL_ICP_SUMS 29     /* 21 = upper triangle of A row by row (A00 A01 .. A05 A11 ..), 6 = b, sum r^2, count */

/* w, h: size of level 0; both must be divisible by 2^(levels-1); levels in 1..6; opts nullable. */
int vol_frontend_create(vol_frontend_t **out, int32_t w, int32_t h, int32_t levels, const vol_frontend_opts_t *opts);
void vol_frontend_destroy(vol_frontend_t *fe);

/* The measured side: F1 on the raw depth frame (DEVICE, w*h uint16 mm, 0 = invalid), then F2-F4 for every level.
 * K: HOST.  Asynchronous on `stream`. */
int vol_frontend_measure(vol_frontend_t *fe, const uint16_t *depth_u16_dev, const float K[9], void *stream);

/* The predicted side from a float depth map (DEVICE, w*h float32 metres along the camera's z axis, 0 = no surface -- the
 * output of vol_raycast).  filter != 0: F8 (round to millimetres, F1), then F2-F4 -- for ray-cast maps; filter == 0: F2-F4
 * directly -- for maps that are already smooth.  Asynchronous. */
int vol_frontend_predict_depth(vol_frontend_t *fe, const float *depth_m_dev, const float K[9], int32_t filter, void *stream);

/* The same with the ray casting included: vol_raycast of `v` from T_world_cam (the pose the prediction is made from,
 * normally the previous frame's), then vol_frontend_predict_depth with the filter (F8) -- or, with
 * opts.trilinear_prediction, vol_raycast_trilinear and no filter.  Unsharded volumes only.  Asynchronous. */
int vol_frontend_predict(vol_frontend_t *fe, const vol_t *v, const float T_world_cam[16], const float K[9], float t_near_m,
                         float t_far_m, void *stream);

/* One F5 step at `level` with the estimate T_pred_cur (HOST: current camera -> prediction camera).  sums_host: HOST,
 * VOL_ICP_SUMS doubles.  The sums are bit-reproducible from run to run on one device: threads, warps and blocks add in a
 * fixed order and the blocks' partial sums meet in integer accumulators (resolution 2^-60), whose result does not depend
 * on the order of arrival.  Synchronises `stream`. */
int vol_frontend_icp_step(vol_frontend_t *fe, int32_t level, const float T_pred_cur[16], double *sums_host, void *stream);

/* F7: the whole coarse-to-fine loop in one cooperative launch (F5 and F6 on the device, F6 in binary64).  T_init: HOST, nullable (identity);
 * iterations: HOST int32[levels], iterations[l] steps at level l; T_out: HOST, the final estimate current camera ->
 * prediction camera (so T_world_cur = T_world_pred * T_out); rms_out / count_out: nullable, residual and number of
 * correspondences of the last step.  Returns VOL_E_ARG for invalid arguments (nothing was launched) and VOL_E_LOST when
 * tracking is lost: a step found fewer than 100 correspondences (status 1), A was not positive definite (2), or A was
 * too close to singular (3): the smallest Cholesky pivot relative to its diagonal entry, min_j d_j / A_jj in (0, 1], fell
 * below cond_min -- some motion is then not observable from the maps (a sphere, a plane, a scene symmetric about the axis
 * the camera turns about) and the solve would return noise along it.  The default, 1e-3, lies between what structured
 * scenes give (0.3 .. 0.5 for rooms and table tops, 8e-3 for a 10 cm object filling a twentieth of the image) and what a
 * sphere or a wall gives through sensor noise (1e-4 .. 4e-4 at the coarsest level; below 1e-6 on exact depth).  What the
 * gate cannot see: sensor noise in the normals adds information that is not there, so a NOISY surface of revolution turned
 * about its axis reads 0.3 like any scene, the images carry no trace of the motion, and F7 returns "no motion" with a small
 * residual; no geometric tracker can do better.  T_out then holds the last estimate that was
 * accepted, rms / count those of the failing step.  The result is bit-reproducible (see vol_frontend_icp_step).
 * Synchronises `stream`. */
int vol_frontend_track(vol_frontend_t *fe, const float T_init[16], const int32_t *iterations, float T_out[16], double *rms_out,
                       int64_t *count_out, void *stream);

/* Status (0 ok, 1, 2, 3 as above), pyramid level and conditioning min_j d_j / A_jj of the last step of the most recent
 * vol_frontend_track; every pointer nullable.  HOST values, no device work. */
int vol_frontend_track_info(const vol_frontend_t *fe, int32_t *status_out, int32_t *level_out, double *conditioning_out);

/* One F5 step that ALLOCATES NOTHING -- for callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid it).  No front-end object: the caller passes the maps of one level and receives the sums, all
 * DEVICE memory.  V_dev / N_dev: vertex and normal map of the current (measured) frame, Vp_dev / Np_dev: of the prediction;
 * each w*h pixels of 4 floats (x, y, z, 0), 16-byte aligned, row-major, invalid = normal (0, 0, 0) -- the layout the front end
 * keeps on the device.  K: HOST, intrinsics of THIS level.  T_pred_cur: HOST, current camera -> prediction camera.  dist_m /
 * cos_min: the F5 gates (<= 0 selects 0.10 / 0.94).  sums_dev: DEVICE, VOL_ICP_SUMS doubles, written in stream order.
 * Asynchronous on `stream`; calls no cudaMalloc, cudaFree, cudaMallocHost or any other allocating routine, and does not
 * synchronise.  The same sums as vol_frontend_icp_step up to binary64 summation order (blocks' partial sums are added in a
 * fixed order, so the result is bit-reproducible as well).
 * Limit: the step's scratch (29 doubles per block of 32 x 8 pixels) is a static device array of VOL_ICP_STATIC_MAX_BLOCKS
 * slots, 1.8 MiB, held by every GPU that loads the library until the process exits; ceil(w / 32) * ceil(h / 8) beyond that
 * is VOL_E_TOOBIG (vol_strerror names the sizes) -- 8192 blocks cover maps up to 1920 x 1088 or 2048 x 1024.  The device is
 * the CURRENT device (ordinals 0..63).  ALL calls share the one array per device: calls that may overlap on the GPU (two
 * streams, two host threads on two streams) RACE on it and return garbage; order them on one stream or with events. */
#define VOL_ICP_STATIC_MAX_BLOCKS 8192
int vol_icp_step_static(const float *V_dev, const float *N_dev, const float *Vp_dev, const float *Np_dev, int32_t w, int32_t h,
                        const float K[9], const float T_pred_cur[16], float dist_m, float cos_min, double *sums_dev, void *stream);

/* Copy the maps of one level to the host (tests, debugging): which = 0 measured, 1 predicted; depth_host: wl*hl floats,
 * vertex_host / normal_host: wl*hl*3 floats; any may be NULL.  Synchronises `stream`. */
int vol_frontend_maps(const vol_frontend_t *fe, int32_t which, int32_t level, float *depth_host, float *vertex_host,
                      float *normal_host, void *stream);

#ifdef __cplusplus
}
#endif
#endif
