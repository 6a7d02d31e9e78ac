/*
 * volfusion.h -- C ABI of the B200-native per-frame volumetric fusion of arXiv 1602.06645
 * ("Creating Simplified 3D Models with High Quality Textures", Liu, Li, Ogunbona, Chow).
 *
 * One call, vol_integrate(), fuses one RGB-D frame into two device-resident volumes:
 *   - the geometry volume: projective TSDF integration of the depth map (the paper defers to
 *     KinectFusion/PCL, the exact definition is DESIGN.md readings A5/A6);
 *   - the asymmetrical colour volume: r x more voxels per axis over the same physical cube,
 *     updated from the calibrated HD RGB frame by eq. 5-10.
 * Every step runs in hand-written sm_100a CUDA kernels; there is no CPU fallback.
 *
 * Conventions
 *   - "T_a_b" is a row-major rigid 4x4 that maps b-coordinates to a-coordinates.
 *     (R_n, t_n) of eq. 5 = inverse(T_world_depth); (R_calib, t_calib) of eq. 3 = inverse(T_depth_rgb).
 *   - K matrices are row-major [fx 0 cx; 0 fy cy; 0 0 1] (eq. 1); pixel centres at integers.
 *   - Voxel (i,j,k) of a grid with voxel size s has its centre at origin + (idx + 0.5) * s (reading A1); both
 *     grids share origin and extent; geometry voxel i spans colour voxels r*i .. r*i + r - 1 per axis.
 *   - Layouts (little-endian, x fastest, linear index ((k*Ny + j)*Nx + i)):
 *       geometry word = int16 tsdf_q (bytes 0-1) | int16 w (bytes 2-3),  F = tsdf_q / 32767
 *       colour word   = u8 R | u8 G | u8 B | u8 wq (bytes 0..3),         W = wq / 255
 *     All-zero bytes = "never observed" (initial state).
 *   - Pointers are marked HOST or DEVICE.  Matrix arguments are HOST and copied at call time.  Frame buffers are
 *     borrowed and must stay valid until the stream has finished the enqueued work.
 *   - Every function returns VOL_OK (0) or a negative VOL_E_* code; validation happens before any launch, so a
 *     failed call leaves the volumes untouched.  Nothing throws or aborts across this boundary.
 *   - `stream` is a cudaStream_t passed as void* (NULL = default stream).  vol_integrate* and vol_reset are
 *     asynchronous on it; vol_download*, vol_upload and vol_frame_stats synchronise it before returning.
 *   - All calls on ONE vol_t must be ordered with respect to each other (one stream, or events between streams): the
 *     per-frame scratch of a volume -- control words, shell marks, work lists, pixel map, depth pyramid, staging sets,
 *     per-tile summaries -- exists once per volume, and two vol_integrate* / vol_frame_stats* / vol_raycast calls in
 *     flight on unordered streams would corrupt it (and the volumes).  Different vol_t are independent.
 *   - Frames enqueued directly one after the other are pipelined: the first kernel of vol_integrate (the per-pixel
 *     pre-pass, which reads only the frame and writes scratch kept in two sets) is a programmatic dependent launch, so
 *     behind the fused kernel of the previous frame it starts as that kernel's thread blocks retire, and it completes
 *     only after that kernel has.  Behind a copy, an event or any kernel that does not itself issue
 *     griddepcontrol.launch_dependents it starts in plain stream order.  The one obligation this puts on a caller: a
 *     kernel of the caller's own that PRODUCES the frame buffers, is enqueued immediately before vol_integrate and
 *     issues griddepcontrol.launch_dependents must issue it after its last write to them (as for any dependent).
 */
#ifndef VOLFUSION_H
#define VOLFUSION_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define VOL_OK       0
#define VOL_E_ARG   -1   /* null pointer, dims <= 0, dims_geo > 4096 x 2048 x 2048 (per shard), r not in 1..4, mu <= 0, unknown or combined variant, w_max not in 1..512,
                            non-zero skew, non-rigid T, image size <= 0, buffer too small, bad shard */
#define VOL_E_OOM   -2   /* device allocation failed */
#define VOL_E_CUDA  -3   /* a CUDA call failed (sticky: see vol_strerror) */
#define VOL_E_LOST  -4   /* vol_frontend_track only: the arguments were valid but the pose could not be estimated (too few
                            correspondences, normal equations not positive definite or too close to singular); the
                            volumes and the front end are intact and the caller may re-localise or skip the frame */
#define VOL_E_TOOBIG -5  /* vol_icp_step_static only: the maps need more scratch than the fixed static array holds */

/* geometry layers per shard slab (and per culling tile along z): rank `shard_rank` of `shard_world` owns the
 * geometry layers k with (k / VOL_SLAB) % shard_world == shard_rank, and the r*VOL_SLAB colour layers under each */
#define VOL_SLAB 8

typedef struct vol vol_t;   /* opaque; owns (or borrows) the two device buffers */

/* Alternative readings of passages the paper leaves open: each is the same
 * per-frame path with one step read differently, selected per volume at vol_create (vol_opts_t.variant); combinations
 * are rejected (VOL_E_ARG).
 *   VOL_VARIANT_HD_FROM_DEPTH_POINT  PAPER.md L115 read with eq. 2-4 (L71-81) literally: the HD pixel of a colour voxel is
 *                                    located from the 3D point of its depth pixel (eq. 7), not from the voxel's own position
 *   VOL_VARIANT_TSDF_ALONG_RAY       L33-35: the signed distance is measured along the voxel's viewing ray,
 *                                    (D - Z_vc) |P_vc| / Z_vc, not along the optical axis
 *   VOL_VARIANT_ADDITIVE_WEIGHT      W_new = min(W_pre + W, 1) instead of eq. 10 (L122) */
#define VOL_VARIANT_HD_FROM_DEPTH_POINT 1
#define VOL_VARIANT_TSDF_ALONG_RAY      2
#define VOL_VARIANT_ADDITIVE_WEIGHT     4

typedef struct {
    float   sigma_m;        /* colour distance gate sigma, metres; <= 0 selects the paper's 0.020 */
    float   gate;           /* weight gate factor; <= 0 selects the paper's 0.8 */
    void   *geo_dev;        /* DEVICE, optional caller-owned storage of info.geo_bytes (e.g. a torch tensor); NULL = library allocates.
                               16-byte aligned; zeroed by vol_create.  While the volume exists the library must stay its only
                               writer (it keeps per-tile summaries of the content): change it through vol_upload / vol_reset */
    void   *col_dev;        /* DEVICE, optional caller-owned storage of info.col_bytes; same rules */
    int32_t device;         /* CUDA device ordinal; < 0 = current device */
    int32_t shard_rank;     /* multi-GPU z-slab sharding; rank 0 of world 1 = whole volume */
    int32_t shard_world;    /* <= 0 is read as 1 */
    int32_t variant;        /* 0 = the method as DESIGN.md reads it, or ONE of VOL_VARIANT_* below */
} vol_opts_t;

typedef struct {
    int32_t  dims_geo[3];   /* full (unsharded) geometry dims Nx, Ny, Nz */
    int32_t  r;
    int32_t  dims_col[3];   /* r * dims_geo */
    int32_t  local_nz_geo;  /* geometry layers stored by this shard (== dims_geo[2] when unsharded) */
    float    voxel_geo_m, voxel_col_m;
    float    origin_m[3], extent_m, trunc_mu_m, sigma_m, gate;
    int32_t  w_max, device, shard_rank, shard_world, variant;
    uint64_t geo_bytes, col_bytes;      /* bytes stored by this shard */
    void    *geo_dev, *col_dev;         /* DEVICE pointers of this shard's storage */
} vol_info_t;

/* Per-frame statistics of the last vol_integrate* call.  tiles_total, tiles_geo and items_col are always valid; everything
 * else is only filled when counting is enabled (vol_set_counting), otherwise 0.
 * A voxel is *read* when the method reaches the load of its stored word (geometry: passes the frustum, non-zero-depth
 * and truncation tests; colour: passes the sigma gate with a valid view weight) and *changed* when the stored word
 * differs after the update.  The *_sectors_* figures count the distinct 32-byte sectors (8 x-adjacent words,
 * aligned in this shard's storage) that hold at least one read / changed voxel: the DRAM granularity of the same sets. */
typedef struct {
    uint64_t geo_read, geo_changed, col_read, col_changed;
    uint32_t tiles_total;   /* geometry tiles owned by this shard */
    uint32_t tiles_geo;     /* geometry tiles (32x4x8 voxels) with at least one sub-box to visit */
    uint32_t items_col;     /* colour work items (non-zero nibbles of the shell-mark words: up to 4 colour cells each) */
    uint32_t cells_col;     /* colour cells (8x4x4 colour voxels) visited */
    uint64_t geo_sectors_read, geo_sectors_written, col_sectors_read, col_sectors_written;
    uint64_t geo_visited;   /* geometry voxels the kernel projected (the read ones are a subset) */
    uint64_t col_gated;     /* colour voxels that went through the sigma gate (S4-S5; the read ones are a subset) */
    uint64_t geo_skippable; /* of geo_read: voxels of sub-boxes that hold nothing but saturated free space (tsdf_q = 32767,
                               w = w_max) and stay in free space this frame -- read and unchanged by definition; the plain
                               (non-counting) kernel leaves those sub-boxes out, so it touches geo_read - geo_skippable */
    uint64_t geo_sectors_skippable;  /* the same in 32-byte sectors (of geo_sectors_read) */
    uint32_t subs_geo;      /* geometry sub-boxes (8x4x4 voxels) visited */
    uint32_t jobs_mark;     /* shell-mark jobs (one or two per 4 x 4 pixel patch with colour-eligible pixels) */
} vol_stats_t;

/* size of the raw record vol_frame_stats_async copies out */
#define VOL_STATS_RAW_BYTES 128

/* Create a volume pair.  dims_geo: HOST int32[3]; r in 1..4; origin_m: HOST
 * float[3], world position of the volume corner; extent_m: side length along x (cubic voxels of extent/dims_geo[0]);
 * trunc_mu_m > 0; w_max in 1..512 (exactness bound of the fp32 running average); opts nullable.
 * Both volumes start zeroed.  *out is only written on success. */
int vol_create(vol_t **out, const int32_t dims_geo[3], int32_t r, const float origin_m[3], float extent_m,
               float trunc_mu_m, int32_t w_max, const vol_opts_t *opts);

/* Fuse one frame (PAPER.md L91-124 per colour voxel; TSDF per geometry voxel).
 * depth_u16_dev: DEVICE, wd*hd uint16 millimetres, 0 = invalid; rgb8_dev: DEVICE, wh*hh*3 bytes
 * interleaved R,G,B; the four matrices are HOST float arrays (see conventions).  Asynchronous on `stream`. */
int vol_integrate(vol_t *v, const uint16_t *depth_u16_dev, int32_t wd, int32_t hd,
                  const uint8_t *rgb8_dev, int32_t wh, int32_t hh,
                  const float T_world_depth[16], const float K_depth[9], const float K_rgb[9],
                  const float T_depth_rgb[16], void *stream);

/* Same, with HOST frame buffers (ideally pinned): copies both images to library-owned device staging buffers, then runs
 * vol_integrate on them, all ordered on `stream`.  The copies use a stream of the library's own and two staging sets, so
 * frames enqueued back to back overlap: the images of frame n + 1 travel while the kernels of frame n run.  The host
 * buffers may be reused once `stream` has passed this call's work. */
int vol_integrate_host(vol_t *v, const uint16_t *depth_u16_host, int32_t wd, int32_t hd,
                       const uint8_t *rgb8_host, int32_t wh, int32_t hh,
                       const float T_world_depth[16], const float K_depth[9], const float K_rgb[9],
                       const float T_depth_rgb[16], void *stream);

/* Ray-cast both volumes into the image of a virtual pinhole camera (the prediction for tracking and the
 * live preview; the paper gives no equations, the definition is DESIGN.md "Ray casting", readings R1-R6): per pixel the
 * ray ((x-cx)/fx, (y-cy)/fy, 1) is sampled every geometry-voxel of camera depth from t_near_m to t_far_m; the first
 * front-face zero crossing of the TSDF (nearest voxel, observed voxels only) gives the depth by linear interpolation, the
 * colour voxel containing the hit point gives the colour.
 * depth_dev: DEVICE, w*h float32, metres along the camera's z axis, 0 = no surface; rgb8_dev: DEVICE, w*h*3 bytes R,G,B
 * (black where there is no surface or no colour), nullable.  T_world_cam / K: HOST, as for vol_integrate.  Unsharded
 * volumes only (VOL_E_ARG otherwise).  Asynchronous on `stream`; reads the volumes and writes, beside its outputs, only
 * per-volume scratch of its own: the first cast after the geometry volume has changed (vol_integrate*, vol_upload,
 * vol_reset) rebuilds the flags that let rays skip bricks, tiles and 8 x 4 x 4 sub-boxes without an observed tsdf <= 0
 * (about 30 us on a 512^3 volume) -- which is why ray casts on one volume fall under the stream-ordering rule above too. */
int vol_raycast(const vol_t *v, int32_t w, int32_t h, const float T_world_cam[16], const float K[9], float t_near_m,
                float t_far_m, float *depth_dev, uint8_t *rgb8_dev, void *stream);

/* The same with the TSDF of a sample interpolated trilinearly from the 8 voxels whose centres surround it (reading R7; a
 * sample with a never-observed or outside voxel among the 8 is unknown).  A plane inside the truncation band is rendered
 * at its exact depth whatever the phase of the samples, and the depth map has no voxel-sized terraces: the tracker can
 * build its prediction from it without the millimetre rounding and bilateral pass that the nearest-voxel map needs (F8).
 * Same arguments, same rules. */
int vol_raycast_trilinear(const vol_t *v, int32_t w, int32_t h, const float T_world_cam[16], const float K[9], float t_near_m,
                float t_far_m, float *depth_dev, uint8_t *rgb8_dev, void *stream);

/* Look up the colour volume at n world points ("given the 3D world positions, the RGB value of any pixel can
 * be found by accessing the colour volume" -- the positions of a polygon's texture map are V_a + i V_aV_green + j V_aV_blue
 * of eq. 11-14, computed by the caller).  points_dev: DEVICE, n x 3 float32 (x, y, z in world metres); words_dev: DEVICE,
 * n uint32: the packed colour word (layout above) of the colour voxel whose cell contains the point (nearest voxel), 0 for
 * a point outside the volume.  Unsharded volumes only.  Asynchronous on `stream`. */
int vol_sample_colour(const vol_t *v, const float *points_dev, int64_t n, uint32_t *words_dev, void *stream);
/* The same with trilinear interpolation between the 8 surrounding voxel centres (reading S2): voxels outside
 * the volume or never observed (wq = 0) are left out and the colour is normalised over the others; the weight byte of the
 * returned word is the trilinear interpolation of the stored weights with those voxels counted as 0 (coverage of the
 * footprint).  0 where no observed voxel is in reach or the point is not finite.  Same arguments and rules. */
int vol_sample_colour_trilinear(const vol_t *v, const float *points_dev, int64_t n, uint32_t *words_dev, void *stream);

/* Copy this shard's volumes to HOST buffers of at least info.geo_bytes / info.col_bytes (either may be NULL to skip). */
int vol_download(const vol_t *v, void *geo_host, size_t geo_bytes, void *col_host, size_t col_bytes, void *stream);
/* Gather single voxels: geo_idx / col_idx are HOST int64 linear indices into the FULL grids (must be owned by this
 * shard); the packed words are written to HOST geo_words / col_words.  Used for sampled parity at full size. */
int vol_download_voxels(const vol_t *v, const int64_t *geo_idx, int64_t n_geo, uint32_t *geo_words,
                        const int64_t *col_idx, int64_t n_col, uint32_t *col_words, void *stream);
/* Overwrite this shard's volumes from HOST buffers (resume / test seeding); either may be NULL to skip.  Synchronises. */
int vol_upload(vol_t *v, const void *geo_host, const void *col_host, void *stream);
/* Zero both volumes (asynchronous). */
int vol_reset(vol_t *v, void *stream);
int vol_info(const vol_t *v, vol_info_t *out);
/* Host-only helper (no CUDA call): the geometry layers rank `shard_rank` of `shard_world` owns out of nz, in storage order.
 * Writes at most `cap` of them to layers_out (HOST, nullable) and returns how many there are, or VOL_E_ARG. */
int vol_shard_layers(int32_t nz, int32_t shard_rank, int32_t shard_world, int32_t *layers_out, int32_t cap);
/* Enable (1) / disable (0) the four voxel counters of vol_stats_t (a separately compiled kernel variant). */
int vol_set_counting(vol_t *v, int32_t on);
/* Statistics of the last frame (synchronises `stream`; copies VOL_STATS_RAW_BYTES device -> host). */
int vol_frame_stats(vol_t *v, vol_stats_t *out, void *stream);
/* The same without the synchronisation, for callers that enqueue frames back to back: copies the raw record of the
 * frame last enqueued on `stream` to raw_host (HOST, pinned, 8-byte aligned, >= VOL_STATS_RAW_BYTES), asynchronously, in stream order;
 * once the stream has passed it, vol_stats_decode (host only, no CUDA call) turns it into a vol_stats_t. */
int vol_frame_stats_async(vol_t *v, void *raw_host, void *stream);
int vol_stats_decode(const vol_t *v, const void *raw_host, vol_stats_t *out);
/* Enable per-kernel CUDA-event timing of subsequent vol_integrate calls / read the last frame's kernel times in
 * milliseconds: ms[0] the per-pixel pre-pass (S1), ms[1] always 0 (kept for the layout: the classification of tiles and sub-boxes
 * for both volumes (S9) runs inside the fused kernel), ms[2] the fused kernel (S2-S9).  Synchronises. */
int vol_set_profiling(vol_t *v, int32_t on);
int vol_last_kernel_ms(vol_t *v, float ms[3]);
/* Number of kernels one vol_integrate call launches (vol_integrate_host may launch one more: its fused kernel runs as a
 * depth-only part and a colour part around the arrival of the HD frame). */
int vol_launches_per_frame(const vol_t *v);
/* Device self-test of the branch-free exact reciprocal / division used on the hot path against the correctly rounded
 * library intrinsics: mismatches[0] = reciprocal over every binary32 in its operand range, mismatches[1] = TSDF
 * running-average quotient over its operand domain (every denominator 1..513 x numerators; all of them when
 * exhaustive != 0, every 257th otherwise), mismatches[2] = colour quotient of eq. 9 and the two weight roundings over
 * stored weights x a sweep of new-sample weights (every binary32 in [2^-20, 255] when exhaustive != 0, every 1021st
 * otherwise) x 16 colour / HD byte pairs.  All must be 0.  Runs on the current device; synchronises. */
int vol_selftest(uint64_t mismatches[3], int32_t exhaustive);
void vol_destroy(vol_t *v);
/* Text for a return code.  For VOL_E_OOM / VOL_E_CUDA it names the failing CUDA call of the most recent failure in this
 * process (one process-global buffer: not meant to be read while other threads are making calls). */
const char *vol_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* VOLFUSION_H */
