// volfusion.cu -- C ABI (include/volfusion.h) and host side (S0, launches) of the fused integration.
//
// Build: nvcc -gencode arch=compute_100a,code=sm_100a -O3 -lineinfo --fmad=false -Xcompiler -fPIC,-ffp-contract=off
//             -shared volfusion.cu -o libvolfusion.so
#include "../../include/volfusion.h"

#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>

#include "fused.cuh"
#include "params.cuh"
#include "prepass.cuh"
#include "raycast.cuh"

using vf::Params;

static char g_err[256] = "";

#define CK(call)                                                                                         \
    do {                                                                                                 \
        cudaError_t e_ = (call);                                                                         \
        if (e_ != cudaSuccess) {                                                                         \
            snprintf(g_err, sizeof g_err, "%s:%d %s: %s", __FILE__, __LINE__, #call, cudaGetErrorString(e_)); \
            return e_ == cudaErrorMemoryAllocation ? VOL_E_OOM : VOL_E_CUDA;                             \
        }                                                                                                \
    } while (0)

constexpr int N_STAGE = 2;          // staging sets of vol_integrate_host

struct vol {
    Params p;                       // volume fields filled at create; frame fields per call
    int device;
    bool own_geo, own_col;
    size_t geo_bytes, col_bytes;
    // per-frame-size scratch
    int scratch_wd, scratch_hd;
    size_t pyr_entries;
    // staging for vol_integrate_host
    // staging for vol_integrate_host: two sets used alternately, so that the copies of one frame overlap the kernels of the
    // frame before it (ev_used[i]: the kernels that last read set i have finished)
    uint16_t *stage_depth[N_STAGE]; size_t stage_depth_bytes;
    uint8_t *stage_rgb[N_STAGE]; size_t stage_rgb_bytes;
    cudaEvent_t ev_depth[N_STAGE], ev_rgb[N_STAGE], ev_used[N_STAGE];
    bool used_valid[N_STAGE];
    unsigned host_seq;
    // fused-kernel launch shape
    int n_sms, fused_blocks;
    bool counting, profiling;
    unsigned frame_seq;             // frames enqueued so far: selects the scratch set (parity) and the control block (mod CTRL_SETS)
    // per-frame scratch, two sets used alternately (Params::pixmap, depthf, pyr, jobs point into set frame_seq & 1), and the
    // CTRL_SETS control blocks (Params::ctrl = ctrl_base + (frame_seq % CTRL_SETS) * CTRL_N): the pre-pass of a frame may run
    // while the fused kernel of the frame before it is still reading its own set
    float4 *scr_pixmap[2]; float *scr_depthf[2]; uint32_t *scr_pyr[2]; uint4 *scr_jobs[2];
    uint32_t *ctrl_base, *ctrl_last;    // ctrl_last: block of the most recent frame (vol_frame_stats*)
    // ray casting: exact "holds an observed tsdf <= 0" flags per sub-box (raycast.cuh, k_sub_neg), rebuilt by the first ray
    // cast after the geometry volume has changed (content_version counts vol_integrate*, vol_upload, vol_reset)
    uint8_t *sub_neg, *tile_any, *brick_any, *sub_dil, *tile_dil, *brick_dil; int sbx, sby, sbz;
    mutable unsigned long long content_version, sub_neg_version, dil_version;
    cudaEvent_t ev[4];
    bool ev_valid;
    // vol_integrate_host: the frames are copied on a stream of the library's own
    cudaStream_t copy_stream;
};

#ifndef VF_PIPELINE
#define VF_PIPELINE true
#endif
// one kernel launch; `dependent` = programmatic dependent launch on the previous kernel of the stream
template <typename... Args>
static cudaError_t launch(void (*kernel)(const Params, Args...), dim3 grid, int block, cudaStream_t s, bool dependent, const Params &p, Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = dim3(block); cfg.dynamicSmemBytes = 0; cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = dependent ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kernel, p, args...);
}

// the fused kernel for colour ratio R, with or without the voxel counters, in the volume's reading of the method
using FusedFn = void (*)(const Params, int);
template <int R>
static FusedFn fused_kernel(bool counting, int variant)
{
    switch (variant) {
        case vf::VAR_HD_FROM_DEPTH_POINT: return counting ? vf::k_fused<R, true, vf::VAR_HD_FROM_DEPTH_POINT> : vf::k_fused<R, false, vf::VAR_HD_FROM_DEPTH_POINT>;
        case vf::VAR_TSDF_ALONG_RAY:      return counting ? vf::k_fused<R, true, vf::VAR_TSDF_ALONG_RAY> : vf::k_fused<R, false, vf::VAR_TSDF_ALONG_RAY>;
        case vf::VAR_ADDITIVE_WEIGHT:     return counting ? vf::k_fused<R, true, vf::VAR_ADDITIVE_WEIGHT> : vf::k_fused<R, false, vf::VAR_ADDITIVE_WEIGHT>;
        default:                          return counting ? vf::k_fused<R, true, vf::VAR_PAPER> : vf::k_fused<R, false, vf::VAR_PAPER>;
    }
}

static int set_device(const vol *v) { CK(cudaSetDevice(v->device)); return VOL_OK; }

// counting variant: bytes of sector map i (one bit per 8 words of the geometry (i < 2) or colour volume, rounded up to words)
static size_t sec_map_bytes(const vol *v, int i)
{
    const size_t words = (i < 2 ? v->geo_bytes : v->col_bytes) / 4u;
    return ((words + 7u) / 8u + 31u) / 32u * 4u + 4u;
}

// rigid inverse in fp64 with left-to-right sums, rounded once to fp32 (S0).  Returns false if T is not rigid.
static bool rigid_inverse(const float T[16], float Rout[9], float tout[3])
{
    if (T[12] != 0.0f || T[13] != 0.0f || T[14] != 0.0f || T[15] != 1.0f) return false;
    for (int i = 0; i < 16; ++i) if (!(std::fabs(T[i]) <= 1e6f)) return false;      // also rejects NaN / inf
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {
            double s = 0.0;
            for (int k = 0; k < 3; ++k) s += (double)T[4 * k + i] * (double)T[4 * k + j];
            if (std::fabs(s - (i == j ? 1.0 : 0.0)) > 1e-4) return false;
        }
    const double det = (double)T[0] * ((double)T[5] * T[10] - (double)T[6] * T[9]) - (double)T[1] * ((double)T[4] * T[10] - (double)T[6] * T[8]) +
                       (double)T[2] * ((double)T[4] * T[9] - (double)T[5] * T[8]);
    if (!(det > 0.0)) return false;
    for (int i = 0; i < 3; ++i) {
        for (int j = 0; j < 3; ++j) Rout[3 * i + j] = T[4 * j + i];
        double s = (double)T[4 * 0 + i] * (double)T[4 * 0 + 3];
        s = s + (double)T[4 * 1 + i] * (double)T[4 * 1 + 3];
        s = s + (double)T[4 * 2 + i] * (double)T[4 * 2 + 3];
        tout[i] = (float)(-s);
    }
    return true;
}

static bool intrinsics_ok(const float K[9])
{
    for (int i = 0; i < 9; ++i) if (!std::isfinite(K[i])) return false;
    return K[0] > 0.0f && K[4] > 0.0f && K[1] == 0.0f && K[3] == 0.0f && K[6] == 0.0f && K[7] == 0.0f && K[8] == 1.0f;
}

// conservative camera-axis half extents of a world-axis box with half sizes (hx, hy, hz)
static void box_extents(const float R[9], double hx, double hy, double hz, double slack, float &ex, float &ey, float &ez)
{
    ex = (float)(std::fabs(R[0]) * hx + std::fabs(R[1]) * hy + std::fabs(R[2]) * hz + slack);
    ey = (float)(std::fabs(R[3]) * hx + std::fabs(R[4]) * hy + std::fabs(R[5]) * hz + slack);
    ez = (float)(std::fabs(R[6]) * hx + std::fabs(R[7]) * hy + std::fabs(R[8]) * hz + slack);
}

// culling only: exact (fp64) inverse of the fp32 world->camera map (R, t), rounded to fp32: camera -> world
static void camera_to_world(const float R[9], const float t[3], float Rw[9], float tw[3])
{
    const double a = R[0], b = R[1], c = R[2], d = R[3], e = R[4], f = R[5], g = R[6], h = R[7], i = R[8];
    const double det = a * (e * i - f * h) - b * (d * i - f * g) + c * (d * h - e * g);
    const double inv[9] = {(e * i - f * h) / det, (c * h - b * i) / det, (b * f - c * e) / det,
                           (f * g - d * i) / det, (a * i - c * g) / det, (c * d - a * f) / det,
                           (d * h - e * g) / det, (b * g - a * h) / det, (a * e - b * d) / det};
    for (int k = 0; k < 9; ++k) Rw[k] = (float)inv[k];
    for (int k = 0; k < 3; ++k) tw[k] = (float)(-(inv[3 * k] * t[0] + inv[3 * k + 1] * t[1] + inv[3 * k + 2] * t[2]));
}

extern "C" const char *vol_strerror(int code)
{
    switch (code) {
        case VOL_OK: return "ok";
        case VOL_E_ARG: return "invalid argument";
        case VOL_E_OOM: return g_err[0] ? g_err : "out of device memory";
        case VOL_E_CUDA: return g_err[0] ? g_err : "CUDA error";
        case VOL_E_LOST: return g_err[0] ? g_err : "tracking lost";
        case VOL_E_TOOBIG: return g_err[0] ? g_err : "input larger than the static scratch";
        default: return "unknown error code";
    }
}

extern "C" int vol_create(vol_t **out, const int32_t dims_geo[3], int32_t r, const float origin_m[3], float extent_m,
                          float trunc_mu_m, int32_t w_max, const vol_opts_t *opts)
{
    if (!out || !dims_geo || !origin_m) return VOL_E_ARG;
    if (dims_geo[0] <= 0 || dims_geo[1] <= 0 || dims_geo[2] <= 0) return VOL_E_ARG;
    if (r < 1 || r > 4 || !(extent_m > 0.0f) || !(trunc_mu_m > 0.0f) || w_max < 1 || w_max > 512) return VOL_E_ARG;
    if (!(extent_m <= 1e6f) || !(trunc_mu_m <= 1e6f)) return VOL_E_ARG;           // also rejects NaN / inf
    for (int i = 0; i < 3; ++i) if (!(std::fabs(origin_m[i]) <= 1e6f)) return VOL_E_ARG;
    if ((int64_t)dims_geo[0] * r > INT32_MAX / 4 || (int64_t)dims_geo[1] * r > INT32_MAX / 4 || (int64_t)dims_geo[2] * r > INT32_MAX / 4) return VOL_E_ARG;
    int rank = 0, world = 1, device = -1;
    float sigma = 0.020f, gate = 0.8f;
    int variant = 0;
    if (opts) {
        variant = opts->variant;
        if (variant != 0 && variant != VOL_VARIANT_HD_FROM_DEPTH_POINT && variant != VOL_VARIANT_TSDF_ALONG_RAY &&
            variant != VOL_VARIANT_ADDITIVE_WEIGHT) return VOL_E_ARG;
        if (opts->sigma_m > 0.0f) sigma = opts->sigma_m;
        if (opts->gate > 0.0f) gate = opts->gate;
        world = opts->shard_world > 0 ? opts->shard_world : 1;
        rank = opts->shard_rank;
        device = opts->device;
        if (rank < 0 || rank >= world) return VOL_E_ARG;
    }
    if (device < 0) CK(cudaGetDevice(&device));
    CK(cudaSetDevice(device));

    vol *v = new (std::nothrow) vol();
    if (!v) return VOL_E_OOM;
    memset(v, 0, sizeof *v);
    v->device = device;
    Params &p = v->p;
    p.nx = dims_geo[0]; p.ny = dims_geo[1]; p.nz = dims_geo[2]; p.r = r;
    p.cnx = r * p.nx; p.cny = r * p.ny; p.cnz = r * p.nz;
    p.shard_rank = rank; p.shard_world = world;
    const int slabs = (p.nz + vf::TZ - 1) / vf::TZ;
    const int my_slabs = slabs > rank ? (slabs - rank + world - 1) / world : 0;
    // stored layers: full slabs except a possibly partial last global slab
    int local_nz = 0;
    for (int s = 0; s < my_slabs; ++s) {
        const int g = s * world + rank;
        local_nz += (g + 1) * vf::TZ <= p.nz ? vf::TZ : p.nz - g * vf::TZ;
    }
    p.local_nz = local_nz;
    p.tiles_x = (p.nx + vf::TX - 1) / vf::TX; p.tiles_y = (p.ny + vf::TY - 1) / vf::TY; p.tiles_z_local = my_slabs;
    const int64_t n_tiles = (int64_t)p.tiles_x * p.tiles_y * my_slabs;
    if (p.tiles_x > vf::ITEM_MAX_TX || p.tiles_y > vf::ITEM_MAX_TY || my_slabs > vf::ITEM_MAX_TZ || n_tiles > INT32_MAX / 128) { delete v; return VOL_E_ARG; }
    p.n_tiles = (int)n_tiles;
    p.ox = origin_m[0]; p.oy = origin_m[1]; p.oz = origin_m[2];
    p.vs = extent_m / (float)p.nx;
    p.vc = p.vs / (float)r;
    p.inv_vc = 1.0f / p.vc;
    p.mu = trunc_mu_m; p.neg_mu = -trunc_mu_m; p.inv_mu = 1.0f / trunc_mu_m;
    p.sigma = sigma; p.sig2 = sigma * sigma; p.gate = gate; p.w_max = w_max; p.variant = variant;
    v->geo_bytes = (size_t)local_nz * p.ny * p.nx * 4u;
    v->col_bytes = (size_t)local_nz * r * p.cny * p.cnx * 4u;

    int rc = VOL_OK;
    auto fail = [&](int code) { vol_destroy(v); return code; };
    if (opts && opts->geo_dev) p.geo = (uint32_t *)opts->geo_dev;
    else if (v->geo_bytes) {
        if (cudaMalloc(&p.geo, v->geo_bytes) != cudaSuccess) { cudaGetLastError(); snprintf(g_err, sizeof g_err, "cudaMalloc(%zu) geometry volume failed", v->geo_bytes); return fail(VOL_E_OOM); }
        v->own_geo = true;
    }
    if (opts && opts->col_dev) p.col = (uint32_t *)opts->col_dev;
    else if (v->col_bytes) {
        if (cudaMalloc(&p.col, v->col_bytes) != cudaSuccess) { cudaGetLastError(); snprintf(g_err, sizeof g_err, "cudaMalloc(%zu) colour volume failed", v->col_bytes); return fail(VOL_E_OOM); }
        v->own_col = true;
    }
    if (((uintptr_t)p.geo | (uintptr_t)p.col) & 15u) return fail(VOL_E_ARG);       // whole sectors per warp access
    if (v->geo_bytes && cudaMemset(p.geo, 0, v->geo_bytes) != cudaSuccess) rc = VOL_E_CUDA;
    if (v->col_bytes && cudaMemset(p.col, 0, v->col_bytes) != cudaSuccess) rc = VOL_E_CUDA;
    const size_t nt = (size_t)(p.n_tiles > 0 ? p.n_tiles : 1), nw = nt * (size_t)vf::words_per_tile(r);
    if (cudaMalloc(&p.work_geo, sizeof(uint32_t) * nt) != cudaSuccess) rc = VOL_E_OOM;
    if (rc == VOL_OK && cudaMemset(p.work_geo, 0, sizeof(uint32_t) * nt) != cudaSuccess) rc = VOL_E_CUDA;   // empty slots are zero
    p.work_col_cap = (uint32_t)(nw * 8);
    if (cudaMalloc(&p.work_col, sizeof(uint2) * nw * 8) != cudaSuccess) rc = VOL_E_OOM;
    if (cudaMalloc(&p.marks, sizeof(uint32_t) * nw) != cudaSuccess) rc = VOL_E_OOM;
    if (rc == VOL_OK && cudaMemset(p.marks, 0, sizeof(uint32_t) * nw) != cudaSuccess) rc = VOL_E_CUDA;
    if (cudaMalloc(&p.tile_sat, nt) != cudaSuccess || cudaMalloc(&p.tile_skip, nt) != cudaSuccess) rc = VOL_E_OOM;
    if (rc == VOL_OK && (cudaMemset(p.tile_sat, 0, nt) != cudaSuccess || cudaMemset(p.tile_skip, 0, nt) != cudaSuccess)) rc = VOL_E_CUDA;
    v->sbx = p.tiles_x * vf::SUBX; v->sby = p.tiles_y; v->sbz = (p.n_tiles > 0 ? p.n_tiles / (p.tiles_x * p.tiles_y) : 0) * vf::SUBZ;
    if (cudaMalloc(&v->sub_neg, nt * vf::SUBX * vf::SUBZ) != cudaSuccess || cudaMalloc(&v->tile_any, nt) != cudaSuccess ||
        cudaMalloc(&v->sub_dil, nt * vf::SUBX * vf::SUBZ) != cudaSuccess || cudaMalloc(&v->tile_dil, nt) != cudaSuccess) rc = VOL_E_OOM;
    v->content_version = 1; v->sub_neg_version = 0;
    if (cudaMalloc(&p.tile_neg, nt) != cudaSuccess) rc = VOL_E_OOM;
    if (rc == VOL_OK && cudaMemset(p.tile_neg, 0, nt) != cudaSuccess) rc = VOL_E_CUDA;
    p.bricks_x = p.tiles_x; p.bricks_y = (p.tiles_y + 7) / 8; p.bricks_z = (my_slabs + 3) / 4;
    const size_t nb = (size_t)p.bricks_x * p.bricks_y * p.bricks_z + 1;
    if (cudaMalloc(&p.brick_neg, nb) != cudaSuccess || cudaMalloc(&v->brick_any, nb) != cudaSuccess || cudaMalloc(&v->brick_dil, nb) != cudaSuccess) rc = VOL_E_OOM;
    if (rc == VOL_OK && cudaMemset(p.brick_neg, 0, nb) != cudaSuccess) rc = VOL_E_CUDA;
    // one 128-byte statistics record (8 words, then 12 counters: read back together by vol_frame_stats*), then the queue control words
    static_assert(sizeof(uint32_t) * vf::ST_N + sizeof(unsigned long long) * vf::CNT_N == VOL_STATS_RAW_BYTES && vf::CTRL_Q0 * 4 == VOL_STATS_RAW_BYTES,
                  "raw statistics record: 8 words, then 12 counters");
    if (cudaMalloc(&v->ctrl_base, sizeof(uint32_t) * vf::CTRL_N * vf::CTRL_SETS) != cudaSuccess) rc = VOL_E_OOM;
    if (rc == VOL_OK && cudaMemset(v->ctrl_base, 0, sizeof(uint32_t) * vf::CTRL_N * vf::CTRL_SETS) != cudaSuccess) rc = VOL_E_CUDA;
    for (int i = 0; i < vf::CTRL_SETS && rc == VOL_OK; ++i)                                                 // "no valid depth yet"
        if (cudaMemset(v->ctrl_base + i * vf::CTRL_N + vf::Q_DMIN, 0xff, sizeof(uint32_t)) != cudaSuccess) rc = VOL_E_CUDA;
    if (rc == VOL_OK) { p.ctrl = v->ctrl_base; p.ctrl_next = v->ctrl_base + vf::CTRL_N; v->ctrl_last = v->ctrl_base; }
    if (rc == VOL_OK) p.counters = reinterpret_cast<unsigned long long *>(p.ctrl + vf::ST_N);
    if (rc != VOL_OK) { cudaGetLastError(); return fail(rc); }

    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return fail(VOL_E_CUDA);
    v->n_sms = prop.multiProcessorCount;
    int occ = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, vf::k_fused<2, false, 0>, vf::CTA, 0) != cudaSuccess || occ < 1) {
        snprintf(g_err, sizeof g_err, "fused kernel cannot be resident on device %d (built for sm_100a): %s", device, cudaGetErrorString(cudaGetLastError()));
        return fail(VOL_E_CUDA);
    }
    v->fused_blocks = v->n_sms * occ;
    for (int i = 0; i < 4; ++i) if (cudaEventCreate(&v->ev[i]) != cudaSuccess) return fail(VOL_E_CUDA);
    if (cudaStreamCreateWithFlags(&v->copy_stream, cudaStreamNonBlocking) != cudaSuccess) return fail(VOL_E_CUDA);
    for (int i = 0; i < N_STAGE; ++i)
        if (cudaEventCreateWithFlags(&v->ev_depth[i], cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&v->ev_rgb[i], cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&v->ev_used[i], cudaEventDisableTiming) != cudaSuccess) return fail(VOL_E_CUDA);
    v->ev_valid = false;
    if (cudaDeviceSynchronize() != cudaSuccess) return fail(VOL_E_CUDA);
    *out = v;
    return VOL_OK;
}

static void free_scratch(vol *v)
{
    for (int i = 0; i < 2; ++i) {
        if (v->scr_pixmap[i]) cudaFree(v->scr_pixmap[i]);
        if (v->scr_pyr[i]) cudaFree(v->scr_pyr[i]);
        if (v->scr_depthf[i]) cudaFree(v->scr_depthf[i]);
        if (v->scr_jobs[i]) cudaFree(v->scr_jobs[i]);
        v->scr_pixmap[i] = nullptr; v->scr_pyr[i] = nullptr; v->scr_depthf[i] = nullptr; v->scr_jobs[i] = nullptr;
    }
}

extern "C" void vol_destroy(vol_t *v)
{
    if (!v) return;
    cudaSetDevice(v->device);
    cudaDeviceSynchronize();
    if (v->own_geo && v->p.geo) cudaFree(v->p.geo);
    if (v->own_col && v->p.col) cudaFree(v->p.col);
    if (v->p.work_geo) cudaFree(v->p.work_geo);
    if (v->p.work_col) cudaFree(v->p.work_col);
    if (v->p.marks) cudaFree(v->p.marks);
    if (v->p.tile_neg) cudaFree(v->p.tile_neg);
    if (v->sub_neg) cudaFree(v->sub_neg);
    if (v->tile_any) cudaFree(v->tile_any);
    if (v->brick_any) cudaFree(v->brick_any);
    if (v->sub_dil) cudaFree(v->sub_dil);
    if (v->tile_dil) cudaFree(v->tile_dil);
    if (v->brick_dil) cudaFree(v->brick_dil);
    if (v->p.tile_sat) cudaFree(v->p.tile_sat);
    if (v->p.tile_skip) cudaFree(v->p.tile_skip);
    for (int i = 0; i < 4; ++i) if (v->p.sec_map[i]) cudaFree(v->p.sec_map[i]);
    if (v->p.brick_neg) cudaFree(v->p.brick_neg);
    if (v->ctrl_base) cudaFree(v->ctrl_base);
    free_scratch(v);
    for (int i = 0; i < N_STAGE; ++i) {
        if (v->stage_depth[i]) cudaFree(v->stage_depth[i]);
        if (v->stage_rgb[i]) cudaFree(v->stage_rgb[i]);
        if (v->ev_depth[i]) cudaEventDestroy(v->ev_depth[i]);
        if (v->ev_rgb[i]) cudaEventDestroy(v->ev_rgb[i]);
        if (v->ev_used[i]) cudaEventDestroy(v->ev_used[i]);
    }
    for (int i = 0; i < 4; ++i) if (v->ev[i]) cudaEventDestroy(v->ev[i]);
    if (v->copy_stream) cudaStreamDestroy(v->copy_stream);
    cudaGetLastError();
    delete v;
}

// (re)allocate the per-frame-size scratch (both sets): pixel map, float depth map, depth pyramid, shell-mark jobs
static int ensure_scratch(vol *v, int wd, int hd)
{
    if (v->scratch_wd == wd && v->scratch_hd == hd && v->scr_pixmap[0]) return VOL_OK;
    Params &p = v->p;
    v->scratch_wd = v->scratch_hd = 0;                       // nothing is valid until every allocation below has succeeded
    if (v->scr_pixmap[0]) CK(cudaDeviceSynchronize());
    free_scratch(v);
    p.jobs_cap = (uint32_t)((size_t)((wd + 3) / 4 * 4) * (size_t)((hd + 3) / 4 * 4));     // one per pixel at most
    int l = 0; size_t off = 0;
    for (; l < 3; ++l) {                                     // blocks of 8, 16, 32 pixels
        const int bs = 8 << l;
        p.pyr_w[l] = (wd + bs - 1) / bs; p.pyr_h[l] = (hd + bs - 1) / bs; p.pyr_off[l] = (int)off;
        off += (size_t)p.pyr_w[l] * p.pyr_h[l];
    }
    p.pyr_levels = 3;
    v->pyr_entries = off;
    for (int i = 0; i < 2; ++i) {
        CK(cudaMalloc(&v->scr_depthf[i], sizeof(float) * (size_t)wd * hd));
        CK(cudaMalloc(&v->scr_jobs[i], sizeof(uint4) * (size_t)p.jobs_cap));
        CK(cudaMalloc(&v->scr_pixmap[i], sizeof(float4) * (size_t)wd * hd));
        CK(cudaMalloc(&v->scr_pyr[i], sizeof(uint32_t) * off));
    }
    v->scratch_wd = wd; v->scratch_hd = hd;
    return VOL_OK;
}

// rgb_ready: optional event the colour update (the only reader of the HD frame) has to wait for.  split: run the geometry
// half of the fused kernel before that wait and the colour half after it (worth it when the HD frame is still on its way);
// otherwise the stream waits first and the whole queue goes in one launch.
static int integrate_impl(vol_t *v, const uint16_t *depth_u16_dev, int32_t wd, int32_t hd, const uint8_t *rgb8_dev,
                          int32_t wh, int32_t hh, const float T_world_depth[16], const float K_depth[9],
                          const float K_rgb[9], const float T_depth_rgb[16], void *stream, cudaEvent_t rgb_ready, bool split)
{
    if (!v || !depth_u16_dev || !rgb8_dev || !T_world_depth || !K_depth || !K_rgb || !T_depth_rgb) return VOL_E_ARG;
    if (wd <= 0 || hd <= 0 || wh <= 0 || hh <= 0 || wd > 16384 || hd > 16384 || wh > 16384 || hh > 16384) return VOL_E_ARG;
    if (!intrinsics_ok(K_depth) || !intrinsics_ok(K_rgb)) return VOL_E_ARG;
    Params p = v->p;
    if (!rigid_inverse(T_world_depth, p.R, p.t) || !rigid_inverse(T_depth_rgb, p.Rc, p.tc)) return VOL_E_ARG;
    int rc = set_device(v); if (rc) return rc;
    rc = ensure_scratch(v, wd, hd); if (rc) return rc;
    p = v->p;                                                  // scratch pointers / pyramid shape
    rigid_inverse(T_world_depth, p.R, p.t); rigid_inverse(T_depth_rgb, p.Rc, p.tc);
    p.fx = K_depth[0]; p.fy = K_depth[4]; p.cx = K_depth[2]; p.cy = K_depth[5];
    p.fxh = K_rgb[0]; p.fyh = K_rgb[4]; p.cxh = K_rgb[2]; p.cyh = K_rgb[5];
    p.wd = wd; p.hd = hd; p.wh = wh; p.hh = hh;
    p.wd_f = (float)wd; p.hd_f = (float)hd; p.wh_f = (float)wh; p.hh_f = (float)hh;
    p.depth = depth_u16_dev; p.rgb = rgb8_dev;
    // culling only: slack for the fp32 evaluation of box centres / world points, tile extents, camera -> world map
    const double mag = std::fabs((double)p.t[0]) + std::fabs((double)p.t[1]) + std::fabs((double)p.t[2]) +
                       std::fabs((double)p.ox) + std::fabs((double)p.oy) + std::fabs((double)p.oz) + (double)p.vs * (p.nx + p.ny + p.nz);
    const double slack = 1e-4 + 2e-5 * mag;
    p.slack = (float)slack;
    box_extents(p.R, 0.5 * vf::TX * p.vs, 0.5 * vf::TY * p.vs, 0.5 * vf::TZ * p.vs, slack, p.tile_ex, p.tile_ey, p.tile_ez);
    box_extents(p.R, 0.5 * (vf::TX / vf::SUBX) * p.vs, 0.5 * vf::TY * p.vs, 0.5 * (vf::TZ / vf::SUBZ) * p.vs, slack, p.sub_ex, p.sub_ey, p.sub_ez);
    p.parity = (int)(v->frame_seq & 1u);
    p.pixmap = v->scr_pixmap[p.parity]; p.depthf = v->scr_depthf[p.parity]; p.pyr = v->scr_pyr[p.parity]; p.jobs = v->scr_jobs[p.parity];
    p.ctrl = v->ctrl_base + (size_t)(v->frame_seq % (unsigned)vf::CTRL_SETS) * vf::CTRL_N;
    p.ctrl_next = v->ctrl_base + (size_t)((v->frame_seq + 1u) % (unsigned)vf::CTRL_SETS) * vf::CTRL_N;
    p.counters = reinterpret_cast<unsigned long long *>(p.ctrl + vf::ST_N);
    p.counting = v->counting ? 1 : 0;
    p.sigma_g = (float)((double)p.sigma * 1.0001 + slack);
    camera_to_world(p.R, p.t, p.Rw, p.tw);
    if (p.n_tiles == 0) return VOL_OK;

    cudaStream_t s = (cudaStream_t)stream;
    if (rgb_ready && !split) { CK(cudaStreamWaitEvent(s, rgb_ready, 0)); rgb_ready = nullptr; }
    if (v->counting) {
        CK(cudaMemsetAsync(p.counters, 0, sizeof(unsigned long long) * vf::CNT_N, s));
        for (int i = 0; i < 4; ++i) CK(cudaMemsetAsync(p.sec_map[i], 0, sec_map_bytes(v, i), s));
    }
    if (v->profiling) CK(cudaEventRecord(v->ev[0], s));
    const dim3 g0((wd + 31) / 32, (hd + 31) / 32);
    const int g2 = v->fused_blocks;
    const bool cnt = v->counting;
    // Both kernels are launched with programmatic stream serialization.  k_fused's CTAs may be scheduled while the pre-pass
    // drains (it signals griddepcontrol.launch_dependents), and they wait for its completion and memory flush with
    // griddepcontrol.wait before touching anything it wrote.  The pre-pass of the NEXT frame, if it follows directly on the
    // stream, may start while this frame's k_fused is running out of work -- it touches nothing that kernel uses (scratch
    // set, control block) and does not complete before it (k_prepass); behind anything else it starts in stream order.
#define VF_LAUNCH(RR)                                                                   \
    do {                                                                                \
        const FusedFn kf = fused_kernel<RR>(cnt, p.variant);                            \
        CK(launch(vf::k_prepass<RR>, g0, 256, s, VF_PIPELINE, p));                            \
        ++v->frame_seq; ++v->content_version; v->ctrl_last = p.ctrl;                    \
        if (v->profiling) { CK(cudaEventRecord(v->ev[1], s)); CK(cudaEventRecord(v->ev[2], s)); } \
        if (rgb_ready) {   /* everything but the colour items now, those once the HD frame has arrived */ \
            CK(launch(kf, dim3(g2), vf::CTA, s, true, p, (int)vf::PHASE_GEO));          \
            CK(cudaStreamWaitEvent(s, rgb_ready, 0));                                    \
            CK(launch(kf, dim3(g2), vf::CTA, s, false, p, (int)vf::PHASE_COL));         \
        } else {                                                                        \
            CK(launch(kf, dim3(g2), vf::CTA, s, true, p, (int)vf::PHASE_ALL));          \
        }                                                                               \
    } while (0)
    switch (p.r) {
        case 1: VF_LAUNCH(1); break;
        case 2: VF_LAUNCH(2); break;
        case 3: VF_LAUNCH(3); break;
        default: VF_LAUNCH(4); break;
    }
#undef VF_LAUNCH
    if (v->profiling) { CK(cudaEventRecord(v->ev[3], s)); v->ev_valid = true; }
    CK(cudaGetLastError());
    return VOL_OK;
}

extern "C" int vol_integrate(vol_t *v, const uint16_t *depth_u16_dev, int32_t wd, int32_t hd, const uint8_t *rgb8_dev,
                             int32_t wh, int32_t hh, const float T_world_depth[16], const float K_depth[9],
                             const float K_rgb[9], const float T_depth_rgb[16], void *stream)
{
    return integrate_impl(v, depth_u16_dev, wd, hd, rgb8_dev, wh, hh, T_world_depth, K_depth, K_rgb, T_depth_rgb, stream, nullptr, false);
}

extern "C" int vol_integrate_host(vol_t *v, const uint16_t *depth_u16_host, int32_t wd, int32_t hd, const uint8_t *rgb8_host,
                                  int32_t wh, int32_t hh, const float T_world_depth[16], const float K_depth[9],
                                  const float K_rgb[9], const float T_depth_rgb[16], void *stream)
{
    if (!v || !depth_u16_host || !rgb8_host) return VOL_E_ARG;
    if (wd <= 0 || hd <= 0 || wh <= 0 || hh <= 0 || wd > 16384 || hd > 16384 || wh > 16384 || hh > 16384) return VOL_E_ARG;
    if (!T_world_depth || !K_depth || !K_rgb || !T_depth_rgb || !intrinsics_ok(K_depth) || !intrinsics_ok(K_rgb)) return VOL_E_ARG;
    float Rt[9], tt[3];
    if (!rigid_inverse(T_world_depth, Rt, tt) || !rigid_inverse(T_depth_rgb, Rt, tt)) return VOL_E_ARG;
    int rc = set_device(v); if (rc) return rc;
    const size_t db = (size_t)wd * hd * sizeof(uint16_t), cb = (size_t)wh * hh * 3;
    if (v->stage_depth_bytes < db || v->stage_rgb_bytes < cb) {            // (re)allocate both sets
        CK(cudaDeviceSynchronize());
        const size_t nd = db > v->stage_depth_bytes ? db : v->stage_depth_bytes, nc = cb > v->stage_rgb_bytes ? cb : v->stage_rgb_bytes;
        for (int i = 0; i < N_STAGE; ++i) {
            if (v->stage_depth[i]) cudaFree(v->stage_depth[i]);
            if (v->stage_rgb[i]) cudaFree(v->stage_rgb[i]);
            v->stage_depth[i] = nullptr; v->stage_rgb[i] = nullptr; v->used_valid[i] = false;
        }
        v->stage_depth_bytes = v->stage_rgb_bytes = 0;
        for (int i = 0; i < N_STAGE; ++i) { CK(cudaMalloc(&v->stage_depth[i], nd)); CK(cudaMalloc(&v->stage_rgb[i], nc)); }
        v->stage_depth_bytes = nd; v->stage_rgb_bytes = nc;
    }
    cudaStream_t s = (cudaStream_t)stream;
    const int set = (int)(v->host_seq++ % (unsigned)N_STAGE), prev = (set + N_STAGE - 1) % N_STAGE;
    // Both images go over the library's copy stream into staging set `set`, ordered only after the kernels that last read
    // that set (two frames ago) -- so they overlap the previous frame's kernels when the caller enqueues frames back to back.
    if (v->used_valid[set]) CK(cudaStreamWaitEvent(v->copy_stream, v->ev_used[set], 0));
    CK(cudaMemcpyAsync(v->stage_depth[set], depth_u16_host, db, cudaMemcpyHostToDevice, v->copy_stream));
    CK(cudaEventRecord(v->ev_depth[set], v->copy_stream));
    CK(cudaMemcpyAsync(v->stage_rgb[set], rgb8_host, cb, cudaMemcpyHostToDevice, v->copy_stream));
    CK(cudaEventRecord(v->ev_rgb[set], v->copy_stream));
    // Is the previous frame still being worked on?  Then this frame's HD image (91 % of the bytes) will have arrived by the
    // time its kernels start, and the whole queue goes in one launch.  Otherwise (the caller waits for every frame) the
    // geometry half runs while the HD image is still on its way and only the colour half waits for it.
    const bool busy = v->used_valid[prev] && cudaEventQuery(v->ev_used[prev]) == cudaErrorNotReady;
    cudaGetLastError();
    CK(cudaStreamWaitEvent(s, v->ev_depth[set], 0));
    rc = integrate_impl(v, v->stage_depth[set], wd, hd, v->stage_rgb[set], wh, hh, T_world_depth, K_depth, K_rgb, T_depth_rgb, stream,
                        v->ev_rgb[set], !busy);
    if (rc) return rc;
    CK(cudaStreamWaitEvent(s, v->ev_rgb[set], 0));             // (already passed, except on a shard without tiles)
    CK(cudaEventRecord(v->ev_used[set], s));
    v->used_valid[set] = true;
    return VOL_OK;
}

static int raycast_impl(const vol_t *v, int32_t w, int32_t h, const float T_world_cam[16], const float K[9], float t_near_m,
                        float t_far_m, float *depth_dev, uint8_t *rgb8_dev, void *stream, bool trilinear)
{
    if (!v || !T_world_cam || !K || !depth_dev) return VOL_E_ARG;
    if (w <= 0 || h <= 0 || w > 16384 || h > 16384 || !intrinsics_ok(K)) return VOL_E_ARG;
    if (!(t_near_m >= 0.0f) || !(t_far_m >= t_near_m) || !(t_far_m <= 1e6f)) return VOL_E_ARG;
    if (v->p.shard_world != 1) return VOL_E_ARG;               // a shard does not hold the whole volume
    float Rt[9], tt[3];
    if (!rigid_inverse(T_world_cam, Rt, tt)) return VOL_E_ARG;  // only used as the rigidity check
    int rc = set_device(v); if (rc) return rc;
    vf::RayParams q;
    q.w = w; q.h = h; q.fx = K[0]; q.fy = K[4]; q.cx = K[2]; q.cy = K[5];
    for (int i = 0; i < 12; ++i) q.T[i] = T_world_cam[i];
    q.t_near = t_near_m; q.t_far = t_far_m; q.depth = depth_dev; q.rgb = rgb8_dev;
    if (v->p.n_tiles == 0) return VOL_OK;
    q.sub_neg = v->sub_neg; q.sbx = v->sbx; q.sby = v->sby; q.tile_any = v->tile_any; q.brick_any = v->brick_any;
    if (v->sub_neg_version != v->content_version) {            // (stream-ordered with the calls that changed the volume: volfusion.h)
        CK(cudaMemsetAsync(v->brick_any, 0, (size_t)v->p.bricks_x * v->p.bricks_y * v->p.bricks_z, (cudaStream_t)stream));
        vf::k_sub_neg<<<(v->p.n_tiles + 7) / 8, 256, 0, (cudaStream_t)stream>>>(v->p, v->sub_neg, v->sbx, v->sby, v->sbz, v->tile_any, v->brick_any);
        v->sub_neg_version = v->content_version;
    }
    q.sub_dil = v->sub_dil; q.tile_dil = v->tile_dil; q.brick_dil = v->brick_dil;
    if (trilinear && v->dil_version != v->content_version) {
        const int tz = v->p.n_tiles / (v->p.tiles_x * v->p.tiles_y);
        const long long ns = (long long)v->sbx * v->sby * v->sbz, nb = (long long)v->p.bricks_x * v->p.bricks_y * v->p.bricks_z;
        const unsigned b0 = (unsigned)((ns + 255) / 256), b1 = (unsigned)((v->p.n_tiles + 255) / 256), b2 = (unsigned)((nb + 255) / 256);
        const vf::DilateJob j0 = {v->sub_neg, v->sub_dil, v->sbx, v->sby, v->sbz, 0u};
        const vf::DilateJob j1 = {v->tile_any, v->tile_dil, v->p.tiles_x, v->p.tiles_y, tz, b0};
        const vf::DilateJob j2 = {v->brick_any, v->brick_dil, v->p.bricks_x, v->p.bricks_y, v->p.bricks_z, b0 + b1};
        vf::k_dilate<<<b0 + b1 + b2, 256, 0, (cudaStream_t)stream>>>(j0, j1, j2);
        v->dil_version = v->content_version;
    }
    const dim3 grid((w + 7) / 8, (h + 7) / 8);
    if (trilinear) vf::k_raycast_trilinear<<<grid, 64, 0, (cudaStream_t)stream>>>(v->p, q);
    else vf::k_raycast<<<grid, 64, 0, (cudaStream_t)stream>>>(v->p, q);
    CK(cudaGetLastError());
    return VOL_OK;
}

extern "C" int vol_raycast(const vol_t *v, int32_t w, int32_t h, const float T_world_cam[16], const float K[9], float t_near_m,
                           float t_far_m, float *depth_dev, uint8_t *rgb8_dev, void *stream)
{
    return raycast_impl(v, w, h, T_world_cam, K, t_near_m, t_far_m, depth_dev, rgb8_dev, stream, false);
}

extern "C" int vol_raycast_trilinear(const vol_t *v, int32_t w, int32_t h, const float T_world_cam[16], const float K[9], float t_near_m,
                                     float t_far_m, float *depth_dev, uint8_t *rgb8_dev, void *stream)
{
    return raycast_impl(v, w, h, T_world_cam, K, t_near_m, t_far_m, depth_dev, rgb8_dev, stream, true);
}

extern "C" int vol_sample_colour(const vol_t *v, const float *points_dev, int64_t n, uint32_t *words_dev, void *stream)
{
    if (!v || n < 0 || (n > 0 && (!points_dev || !words_dev))) return VOL_E_ARG;
    if (v->p.shard_world != 1) return VOL_E_ARG;               // a shard does not hold the whole volume
    int rc = set_device(v); if (rc) return rc;
    if (n == 0 || v->p.n_tiles == 0) return VOL_OK;
    if ((n + 255) / 256 > 0x7fffffffLL) return VOL_E_ARG;
    vf::k_sample_colour<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(v->p, points_dev, (long long)n, words_dev);
    CK(cudaGetLastError());
    return VOL_OK;
}

extern "C" int vol_sample_colour_trilinear(const vol_t *v, const float *points_dev, int64_t n, uint32_t *words_dev, void *stream)
{
    if (!v || n < 0 || (n > 0 && (!points_dev || !words_dev))) return VOL_E_ARG;
    if (v->p.shard_world != 1) return VOL_E_ARG;               // a shard does not hold the whole volume
    int rc = set_device(v); if (rc) return rc;
    if (n == 0 || v->p.n_tiles == 0) return VOL_OK;
    if ((n + 255) / 256 > 0x7fffffffLL) return VOL_E_ARG;
    vf::k_sample_colour_trilinear<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(v->p, points_dev, (long long)n, words_dev);
    CK(cudaGetLastError());
    return VOL_OK;
}

extern "C" int vol_download(const vol_t *v, void *geo_host, size_t geo_bytes, void *col_host, size_t col_bytes, void *stream)
{
    if (!v) return VOL_E_ARG;
    if ((geo_host && geo_bytes < v->geo_bytes) || (col_host && col_bytes < v->col_bytes)) return VOL_E_ARG;
    int rc = set_device(v); if (rc) return rc;
    cudaStream_t s = (cudaStream_t)stream;
    if (geo_host && v->geo_bytes) CK(cudaMemcpyAsync(geo_host, v->p.geo, v->geo_bytes, cudaMemcpyDeviceToHost, s));
    if (col_host && v->col_bytes) CK(cudaMemcpyAsync(col_host, v->p.col, v->col_bytes, cudaMemcpyDeviceToHost, s));
    CK(cudaStreamSynchronize(s));
    return VOL_OK;
}

extern "C" int vol_upload(vol_t *v, const void *geo_host, const void *col_host, void *stream)
{
    if (!v) return VOL_E_ARG;
    int rc = set_device(v); if (rc) return rc;
    cudaStream_t s = (cudaStream_t)stream;
    if (geo_host && v->geo_bytes) CK(cudaMemcpyAsync(v->p.geo, geo_host, v->geo_bytes, cudaMemcpyHostToDevice, s));
    if (col_host && v->col_bytes) CK(cudaMemcpyAsync(v->p.col, col_host, v->col_bytes, cudaMemcpyHostToDevice, s));
    ++v->content_version;
    if (geo_host && v->p.n_tiles > 0) {                       // unknown content: no tile or brick may be skipped
        CK(cudaMemsetAsync(v->p.tile_sat, 0, (size_t)v->p.n_tiles, s));
        CK(cudaMemsetAsync(v->p.tile_neg, 1, (size_t)v->p.n_tiles, s));
        CK(cudaMemsetAsync(v->p.brick_neg, 1, (size_t)v->p.bricks_x * v->p.bricks_y * v->p.bricks_z, s));
    }
    CK(cudaStreamSynchronize(s));
    return VOL_OK;
}

extern "C" int vol_reset(vol_t *v, void *stream)
{
    if (!v) return VOL_E_ARG;
    int rc = set_device(v); if (rc) return rc;
    cudaStream_t s = (cudaStream_t)stream;
    ++v->content_version;
    if (v->geo_bytes) CK(cudaMemsetAsync(v->p.geo, 0, v->geo_bytes, s));
    if (v->col_bytes) CK(cudaMemsetAsync(v->p.col, 0, v->col_bytes, s));
    if (v->p.n_tiles > 0) {
        CK(cudaMemsetAsync(v->p.tile_sat, 0, (size_t)v->p.n_tiles, s));
        CK(cudaMemsetAsync(v->p.tile_neg, 0, (size_t)v->p.n_tiles, s));
        CK(cudaMemsetAsync(v->p.brick_neg, 0, (size_t)v->p.bricks_x * v->p.bricks_y * v->p.bricks_z, s));
    }
    return VOL_OK;
}

// gather kernel for vol_download_voxels: idx are LOCAL linear indices
__global__ void k_gather(const uint32_t *__restrict__ src, const long long *__restrict__ idx, long long n, uint32_t *__restrict__ dst)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) dst[i] = src[idx[i]];
}

// global linear index of a grid with layers of `scale` x the geometry layers -> this shard's local index (or -1)
static long long to_local(const vol *v, long long idx, int scale)
{
    const Params &p = v->p;
    const long long nx = (long long)p.nx * scale, ny = (long long)p.ny * scale, nz = (long long)p.nz * scale;
    if (idx < 0 || idx >= nx * ny * nz) return -1;
    const long long k = idx / (nx * ny), rem = idx % (nx * ny);
    const long long slab = k / ((long long)vf::TZ * scale), in = k % ((long long)vf::TZ * scale);
    if (slab % p.shard_world != p.shard_rank) return -1;
    return ((slab / p.shard_world) * vf::TZ * scale + in) * nx * ny + rem;
}

static int gather(const vol *v, const uint32_t *src, const int64_t *idx, int64_t n, int scale, uint32_t *out, cudaStream_t s)
{
    if (n == 0) return VOL_OK;
    long long *h = new (std::nothrow) long long[n];
    if (!h) return VOL_E_OOM;
    for (int64_t i = 0; i < n; ++i) { h[i] = to_local(v, idx[i], scale); if (h[i] < 0) { delete[] h; return VOL_E_ARG; } }
    long long *d_idx = nullptr; uint32_t *d_out = nullptr;
    int rc = VOL_OK;
    if (cudaMalloc(&d_idx, sizeof(long long) * n) != cudaSuccess || cudaMalloc(&d_out, sizeof(uint32_t) * n) != cudaSuccess) rc = VOL_E_OOM;
    if (rc == VOL_OK && cudaMemcpyAsync(d_idx, h, sizeof(long long) * n, cudaMemcpyHostToDevice, s) != cudaSuccess) rc = VOL_E_CUDA;
    if (rc == VOL_OK) {
        k_gather<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(src, d_idx, n, d_out);
        if (cudaMemcpyAsync(out, d_out, sizeof(uint32_t) * n, cudaMemcpyDeviceToHost, s) != cudaSuccess) rc = VOL_E_CUDA;
        if (cudaStreamSynchronize(s) != cudaSuccess) rc = VOL_E_CUDA;
    }
    if (rc != VOL_OK) snprintf(g_err, sizeof g_err, "vol_download_voxels: %s", cudaGetErrorString(cudaGetLastError()));
    cudaFree(d_idx); cudaFree(d_out); delete[] h;
    return rc;
}

extern "C" int vol_download_voxels(const vol_t *v, const int64_t *geo_idx, int64_t n_geo, uint32_t *geo_words,
                                   const int64_t *col_idx, int64_t n_col, uint32_t *col_words, void *stream)
{
    if (!v || n_geo < 0 || n_col < 0 || (n_geo && (!geo_idx || !geo_words)) || (n_col && (!col_idx || !col_words))) return VOL_E_ARG;
    int rc = set_device(v); if (rc) return rc;
    rc = gather(v, v->p.geo, geo_idx, n_geo, 1, geo_words, (cudaStream_t)stream); if (rc) return rc;
    return gather(v, v->p.col, col_idx, n_col, v->p.r, col_words, (cudaStream_t)stream);
}

extern "C" int vol_info(const vol_t *v, vol_info_t *o)
{
    if (!v || !o) return VOL_E_ARG;
    const Params &p = v->p;
    memset(o, 0, sizeof *o);
    o->dims_geo[0] = p.nx; o->dims_geo[1] = p.ny; o->dims_geo[2] = p.nz; o->r = p.r;
    for (int i = 0; i < 3; ++i) o->dims_col[i] = o->dims_geo[i] * p.r;
    o->local_nz_geo = p.local_nz; o->voxel_geo_m = p.vs; o->voxel_col_m = p.vc;
    o->origin_m[0] = p.ox; o->origin_m[1] = p.oy; o->origin_m[2] = p.oz; o->extent_m = p.vs * (float)p.nx;
    o->trunc_mu_m = p.mu; o->sigma_m = p.sigma; o->gate = p.gate; o->w_max = p.w_max; o->device = v->device; o->variant = p.variant;
    o->shard_rank = p.shard_rank; o->shard_world = p.shard_world;
    o->geo_bytes = v->geo_bytes; o->col_bytes = v->col_bytes; o->geo_dev = p.geo; o->col_dev = p.col;
    return VOL_OK;
}

extern "C" int vol_shard_layers(int32_t nz, int32_t rank, int32_t world, int32_t *layers_out, int32_t cap)
{
    if (nz <= 0 || world <= 0 || rank < 0 || rank >= world || cap < 0) return VOL_E_ARG;
    int n = 0;
    for (int k = 0; k < nz; ++k)
        if ((k / vf::TZ) % world == rank) { if (layers_out && n < cap) layers_out[n] = k; ++n; }
    return n;
}

extern "C" int vol_set_counting(vol_t *v, int32_t on)
{
    if (!v) return VOL_E_ARG;
    if (on && !v->p.sec_map[0]) {                              // the sector maps of the counting variant, on first use
        int rc = set_device(v); if (rc) return rc;
        for (int i = 0; i < 4; ++i) {
            if (cudaMalloc(&v->p.sec_map[i], sec_map_bytes(v, i)) != cudaSuccess) {
                cudaGetLastError();
                for (int k = 0; k < 4; ++k) if (v->p.sec_map[k]) { cudaFree(v->p.sec_map[k]); v->p.sec_map[k] = nullptr; }
                return VOL_E_OOM;
            }
        }
    }
    v->counting = on != 0;
    return VOL_OK;
}
extern "C" int vol_set_profiling(vol_t *v, int32_t on) { if (!v) return VOL_E_ARG; v->profiling = on != 0; v->ev_valid = false; return VOL_OK; }
extern "C" int vol_launches_per_frame(const vol_t *v) { return v ? 2 : VOL_E_ARG; }

extern "C" int vol_frame_stats_async(vol_t *v, void *raw_host, void *stream)
{
    if (!v || !raw_host) return VOL_E_ARG;
    int rc = set_device(v); if (rc) return rc;
    cudaStream_t s = (cudaStream_t)stream;
    CK(cudaMemcpyAsync(raw_host, v->ctrl_last, VOL_STATS_RAW_BYTES, cudaMemcpyDeviceToHost, s));
    return VOL_OK;
}

extern "C" int vol_stats_decode(const vol_t *v, const void *raw_host, vol_stats_t *out)
{
    if (!v || !raw_host || !out) return VOL_E_ARG;
    uint32_t st[vf::ST_N]; unsigned long long cnt[vf::CNT_N];
    memcpy(st, raw_host, sizeof st); memcpy(cnt, (const char *)raw_host + sizeof st, sizeof cnt);
    memset(out, 0, sizeof *out);
    if (v->counting) {
        out->geo_read = cnt[vf::CNT_GEO_READ]; out->geo_changed = cnt[vf::CNT_GEO_CHANGED];
        out->col_read = cnt[vf::CNT_COL_READ]; out->col_changed = cnt[vf::CNT_COL_CHANGED];
        out->geo_sectors_read = cnt[vf::CNT_GEO_SEC_READ]; out->geo_sectors_written = cnt[vf::CNT_GEO_SEC_WRITTEN];
        out->col_sectors_read = cnt[vf::CNT_COL_SEC_READ]; out->col_sectors_written = cnt[vf::CNT_COL_SEC_WRITTEN];
        out->geo_visited = cnt[vf::CNT_GEO_VISITED]; out->col_gated = cnt[vf::CNT_COL_GATED];
        out->geo_skippable = cnt[vf::CNT_GEO_SKIPPABLE]; out->geo_sectors_skippable = cnt[vf::CNT_GEO_SEC_SKIPPABLE];
        out->cells_col = st[vf::ST_CELLS]; out->subs_geo = st[vf::ST_SUBS];
    }
    out->tiles_total = (uint32_t)v->p.n_tiles;
    out->tiles_geo = st[vf::ST_NGEO];
    out->items_col = st[vf::ST_NCOL] + st[vf::ST_NCOL_SMALL];
    out->jobs_mark = st[vf::ST_NJOBS];
    return VOL_OK;
}

extern "C" int vol_frame_stats(vol_t *v, vol_stats_t *out, void *stream)
{
    if (!v || !out) return VOL_E_ARG;
    unsigned long long raw[VOL_STATS_RAW_BYTES / 8];
    int rc = vol_frame_stats_async(v, raw, stream); if (rc) return rc;
    CK(cudaStreamSynchronize((cudaStream_t)stream));
    return vol_stats_decode(v, raw, out);
}

extern "C" int vol_last_kernel_ms(vol_t *v, float ms[3])
{
    if (!v || !ms || !v->ev_valid) return VOL_E_ARG;
    int rc = set_device(v); if (rc) return rc;
    CK(cudaEventSynchronize(v->ev[3]));
    for (int i = 0; i < 3; ++i) CK(cudaEventElapsedTime(&ms[i], v->ev[i], v->ev[i + 1]));
    return VOL_OK;
}

// ---- vol_selftest: rcp_exact / div_with against the correctly rounded intrinsics -------------------------------
__global__ void k_selftest_rcp(unsigned long long *bad)
{
    // every positive binary32 with RCP_MIN <= a <= RCP_MAX (and its negative)
    const uint32_t lo = __float_as_uint(vf::RCP_MIN), hi = __float_as_uint(vf::RCP_MAX);
    unsigned long long n = 0;
    for (uint64_t b = (uint64_t)lo + (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; b <= hi; b += (uint64_t)gridDim.x * blockDim.x) {
        const float a = __uint_as_float((uint32_t)b);
        n += __float_as_uint(vf::rcp_exact(a)) != __float_as_uint(__frcp_rn(a));
        n += __float_as_uint(vf::rcp_exact(-a)) != __float_as_uint(__frcp_rn(-a));
    }
    if (n) atomicAdd(bad, n);
}

__global__ void k_selftest_div(unsigned long long *bad, uint32_t stride)
{
    // numerators: 0 and every |a| in [2^-40, 2^40] (both signs), denominators 1..513
    const uint32_t lo = __float_as_uint(0x1p-40f), hi = __float_as_uint(0x1p40f);
    unsigned long long n = 0;
    for (uint64_t b = (uint64_t)lo + ((uint64_t)blockIdx.x * blockDim.x + threadIdx.x) * stride; b <= hi; b += (uint64_t)gridDim.x * blockDim.x * stride) {
        const float a = __uint_as_float((uint32_t)b);
        for (int w = 0; w <= 512; ++w) {
            const float den = (float)w + 1.0f, rb = vf::div_prepare(den);
            n += __float_as_uint(vf::div_with(a, den, rb)) != __float_as_uint(__fdiv_rn(a, den));
            n += __float_as_uint(vf::div_with(-a, den, rb)) != __float_as_uint(__fdiv_rn(-a, den));
        }
    }
    if (blockIdx.x == 0 && threadIdx.x == 0)
        for (int w = 0; w <= 512; ++w) { const float den = (float)w + 1.0f; n += __float_as_uint(vf::div_with(0.0f, den, vf::div_prepare(den))) != 0u; }
    if (n) atomicAdd(bad, n);
}

// the colour quotient of eq. 9 and its rounding, as issued by the fast path of colour_update_staged, against the plain
// expression: every stored weight wq, colour C and HD byte h with a sweep of new-sample weights 255 W >= 2^-20
__global__ void k_selftest_colour(unsigned long long *bad, uint32_t stride)
{
    unsigned long long n = 0;
    const uint32_t lo = __float_as_uint(0x1p-20f), hi = __float_as_uint(255.0f);
    for (uint64_t b = (uint64_t)lo + ((uint64_t)blockIdx.x * blockDim.x + threadIdx.x) * stride; b <= hi; b += (uint64_t)gridDim.x * blockDim.x * stride) {
        const float W255 = __uint_as_float((uint32_t)b);
        for (uint32_t wq = 0; wq < 256u; wq += 1u + (uint32_t)(b % 3u)) {
            const float wqf = (float)wq, den = __fadd_rn(wqf, W255), rden = vf::div_prepare(den);
            for (uint32_t k = 0; k < 16u; ++k) {
                const uint32_t C = (uint32_t)((b >> 3) + 37u * k + wq) & 0xffu, h = (uint32_t)((b >> 7) + 101u * k) & 0xffu;
                const float num = __fmaf_rn(W255, (float)h, (float)(C * wq));
                const uint32_t fast = min(__float_as_uint(__fadd_rn(vf::div_with(num, den, rden), 12582912.0f)) & 0x1ffu, 255u);
                const float cn = rintf(__fdiv_rn(num, den));
                const uint32_t ref = (uint32_t)(cn < 0.0f ? 0 : (cn > 255.0f ? 255 : (int)cn));
                n += fast != ref;
            }
            const float W = __fdiv_rn(W255, 255.0f) > 1.0f ? 1.0f : __fdiv_rn(W255, 255.0f);
            const float wnf = __fmaf_rn(W, (float)(255u - wq), wqf);
            n += min(__float_as_uint(__fadd_rn(wnf, 12582912.0f)) & 0x3ffu, 255u) != (uint32_t)min(__float2int_rn(wnf), 255);
            const float wna = __fadd_rn(wqf, W255);
            n += min(__float_as_uint(__fadd_rn(wna, 12582912.0f)) & 0x3ffu, 255u) != (uint32_t)min(__float2int_rn(wna), 255);
        }
    }
    if (n) atomicAdd(bad, n);
}

extern "C" int vol_selftest(uint64_t mismatches[3], int32_t exhaustive)
{
    if (!mismatches) return VOL_E_ARG;
    unsigned long long *d = nullptr;
    CK(cudaMalloc(&d, 3 * sizeof(unsigned long long)));
    int rc = VOL_OK;
    if (cudaMemset(d, 0, 3 * sizeof(unsigned long long)) != cudaSuccess) rc = VOL_E_CUDA;
    if (rc == VOL_OK) {
        k_selftest_rcp<<<148 * 8, 256>>>(d);
        k_selftest_div<<<148 * 8, 256>>>(d + 1, exhaustive ? 1u : 257u);
        k_selftest_colour<<<148 * 8, 256>>>(d + 2, exhaustive ? 1u : 1021u);
        unsigned long long h[3];
        if (cudaMemcpy(h, d, sizeof h, cudaMemcpyDeviceToHost) != cudaSuccess) rc = VOL_E_CUDA;
        else { mismatches[0] = h[0]; mismatches[1] = h[1]; mismatches[2] = h[2]; }
    }
    if (rc != VOL_OK) snprintf(g_err, sizeof g_err, "vol_selftest: %s", cudaGetErrorString(cudaGetLastError()));
    cudaFree(d);
    return rc;
}

#ifdef VF_TRACE
// development aid: copy the per-warp trace of the last k_fused launch (8192 x 16 words) to the host
extern "C" int vol_trace_dump(unsigned long long *host)
{
    CK(cudaDeviceSynchronize());
    CK(cudaMemcpyFromSymbol(host, vf::g_trace, sizeof(unsigned long long) * 8192 * 16));
    return VOL_OK;
}
#endif

#include "frontend_host.cuh"
#include "noalloc.cuh"
