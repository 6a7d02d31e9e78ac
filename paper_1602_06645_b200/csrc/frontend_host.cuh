// frontend_host.cuh -- host side of include/volfrontend.h (included at the end of volfusion.cu: same library, same error
// reporting).  The tracker's whole loop (F5-F7) is one cooperative launch, k_icp_track.
#pragma once
#include "../../include/volfrontend.h"
#include "frontend.cuh"

constexpr int FE_TRACK_OUT = 24;                            // doubles read back by vol_frontend_track (17 used)

struct vol_frontend {
    int device, w, h, levels;
    float sigma_s, sigma_r, dist_m, cos_min;
    int kmax;
    float *ws, *wr;                                         // F1 tables (device)
    float *D[2][vf::FE_MAX_LEVELS];                         // [0] measured, [1] predicted
    float4 *V[2][vf::FE_MAX_LEVELS], *N[2][vf::FE_MAX_LEVELS];
    vf::LevelK k[2][vf::FE_MAX_LEVELS];
    bool have[2];
    float *ray_depth;                                       // vol_frontend_predict: the ray-cast depth map
    unsigned long long *acc_dev, *acc_pinned;               // vol_frontend_icp_step: ICP_ACC integer accumulators
    unsigned long long *track_acc; size_t track_steps;      // vol_frontend_track: one set of accumulators per step
    double *track_out, *track_out_pinned;                   // FE_TRACK_OUT doubles: T (3 x 4), rms, count, status, level, conditioning
    double cond_min;
    bool trilinear_prediction;
    int last_status, last_level; double last_cond;          // of the most recent vol_frontend_track
    int track_blocks;                                       // co-resident blocks of k_icp_track
};

static int fe_set_device(const vol_frontend *fe) { CK(cudaSetDevice(fe->device)); return VOL_OK; }

extern "C" void vol_frontend_destroy(vol_frontend_t *fe)
{
    if (!fe) return;
    cudaSetDevice(fe->device);
    if (fe->ws) cudaFree(fe->ws);
    if (fe->wr) cudaFree(fe->wr);
    for (int s = 0; s < 2; ++s)
        for (int l = 0; l < vf::FE_MAX_LEVELS; ++l) {
            if (fe->D[s][l]) cudaFree(fe->D[s][l]);
            if (fe->V[s][l]) cudaFree(fe->V[s][l]);
            if (fe->N[s][l]) cudaFree(fe->N[s][l]);
        }
    if (fe->ray_depth) cudaFree(fe->ray_depth);
    if (fe->acc_dev) cudaFree(fe->acc_dev);
    if (fe->acc_pinned) cudaFreeHost(fe->acc_pinned);
    if (fe->track_acc) cudaFree(fe->track_acc);
    if (fe->track_out) cudaFree(fe->track_out);
    if (fe->track_out_pinned) cudaFreeHost(fe->track_out_pinned);
    cudaGetLastError();
    delete fe;
}

extern "C" int vol_frontend_create(vol_frontend_t **out, int32_t w, int32_t h, int32_t levels, const vol_frontend_opts_t *opts)
{
    if (!out || w <= 0 || h <= 0 || w > 16384 || h > 16384 || levels < 1 || levels > vf::FE_MAX_LEVELS) return VOL_E_ARG;
    if (w % (1 << (levels - 1)) != 0 || h % (1 << (levels - 1)) != 0) return VOL_E_ARG;
    float sigma_s = 4.5f, sigma_r = 0.030f, dist_m = 0.10f, cos_min = 0.94f, cond_min = VOL_ICP_COND_MIN;
    int device = -1;
    if (opts) {
        if (opts->sigma_s_px > 0.0f) sigma_s = opts->sigma_s_px;
        if (opts->sigma_r_m > 0.0f) sigma_r = opts->sigma_r_m;
        if (opts->dist_m > 0.0f) dist_m = opts->dist_m;
        if (opts->cos_min > 0.0f) cos_min = opts->cos_min;
        if (opts->cond_min > 0.0f) cond_min = opts->cond_min;
        device = opts->device;
    }
    if (!(sigma_s <= 1e3f) || !(sigma_r <= 1.0f) || !(dist_m <= 1e3f) || !(cos_min <= 1.0f) || !(cond_min < 1.0f)) return VOL_E_ARG;
    if (device < 0) CK(cudaGetDevice(&device));
    CK(cudaSetDevice(device));
    vol_frontend *fe = new (std::nothrow) vol_frontend();
    if (!fe) return VOL_E_OOM;
    memset(fe, 0, sizeof *fe);
    fe->device = device; fe->w = w; fe->h = h; fe->levels = levels;
    fe->sigma_s = sigma_s; fe->sigma_r = sigma_r; fe->dist_m = dist_m; fe->cos_min = cos_min; fe->cond_min = (double)cond_min;
    fe->trilinear_prediction = opts && opts->trilinear_prediction != 0;
    // F1 tables: binary64, rounded once
    const double ss = (double)sigma_s, sr = (double)sigma_r * 1000.0;
    fe->kmax = (int)std::ceil(3.0 * sr);
    float ws[49];
    for (int dy = -vf::FE_RADIUS; dy <= vf::FE_RADIUS; ++dy)
        for (int dx = -vf::FE_RADIUS; dx <= vf::FE_RADIUS; ++dx)
            ws[(dy + vf::FE_RADIUS) * 7 + dx + vf::FE_RADIUS] = (float)std::exp(-((double)(dx * dx) + (double)(dy * dy)) / (2.0 * ss * ss));
    float *wr = new (std::nothrow) float[fe->kmax + 1];
    if (!wr) { delete fe; return VOL_E_OOM; }
    for (int k = 0; k <= fe->kmax; ++k) wr[k] = (float)std::exp(-((double)k * (double)k) / (2.0 * sr * sr));
    auto fail = [&](int code) { delete[] wr; vol_frontend_destroy(fe); return code; };
    bool okc = cudaMalloc(&fe->ws, sizeof ws) == cudaSuccess && cudaMalloc(&fe->wr, sizeof(float) * (fe->kmax + 1)) == cudaSuccess &&
               cudaMalloc(&fe->ray_depth, sizeof(float) * (size_t)w * h) == cudaSuccess &&
               cudaMalloc(&fe->acc_dev, sizeof(unsigned long long) * vf::ICP_ACC) == cudaSuccess &&
               cudaMallocHost(&fe->acc_pinned, sizeof(unsigned long long) * vf::ICP_ACC) == cudaSuccess &&
               cudaMalloc(&fe->track_out, sizeof(double) * FE_TRACK_OUT) == cudaSuccess &&
               cudaMallocHost(&fe->track_out_pinned, sizeof(double) * FE_TRACK_OUT) == cudaSuccess;
    for (int s = 0; s < 2 && okc; ++s)
        for (int l = 0; l < levels && okc; ++l) {
            const size_t n = (size_t)(w >> l) * (h >> l);
            okc = cudaMalloc(&fe->D[s][l], n * sizeof(float)) == cudaSuccess && cudaMalloc(&fe->V[s][l], n * sizeof(float4)) == cudaSuccess &&
                  cudaMalloc(&fe->N[s][l], n * sizeof(float4)) == cudaSuccess;
        }
    if (!okc) { cudaGetLastError(); return fail(VOL_E_OOM); }
    if (cudaMemcpy(fe->ws, ws, sizeof ws, cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaMemcpy(fe->wr, wr, sizeof(float) * (fe->kmax + 1), cudaMemcpyHostToDevice) != cudaSuccess) return fail(VOL_E_CUDA);
    delete[] wr;
    int occ = 0, sms = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, vf::k_icp_track, 256, 0) != cudaSuccess || occ < 1 ||
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device) != cudaSuccess) { vol_frontend_destroy(fe); return VOL_E_CUDA; }
    fe->track_blocks = (occ < 2 ? occ : 2) * sms;           // two blocks per SM: measured equal to full occupancy, a quarter of the reductions
    *out = fe;
    return VOL_OK;
}

// F2-F4 for every level of side s, from its level-0 depth map: two launches (all depth levels, then all vertex / normal maps)
static int fe_build_pyramid(vol_frontend *fe, int s, const float K[9], cudaStream_t st)
{
    vf::LevelK k = {K[0], K[4], K[2], K[5]};
    vf::PyramidParams pq; vf::MapParams mq;
    memset(&pq, 0, sizeof pq); memset(&mq, 0, sizeof mq);
    pq.levels = mq.levels = fe->levels; pq.w0 = fe->w; pq.h0 = fe->h; pq.thr = 3.0f * fe->sigma_r;
    unsigned first = 0;
    for (int l = 0; l < fe->levels; ++l) {
        const int w = fe->w >> l, h = fe->h >> l;
        if (l > 0) {
            k.fx = k.fx * 0.5f; k.fy = k.fy * 0.5f;
            k.cx = (k.cx - 0.5f) * 0.5f; k.cy = (k.cy - 0.5f) * 0.5f;
        }
        fe->k[s][l] = k;
        pq.D[l] = fe->D[s][l];
        vf::MapLevel &m = mq.lv[l];
        m.D = fe->D[s][l]; m.V = fe->V[s][l]; m.N = fe->N[s][l]; m.w = w; m.h = h; m.k = k;
        m.first_block = first; m.blocks_x = (unsigned)((w + 31) / 32);
        first += m.blocks_x * (unsigned)((h + 7) / 8);
    }
    if (fe->levels > 1) {
        const int top = fe->levels - 1, wt = fe->w >> top, ht = fe->h >> top;
        vf::k_pyramid_depth<<<dim3((wt + 31) / 32, (ht + 7) / 8), 256, 0, st>>>(pq);
    }
    vf::k_vertex_normal<<<first, 256, 0, st>>>(mq);
    CK(cudaGetLastError());
    fe->have[s] = true;
    return VOL_OK;
}

extern "C" int vol_frontend_measure(vol_frontend_t *fe, const uint16_t *depth_u16_dev, const float K[9], void *stream)
{
    if (!fe || !depth_u16_dev || !K || !intrinsics_ok(K)) return VOL_E_ARG;
    int rc = fe_set_device(fe); if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    vf::k_bilateral<false><<<dim3((fe->w + 31) / 32, (fe->h + 7) / 8), 256, 0, st>>>(depth_u16_dev, fe->w, fe->h, fe->ws, fe->wr, fe->kmax, fe->D[0][0]);
    return fe_build_pyramid(fe, 0, K, st);
}

extern "C" int vol_frontend_predict_depth(vol_frontend_t *fe, const float *depth_m_dev, const float K[9], int32_t filter, void *stream)
{
    if (!fe || !depth_m_dev || !K || !intrinsics_ok(K)) return VOL_E_ARG;
    int rc = fe_set_device(fe); if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const int n = fe->w * fe->h;
    if (filter) {                                            // F8: rounding to millimetres inside the filter's tile load
        vf::k_bilateral<true><<<dim3((fe->w + 31) / 32, (fe->h + 7) / 8), 256, 0, st>>>(depth_m_dev, fe->w, fe->h, fe->ws, fe->wr, fe->kmax, fe->D[1][0]);
    } else {
        CK(cudaMemcpyAsync(fe->D[1][0], depth_m_dev, sizeof(float) * (size_t)n, cudaMemcpyDeviceToDevice, st));
    }
    return fe_build_pyramid(fe, 1, K, st);
}

extern "C" int vol_frontend_predict(vol_frontend_t *fe, const vol_t *v, const float T_world_cam[16], const float K[9], float t_near_m,
                                    float t_far_m, void *stream)
{
    if (!fe || !v || fe->device != v->device) return VOL_E_ARG;
    const bool tri = fe->trilinear_prediction;
    int rc = tri ? vol_raycast_trilinear(v, fe->w, fe->h, T_world_cam, K, t_near_m, t_far_m, fe->ray_depth, nullptr, stream)
                 : vol_raycast(v, fe->w, fe->h, T_world_cam, K, t_near_m, t_far_m, fe->ray_depth, nullptr, stream);
    if (rc) return rc;
    return vol_frontend_predict_depth(fe, fe->ray_depth, K, tri ? 0 : 1, stream);
}

static vf::IcpLevel fe_level(const vol_frontend *fe, int level)
{
    vf::IcpLevel lv;
    lv.V = fe->V[0][level]; lv.N = fe->N[0][level]; lv.Vp = fe->V[1][level]; lv.Np = fe->N[1][level];
    lv.w = fe->w >> level; lv.h = fe->h >> level; lv.k = fe->k[1][level];
    return lv;
}

static int fe_icp_launch(vol_frontend *fe, int level, const float T[16], cudaStream_t st)
{
    vf::IcpParams q;
    q.lv = fe_level(fe, level);
    for (int i = 0; i < 3; ++i) { for (int j = 0; j < 3; ++j) q.R[3 * i + j] = T[4 * i + j]; q.t[i] = T[4 * i + 3]; }
    q.dist2 = fe->dist_m * fe->dist_m; q.cos_min = fe->cos_min; q.acc = fe->acc_dev;
    CK(cudaMemsetAsync(fe->acc_dev, 0, sizeof(unsigned long long) * vf::ICP_ACC, st));
    vf::k_icp<<<dim3((q.lv.w + 31) / 32, (q.lv.h + 7) / 8), 256, 0, st>>>(q);
    CK(cudaGetLastError());
    CK(cudaMemcpyAsync(fe->acc_pinned, fe->acc_dev, sizeof(unsigned long long) * vf::ICP_ACC, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    return VOL_OK;
}

static bool fe_rigid(const float T[16])
{
    float R[9], t[3];
    return rigid_inverse(T, R, t);
}

extern "C" int vol_frontend_icp_step(vol_frontend_t *fe, int32_t level, const float T_pred_cur[16], double *sums_host, void *stream)
{
    if (!fe || !T_pred_cur || !sums_host || level < 0 || level >= fe->levels || !fe->have[0] || !fe->have[1]) return VOL_E_ARG;
    if (!fe_rigid(T_pred_cur)) return VOL_E_ARG;
    int rc = fe_set_device(fe); if (rc) return rc;
    rc = fe_icp_launch(fe, level, T_pred_cur, (cudaStream_t)stream); if (rc) return rc;
    for (int i = 0; i < vf::ICP_SUMS; ++i) sums_host[i] = vf::icp_total((long long)fe->acc_pinned[i], (long long)fe->acc_pinned[vf::ICP_SUMS + i]);
    return VOL_OK;
}

// F7 in one cooperative launch (k_icp_track: F5 and F6 on the device); one read-back of 128 bytes
extern "C" int vol_frontend_track(vol_frontend_t *fe, const float T_init[16], const int32_t *iterations, float T_out[16], double *rms_out,
                                  int64_t *count_out, void *stream)
{
    if (!fe || !iterations || !T_out || !fe->have[0] || !fe->have[1]) return VOL_E_ARG;
    if (T_init && !fe_rigid(T_init)) return VOL_E_ARG;
    size_t steps = 0;
    for (int l = 0; l < fe->levels; ++l) { if (iterations[l] < 0 || iterations[l] > 1000) return VOL_E_ARG; steps += (size_t)iterations[l]; }
    int rc = fe_set_device(fe); if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    if (steps > fe->track_steps) {
        if (fe->track_acc) { CK(cudaDeviceSynchronize()); cudaFree(fe->track_acc); fe->track_acc = nullptr; fe->track_steps = 0; }
        CK(cudaMalloc(&fe->track_acc, steps * vf::TRACK_STRIDE * sizeof(unsigned long long)));
        fe->track_steps = steps;
    }
    vf::TrackParams q;
    memset(&q, 0, sizeof q);
    for (int l = 0; l < fe->levels; ++l) { q.lv[l] = fe_level(fe, l); q.iters[l] = iterations[l]; }
    q.levels = fe->levels; q.min_count = 100;
    q.dist2 = fe->dist_m * fe->dist_m; q.cos_min = fe->cos_min;
    for (int i = 0; i < 12; ++i) q.T0[i] = T_init ? (double)T_init[i] : (i % 5 == 0 ? 1.0 : 0.0);
    q.acc = fe->track_acc; q.out = fe->track_out; q.cond_min = fe->cond_min;
    if (steps > 0) CK(cudaMemsetAsync(fe->track_acc, 0, steps * vf::TRACK_STRIDE * sizeof(unsigned long long), st));
    const int tiles0 = ((fe->w + 31) / 32) * ((fe->h + 7) / 8);
    const int blocks = fe->track_blocks < tiles0 ? fe->track_blocks : tiles0;
    void *args[] = {&q};
    CK(cudaLaunchCooperativeKernel((const void *)vf::k_icp_track, dim3(blocks), dim3(256), args, 0, st));
    CK(cudaMemcpyAsync(fe->track_out_pinned, fe->track_out, sizeof(double) * FE_TRACK_OUT, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    const double *o = fe->track_out_pinned;
    fe->last_status = (int)o[14]; fe->last_level = (int)o[15]; fe->last_cond = o[16];
    for (int i = 0; i < 12; ++i) T_out[i] = (float)o[i];
    T_out[12] = T_out[13] = T_out[14] = 0.0f; T_out[15] = 1.0f;
    if (rms_out) *rms_out = o[12];
    if (count_out) *count_out = (int64_t)o[13];
    if (o[14] == 1.0) { snprintf(g_err, sizeof g_err, "vol_frontend_track: %lld correspondences at level %d", (long long)o[13], (int)o[15]); return VOL_E_LOST; }
    if (o[14] == 2.0) { snprintf(g_err, sizeof g_err, "vol_frontend_track: normal equations not positive definite at level %d", (int)o[15]); return VOL_E_LOST; }
    if (o[14] == 3.0) { snprintf(g_err, sizeof g_err, "vol_frontend_track: motion unobservable at level %d (conditioning %.3g < %.3g)", (int)o[15], o[16], fe->cond_min); return VOL_E_LOST; }
    return VOL_OK;
}

extern "C" int vol_frontend_track_info(const vol_frontend_t *fe, int32_t *status_out, int32_t *level_out, double *conditioning_out)
{
    if (!fe) return VOL_E_ARG;
    if (status_out) *status_out = fe->last_status;
    if (level_out) *level_out = fe->last_level;
    if (conditioning_out) *conditioning_out = fe->last_cond;
    return VOL_OK;
}

extern "C" int vol_frontend_maps(const vol_frontend_t *fe, int32_t which, int32_t level, float *depth_host, float *vertex_host,
                                 float *normal_host, void *stream)
{
    if (!fe || which < 0 || which > 1 || level < 0 || level >= fe->levels || !fe->have[which]) return VOL_E_ARG;
    int rc = fe_set_device(fe); if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t n = (size_t)(fe->w >> level) * (fe->h >> level);
    if (depth_host) CK(cudaMemcpyAsync(depth_host, fe->D[which][level], n * sizeof(float), cudaMemcpyDeviceToHost, st));
    float4 *tmp = nullptr;
    if (vertex_host || normal_host) { tmp = new (std::nothrow) float4[n]; if (!tmp) return VOL_E_OOM; }
    for (int m = 0; m < 2; ++m) {
        float *dst = m == 0 ? vertex_host : normal_host;
        if (!dst) continue;
        cudaError_t e = cudaMemcpyAsync(tmp, m == 0 ? fe->V[which][level] : fe->N[which][level], n * sizeof(float4), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) { delete[] tmp; CK(e); }
        for (size_t i = 0; i < n; ++i) { dst[3 * i] = tmp[i].x; dst[3 * i + 1] = tmp[i].y; dst[3 * i + 2] = tmp[i].z; }
    }
    delete[] tmp;
    CK(cudaStreamSynchronize(st));
    return VOL_OK;
}
