// noalloc.cuh -- vol_icp_step_static (include/volfrontend.h): one F5 step that allocates nothing.
//
// For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it).
// The scratch the step needs -- one set of 29 binary64 partial sums per thread block and a ticket counter -- lives in a
// file-scope __device__ array of fixed size; the caller passes the maps in and the sums out, all DEVICE memory.  Every GPU
// that loads the library holds the array (1.8 MiB) until exit.
//
// Included at the end of volfusion.cu: the array, the kernel that is handed its address and the cudaGetSymbolAddress call
// that obtains that address are in one translation unit.  In HOST code the array's name is only a stand-in for the symbol,
// not a device address; the address is looked up once per device, with that device current, and passed to the kernel.
#pragma once
#include <mutex>
#include "frontend.cuh"

namespace vf {

constexpr int STATIC_MAX_BLOCKS = VOL_ICP_STATIC_MAX_BLOCKS;     // thread blocks of 32 x 8 pixels
constexpr int STATIC_HEAD = 32;                                  // doubles: a 256-byte header, its first word the ticket counter

}  // namespace vf

// file scope: 256-byte header + STATIC_MAX_BLOCKS slots of ICP_SUMS doubles = 1 900 800 bytes
static __device__ __align__(256) double g_icp_static_scratch[vf::STATIC_HEAD + (size_t)vf::STATIC_MAX_BLOCKS * vf::ICP_SUMS];

namespace vf {

// F5, one step, one thread per measured pixel like k_icp; but the blocks' partial sums are not added into shared
// accumulators: block b stores its 29 sums in slot b of the scratch, and the block that draws the last ticket adds the slots
// up in a fixed order (8 interleaved slices, block index ascending within a slice, then the slices in turn).  The result does
// not depend on the order in which the blocks ran.  `scratch` is g_icp_static_scratch's device address; its ticket word is
// zero at launch (cleared by the entry point on the stream); every slot that is read was written by this launch.
__global__ void __launch_bounds__(256) k_icp_static(const __grid_constant__ IcpParams q, double *scratch, double *out)
{
    __shared__ double sh[8][ICP_SUMS];
    __shared__ bool s_last;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int x = blockIdx.x * 32 + lane, y = blockIdx.y * 8 + wid;
    const unsigned n_blocks = gridDim.x * gridDim.y, block = blockIdx.y * gridDim.x + blockIdx.x;
    double *slots = scratch + STATIC_HEAD;
    double s[ICP_SUMS];
#pragma unroll
    for (int i = 0; i < ICP_SUMS; ++i) s[i] = 0.0;
    float J[6], r;
    if (x < q.lv.w && y < q.lv.h && icp_pixel(q.lv, q.R, q.t, q.dist2, q.cos_min, x, y, J, r)) icp_accumulate(s, J, r);
#pragma unroll
    for (int i = 0; i < ICP_SUMS; ++i) {
        double a = s[i];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
        if (lane == 0) sh[wid][i] = a;
    }
    __syncthreads();
    if (threadIdx.x < ICP_SUMS) {
        double a = 0.0;
#pragma unroll
        for (int k = 0; k < 8; ++k) a += sh[k][threadIdx.x];
        __stcg(slots + (size_t)block * ICP_SUMS + threadIdx.x, a);
        __threadfence();                                         // the slot is visible before the ticket is drawn
    }
    __syncthreads();
    if (threadIdx.x == 0) s_last = atomicAdd(reinterpret_cast<unsigned *>(scratch), 1u) == n_blocks - 1u;
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    double a = 0.0;
    if (lane < ICP_SUMS)
        for (unsigned b = (unsigned)wid; b < n_blocks; b += 8u) a += __ldcg(slots + (size_t)b * ICP_SUMS + lane);
    __syncthreads();                                             // (sh is reused)
    if (lane < ICP_SUMS) sh[wid][lane] = a;
    __syncthreads();
    if (threadIdx.x < ICP_SUMS) {
        double t = 0.0;
#pragma unroll
        for (int k = 0; k < 8; ++k) t += sh[k][threadIdx.x];
        out[threadIdx.x] = t;
    }
}

}  // namespace vf

// device address of the scratch array, looked up once per device
static std::mutex g_static_mutex;
static double *g_static_ptr[64];

static int static_scratch(double **out)
{
    int dev = -1;
    CK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) { snprintf(g_err, sizeof g_err, "vol_icp_step_static: device ordinal %d not supported", dev); return VOL_E_TOOBIG; }
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_ptr[dev]) {
        double *ptr = nullptr;
        CK(cudaGetSymbolAddress((void **)&ptr, g_icp_static_scratch));
        if (!ptr) { snprintf(g_err, sizeof g_err, "vol_icp_step_static: cudaGetSymbolAddress returned a null address"); return VOL_E_CUDA; }
        g_static_ptr[dev] = ptr;
    }
    *out = g_static_ptr[dev];
    return VOL_OK;
}

extern "C" int vol_icp_step_static(const float *V_dev, const float *N_dev, const float *Vp_dev, const float *Np_dev, int32_t w, int32_t h,
                                   const float K[9], const float T_pred_cur[16], float dist_m, float cos_min, double *sums_dev,
                                   void *stream)
{
    if (!V_dev || !N_dev || !Vp_dev || !Np_dev || !K || !T_pred_cur || !sums_dev) return VOL_E_ARG;
    if (w <= 0 || h <= 0 || !intrinsics_ok(K) || !fe_rigid(T_pred_cur)) return VOL_E_ARG;
    if (!(dist_m <= 1e3f) || !(cos_min <= 1.0f)) return VOL_E_ARG;
    if (((uintptr_t)V_dev | (uintptr_t)N_dev | (uintptr_t)Vp_dev | (uintptr_t)Np_dev) & 15u) return VOL_E_ARG;    // float4 loads
    if (((uintptr_t)sums_dev) & 7u) return VOL_E_ARG;
    const long long bx = ((long long)w + 31) / 32, by = ((long long)h + 7) / 8;
    if (bx * by > (long long)vf::STATIC_MAX_BLOCKS) {
        snprintf(g_err, sizeof g_err, "vol_icp_step_static: a %d x %d map needs %lld blocks of 32 x 8 pixels, the static scratch holds %d "
                                      "(VOL_ICP_STATIC_MAX_BLOCKS); use vol_frontend_icp_step", w, h, bx * by, vf::STATIC_MAX_BLOCKS);
        return VOL_E_TOOBIG;
    }
    double *scratch = nullptr;
    int rc = static_scratch(&scratch); if (rc) return rc;
    vf::IcpParams q;
    q.lv.V = reinterpret_cast<const float4 *>(V_dev); q.lv.N = reinterpret_cast<const float4 *>(N_dev);
    q.lv.Vp = reinterpret_cast<const float4 *>(Vp_dev); q.lv.Np = reinterpret_cast<const float4 *>(Np_dev);
    q.lv.w = w; q.lv.h = h; q.lv.k.fx = K[0]; q.lv.k.fy = K[4]; q.lv.k.cx = K[2]; q.lv.k.cy = K[5];
    for (int i = 0; i < 3; ++i) { for (int j = 0; j < 3; ++j) q.R[3 * i + j] = T_pred_cur[4 * i + j]; q.t[i] = T_pred_cur[4 * i + 3]; }
    const float d = dist_m > 0.0f ? dist_m : 0.10f;
    q.dist2 = d * d; q.cos_min = cos_min > 0.0f ? cos_min : 0.94f; q.acc = nullptr;
    cudaStream_t st = (cudaStream_t)stream;
    CK(cudaMemsetAsync(scratch, 0, sizeof(double) * vf::STATIC_HEAD, st));          // the ticket counter starts at zero
    vf::k_icp_static<<<dim3((unsigned)bx, (unsigned)by), 256, 0, st>>>(q, scratch, sums_dev);
    CK(cudaGetLastError());
    return VOL_OK;
}
