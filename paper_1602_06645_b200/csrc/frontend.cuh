// frontend.cuh -- kernels of the depth front end and the ICP step (volfrontend.h readings F1-F5).
//
// Image-sized work (307 K pixels at most): one thread per pixel, whole-warp rows, no tiling -- these kernels are bound by
// launch latency and L2, not by HBM.  All map arithmetic is binary32, one rounding per operation, NO fused multiply-add
// (explicit __fmul_rn / __fadd_rn; the file is compiled with --fmad=false as well), in the order the oracle states, so
// depth, vertex and normal maps are bit-identical to oracle/frontend.py.  The ICP sums are binary64.
#pragma once
#include <cstdint>
#include <cooperative_groups.h>
#include <cuda_runtime.h>

namespace vf {

constexpr int FE_RADIUS = 3;                  // F1: 7 x 7 window
constexpr int FE_MAX_LEVELS = 6;
constexpr int ICP_SUMS = 29;                  // 21 (upper triangle of A) + 6 (b) + sum r^2 + count

struct LevelK { float fx, fy, cx, cy; };

// F1: bilateral filter of the raw depth.  ws: 49 spatial weights [dy + 3][dx + 3]; wr: kmax + 1 range weights over whole mm.
// A CTA filters 32 x 8 pixels from a shared-memory tile of 38 x 14 (the 7 x 7 windows of neighbouring pixels overlap in 42 of
// their 49 pixels).  FROM_FLOAT: the input is float metres and F8's rounding to whole millimetres (half-even, clamped to
// 65535) is done while the tile is loaded.
template <bool FROM_FLOAT>
__global__ void __launch_bounds__(256) k_bilateral(const void *__restrict__ in, int w, int h, const float *__restrict__ ws,
                                                   const float *__restrict__ wr, int kmax, float *__restrict__ out)
{
    constexpr int TW = 32 + 2 * FE_RADIUS, TH = 8 + 2 * FE_RADIUS;
    __shared__ uint16_t tile[TH][TW + 2];
    __shared__ float s_ws[49];
    const int x0 = blockIdx.x * 32 - FE_RADIUS, y0 = blockIdx.y * 8 - FE_RADIUS;
    for (int i = threadIdx.x; i < TW * TH; i += 256) {
        const int tx = i % TW, ty = i / TW, xx = x0 + tx, yy = y0 + ty;
        uint16_t v = 0;                                       // outside the image: never used (the window is clipped below)
        if (xx >= 0 && xx < w && yy >= 0 && yy < h) {
            if (FROM_FLOAT) v = (uint16_t)fminf(rintf(__fmul_rn(__ldg(static_cast<const float *>(in) + (size_t)yy * w + xx), 1000.0f)), 65535.0f);
            else v = __ldg(static_cast<const uint16_t *>(in) + (size_t)yy * w + xx);
        }
        tile[ty][tx] = v;
    }
    if (threadIdx.x < 49) s_ws[threadIdx.x] = __ldg(ws + threadIdx.x);
    __syncthreads();
    const int lx = threadIdx.x & 31, ly = threadIdx.x >> 5;
    const int x = blockIdx.x * 32 + lx, y = blockIdx.y * 8 + ly;
    if (x >= w || y >= h) return;
    const int d = (int)tile[ly + FE_RADIUS][lx + FE_RADIUS];
    float r = 0.0f;
    if (d > 0) {
        float sw = 0.0f, sd = 0.0f;
#pragma unroll
        for (int dy = -FE_RADIUS; dy <= FE_RADIUS; ++dy) {
            const int yy = y + dy;
            if (yy < 0 || yy >= h) continue;
#pragma unroll
            for (int dx = -FE_RADIUS; dx <= FE_RADIUS; ++dx) {
                const int xx = x + dx;
                if (xx < 0 || xx >= w) continue;
                const int q = (int)tile[ly + FE_RADIUS + dy][lx + FE_RADIUS + dx];
                const int delta = abs(q - d);
                if (q > 0 && delta <= kmax) {
                    const float wgt = __fmul_rn(s_ws[(dy + FE_RADIUS) * 7 + (dx + FE_RADIUS)], __ldg(wr + delta));
                    sw = __fadd_rn(sw, wgt);
                    sd = __fadd_rn(sd, __fmul_rn(wgt, (float)q));
                }
            }
        }
        r = __fmul_rn(__fdiv_rn(sd, sw), 0.001f);                         // mm -> m
    }
    out[(size_t)y * w + x] = r;
}

// F2 for one output pixel: the 2 x 2 block (v[0] = the block's first pixel) -> its mean over the valid pixels within thr of v[0]
__device__ __forceinline__ float fe_half_sample(const float (&v)[4], float thr)
{
    const float c = v[0];
    float res = 0.0f;
    if (c > 0.0f) {
        float s = 0.0f, n = 0.0f;
#pragma unroll
        for (int i = 0; i < 4; ++i)
            if (v[i] > 0.0f && fabsf(__fsub_rn(v[i], c)) <= thr) { s = __fadd_rn(s, v[i]); n = __fadd_rn(n, 1.0f); }
        res = __fdiv_rn(s, n);
    }
    return res;
}

// F2, every level in ONE launch: a thread owns one pixel of the coarsest level, i.e. a square block of 2^(levels-1) pixels
// of level 0, and builds the levels of that block one after the other (level l reads the values the same thread has just
// written for level l - 1).  D[l]: depth map of level l, w0 x h0 the size of level 0.
struct PyramidParams { float *D[FE_MAX_LEVELS]; int levels, w0, h0; float thr; };
__global__ void __launch_bounds__(256) k_pyramid_depth(const __grid_constant__ PyramidParams q)
{
    const int top = q.levels - 1, wt = q.w0 >> top, ht = q.h0 >> top;
    const int X = blockIdx.x * 32 + (threadIdx.x & 31), Y = blockIdx.y * 8 + (threadIdx.x >> 5);
    if (X >= wt || Y >= ht) return;
    for (int l = 1; l <= top; ++l) {
        const int wl = q.w0 >> l, side = 1 << (top - l);                  // this thread's block at level l is side x side
        const float *in = q.D[l - 1];
        float *out = q.D[l];
        for (int by = 0; by < side; ++by)
            for (int bx = 0; bx < side; ++bx) {
                const int x = X * side + bx, y = Y * side + by;
                const float2 r0 = *reinterpret_cast<const float2 *>(in + (size_t)(2 * y) * (2 * wl) + 2 * x);
                const float2 r1 = *reinterpret_cast<const float2 *>(in + (size_t)(2 * y + 1) * (2 * wl) + 2 * x);
                const float v[4] = {r0.x, r0.y, r1.x, r1.y};
                out[(size_t)y * wl + x] = fe_half_sample(v, q.thr);
            }
    }
}

// F3 = eq. 7: the vertex of pixel (x, y) with depth D
__device__ __forceinline__ float3 fe_vertex(const LevelK k, int x, int y, float D)
{
    return make_float3(__fdiv_rn(__fmul_rn(__fsub_rn((float)x, k.cx), D), k.fx), __fdiv_rn(__fmul_rn(__fsub_rn((float)y, k.cy), D), k.fy), D);
}

// F3 + F4 of every level in ONE launch: V (xyz, w = 0) and N (eq. 8 normalised; zero where a neighbour is missing or invalid).
// The CTAs of the levels follow one another in the grid (first_block).
struct MapLevel { const float *D; float4 *V, *N; int w, h; LevelK k; unsigned first_block, blocks_x; };
struct MapParams { MapLevel lv[FE_MAX_LEVELS]; int levels; };
__global__ void __launch_bounds__(256) k_vertex_normal(const __grid_constant__ MapParams q)
{
    int l = 0;
    while (l + 1 < q.levels && blockIdx.x >= q.lv[l + 1].first_block) ++l;
    const MapLevel &m = q.lv[l];
    const unsigned blk = blockIdx.x - m.first_block;
    const int w = m.w, h = m.h;
    const LevelK k = m.k;
    const float *__restrict__ D = m.D;
    const int x = (int)(blk % m.blocks_x) * 32 + (threadIdx.x & 31), y = (int)(blk / m.blocks_x) * 8 + (threadIdx.x >> 5);
    if (x >= w || y >= h) return;
    const size_t o = (size_t)y * w + x;
    const float d0 = __ldg(D + o);
    float4 v = make_float4(0.0f, 0.0f, 0.0f, 0.0f), n = v;
    if (d0 > 0.0f) {
        const float3 p0 = fe_vertex(k, x, y, d0);
        v = make_float4(p0.x, p0.y, p0.z, 0.0f);
        if (x + 1 < w && y + 1 < h) {
            const float d1 = __ldg(D + o + 1), d2 = __ldg(D + o + w);
            if (d1 > 0.0f && d2 > 0.0f) {
                const float3 p1 = fe_vertex(k, x + 1, y, d1), p2 = fe_vertex(k, x, y + 1, d2);
                const float ax = __fsub_rn(p1.x, p0.x), ay = __fsub_rn(p1.y, p0.y), az = __fsub_rn(p1.z, p0.z);
                const float bx = __fsub_rn(p2.x, p0.x), by = __fsub_rn(p2.y, p0.y), bz = __fsub_rn(p2.z, p0.z);
                const float nx = __fsub_rn(__fmul_rn(ay, bz), __fmul_rn(az, by));
                const float ny = __fsub_rn(__fmul_rn(az, bx), __fmul_rn(ax, bz));
                const float nz = __fsub_rn(__fmul_rn(ax, by), __fmul_rn(ay, bx));
                const float ln = __fsqrt_rn(__fadd_rn(__fadd_rn(__fmul_rn(nx, nx), __fmul_rn(ny, ny)), __fmul_rn(nz, nz)));
                if (ln > 0.0f) n = make_float4(__fdiv_rn(nx, ln), __fdiv_rn(ny, ln), __fdiv_rn(nz, ln), 0.0f);
            }
        }
    }
    m.V[o] = v; m.N[o] = n;
}


__device__ __forceinline__ float fe_dot3(float a0, float a1, float a2, float b0, float b1, float b2)
{
    return __fadd_rn(__fadd_rn(__fmul_rn(a0, b0), __fmul_rn(a1, b1)), __fmul_rn(a2, b2));
}

// the maps of one level, both sides
struct IcpLevel {
    const float4 *V, *N, *Vp, *Np;
    int w, h;
    LevelK k;
};

// F5 for one measured pixel: J and r in binary32 exactly as the oracle; false if the pixel has no correspondence
__device__ __forceinline__ bool icp_pixel(const IcpLevel &q, const float (&R)[9], const float (&t)[3], float dist2_max, float cos_min,
                                          int x, int y, float (&J)[6], float &r)
{
    const size_t o = (size_t)y * q.w + x;
    const float4 n = __ldg(q.N + o);
    if (!(n.x != 0.0f || n.y != 0.0f || n.z != 0.0f)) return false;
    const float4 v = __ldg(q.V + o);
    const float px = __fadd_rn(fe_dot3(R[0], R[1], R[2], v.x, v.y, v.z), t[0]);
    const float py = __fadd_rn(fe_dot3(R[3], R[4], R[5], v.x, v.y, v.z), t[1]);
    const float pz = __fadd_rn(fe_dot3(R[6], R[7], R[8], v.x, v.y, v.z), t[2]);
    const float mx = fe_dot3(R[0], R[1], R[2], n.x, n.y, n.z);
    const float my = fe_dot3(R[3], R[4], R[5], n.x, n.y, n.z);
    const float mz = fe_dot3(R[6], R[7], R[8], n.x, n.y, n.z);
    if (!(pz > 0.0f)) return false;
    const float u = __fadd_rn(__fmul_rn(q.k.fx, __fdiv_rn(px, pz)), q.k.cx);
    const float vv = __fadd_rn(__fmul_rn(q.k.fy, __fdiv_rn(py, pz)), q.k.cy);
    const float xf = floorf(__fadd_rn(u, 0.5f)), yf = floorf(__fadd_rn(vv, 0.5f));
    if (!(xf >= 0.0f && xf < (float)q.w && yf >= 0.0f && yf < (float)q.h)) return false;
    const size_t op = (size_t)(int)yf * q.w + (int)xf;
    const float4 nq = __ldg(q.Np + op);
    if (!(nq.x != 0.0f || nq.y != 0.0f || nq.z != 0.0f)) return false;
    const float4 vq = __ldg(q.Vp + op);
    const float dx = __fsub_rn(vq.x, px), dy = __fsub_rn(vq.y, py), dz = __fsub_rn(vq.z, pz);
    const float dist2 = fe_dot3(dx, dy, dz, dx, dy, dz);
    const float cosang = fe_dot3(mx, my, mz, nq.x, nq.y, nq.z);
    if (dist2 > dist2_max || cosang < cos_min) return false;
    r = fe_dot3(nq.x, nq.y, nq.z, dx, dy, dz);
    J[0] = __fsub_rn(__fmul_rn(py, nq.z), __fmul_rn(pz, nq.y));
    J[1] = __fsub_rn(__fmul_rn(pz, nq.x), __fmul_rn(px, nq.z));
    J[2] = __fsub_rn(__fmul_rn(px, nq.y), __fmul_rn(py, nq.x));
    J[3] = nq.x; J[4] = nq.y; J[5] = nq.z;
    return true;
}

// add one correspondence to a thread's 29 binary64 sums
__device__ __forceinline__ void icp_accumulate(double (&s)[ICP_SUMS], const float (&J)[6], float r)
{
    int idx = 0;
#pragma unroll
    for (int i = 0; i < 6; ++i)
#pragma unroll
        for (int j = i; j < 6; ++j) s[idx++] += (double)J[i] * (double)J[j];
#pragma unroll
    for (int i = 0; i < 6; ++i) s[21 + i] += (double)J[i] * (double)r;
    s[27] += (double)r * (double)r;
    s[28] += 1.0;
}

// A block's partial sum a goes into TWO 64-bit integer accumulators, a = hi * 2^-20 + lo * 2^-60: hi = rint(a * 2^20), the
// remainder a - hi * 2^-20 is exact in binary64 (|.| <= 2^-21) and lo = rint(remainder * 2^60) drops only bits below 2^-60.
// Integer addition is associative, so the totals -- and with them the estimated pose -- do not depend on the order in which
// the blocks arrive (binary64 atomicAdd would).  |a| is far below 2^42 for maps in metres (at most 2^19 pixels x (10 m)^2);
// it is clamped there so that a corrupt map cannot overflow the integers.
constexpr int ICP_ACC = 2 * ICP_SUMS;          // int64 words per set of accumulators: hi[ICP_SUMS], lo[ICP_SUMS]
constexpr int TRACK_STRIDE = 64;               // k_icp_track: words per step -- ICP_ACC accumulators, then the step's arrival counter

__device__ __forceinline__ void icp_publish(double a, unsigned long long *acc)
{
    a = fmin(fmax(a, -0x1p42), 0x1p42);
    const double hi = rint(a * 0x1p20);
    const double lo = rint((a - hi * 0x1p-20) * 0x1p60);
    atomicAdd(acc, (unsigned long long)(long long)hi);
    atomicAdd(acc + ICP_SUMS, (unsigned long long)(long long)lo);
}

__host__ __device__ __forceinline__ double icp_total(long long hi, long long lo) { return (double)hi * 0x1p-20 + (double)lo * 0x1p-60; }

// block reduction (256 threads) of the per-thread sums in a fixed order (shuffle tree, then the 8 warps in turn), then
// icp_publish of the block's 29 partial sums
__device__ __forceinline__ void icp_block_reduce(const double (&s)[ICP_SUMS], double (*sh)[ICP_SUMS], unsigned long long *acc)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
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
        if (a != 0.0) icp_publish(a, acc + threadIdx.x);
    }
    __syncthreads();
}

struct IcpParams {
    IcpLevel lv;
    float R[9], t[3];               // current camera -> prediction camera
    float dist2, cos_min;
    unsigned long long *acc;        // ICP_ACC integer accumulators (zeroed before the launch), see icp_publish
};

// F5, one step (vol_frontend_icp_step): one thread per measured pixel
__global__ void __launch_bounds__(256) k_icp(const __grid_constant__ IcpParams q)
{
    __shared__ double sh[8][ICP_SUMS];
    const int x = blockIdx.x * 32 + (threadIdx.x & 31), y = blockIdx.y * 8 + (threadIdx.x >> 5);
    double s[ICP_SUMS];
#pragma unroll
    for (int i = 0; i < ICP_SUMS; ++i) s[i] = 0.0;
    float J[6], r;
    if (x < q.lv.w && y < q.lv.h && icp_pixel(q.lv, q.R, q.t, q.dist2, q.cos_min, x, y, J, r)) icp_accumulate(s, J, r);
    icp_block_reduce(s, sh, q.acc);
}

// F6 in binary64: A xi = b by Cholesky, then T <- [exp(omega) R, exp(omega) t + v].  T: 12 doubles (3 x 4, row-major).
// Returns 0, or 2 if A is not positive definite, or 3 if A is too close to singular: *cond = min_j d_j / A_jj, the smallest
// Cholesky pivot relative to its diagonal entry (the part of parameter j's information that the parameters before it do
// not already explain; 1 for a diagonal A, 0 for a singular one, and invariant under rescaling the parameters), and a
// motion is unobservable where it falls below cond_min -- a sphere seen from its centre line, a scene that is
// symmetric about the axis the camera turns about.  T is left alone in both failure cases.  One thread of every block runs this between two steps while the others
// wait, so the chain of slow binary64 operations is kept short: one rsqrt per column instead of a sqrt and the divisions,
// and the two Rodrigues coefficients from their series (ICP increments are far below 0.1 rad; sin / cos otherwise).
__device__ inline int icp_se3_update(double *T, const double *sums, double cond_min, double *cond)
{
    double A[6][6], L[6][6], inv[6], b[6], y[6], xi[6];
    int idx = 0;
    for (int i = 0; i < 6; ++i) for (int j = i; j < 6; ++j) { A[i][j] = sums[idx]; A[j][i] = sums[idx]; ++idx; }
    for (int i = 0; i < 6; ++i) { b[i] = sums[21 + i]; for (int j = 0; j < 6; ++j) L[i][j] = 0.0; }
    double worst = 1.0;
    for (int j = 0; j < 6; ++j) {                                    // column by column
        double d = A[j][j];
        for (int k = 0; k < j; ++k) d -= L[j][k] * L[j][k];
        if (!(d > 0.0)) { *cond = 0.0; return 2; }
        worst = fmin(worst, d / A[j][j]);
        inv[j] = rsqrt(d);
        L[j][j] = d * inv[j];
        for (int i = j + 1; i < 6; ++i) {
            double a = A[i][j];
            for (int k = 0; k < j; ++k) a -= L[i][k] * L[j][k];
            L[i][j] = a * inv[j];
        }
    }
    *cond = worst;
    if (worst < cond_min) return 3;
    for (int i = 0; i < 6; ++i) { double a = b[i]; for (int k = 0; k < i; ++k) a -= L[i][k] * y[k]; y[i] = a * inv[i]; }
    for (int i = 5; i >= 0; --i) { double a = y[i]; for (int k = i + 1; k < 6; ++k) a -= L[k][i] * xi[k]; xi[i] = a * inv[i]; }
    const double ox = xi[0], oy = xi[1], oz = xi[2], t2 = ox * ox + oy * oy + oz * oz;
    double ca, cb;                                                   // sin(th) / th and (1 - cos(th)) / th^2, th^2 = t2
    if (t2 < 1e-2) {
        ca = 1.0 - t2 / 6.0 * (1.0 - t2 / 20.0 * (1.0 - t2 / 42.0 * (1.0 - t2 / 72.0 * (1.0 - t2 / 110.0))));
        cb = 0.5 - t2 / 24.0 * (1.0 - t2 / 30.0 * (1.0 - t2 / 56.0 * (1.0 - t2 / 90.0 * (1.0 - t2 / 132.0))));
    } else {
        const double th = sqrt(t2);
        ca = sin(th) / th; cb = (1.0 - cos(th)) / t2;
    }
    const double Kx[3][3] = {{0.0, -oz, oy}, {oz, 0.0, -ox}, {-oy, ox, 0.0}};
    double Ri[3][3];
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {
            double k2 = 0.0;
            for (int k = 0; k < 3; ++k) k2 += Kx[i][k] * Kx[k][j];
            Ri[i][j] = (i == j ? 1.0 : 0.0) + ca * Kx[i][j] + cb * k2;
        }
    double out[12];
    for (int i = 0; i < 3; ++i) {
        for (int j = 0; j < 3; ++j) { double a = 0.0; for (int k = 0; k < 3; ++k) a += Ri[i][k] * T[4 * k + j]; out[4 * i + j] = a; }
        double a = 0.0; for (int k = 0; k < 3; ++k) a += Ri[i][k] * T[4 * k + 3];
        out[4 * i + 3] = a + xi[3 + i];
    }
    for (int i = 0; i < 12; ++i) T[i] = out[i];
    return 0;
}

// F7 in ONE cooperative launch (vol_frontend_track): every step is a grid-stride pass over the level's pixels into its own
// set of accumulators (all zeroed before the launch), one grid-wide barrier (an arrival counter), and the 6 x 6 solve -- done redundantly by one
// thread of every block (29 values in, 12 out: cheaper than a second barrier to broadcast the result).
struct TrackParams {
    IcpLevel lv[FE_MAX_LEVELS];
    int levels, iters[FE_MAX_LEVELS], min_count;
    float dist2, cos_min;
    double T0[12];                  // initial estimate
    double cond_min;                // icp_se3_update's threshold
    unsigned long long *acc;        // total steps x TRACK_STRIDE words (accumulators and arrival counter of every step), zeroed
    double *out;                    // 12 (T) + rms + count + status (0 ok, 1 too few correspondences, 2 not positive definite,
                                    // 3 unobservable) + level + conditioning of the last step solved
};

__global__ void __launch_bounds__(256) k_icp_track(const __grid_constant__ TrackParams q)
{
    __shared__ double sh[8][ICP_SUMS], shT[16];
    double T[12];
#pragma unroll
    for (int i = 0; i < 12; ++i) T[i] = q.T0[i];
    double rms = 0.0, count = 0.0, status = 0.0, at_level = 0.0, cond = 1.0;
    int step = 0;
    for (int l = q.levels - 1; l >= 0 && status == 0.0; --l) {
        const IcpLevel &lv = q.lv[l];
        const int tx = (lv.w + 31) / 32, tiles = tx * ((lv.h + 7) / 8);
        for (int it = 0; it < q.iters[l] && status == 0.0; ++it, ++step) {
            float R[9], t[3];
#pragma unroll
            for (int i = 0; i < 3; ++i) { R[3 * i] = (float)T[4 * i]; R[3 * i + 1] = (float)T[4 * i + 1]; R[3 * i + 2] = (float)T[4 * i + 2]; t[i] = (float)T[4 * i + 3]; }
            double s[ICP_SUMS];
#pragma unroll
            for (int i = 0; i < ICP_SUMS; ++i) s[i] = 0.0;
            for (int tile = blockIdx.x; tile < tiles; tile += gridDim.x) {
                const int x = (tile % tx) * 32 + (threadIdx.x & 31), y = (tile / tx) * 8 + (threadIdx.x >> 5);
                float J[6], r;
                if (x < lv.w && y < lv.h && icp_pixel(lv, R, t, q.dist2, q.cos_min, x, y, J, r)) icp_accumulate(s, J, r);
            }
            unsigned long long *acc = q.acc + (size_t)step * TRACK_STRIDE;
            icp_block_reduce(s, sh, acc);                        // (ends with a block barrier: this block's reductions have been issued)
            if (threadIdx.x == 0) {                              // one thread per block solves; the others take its result
                // the grid-wide barrier of this step: one arrival counter per step (zeroed with the accumulators), bumped with
                // release semantics -- cumulative over the block's reductions through the block barrier above -- and polled with
                // acquire loads.  All blocks are co-resident (cooperative launch).  Lighter than grid.sync(): no system-scope
                // fence, no L1 invalidation, and only the thread that needs the sums waits for them.
                unsigned *arrive = reinterpret_cast<unsigned *>(acc + ICP_ACC);
                asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(arrive) : "memory");
                unsigned seen;
                do { asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(arrive) : "memory"); } while (seen < gridDim.x);
                double g[ICP_SUMS];
#pragma unroll
                for (int i = 0; i < ICP_SUMS; ++i) g[i] = icp_total((long long)__ldcg(acc + i), (long long)__ldcg(acc + ICP_SUMS + i));
                count = g[28];
                if (count < (double)q.min_count) status = 1.0;
                else {
                    rms = sqrt(g[27] / count);
                    status = (double)icp_se3_update(T, g, q.cond_min, &cond);
                }
#pragma unroll
                for (int i = 0; i < 12; ++i) shT[i] = T[i];
                shT[12] = rms; shT[13] = count; shT[14] = status; shT[15] = cond;
            }
            __syncthreads();
#pragma unroll
            for (int i = 0; i < 12; ++i) T[i] = shT[i];
            rms = shT[12]; count = shT[13]; status = shT[14]; cond = shT[15]; at_level = (double)l;
            __syncthreads();
        }
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        for (int i = 0; i < 12; ++i) q.out[i] = T[i];
        q.out[12] = rms; q.out[13] = count; q.out[14] = status; q.out[15] = at_level; q.out[16] = cond;
    }
}

}  // namespace vf
