// fused.cuh -- K2: the fused integration kernel (S2-S9), warp-centric and persistent.
//
// One launch does everything that follows the per-pixel pre-pass.  Every warp first helps with the producer roles
// (prepass.cuh: geometry tile classification, shell marking -- chunks claimed from counters, so nobody waits for work that
// has not been claimed), then consumes work items until none is left:
//   geometry items (one tile of 32x4x8 TSDF voxels + the mask of its 8x4x4 sub-boxes that may be updated) are published by
//     the classification as it goes and consumed from the first microsecond; a warp takes them while there are any;
//   colour items (one non-zero shell-mark nibble = up to 4 colour cells of 8x4x4 voxels of one tile) exist once every mark
//     has been set and the mark words have been scanned (two grid-wide conditions, observed through counters); the items of
//     3-4 cells are taken first, those of 1-2 cells last, so that the kernel ends on short items.
// A lane owns an (x, y) column of a sub-box or cell (4 voxels along z), so a warp reads whole 32-byte sectors and the
// per-column part of eq. 5 is hoisted.  Colour voxels that pass the gate are compacted in a per-warp shared-memory stage and
// updated one per lane.  No block-level barriers; the state of a warp's loop lives in shared memory.
//
// The per-voxel arithmetic is the canonical sequence of DESIGN.md, issued branch-free for 4 voxels at a time
// (projection -> gathers -> update); operands outside the range of the branch-free exact reciprocal (exact.cuh) send
// the whole warp through the plain reference routines below, which use the library intrinsics.
#pragma once
#include "exact.cuh"
#include "params.cuh"
#include "prepass.cuh"

namespace vf {

// ---------------------------------------------------------------------------------------------------------------
// plain per-voxel routines (any operand range) -- the slow path, and the definition the fast path must reproduce
// ---------------------------------------------------------------------------------------------------------------

// O-G for one geometry voxel (readings A5/A6).  (X, Y, Z) = voxel centre in the depth camera (eq. 5).
__device__ __noinline__ uint32_t geo_voxel_ref(const Params &p, float X, float Y, float Z, uint32_t word, bool &read)
{
    int x, y;
    read = false;
    if (!project_px(p.fx, p.fy, p.cx, p.cy, p.wd_f, p.hd_f, X, Y, Z, x, y)) return word;
    const uint32_t d = __ldg(p.depth + y * p.wd + x);
    if (d == 0u) return word;                                             // "if non-zero" (L103)
    const float D = __fmul_rn((float)d, 0.001f);
    float sdf = __fsub_rn(D, Z);
    if (p.variant == VAR_TSDF_ALONG_RAY)                                  // measured along the voxel's viewing ray
        sdf = __fmul_rn(sdf, __fmul_rn(__fsqrt_rn(__fmaf_rn(Z, Z, __fmaf_rn(Y, Y, __fmul_rn(X, X)))), __fdiv_rn(1.0f, Z)));
    if (sdf < p.neg_mu) return word;                                      // behind the truncation band: unchanged
    read = true;
    const float tsdf = fminf(1.0f, __fmul_rn(sdf, p.inv_mu));
    const int q = (int)(short)(word & 0xffffu);
    const int w = (int)(short)(word >> 16);
    const float num = __fmaf_rn((float)q, (float)w, __fmul_rn(tsdf, 32767.0f));
    const int qn = __float2int_rn(__fdiv_rn(num, __fadd_rn((float)w, 1.0f)));
    const int wn = min(w + 1, p.w_max);
    return ((uint32_t)qn & 0xffffu) | ((uint32_t)wn << 16);
}

// sigma gate of one colour voxel (eq. 6-8 via the pixel map, L101-110).  Returns the pixel-map entry of its depth pixel
// (eq. 7's point; w = the view weight W > 0) if the voxel passes, w = 0 otherwise.
__device__ __noinline__ float4 col_voxel_gate_ref(const Params &p, float X, float Y, float Z)
{
    int x, y;
    const float4 none = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
    if (!project_px(p.fx, p.fy, p.cx, p.cy, p.wd_f, p.hd_f, X, Y, Z, x, y)) return none;
    const float4 pm = __ldg(p.pixmap + y * p.wd + x);
    if (!(pm.w > 0.0f)) return none;
    const float dx = __fsub_rn(X, pm.x), dy = __fsub_rn(Y, pm.y), dz = __fsub_rn(Z, pm.z);
    const float d2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
    return d2 > p.sig2 ? none : pm;
}

// ---------------------------------------------------------------------------------------------------------------
// branch-free projection of one voxel (fast path): pixel offset y * w + x, or ok = false.
// Precondition (tile_is_near() false for the voxel's tile): RCP_MIN <= Z <= RCP_MAX.
// ---------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void project_fast(float fx, float fy, float cx, float cy, uint32_t w, uint32_t wbits, uint32_t hbits, uint32_t koff,
                                             float X, float Y, float Z, bool &ok, uint32_t &off)
{
    const float iz = rcp_exact(Z);
    const float u = __fmaf_rn(fx, __fmul_rn(X, iz), cx);
    const float v = __fmaf_rn(fy, __fmul_rn(Y, iz), cy);
    const float tu = __fadd_rn(u, 0.5f), tv = __fadd_rn(v, 0.5f);
    // A2/A3: floor(t) in [0, w)  <=>  0 <= t < w.  t is finite and never -0, so on the bit patterns (monotonic for t >= 0,
    // sign bit set for t < 0) this is one unsigned compare against the bits of (float)w.
    ok = (__float_as_uint(tu) < wbits) && (__float_as_uint(tv) < hbits);
    // floor without the conversion pipe: for |t| < 2^22, t + 1.5 * 2^23 rounded towards -inf has floor(t) in its low
    // mantissa bits; koff = bits(1.5 * 2^23) * (w + 1) folds both biases of y * w + x into one subtraction (mod 2^32)
    const uint32_t bu = __float_as_uint(__fadd_rd(tu, 12582912.0f)), bv = __float_as_uint(__fadd_rd(tv, 12582912.0f));
    off = ok ? bv * w + bu - koff : 0u;
}

// the same without the final select: off is only meaningful when ok
__device__ __forceinline__ void project_fast_raw(float fx, float fy, float cx, float cy, uint32_t w, uint32_t wbits, uint32_t hbits, uint32_t koff,
                                                 float X, float Y, float Z, bool &ok, uint32_t &off, float &iz)
{
    iz = rcp_exact(Z);
    const float u = __fmaf_rn(fx, __fmul_rn(X, iz), cx);
    const float v = __fmaf_rn(fy, __fmul_rn(Y, iz), cy);
    const float tu = __fadd_rn(u, 0.5f), tv = __fadd_rn(v, 0.5f);
    ok = (__float_as_uint(tu) < wbits) && (__float_as_uint(tv) < hbits);
    const uint32_t bu = __float_as_uint(__fadd_rd(tu, 12582912.0f)), bv = __float_as_uint(__fadd_rd(tv, 12582912.0f));
    off = bv * w + bu - koff;
}

// lane 0 draws the next queue ticket.  A predicated instruction, not a branch: the warp must not diverge here, or the
// compiler may run the whole item once for lane 0 and once for the other lanes.
__device__ __forceinline__ void next_ticket(uint32_t *cursor, int lane, uint32_t &ticket)
{
    asm volatile("{\n\t.reg .pred q;\n\tsetp.eq.s32 q, %1, 0;\n\t@q atom.global.add.u32 %0, [%2], 1;\n\t}"
                 : "+r"(ticket) : "r"(lane), "l"(cursor) : "memory");
}
// the same for `n` consecutive tickets
__device__ __forceinline__ void next_tickets(uint32_t *cursor, uint32_t n, int lane, uint32_t &ticket)
{
    asm volatile("{\n\t.reg .pred q;\n\tsetp.eq.s32 q, %1, 0;\n\t@q atom.global.add.u32 %0, [%2], %3;\n\t}"
                 : "+r"(ticket) : "r"(lane), "l"(cursor), "r"(n) : "memory");
}
// n consecutive tickets, the first one returned to every lane at once
__device__ __forceinline__ uint32_t claim_n(uint32_t *counter, uint32_t n, int lane)
{
    uint32_t t = 0;
    next_tickets(counter, n, lane, t);
    return __shfl_sync(0xffffffffu, t, 0);
}
// one ticket, returned to every lane at once (producer chunks: the result is needed right away)
__device__ __forceinline__ uint32_t claim(uint32_t *counter, int lane)
{
    uint32_t t = 0;
    next_ticket(counter, lane, t);
    return __shfl_sync(0xffffffffu, t, 0);
}
// a chunk of producer work is finished: the counter the consumers watch is bumped with release semantics (a MEMBAR before
// the reduction, and -- unlike __threadfence() -- no invalidation of this SM's L1, which the other warps' gathers live on)
__device__ __forceinline__ void chunk_done(uint32_t *counter, int lane)
{
    __syncwarp();
    if (lane == 0) asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(counter) : "memory");
}
// polling load of a control word or a work-list slot: served by L2, no acquire (an acquire invalidates L1 every time).
// What the flag guards is only ever read through L2 afterwards (ld.cg, atomics), and only in code that is control-dependent
// on the polled value.
__device__ __forceinline__ uint32_t ld_relaxed(const uint32_t *ptr)
{
    uint32_t v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(ptr) : "memory");
    return v;
}

struct Counts { unsigned long long n[CNT_N]; };

#ifndef VF_COL_BATCH
#define VF_COL_BATCH 4
#endif
constexpr uint32_t COL_BATCH = VF_COL_BATCH, COL_BATCH_TAIL = 12, GEO_BATCH = 1;
// per-warp state of the consumer loop (shared memory; written by lane 0 between __syncwarp()s, read by every lane): the items
// need every register, and what is kept in shared memory is not spilled to (cached, evictable) local memory around them
enum : uint32_t { F_GEO_DONE = 1u, F_COL_DONE = 2u, F_MARKS_SET = 4u, F_SCAN_CLAIMED = 8u, F_COL_READY = 16u, F_CLS_COMPLETE = 32u };
struct WarpState {
    uint32_t flags;                 // F_*
    uint32_t gt, gt_left;           // next geometry ticket of the warp and how many of its batch are left
    uint32_t ct, ct_size;           // first ticket and size of the NEXT batch of colour items
    uint32_t cb_left, cb_idx;       // the current batch: items left, index of the next one
    uint32_t n_col, n_col_big;      // length of the colour work list (once it is final), and how many of its items are long ones
    int      n_staged;              // fill level of the warp's stage
    uint32_t cb_item[COL_BATCH][2]; // the current batch
};

// development aid (compile with -DVF_TRACE): per-warp timestamps of the phase transitions of k_fused, 16 words per warp
#ifdef VF_TRACE
__device__ unsigned long long g_trace[8192 * 16];
__device__ __forceinline__ unsigned long long vf_now() { unsigned long long t; asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t)); return t; }
#define VF_T(slot) do { if (lane == 0 && gw < 8192u) g_trace[gw * 16u + (slot)] = vf_now(); } while (0)
#define VF_TC(slot, v) do { if (lane == 0 && gw < 8192u) g_trace[gw * 16u + (slot)] = (v); } while (0)
#else
#define VF_T(slot) do { } while (0)
#define VF_TC(slot, v) do { } while (0)
#endif

// COUNT only: 1 if the lane is the first of the whole frame to touch the 32-byte sector (8 words) of word index `word` in
// volume map `which` (Params::sec_map)
__device__ __forceinline__ unsigned sector_first(const Params &p, int which, bool pred, unsigned long long word)
{
    if (!pred) return 0u;
    const unsigned long long s = word >> 3;
    const uint32_t bit = 1u << (unsigned)(s & 31ull);
    return (atomicOr(p.sec_map[which] + (s >> 5), bit) & bit) ? 0u : 1u;
}

// ptr + e layers (e = 0..3 a compile-time constant after unrolling): one mad.wide with an immediate
__device__ __forceinline__ uint32_t *layer_ptr(uint32_t *ptr, int e, uint32_t layer_b)
{
    unsigned long long a = (unsigned long long)ptr;
    if (e == 1) asm("mad.wide.u32 %0, %1, 1, %2;" : "=l"(a) : "r"(layer_b), "l"(a));
    if (e == 2) asm("mad.wide.u32 %0, %1, 2, %2;" : "=l"(a) : "r"(layer_b), "l"(a));
    if (e == 3) asm("mad.wide.u32 %0, %1, 3, %2;" : "=l"(a) : "r"(layer_b), "l"(a));
    return reinterpret_cast<uint32_t *>(a);
}


// COUNT only: how many distinct 32-byte sectors (8 words) the lanes with `pred` touch at word index `word`
__device__ __forceinline__ unsigned sectors_touched(bool pred, unsigned long long word, int lane)
{
    const unsigned act = __ballot_sync(0xffffffffu, pred);
    unsigned first = 0;
    if (pred) {
        const unsigned peers = __match_any_sync(act, word >> 3);
        first = (__ffs(peers) - 1 == lane) ? 1u : 0u;
    }
    return first;
}

// S3 for four voxels of one lane (stored words o, camera depth Z of the voxel, depth D of its pixel -- 0 = none --, and, for
// VAR_TSDF_ALONG_RAY, the factor L from the distance along z to the distance along the ray): truncation test and running
// average; w4 = the new words.  Votes with the whole warp: every lane must call it.
template <bool COUNT, int VAR>
__device__ __forceinline__ void tsdf_update4(const uint32_t (&o)[4], const float (&Z)[4], const float (&D)[4], const float (&L)[4],
                                             float neg_mu, float inv_mu, int w_max, uint32_t (&w4)[4], bool (&upd)[4])
{
    float sdf[4];
    bool easy = true;
#pragma unroll
    for (int e = 0; e < 4; ++e) {
        sdf[e] = __fsub_rn(D[e], Z[e]);
        if (VAR == VAR_TSDF_ALONG_RAY) sdf[e] = __fmul_rn(sdf[e], L[e]);
        upd[e] = (D[e] != 0.0f) & !(sdf[e] < neg_mu);
        // saturated free space (tsdf = 1 onto q = 32767) or first touch (w = 0): the running average is 32767 exactly,
        // fma(32767, w, 32767) / (w + 1) with every intermediate below 2^24.  (Bitwise on purpose: no branches.)
        easy = easy & (!upd[e] | ((__fmul_rn(sdf[e], inv_mu) >= 1.0f) & (((o[e] & 0xffffu) == 0x7fffu) | (o[e] < 0x10000u))));
    }
    if (__all_sync(0xffffffffu, easy)) {                              // whole warp in free space: no division needed
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const int wn = min((int)(short)(o[e] >> 16) + 1, w_max);
            w4[e] = upd[e] ? (0x7fffu | ((uint32_t)wn << 16)) : o[e];
        }
    } else {
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const float tsdf = fminf(1.0f, __fmul_rn(sdf[e], inv_mu));
            const int q = (int)(short)(o[e] & 0xffffu);
            const int wi = (int)(short)(o[e] >> 16);
            const float wf = (float)wi;
            // num is 0 or 2^-40 <= |num| < 2^26 (vol_create bounds mu), den in [1, 513]
            const float num = __fmaf_rn((float)q, wf, __fmul_rn(tsdf, 32767.0f));
            const float den = __fadd_rn(wf, 1.0f);
            // rint (half-even) without the conversion pipe: |quotient| <= 32767, so adding 1.5 * 2^23 leaves it in the
            // low mantissa bits, already in two's complement
            const uint32_t qn = __float_as_uint(__fadd_rn(div_with(num, den, div_prepare(den)), 12582912.0f));
            const int wn = min(wi + 1, w_max);
            const uint32_t nw = (qn & 0xffffu) | ((uint32_t)wn << 16);
            w4[e] = upd[e] ? nw : o[e];
        }
    }
}

// NEAR tiles (may hold voxels with Z <= 0 or outside rcp_exact's range) take the plain per-voxel routine, whole.
template <bool COUNT>
__device__ __noinline__ void geometry_tile_near(const Params &p, int ttx, int tty, int ttz, int lane, Counts &c)
{
    const int xl = lane & 7, j = tty * TY + (lane >> 3);
    const int gz0 = local_to_global_tz(p, ttz) * TZ, lz0 = ttz * TZ;
    const float py = __fmaf_rn((float)j + 0.5f, p.vs, p.oy);
    for (int bx = 0; bx < SUBX; ++bx) {
        const int i = ttx * TX + 8 * bx + xl;
        if (!(i < p.nx && j < p.ny)) continue;
        const float px = __fmaf_rn((float)i + 0.5f, p.vs, p.ox);
        const float bX = __fmaf_rn(p.R[1], py, __fmaf_rn(p.R[0], px, p.t[0]));
        const float bY = __fmaf_rn(p.R[4], py, __fmaf_rn(p.R[3], px, p.t[1]));
        const float bZ = __fmaf_rn(p.R[7], py, __fmaf_rn(p.R[6], px, p.t[2]));
#pragma unroll 1
        for (int z = 0; z < TZ && gz0 + z < p.nz; ++z) {
            uint32_t *ptr = p.geo + ((size_t)(lz0 + z) * p.ny + j) * p.nx + i;
            const uint32_t o = *ptr;
            const float pz = __fmaf_rn((float)(gz0 + z) + 0.5f, p.vs, p.oz);
            bool rd = false;
            const uint32_t w = geo_voxel_ref(p, __fmaf_rn(p.R[2], pz, bX), __fmaf_rn(p.R[5], pz, bY), __fmaf_rn(p.R[8], pz, bZ), o, rd);
            if (COUNT) {
                c.n[CNT_GEO_VISITED] += 1; c.n[CNT_GEO_READ] += rd; c.n[CNT_GEO_CHANGED] += w != o;
                const unsigned long long wi = (unsigned long long)(ptr - p.geo);
                c.n[CNT_GEO_SEC_READ] += sector_first(p, 0, rd, wi); c.n[CNT_GEO_SEC_WRITTEN] += sector_first(p, 1, w != o, wi);
            }
            if (w != o) *ptr = w;
        }
    }
}

// The wanted sub-boxes (bits of m4: bx = 0..3) of one z half of a geometry tile, one warp pass each: lane = (x = lane & 7,
// y = lane >> 3) owns the column of 4 voxels along z, so every access of the warp is four whole 32-byte sectors and the
// per-column part of eq. 5 is hoisted.  The passes are software-pipelined over two alternating register sets: while
// sub-box n is updated, sub-box n + 1 has already been projected and its depth gathers and voxel loads are in flight.
// FULL: the half lies wholly inside the volume (no voxel of it needs a bounds test).
// Returns, in visiting order (bit n = the n-th wanted sub-box), which sub-boxes hold nothing but the saturated free-space
// word afterwards.  COUNT: sk4 = the sub-boxes (bits bx) the plain variant would not have been given (their voxels are
// counted as skippable too).
template <bool COUNT, int VAR, bool FULL>
__device__ __forceinline__ uint32_t geometry_half_boxes(const Params &p, int ttx, int tty, int gz0, int lz0, uint32_t m4, uint32_t sk4, int lane, Counts &c)
{
    const int xl = lane & 7, j = tty * TY + (lane >> 3);
    const float fx = p.fx, fy = p.fy, cx = p.cx, cy = p.cy, vs = p.vs;
    const float neg_mu = p.neg_mu, inv_mu = p.inv_mu;
    const uint32_t wd = (uint32_t)p.wd, wbits = __float_as_uint(p.wd_f), hbits = __float_as_uint(p.hd_f), koff = 0x4B400000u * (wd + 1u);
    const int w_max = p.w_max;
    const float *__restrict__ depthf = p.depthf;
    const float py = __fmaf_rn((float)j + 0.5f, vs, p.oy);
    const float r02 = p.R[2], r12 = p.R[5], r22 = p.R[8];
    const uint32_t layer_b = (uint32_t)((size_t)p.ny * p.nx * 4u);
    const int nrem_row = FULL ? 4 : (j < p.ny ? p.nz - gz0 : 0);      // layers of this half the lane's row really has
    const int i0 = ttx * TX + xl;
    uint32_t *const row_ptr = p.geo + ((size_t)lz0 * p.ny + j) * p.nx + i0;   // the lane's voxel of the half's first layer in sub-box 0
    float pz[4];
#pragma unroll
    for (int e = 0; e < 4; ++e) pz[e] = __fmaf_rn((float)(gz0 + e) + 0.5f, vs, p.oz);
    // S2 of one sub-box: eq. 5, projection, the four depth gathers and the four voxel loads.  A voxel outside the frustum
    // or the volume keeps D = 0 ("invalid depth": not updated); its gather is predicated off.
    auto load_project = [&](int bx, uint32_t *&ptr, uint32_t (&o)[4], float (&Z)[4], float (&D)[4], float (&L)[4]) {
        const int i = i0 + 8 * bx;
        const int nrem = FULL ? 4 : (i < p.nx ? nrem_row : 0);
        const float px = __fmaf_rn((float)i + 0.5f, vs, p.ox);
        const float bX = __fmaf_rn(p.R[1], py, __fmaf_rn(p.R[0], px, p.t[0]));
        const float bY = __fmaf_rn(p.R[4], py, __fmaf_rn(p.R[3], px, p.t[1]));
        const float bZ = __fmaf_rn(p.R[7], py, __fmaf_rn(p.R[6], px, p.t[2]));
        ptr = row_ptr + 8 * bx;
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const bool in = FULL || e < nrem;
            // the voxel stream bypasses L1 (__ldcg): every sector is used once, and L1 is better spent on the depth image
            if (FULL) o[e] = __ldcg(layer_ptr(ptr, e, layer_b));
            else { o[e] = 0u; if (in) o[e] = __ldcg(layer_ptr(ptr, e, layer_b)); }
            const float X = __fmaf_rn(r02, pz[e], bX), Y = __fmaf_rn(r12, pz[e], bY);
            Z[e] = __fmaf_rn(r22, pz[e], bZ);
            bool ok; uint32_t off; float iz;
            project_fast_raw(fx, fy, cx, cy, wd, wbits, hbits, koff, X, Y, Z[e], ok, off, iz);
            if (VAR == VAR_TSDF_ALONG_RAY)
                L[e] = __fmul_rn(__fsqrt_rn(__fmaf_rn(Z[e], Z[e], __fmaf_rn(Y, Y, __fmul_rn(X, X)))), iz);
            D[e] = 0.0f;
            if (ok && in) D[e] = __ldg(depthf + off);
        }
    };
    // S3 of one sub-box (the n-th of the half, bx its number): truncation test, running average, store of the words that
    // changed; true if the sub-box holds nothing but the saturated free-space word afterwards.  (A column that is partly
    // outside the volume never does: its missing voxels read as 0.)
    auto update = [&](int bx, uint32_t *ptr, const uint32_t (&o)[4], const float (&Z)[4], const float (&D)[4], const float (&L)[4]) -> bool {
        uint32_t w4[4]; bool upd[4];
        tsdf_update4<COUNT, VAR>(o, Z, D, L, neg_mu, inv_mu, w_max, w4, upd);
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            if (COUNT) {
                const unsigned long long wi = (unsigned long long)(layer_ptr(ptr, e, layer_b) - p.geo);
                c.n[CNT_GEO_VISITED] += 1; c.n[CNT_GEO_READ] += upd[e]; c.n[CNT_GEO_CHANGED] += w4[e] != o[e];
                const unsigned sr = sector_first(p, 0, upd[e], wi);
                c.n[CNT_GEO_SEC_READ] += sr;
                c.n[CNT_GEO_SEC_WRITTEN] += sector_first(p, 1, w4[e] != o[e], wi);
                if ((sk4 >> bx) & 1u) { c.n[CNT_GEO_SKIPPABLE] += upd[e]; c.n[CNT_GEO_SEC_SKIPPABLE] += sr; }
            }
            if (w4[e] != o[e]) __stcg(layer_ptr(ptr, e, layer_b), w4[e]);   // skip the store when nothing changed
        }
        const uint32_t sat_word = 0x7fffu | ((uint32_t)w_max << 16);
        return __all_sync(0xffffffffu, (((w4[0] ^ sat_word) | (w4[1] ^ sat_word)) | ((w4[2] ^ sat_word) | (w4[3] ^ sat_word))) == 0u);
    };
    if (COUNT && lane == 0) atomicAdd(&p.ctrl[ST_SUBS], (uint32_t)__popc(m4));
    uint32_t m = m4, satseq = 0u;
    if (!FULL) {
        // a half that sticks out of the volume (the last tiles of an axis): one sub-box after the other, no pipeline
        uint32_t *pA, oA[4];
        float ZA[4], DA[4], LA[4];
#pragma unroll 1
        for (uint32_t n = 0; m != 0u; ++n) {
            const int bx = __ffs(m) - 1; m &= m - 1u;
            load_project(bx, pA, oA, ZA, DA, LA);
            satseq |= (update(bx, pA, oA, ZA, DA, LA) ? 1u : 0u) << n;
        }
        return satseq;
    }
    // Two register sets, A and B, used alternately (no register-to-register rotation).  n = position of set A's sub-box in
    // the visiting order (set B's is n + 1).
    uint32_t *pA, *pB, oA[4], oB[4];
    float ZA[4], ZB[4], DA[4], DB[4], LA[4], LB[4];
    int b = __ffs(m) - 1, bxA = b, bxB = 0;                              // (bxA / bxB: only the counting variant keeps them)
    m &= m - 1u;
    load_project(b, pA, oA, ZA, DA, LA);
#pragma unroll 1
    for (uint32_t n = 0;; n += 2) {
        const bool hasB = m != 0u;
        if (hasB) { b = __ffs(m) - 1; m &= m - 1u; bxB = b; load_project(b, pB, oB, ZB, DB, LB); }   // sub-box n + 1 in flight
        satseq |= (update(COUNT ? bxA : 0, pA, oA, ZA, DA, LA) ? 1u : 0u) << n;
        if (!hasB) break;
        const bool hasA = m != 0u;
        if (hasA) { b = __ffs(m) - 1; m &= m - 1u; bxA = b; load_project(b, pA, oA, ZA, DA, LA); }   // sub-box n + 2 in flight
        satseq |= (update(COUNT ? bxB : 0, pB, oB, ZB, DB, LB) ? 2u : 0u) << n;
        if (!hasA) break;
    }
    return satseq;
}

// one geometry tile, one warp.  The item names the tile's 8x4x4 sub-boxes that may hold a voxel this frame updates; they
// are visited z half by z half (4 layers).
// (A whole-row path for z halves whose four sub-boxes are all wanted -- 16-byte vectors, everything per layer shared by four
// voxels -- was measured: 14 % faster on a saturating frame, but its registers cost the scan frames 8 % even when it is not
// taken, so it is not in the kernel.)
template <bool COUNT, int VAR>
__device__ __forceinline__ void geometry_tile(const Params &p, uint32_t item, int lane, Counts &c)
{
    int ttx, tty, ttz, mask;
    item_unpack(item, ttx, tty, ttz, mask);
    const uint32_t tile = (uint32_t)((ttz * p.tiles_y + tty) * p.tiles_x + ttx);
    if (tile_is_near(p, ttx, tty, ttz)) {
        if (lane == 0) p.tile_sat[tile] = 0;
        geometry_tile_near<COUNT>(p, ttx, tty, ttz, lane, c);
        return;
    }
    const int gz0 = local_to_global_tz(p, ttz) * TZ, lz0 = ttz * TZ;
    uint32_t sat = (uint32_t)__ldg(p.tile_sat + tile) & ~(uint32_t)mask;   // the visited sub-boxes are looked at afresh
    const uint32_t skippable = COUNT ? (uint32_t)__ldcg(p.tile_skip + tile) : 0u;
    const bool full_xy = ttx * TX + TX <= p.nx && tty * TY + TY <= p.ny;
#pragma unroll 1
    for (int zh = 0; zh < SUBZ; ++zh) {
        uint32_t m = ((uint32_t)mask >> zh) & 0x55u;                  // bit 2 bx: sub-box bx of this half
        if (m == 0u) continue;
        m = (m | (m >> 1)) & 0x33u; m = (m | (m >> 2)) & 0x0fu;       // bit bx
        uint32_t sk = (skippable >> zh) & 0x55u;
        sk = (sk | (sk >> 1)) & 0x33u; sk = (sk | (sk >> 2)) & 0x0fu;
        const int g = gz0 + zh * (TZ / SUBZ), l = lz0 + zh * (TZ / SUBZ);
        uint32_t seq = full_xy && g + TZ / SUBZ <= p.nz ? geometry_half_boxes<COUNT, VAR, true>(p, ttx, tty, g, l, m, sk, lane, c)
                                                        : geometry_half_boxes<COUNT, VAR, false>(p, ttx, tty, g, l, m, sk, lane, c);
        for (; seq != 0u && m != 0u; seq >>= 1, m &= m - 1u)           // visiting order -> item mask bit 2 bx + zh
            if (seq & 1u) sat |= 1u << (2 * (__ffs(m) - 1) + zh);
    }
    if (lane == 0) p.tile_sat[tile] = (uint8_t)sat;
}

// pull the sectors of a geometry tile into L2 when the tile is started: lane = (row, layer); a layer is wanted when its z
// half holds a sub-box of the mask.  (Whole 128-byte lines: the x sub-boxes a tile leaves out are the minority.)
__device__ __forceinline__ void geometry_prefetch(const Params &p, uint32_t item, int lane)
{
    int ttx, tty, ttz, mask;
    item_unpack(item, ttx, tty, ttz, mask);
    const int j = tty * TY + (lane & 3), lz = ttz * TZ + (lane >> 2);
    const bool wanted = ((mask >> ((lane >> 2) / (TZ / SUBZ))) & 0x55) != 0;
    if (j < p.ny && lz < p.local_nz && wanted)
        asm volatile("prefetch.global.L2 [%0];" ::"l"(p.geo + ((size_t)lz * p.ny + j) * p.nx + ttx * TX));
}

// Per-warp staging buffer of colour voxels that passed the sigma gate.  The gate (S4-S5) runs on whole cells, 4 voxels
// per lane, and only a fraction of them passes; the update (S6-S8: weight gate, HD lookup, eq. 9-10) is several times
// longer.  Passing voxels are therefore compacted here and updated 32 at a time with every lane busy.
constexpr int STAGE_CAP = 64;             // up to 31 carried over + the 32 of one layer of a cell
struct Stage {
    float4 rec[STAGE_CAP];                // {X, Y, Z} = voxel centre in the depth camera (eq. 5) -- or, VAR_HD_FROM_DEPTH_POINT, the
                                          // 3D point of its depth pixel (eq. 7); W = view weight of its pixel
    uint2  adr[STAGE_CAP];                // word index of the voxel in this shard's colour volume (lo, hi)
};

// S6-S8 (weight gate L115, HD pixel eq. 3-4, eq. 9, eq. 10) for up to 32 staged voxels [first, first + n): one voxel per
// lane.  The HD pixel (eq. 3-4) is computed and its three bytes requested BEFORE the stored word arrives: the two gathers do
// not depend on each other, so their latencies overlap instead of adding up (the word is a DRAM access, and one warp
// works through its stage round after round).  A voxel that then fails the weight gate has fetched 3 bytes in vain.
// Like the gate, the update issues the exact reciprocal / quotient sequences directly (exact.cuh) when every lane's operands
// are in their range -- Z_hd in [RCP_MIN, RCP_MAX] or <= 0, and a new-sample weight 255 W >= 2^-20 -- and integer
// conversions as magic-number additions; otherwise the whole round takes the plain routines.
template <bool COUNT, int VAR>
__device__ __forceinline__ void colour_update_staged(const Params &p, const Stage &st, int first, int n, int lane, Counts &c)
{
    const bool have = lane < n;
    uint32_t old = 0u, nw = 0u;
    unsigned long long wi = 0ull;
    float4 r = make_float4(0.f, 0.f, 1.f, 1.f);
    uint32_t *ptr = p.col;
    if (have) {
        r = st.rec[first + lane];
        const uint2 a = st.adr[first + lane];
        wi = ((unsigned long long)a.y << 32) | (unsigned long long)a.x;
        ptr = p.col + wi;
        old = __ldcg(ptr);                                            // first HBM touch of this colour voxel (S6); L2 only
    }
    // HD pixel of the voxel's own position (eq. 3-4; A10, A11)
    const float Xh = __fmaf_rn(p.Rc[2], r.z, __fmaf_rn(p.Rc[1], r.y, __fmaf_rn(p.Rc[0], r.x, p.tc[0])));
    const float Yh = __fmaf_rn(p.Rc[5], r.z, __fmaf_rn(p.Rc[4], r.y, __fmaf_rn(p.Rc[3], r.x, p.tc[1])));
    const float Zh = __fmaf_rn(p.Rc[8], r.z, __fmaf_rn(p.Rc[7], r.y, __fmaf_rn(p.Rc[6], r.x, p.tc[2])));
    const float W = r.w, W255 = __fmul_rn(W, 255.0f);
    const bool tame = !have || ((!(Zh > 0.0f) || (Zh >= RCP_MIN && Zh <= RCP_MAX)) && W255 >= 0x1p-20f);
    if (__all_sync(0xffffffffu, tame)) {
        const uint32_t wh = (uint32_t)p.wh;
        bool okh; uint32_t off;
        project_fast(p.fxh, p.fyh, p.cxh, p.cyh, wh, __float_as_uint(p.wh_f), __float_as_uint(p.hh_f), 0x4B400000u * (wh + 1u),
                     Xh, Yh, Zh > 0.0f ? Zh : 1.0f, okh, off);                 // A13; A14: nearest pixel (offset 0 when outside: a valid address)
        okh = okh && Zh > 0.0f && have;
        unsigned long long addr;
        asm("mad.wide.u32 %0, %1, 3, %2;" : "=l"(addr) : "r"(okh ? off : 0u), "l"(p.rgb));
        const uint8_t *hd = reinterpret_cast<const uint8_t *>(addr);
        const uint32_t h0 = __ldg(hd), h1 = __ldg(hd + 1), h2 = __ldg(hd + 2);
        const uint32_t wq = old >> 24;
        const float wqf = (float)wq;
        nw = old;
        if (okh && W255 > __fmul_rn(p.gate, wqf)) {                   // L115, A9
            const float den = __fadd_rn(wqf, W255), rden = div_prepare(den);   // den in [2^-20, 510]
            const uint32_t h[3] = {h0, h1, h2};
            nw = 0u;
#pragma unroll
            for (int ch = 0; ch < 3; ++ch) {                          // eq. 9: the quotient lies in [0, 255], so the clamp is idle
                const uint32_t C = (old >> (8 * ch)) & 0xffu;
                const float num = __fmaf_rn(W255, (float)h[ch], (float)(C * wq));   // 0 or in [2^-20, 2^17]
                const uint32_t ci = __float_as_uint(__fadd_rn(div_with(num, den, rden), 12582912.0f)) & 0x1ffu;   // rint, half-even
                nw |= min(ci, 255u) << (8 * ch);
            }
            const float wnf = VAR == VAR_ADDITIVE_WEIGHT ? __fadd_rn(wqf, W255)                    // W_pre + W
                                                         : __fmaf_rn(W, (float)(255u - wq), wqf); // eq. 10, A12
            const uint32_t wn = __float_as_uint(__fadd_rn(wnf, 12582912.0f)) & 0x3ffu;             // rint; wnf in [0, 510]
            nw |= min(wn, 255u) << 24;
            if (nw != old) *ptr = nw;
        }
    } else if (have) {
        int xh = 0, yh = 0;
        const bool okh = project_px(p.fxh, p.fyh, p.cxh, p.cyh, p.wh_f, p.hh_f, Xh, Yh, Zh, xh, yh);   // A13
        const uint8_t *hd = p.rgb + (size_t)(yh * p.wh + xh) * 3;     // A14: nearest pixel ((0, 0) when outside: a valid address)
        const uint32_t h0 = __ldg(hd), h1 = __ldg(hd + 1), h2 = __ldg(hd + 2);
        const int wq = (int)(old >> 24);
        nw = old;
        if (okh && W255 > __fmul_rn(p.gate, (float)wq)) {             // L115, A9
            const float den = __fadd_rn((float)wq, W255);
            const uint32_t h[3] = {h0, h1, h2};
            nw = 0;
#pragma unroll
            for (int ch = 0; ch < 3; ++ch) {                          // eq. 9
                const int C = (int)((old >> (8 * ch)) & 0xffu);
                const float num = __fmaf_rn(W255, (float)h[ch], (float)(C * wq));
                const float cn = rintf(__fdiv_rn(num, den));
                const int ci = cn < 0.0f ? 0 : (cn > 255.0f ? 255 : (int)cn);
                nw |= (uint32_t)ci << (8 * ch);
            }
            int wn = VAR == VAR_ADDITIVE_WEIGHT ? __float2int_rn(__fadd_rn((float)wq, W255))          // W_pre + W
                                                : __float2int_rn(__fmaf_rn(W, (float)(255 - wq), (float)wq)); // eq. 10, A12
            nw |= (uint32_t)min(wn, 255) << 24;
            if (nw != old) *ptr = nw;
        }
    }
    if (COUNT) {
        c.n[CNT_COL_READ] += have; c.n[CNT_COL_CHANGED] += have && nw != old;
        c.n[CNT_COL_SEC_READ] += sector_first(p, 2, have, wi);
        c.n[CNT_COL_SEC_WRITTEN] += sector_first(p, 3, have && nw != old, wi);
    }
}

// one colour cell of 8 x 4 x 4 voxels, one warp: lane = (x = lane & 7, y = lane >> 3) owns the column of 4 voxels along z,
// so the per-column part of eq. 5 is hoisted.  (ic, jc) = the lane's column in the full colour grid, kcg / kcl = the cell's
// first layer in the full grid / in this shard.  Voxels that pass the gate are appended to the warp's stage, layer by
// layer (n = its fill level, warp-uniform); full groups of 32 are updated at once.
template <bool COUNT, int VAR>
__device__ __forceinline__ void colour_cell(const Params &p, bool near, int ic, int jc, int kcg, int kcl, Stage &st, int &n, int lane, Counts &c)
{
    const float fx = p.fx, fy = p.fy, cx_ = p.cx, cy_ = p.cy, sig2 = p.sig2;
    const uint32_t wd = (uint32_t)p.wd, wbits = __float_as_uint(p.wd_f), hbits = __float_as_uint(p.hd_f), koff = 0x4B400000u * (wd + 1u);
    const float4 *__restrict__ pixmap = p.pixmap;
    const bool in_xy = ic < p.cnx && jc < p.cny;
    const float px = __fmaf_rn((float)ic + 0.5f, p.vc, p.ox);
    const float py = __fmaf_rn((float)jc + 0.5f, p.vc, p.oy);
    const float bX = __fmaf_rn(p.R[1], py, __fmaf_rn(p.R[0], px, p.t[0]));      // S4: eq. 5, the part that does not depend on z
    const float bY = __fmaf_rn(p.R[4], py, __fmaf_rn(p.R[3], px, p.t[1]));
    const float bZ = __fmaf_rn(p.R[7], py, __fmaf_rn(p.R[6], px, p.t[2]));
    const float kf0 = (float)kcg + 0.5f;
    float X[4], Y[4], Z[4];
    float4 pm[4];
    bool pass[4];
    if (near) {
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const float pz = __fmaf_rn(__fadd_rn(kf0, (float)e), p.vc, p.oz);
            X[e] = __fmaf_rn(p.R[2], pz, bX); Y[e] = __fmaf_rn(p.R[5], pz, bY); Z[e] = __fmaf_rn(p.R[8], pz, bZ);
            const bool act = in_xy && kcg + e < p.cnz;
            pm[e] = act ? col_voxel_gate_ref(p, X[e], Y[e], Z[e]) : make_float4(0.0f, 0.0f, 0.0f, 0.0f);
            pass[e] = pm[e].w > 0.0f;
        }
    } else {
        uint32_t off[4]; bool ok[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const float pz = __fmaf_rn(__fadd_rn(kf0, (float)e), p.vc, p.oz);
            X[e] = __fmaf_rn(p.R[2], pz, bX); Y[e] = __fmaf_rn(p.R[5], pz, bY); Z[e] = __fmaf_rn(p.R[8], pz, bZ);
            project_fast(fx, fy, cx_, cy_, wd, wbits, hbits, koff, X[e], Y[e], Z[e], ok[e], off[e]);   // eq. 6
        }
#pragma unroll
        for (int e = 0; e < 4; ++e) pm[e] = __ldg(pixmap + off[e]);      // eq. 7-8 and W per pixel (S1)
#pragma unroll
        for (int e = 0; e < 4; ++e) {                                 // S5: sigma gate (L108)
            const float dx = __fsub_rn(X[e], pm[e].x), dy = __fsub_rn(Y[e], pm[e].y), dz = __fsub_rn(Z[e], pm[e].z);
            const float d2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
            pass[e] = in_xy && kcg + e < p.cnz && ok[e] && (pm[e].w > 0.0f) && !(d2 > sig2);
        }
    }
    if (COUNT) c.n[CNT_COL_GATED] += in_xy ? (unsigned long long)max(0, min(4, p.cnz - kcg)) : 0ull;
    // compact, layer by layer: one vote each; a full group of 32 is updated at once
    const unsigned lt = (1u << lane) - 1u;
    const size_t col0 = ((size_t)kcl * (size_t)p.cny + (size_t)jc) * (size_t)p.cnx + (size_t)ic, clayer = (size_t)p.cny * (size_t)p.cnx;
#pragma unroll
    for (int e = 0; e < 4; ++e) {
        const unsigned b = __ballot_sync(0xffffffffu, pass[e]);
        if (b == 0u) continue;                                        // warp-uniform
        if (pass[e]) {
            const size_t a = col0 + (size_t)e * clayer;
            // start the DRAM access of the stored word now; the update reads it a few hundred cycles later
            asm volatile("prefetch.global.L2 [%0];" ::"l"(p.col + a));
            const int slot = n + __popc(b & lt);
            st.rec[slot] = VAR == VAR_HD_FROM_DEPTH_POINT ? pm[e] : make_float4(X[e], Y[e], Z[e], pm[e].w);
            st.adr[slot] = make_uint2((uint32_t)a, (uint32_t)(a >> 32));
        }
        n += __popc(b);
        __syncwarp();
        if (n >= 32) { n -= 32; colour_update_staged<COUNT, VAR>(p, st, n, 32, lane, c); __syncwarp(); }
    }
}

// one colour work item, one warp: the set bits of one nibble of a shell-mark word are up to 4 colour cells of one tile.
template <int R, bool COUNT, int VAR>
__device__ __forceinline__ void colour_item(const Params &p, uint2 item, Stage &st, int &n, int lane, Counts &c)
{
    constexpr int CX = cells_x(R), CY = cells_y(R);
    int ttx, tty, ttz, sub;
    item_unpack(item.x, ttx, tty, ttz, sub);
    const bool near = tile_is_near(p, ttx, tty, ttz);
    const int word = sub >> 3;
    uint32_t bits = item.y;
    const int cgx0 = ttx * TX * R, cgy0 = tty * TY * R;
    const int cgz0 = local_to_global_tz(p, ttz) * TZ * R, clz0 = ttz * TZ * R;
    if (COUNT && lane == 0) atomicAdd(&p.ctrl[ST_CELLS], (uint32_t)__popc(bits));
    while (bits) {
        const int b = word * 32 + (__ffs(bits) - 1);
        bits &= bits - 1;
        const int cx = b % CX, cy = (b / CX) % CY, cz = b / (CX * CY);
        colour_cell<COUNT, VAR>(p, near, cgx0 + cx * CLX + (lane & 7), cgy0 + cy * CLY + (lane >> 3), cgz0 + cz * CLZ, clz0 + cz * CLZ, st, n, lane, c);
    }
}

// phase: PHASE_ALL = everything in one launch (frames already on the device); PHASE_GEO = the producer roles and the
// geometry items; PHASE_COL = the colour items only -- so that vol_integrate_host can run everything that only needs the
// depth image while the HD frame is still being copied (only the colour update reads it).
enum { PHASE_ALL = 0, PHASE_GEO = 1, PHASE_COL = 2 };
#ifndef VF_MIN_CTAS
#define VF_MIN_CTAS 4
#endif

template <int R, bool COUNT, int VAR>
__global__ void __launch_bounds__(CTA, VF_MIN_CTAS) k_fused(const __grid_constant__ Params p, int phase)
{
    __shared__ Stage s_stage[WARPS_PER_CTA];
    __shared__ WarpState s_state[WARPS_PER_CTA];
    const int lane = threadIdx.x & 31;
    Stage &st = s_stage[threadIdx.x >> 5];
    pdl_wait();
    pdl_launch_dependents();      // the next frame's pre-pass may fill the SMs as this grid's CTAs retire (k_prepass)
    uint32_t *ctrl = p.ctrl;
    const uint32_t n_tiles = (uint32_t)p.n_tiles;
    const uint32_t n_cls = (n_tiles + CLS_CHUNK - 1) / CLS_CHUNK, n_scan = (n_tiles + SCAN_CHUNK - 1) / SCAN_CHUNK;
    uint32_t n_mark = 0;
    Counts c;
    if (COUNT) {
#pragma unroll
        for (int k = 0; k < CNT_N; ++k) c.n[k] = 0ull;
    }
    const uint32_t gw = blockIdx.x * WARPS_PER_CTA + (threadIdx.x >> 5), n_warps = gridDim.x * WARPS_PER_CTA;
    VF_T(0);
    // ---- producer roles: the classification (it feeds the geometry queue), then the shell marks.  The first classification
    //      chunk of a warp is its own number in the grid (no atomic: thousands of warps start at the same moment); every other
    //      chunk is claimed from a counter, so that no chunk ever waits for a warp that is busy with an item.
    if (phase != PHASE_COL) {
        const uint32_t njobs = min(__ldcg(&ctrl[Q_NJOBS]), p.jobs_cap);
        n_mark = (njobs + MARK_CHUNK - 1) / MARK_CHUNK;
        if (gw == 0 && lane == 0) ctrl[ST_NJOBS] = njobs;
        for (uint32_t k = gw; k < n_cls; k = n_cls <= n_warps ? n_cls : n_warps + claim(&ctrl[Q_CLS_CLAIM], lane)) {
            classify_chunk(p, k, lane);
            chunk_done(&ctrl[Q_CLS_DONE], lane);
        }
        VF_T(1);
        for (;;) {
            const uint32_t k = claim(&ctrl[Q_MARK_CLAIM], lane);
            if (k >= n_mark) break;
            mark_chunk<R>(p, k, njobs, lane);
            chunk_done(&ctrl[Q_MARK_DONE], lane);
        }
    }
    VF_T(2);
#ifdef VF_TRACE
    unsigned long long tr_ngeo = 0, tr_ncol = 0, tr_sleep = 0, tr_tgeo = 0, tr_tcol = 0, tr_tscan = 0, tr_ovg = 0, tr_ovc = 0, tr_top = 0;
#endif
    // ---- consumer: colour items once they exist (they are the longer ones), geometry items otherwise.
    // Every access to the queues is an L2 round trip of the order of a microsecond under load, so a round of the loop first
    // ISSUES whatever it may need (the progress counter it is watching, the slot of its geometry ticket) and only then looks at
    // the answers; colour tickets are drawn for several items at once (geometry tickets one by one: measured, balance is worth more).  The state of the loop lives in shared memory: the items need
    // every register, and what is kept in shared memory is not spilled to (cached, evictable) local memory around them.
    volatile WarpState &ws = s_state[threadIdx.x >> 5];
    if (lane == 0) {
        ws.flags = phase == PHASE_COL ? (F_GEO_DONE | F_MARKS_SET | F_SCAN_CLAIMED) : 0u;
        ws.gt = 0u; ws.gt_left = 0u; ws.ct = 0u; ws.ct_size = 1u; ws.cb_left = 0u; ws.cb_idx = 0u; ws.n_col = 0u; ws.n_staged = 0;
    }
    __syncwarp();
    for (;;) {
#ifdef VF_TRACE
        tr_top = clock64();
#endif
        uint32_t flags = ws.flags;
        // -- requests
        uint32_t v_poll = 0u, v_slot = 0u;
        const int watching = (flags & (F_COL_DONE | F_COL_READY)) ? 0 : (!(flags & F_MARKS_SET) ? 1 : ((flags & F_SCAN_CLAIMED) ? 2 : 0));
        if (watching == 1) v_poll = ld_relaxed(&ctrl[Q_MARK_DONE]);
        if (watching == 2) v_poll = ld_relaxed(&ctrl[Q_SCAN_DONE]);
        const bool geo_turn = !(flags & F_GEO_DONE);              // geometry tiles first: the colour list ends on short items
        uint32_t gt = ws.gt;
        if (geo_turn && ws.gt_left == 0u) {
            gt = claim_n(&ctrl[Q_GEO_CURSOR], GEO_BATCH, lane);
            __syncwarp();
            if (lane == 0) { ws.gt = gt; ws.gt_left = GEO_BATCH; }
        }
        if (geo_turn && gt < n_tiles) v_slot = ld_relaxed(p.work_geo + gt);
        // -- answers
        if (watching == 1 && v_poll >= n_mark) { flags |= F_MARKS_SET; VF_T(3); }
        if (watching == 2 && v_poll >= (phase == PHASE_COL ? 0u : n_scan)) {
            flags |= F_COL_READY;
            VF_T(5);
            const uint32_t nb = __ldcg(&ctrl[ST_NCOL]), nc = nb + __ldcg(&ctrl[ST_NCOL_SMALL]), t = claim_n(&ctrl[Q_COL_CURSOR], 1u, lane);
            __syncwarp();
            if (lane == 0) { ws.n_col = nc; ws.n_col_big = nb; ws.ct = t; ws.ct_size = 1u; }
        }
        if ((flags & (F_MARKS_SET | F_SCAN_CLAIMED)) == F_MARKS_SET) {
            const uint32_t k = claim(&ctrl[Q_SCAN_CLAIM], lane);
            if (k < n_scan) {
#ifdef VF_TRACE
                const unsigned long long t0 = clock64();
#endif
                scan_chunk<R>(p, k, lane);
                chunk_done(&ctrl[Q_SCAN_DONE], lane);
#ifdef VF_TRACE
                tr_tscan += clock64() - t0;
                VF_T(11);
#endif
            } else {
                flags |= F_SCAN_CLAIMED;
                VF_T(4);
                if (phase == PHASE_GEO) flags |= F_COL_DONE;          // the colour items are left to the next launch
            }
        }
        __syncwarp();
        if (lane == 0) ws.flags = flags;
        __syncwarp();
        if ((flags & (F_COL_READY | F_COL_DONE)) == F_COL_READY && !geo_turn) {
            // Colour items are taken in batches: one ticket and one load for up to COL_BATCH of them; single items towards
            // the end of the list, where balance matters.
            uint32_t cb_left = ws.cb_left;
            if (cb_left == 0u) {
                const uint32_t ct = ws.ct, n_col = ws.n_col;
                if (ct < n_col) {
                    cb_left = min(ws.ct_size, n_col - ct);
                    if ((uint32_t)lane < cb_left) {                 // the long items from the front of the list, then the short ones from its back
                        const uint32_t t = ct + (uint32_t)lane, nb = ws.n_col_big;
                        const uint2 it = __ldcg(p.work_col + (t < nb ? t : p.work_col_cap - 1u - (t - nb)));
                        ws.cb_item[lane][0] = it.x; ws.cb_item[lane][1] = it.y;
                    }
                    const uint32_t sz = n_col - ct > COL_BATCH_TAIL * n_warps ? COL_BATCH : 1u;
                    const uint32_t t = claim_n(&ctrl[Q_COL_CURSOR], sz, lane);
                    __syncwarp();
                    if (lane == 0) { ws.ct = t; ws.ct_size = sz; ws.cb_idx = 0u; ws.cb_left = cb_left; }
                } else {
                    if (lane == 0) ws.flags = flags | F_COL_DONE;
                    VF_T(6);
                }
                __syncwarp();
            }
            if (cb_left != 0u) {
                const uint32_t idx = ws.cb_idx;
                const uint2 item = make_uint2(ws.cb_item[idx][0], ws.cb_item[idx][1]);
                int n_staged = ws.n_staged;
                __syncwarp();
                if (lane == 0) { ws.cb_idx = idx + 1u; ws.cb_left = cb_left - 1u; }
#ifdef VF_TRACE
                const unsigned long long t0 = clock64();
                tr_ovc += t0 - tr_top;
#endif
                colour_item<R, COUNT, VAR>(p, item, st, n_staged, lane, c);
#ifdef VF_TRACE
                tr_ncol++; tr_tcol += clock64() - t0;
#endif
                __syncwarp();
                if (lane == 0) ws.n_staged = n_staged;
                __syncwarp();
            }
            continue;
        }
        if (geo_turn) {
            bool complete = (flags & F_CLS_COMPLETE) != 0u || gt >= n_tiles;
            if (v_slot == 0u && !complete) {                          // not published yet -- or beyond the end of the list?
                complete = ld_relaxed(&ctrl[Q_CLS_DONE]) >= n_cls;
                if (complete && gt < n_tiles) v_slot = ld_relaxed(p.work_geo + gt);
            }
            if (v_slot != 0u) {
                if (lane == 0) { p.work_geo[gt] = 0u; ws.gt = gt + 1u; ws.gt_left = ws.gt_left - 1u; }   // the list is all zero again when the frame is done
                geometry_prefetch(p, v_slot, lane);
#ifdef VF_TRACE
                const unsigned long long t0 = clock64();
                tr_ovg += t0 - tr_top;
#endif
                geometry_tile<COUNT, VAR>(p, v_slot, lane, c);
#ifdef VF_TRACE
                tr_ngeo++; tr_tgeo += clock64() - t0;
#endif
                __syncwarp();
                continue;
            }
            if (complete) {                                           // every item below the final count has been taken
                flags |= F_CLS_COMPLETE | F_GEO_DONE;
                __syncwarp();
                if (lane == 0) ws.flags = flags;
                __syncwarp();
            }
        }
        if ((flags & (F_GEO_DONE | F_COL_DONE)) == (F_GEO_DONE | F_COL_DONE)) break;
        if (watching == 0 && !geo_turn) continue;
        if (flags & F_GEO_DONE || v_slot == 0u) {
            __nanosleep(1000);                                        // waiting for claimed producer chunks to finish (a round costs ~100 instructions)
#ifdef VF_TRACE
            tr_sleep++;
#endif
        }
    }
    int n_staged = ws.n_staged;
    VF_T(8);
    VF_TC(9, tr_ngeo); VF_TC(10, tr_ncol); VF_TC(12, tr_tgeo); VF_TC(13, tr_tcol); VF_TC(14, tr_tscan); VF_TC(15, tr_ovg); VF_TC(7, tr_ovc);
    if (n_staged > 0) colour_update_staged<COUNT, VAR>(p, st, 0, n_staged, lane, c);
    if (COUNT) {
#pragma unroll
        for (int k = 0; k < CNT_N; ++k) {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) c.n[k] += __shfl_xor_sync(0xffffffffu, c.n[k], o);
            if (lane == 0 && c.n[k]) atomicAdd(&p.counters[k], c.n[k]);
        }
    }
}

}  // namespace vf
