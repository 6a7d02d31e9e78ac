// fused.cuh -- K2: the fused integration kernel (S2-S8), warp-centric and persistent.
//
// Every warp pops work items from one queue until it is empty -- first the colour items (one non-zero shell-mark
// nibble = up to 4 colour cells of 8x4x4 voxels of one tile), then the geometry items (one tile of 32x4x8 TSDF voxels, marched
// along z with per-column bases hoisted).  A lane always owns one 16-byte vector of 4 x-adjacent voxels, so a warp
// reads whole 32-byte sectors (colour gate) or 128-byte lines (geometry rows).  Colour voxels that pass the gate are
// compacted in a per-warp shared-memory stage and updated one per lane.  No block-level barriers.
//
// The per-voxel arithmetic is the canonical sequence of DESIGN.md, issued branch-free for 4 voxels at a time
// (projection -> gathers -> update); operands outside the range of the branch-free exact reciprocal (exact.cuh) send
// the whole warp through the plain reference routines below, which use the library intrinsics.
#pragma once
#include "exact.cuh"
#include "params.cuh"

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
// Precondition (established per tile by k_mark_classify / k_items_col, bit ITEM_NEAR clear): RCP_MIN <= Z <= RCP_MAX.
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

struct Counts { unsigned long long gr, gc, cr, cc; };

// one geometry tile, one warp: lane = (vx = lane & 7, y = lane >> 3) owns voxels (gx0 + 4 vx .. + 3, gy0 + y) of every layer.
// NEAR tiles (may hold voxels with Z <= 0 or outside rcp_exact's range) take the plain per-voxel routine.
// Otherwise the layers are software-pipelined: while layer z is updated, layer z + 1 has already been projected and its
// four depth gathers and its voxel vector are in flight.
template <bool COUNT, int VAR>
__device__ __forceinline__ void geometry_tile(const Params &p, uint32_t item, int lane, Counts &c)
{
    const bool near = (item & ITEM_NEAR) != 0u;
    int ttx, tty, ttz, sub;
    item_unpack(item, ttx, tty, ttz, sub);
    const int i0 = ttx * TX + 4 * (lane & 7), j = tty * TY + (lane >> 3);
    // the classification tested the tile's two z-halves separately (bits 0 and 1 of sub): a half that failed holds no
    // voxel this frame can update, and its four layers are left out -- the march starts at layer zb and covers nl layers
    const int zb = (near || (sub & 1)) ? 0 : TZ / 2;
    const int gz0 = local_to_global_tz(p, ttz) * TZ + zb, lz0 = ttz * TZ + zb;
    const bool inside = i0 < p.nx && j < p.ny;
    const unsigned lanes = __ballot_sync(0xffffffffu, inside);    // ragged tile: the votes below name only these lanes
    if (!inside) return;
    const int nl = min((near || (sub & 2)) ? TZ - zb : TZ / 2, p.nz - gz0);
    // per-column bases of eq. 5: fma(R_1, py, fma(R_0, px, t)) -- the z term is added per layer with one fma each
    const float py = __fmaf_rn((float)j + 0.5f, p.vs, p.oy);
    float bX[4], bY[4], bZ[4];
#pragma unroll
    for (int e = 0; e < 4; ++e) {
        const float px = __fmaf_rn((float)(i0 + e) + 0.5f, p.vs, p.ox);
        bX[e] = __fmaf_rn(p.R[1], py, __fmaf_rn(p.R[0], px, p.t[0]));
        bY[e] = __fmaf_rn(p.R[4], py, __fmaf_rn(p.R[3], px, p.t[1]));
        bZ[e] = __fmaf_rn(p.R[7], py, __fmaf_rn(p.R[6], px, p.t[2]));
    }
    const float r02 = p.R[2], r12 = p.R[5], r22 = p.R[8];
    const size_t layer = (size_t)p.ny * p.nx;
    uint4 *ptr = reinterpret_cast<uint4 *>(p.geo + ((size_t)lz0 * p.ny + j) * p.nx + i0);
    if (near) {
        for (int z = 0; z < nl; ++z) {
            const uint4 cur = *ptr;
            const float pz = __fmaf_rn((float)(gz0 + z) + 0.5f, p.vs, p.oz);
            const uint32_t o4[4] = {cur.x, cur.y, cur.z, cur.w};
            uint32_t w4[4];
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                bool rd = false;
                w4[e] = geo_voxel_ref(p, __fmaf_rn(r02, pz, bX[e]), __fmaf_rn(r12, pz, bY[e]), __fmaf_rn(r22, pz, bZ[e]), o4[e], rd);
                if (COUNT) { c.gr += rd; c.gc += w4[e] != o4[e]; }
            }
            if ((w4[0] != o4[0]) | (w4[1] != o4[1]) | (w4[2] != o4[2]) | (w4[3] != o4[3])) *ptr = make_uint4(w4[0], w4[1], w4[2], w4[3]);
            ptr = reinterpret_cast<uint4 *>(reinterpret_cast<uint32_t *>(ptr) + layer);
        }
        return;
    }
    const float fx = p.fx, fy = p.fy, cx = p.cx, cy = p.cy;
    const float neg_mu = p.neg_mu, inv_mu = p.inv_mu;
    const uint32_t wd = (uint32_t)p.wd, wbits = __float_as_uint(p.wd_f), hbits = __float_as_uint(p.hd_f), koff = 0x4B400000u * (wd + 1u);
    const int w_max = p.w_max;
    const uint16_t *__restrict__ depth = p.depth;
    // S2 of one layer: eq. 5 z term, projection, and the four depth gathers (offset 0 when outside: a valid address)
    // A voxel outside the frustum keeps d = 0 ("invalid depth": not updated); its gather is predicated off.  The address is
    // one mad.wide (FMA pipe) instead of a 64-bit add pair: the ALU pipe is the busiest one in this loop.
    // (VAR_TSDF_ALONG_RAY only: L = |P_vc| / Z_vc, the factor from the distance along z to the distance along the ray)
    auto project_layer = [&](int z, float (&Z)[4], uint32_t (&d)[4], float (&L)[4]) {
        const float pz = __fmaf_rn((float)(gz0 + z) + 0.5f, p.vs, p.oz);
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const float X = __fmaf_rn(r02, pz, bX[e]), Y = __fmaf_rn(r12, pz, bY[e]);
            Z[e] = __fmaf_rn(r22, pz, bZ[e]);
            bool ok; uint32_t off; float iz;
            project_fast_raw(fx, fy, cx, cy, wd, wbits, hbits, koff, X, Y, Z[e], ok, off, iz);
            if (VAR == VAR_TSDF_ALONG_RAY)
                L[e] = __fmul_rn(__fsqrt_rn(__fmaf_rn(Z[e], Z[e], __fmaf_rn(Y, Y, __fmul_rn(X, X)))), iz);
            d[e] = 0u;
            if (ok) {
                unsigned long long addr;
                asm("mad.wide.u32 %0, %1, 2, %2;" : "=l"(addr) : "r"(off), "l"(depth));
                d[e] = __ldg(reinterpret_cast<const uint16_t *>(addr));
            }
        }
    };
    // S3 of one layer: truncation test, running average, store if a word changed
    auto update_layer = [&](uint4 *ptr, const uint4 &cur, const float (&Z)[4], const uint32_t (&d)[4], const float (&L)[4]) {
        const uint32_t o4[4] = {cur.x, cur.y, cur.z, cur.w};
        uint32_t w4[4];
        float sdf[4]; bool upd[4];
        bool easy = true;
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const float D = __fmul_rn((float)d[e], 0.001f);
            sdf[e] = __fsub_rn(D, Z[e]);
            if (VAR == VAR_TSDF_ALONG_RAY) sdf[e] = __fmul_rn(sdf[e], L[e]);
            upd[e] = (d[e] != 0u) & !(sdf[e] < neg_mu);
            // saturated free space (tsdf = 1 onto q = 32767) or first touch (w = 0): the running average is 32767 exactly,
            // fma(32767, w, 32767) / (w + 1) with every intermediate below 2^24.  (Bitwise on purpose: no branches.)
            easy = easy & (!upd[e] | ((__fmul_rn(sdf[e], inv_mu) >= 1.0f) & (((o4[e] & 0xffffu) == 0x7fffu) | (o4[e] < 0x10000u))));
            if (COUNT) c.gr += upd[e];
        }
        if (__all_sync(lanes, easy)) {                            // whole warp in free space: no division needed
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const int wn = min((int)(short)(o4[e] >> 16) + 1, w_max);
                w4[e] = upd[e] ? (0x7fffu | ((uint32_t)wn << 16)) : o4[e];
            }
        } else {
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const float tsdf = fminf(1.0f, __fmul_rn(sdf[e], inv_mu));
                const int q = (int)(short)(o4[e] & 0xffffu);
                const int wi = (int)(short)(o4[e] >> 16);
                const float wf = (float)wi;
                // num is 0 or 2^-40 <= |num| < 2^26 (vol_create bounds mu), den in [1, 513]
                const float num = __fmaf_rn((float)q, wf, __fmul_rn(tsdf, 32767.0f));
                const float den = __fadd_rn(wf, 1.0f);
                // rint (half-even) without the conversion pipe: |quotient| <= 32767, so adding 1.5 * 2^23 leaves it in the
                // low mantissa bits, already in two's complement
                const uint32_t qn = __float_as_uint(__fadd_rn(div_with(num, den, div_prepare(den)), 12582912.0f));
                const int wn = min(wi + 1, w_max);
                const uint32_t nw = (qn & 0xffffu) | ((uint32_t)wn << 16);
                w4[e] = upd[e] ? nw : o4[e];
            }
        }
        const bool any = (w4[0] != o4[0]) | (w4[1] != o4[1]) | (w4[2] != o4[2]) | (w4[3] != o4[3]);
        if (COUNT) c.gc += (w4[0] != o4[0]) + (w4[1] != o4[1]) + (w4[2] != o4[2]) + (w4[3] != o4[3]);
        if (any) *ptr = make_uint4(w4[0], w4[1], w4[2], w4[3]);   // skip the store when nothing changed
    };
    // Two register sets, A (even layers) and B (odd layers), used alternately: the pipeline needs no register-to-register
    // rotation, which would make the warp wait for the loads it has just issued.
    float ZA[4], ZB[4], LA[4], LB[4]; uint32_t dA[4], dB[4];
    // the voxel stream bypasses L1 (__ldcg): every line is used once, and L1 is better spent on the depth image
    uint4 curA = __ldcg(ptr), curB = curA;
    project_layer(0, ZA, dA, LA);
    for (int z = 0; z < nl; z += 2) {
        uint4 *pB = reinterpret_cast<uint4 *>(reinterpret_cast<uint32_t *>(ptr) + layer);
        uint4 *pA2 = reinterpret_cast<uint4 *>(reinterpret_cast<uint32_t *>(pB) + layer);
        const bool hasB = z + 1 < nl, hasA2 = z + 2 < nl;
        if (hasB) { curB = __ldcg(pB); project_layer(z + 1, ZB, dB, LB); }               // layer z + 1 in flight
        update_layer(ptr, curA, ZA, dA, LA);
        if (hasB) {
            if (hasA2) { curA = __ldcg(pA2); project_layer(z + 2, ZA, dA, LA); }         // layer z + 2 in flight
            update_layer(pB, curB, ZB, dB, LB);
        }
        ptr = pA2;
    }
}

// pull the 32 lines (8 layers x 4 rows x 128 bytes) of a geometry tile into L2: one line per lane, no register is tied up.
// Issued when the tile is started: its later layers are then L2 hits by the time the layer pipeline reaches them.
__device__ __forceinline__ void geometry_prefetch(const Params &p, uint32_t item, int lane)
{
    int ttx, tty, ttz, sub;
    item_unpack(item, ttx, tty, ttz, sub);
    const int j = tty * TY + (lane & 3), lz = ttz * TZ + (lane >> 2);
    const bool wanted = (item & ITEM_NEAR) != 0u || ((sub >> ((lane >> 2) / (TZ / 2))) & 1) != 0;   // its z-half is processed
    if (j < p.ny && lz < p.local_nz && wanted)
        asm volatile("prefetch.global.L2 [%0];" ::"l"(p.geo + ((size_t)lz * p.ny + j) * p.nx + ttx * TX));
}

// Per-warp staging buffer of colour voxels that passed the sigma gate.  The gate (S4-S5) runs on whole cells, 4 voxels
// per lane, and only a fraction of them passes; the update (S6-S8: weight gate, HD lookup, eq. 9-10) is several times
// longer.  Passing voxels are therefore compacted here and updated 32 at a time with every lane busy.
constexpr int STAGE_CAP = 160;            // up to 31 carried over + 128 of one cell
struct Stage {
    float4 rec[STAGE_CAP];                // {X, Y, Z} = voxel centre in the depth camera (eq. 5) -- or, VAR_HD_FROM_DEPTH_POINT, the
                                          // 3D point of its depth pixel (eq. 7); W = view weight of its pixel
    uint2  adr[STAGE_CAP];                // word index of the voxel in this shard's colour volume (lo, hi)
};

// S6-S8 (weight gate L115, HD pixel eq. 3-4, eq. 9, eq. 10) for up to 32 staged voxels [first, first + n): one voxel per
// lane.  The HD pixel (eq. 3-4) is computed and its three bytes requested BEFORE the stored word arrives: the two gathers do
// not depend on each other, so their latencies overlap instead of adding up (the word is a DRAM access, and one warp
// works through its stage round after round).  A voxel that then fails the weight gate has fetched 3 bytes in vain.
template <bool COUNT, int VAR>
__device__ __forceinline__ void colour_update_staged(const Params &p, const Stage &st, int first, int n, int lane, Counts &c)
{
    if (lane < n) {
        const float4 r = st.rec[first + lane];
        const uint2 a = st.adr[first + lane];
        uint32_t *ptr = p.col + (((size_t)a.y << 32) | (size_t)a.x);
        const uint32_t old = __ldcg(ptr);                         // first HBM touch of this colour voxel (S6); L2 only
        // HD pixel of the voxel's own position (eq. 3-4; A10, A11)
        const float Xh = __fmaf_rn(p.Rc[2], r.z, __fmaf_rn(p.Rc[1], r.y, __fmaf_rn(p.Rc[0], r.x, p.tc[0])));
        const float Yh = __fmaf_rn(p.Rc[5], r.z, __fmaf_rn(p.Rc[4], r.y, __fmaf_rn(p.Rc[3], r.x, p.tc[1])));
        const float Zh = __fmaf_rn(p.Rc[8], r.z, __fmaf_rn(p.Rc[7], r.y, __fmaf_rn(p.Rc[6], r.x, p.tc[2])));
        int xh = 0, yh = 0;
        const bool okh = project_px(p.fxh, p.fyh, p.cxh, p.cyh, p.wh_f, p.hh_f, Xh, Yh, Zh, xh, yh);   // A13
        const uint8_t *hd = p.rgb + (size_t)(yh * p.wh + xh) * 3;     // A14: nearest pixel ((0, 0) when outside: a valid address)
        const uint32_t h0 = __ldg(hd), h1 = __ldg(hd + 1), h2 = __ldg(hd + 2);
        const int wq = (int)(old >> 24);
        const float W = r.w, W255 = __fmul_rn(W, 255.0f);
        uint32_t nw = old;
        if (okh && W255 > __fmul_rn(p.gate, (float)wq)) {         // L115, A9
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
        if (COUNT) { c.cr += 1; c.cc += nw != old; }
    }
}

// one colour cell of 8 x 4 x 4 voxels, one warp: lane = (vx = lane & 1, y = (lane >> 1) & 3, z = lane >> 3) owns 4
// x-adjacent voxels.  (ic0, jc, kcg) = the lane's first voxel in the full colour grid, kcl = its layer in this shard.
// Voxels that pass the gate are appended to the warp's stage (n = its fill level, warp-uniform); full groups of 32 are
// updated at once.
template <bool COUNT, int VAR>
__device__ __forceinline__ void colour_cell(const Params &p, bool near, int ic0, int jc, int kcg, int kcl, Stage &st, int &n, int lane, Counts &c)
{
    const float fx = p.fx, fy = p.fy, cx_ = p.cx, cy_ = p.cy, sig2 = p.sig2;
    const uint32_t wd = (uint32_t)p.wd, wbits = __float_as_uint(p.wd_f), hbits = __float_as_uint(p.hd_f), koff = 0x4B400000u * (wd + 1u);
    const float4 *__restrict__ pixmap = p.pixmap;
    const bool act = ic0 < p.cnx && jc < p.cny && kcg < p.cnz;
    const float py = __fmaf_rn((float)jc + 0.5f, p.vc, p.oy);
    const float pz = __fmaf_rn((float)kcg + 0.5f, p.vc, p.oz);
    float X[4], Y[4], Z[4], W[4];
#pragma unroll
    for (int e = 0; e < 4; ++e) {                                     // S4: eq. 5
        const float px = __fmaf_rn((float)(ic0 + e) + 0.5f, p.vc, p.ox);
        X[e] = __fmaf_rn(p.R[2], pz, __fmaf_rn(p.R[1], py, __fmaf_rn(p.R[0], px, p.t[0])));
        Y[e] = __fmaf_rn(p.R[5], pz, __fmaf_rn(p.R[4], py, __fmaf_rn(p.R[3], px, p.t[1])));
        Z[e] = __fmaf_rn(p.R[8], pz, __fmaf_rn(p.R[7], py, __fmaf_rn(p.R[6], px, p.t[2])));
    }
    unsigned pass = 0;
    float4 pm[4];
    if (near) {
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            pm[e] = act ? col_voxel_gate_ref(p, X[e], Y[e], Z[e]) : make_float4(0.0f, 0.0f, 0.0f, 0.0f);
            W[e] = pm[e].w;
            if (W[e] > 0.0f) pass |= 1u << e;
        }
    } else {
        uint32_t off[4]; bool ok[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) project_fast(fx, fy, cx_, cy_, wd, wbits, hbits, koff, X[e], Y[e], Z[e], ok[e], off[e]);   // eq. 6
#pragma unroll
        for (int e = 0; e < 4; ++e) pm[e] = __ldg(pixmap + off[e]);      // eq. 7-8 and W per pixel (S1)
#pragma unroll
        for (int e = 0; e < 4; ++e) {                                 // S5: sigma gate (L108)
            const float dx = __fsub_rn(X[e], pm[e].x), dy = __fsub_rn(Y[e], pm[e].y), dz = __fsub_rn(Z[e], pm[e].z);
            const float d2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
            const bool in = act && ok[e] && (pm[e].w > 0.0f) && !(d2 > sig2);
            W[e] = pm[e].w;
            if (in) pass |= 1u << e;
        }
    }
    // compact: exclusive prefix of the per-lane counts
    const int cnt = __popc(pass);
    int pre = cnt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const int v = __shfl_up_sync(0xffffffffu, pre, o); if (lane >= o) pre += v; }
    const int total = __shfl_sync(0xffffffffu, pre, 31);
    if (total == 0) return;
    int slot = n + pre - cnt;
    const size_t base = ((size_t)kcl * (size_t)p.cny + (size_t)jc) * (size_t)p.cnx + (size_t)ic0;
    // start the DRAM access of the stored words now; the update reads them a few hundred cycles later
    if (pass) asm volatile("prefetch.global.L2 [%0];" ::"l"(p.col + base));
#pragma unroll
    for (int e = 0; e < 4; ++e)
        if (pass & (1u << e)) {
            st.rec[slot] = VAR == VAR_HD_FROM_DEPTH_POINT ? make_float4(pm[e].x, pm[e].y, pm[e].z, W[e]) : make_float4(X[e], Y[e], Z[e], W[e]);
            const size_t a = base + (size_t)e;
            st.adr[slot] = make_uint2((uint32_t)a, (uint32_t)(a >> 32));
            ++slot;
        }
    n += total;
    __syncwarp();
    while (n >= 32) { n -= 32; colour_update_staged<COUNT, VAR>(p, st, n, 32, lane, c); }
    __syncwarp();
}

// one colour work item, one warp: the set bits of one nibble of a shell-mark word are up to 4 colour cells of one tile.
// The ticket of the next item is drawn before the LAST cell: its latency is hidden, yet no item waits reserved behind a
// long one.
template <int R, bool COUNT, int VAR>
__device__ __forceinline__ void colour_item(const Params &p, uint32_t item, Stage &st, int &n, int lane, Counts &c, uint32_t *cursor, uint32_t &ticket)
{
    const bool near = (item & ITEM_NEAR) != 0u;
    constexpr int CX = cells_x(R), CY = cells_y(R), WPT = words_per_tile(R);
    int ttx, tty, ttz, sub;
    item_unpack(item, ttx, tty, ttz, sub);
    const int word = sub >> 3;
    const uint32_t wi = (uint32_t)((ttz * p.tiles_y + tty) * p.tiles_x + ttx) * WPT + (uint32_t)word, sh = 4u * ((uint32_t)sub & 7u);
    uint32_t bits = 0;
    if (lane == 0) {                                                      // consume this item's nibble of the marks (self-cleaning)
        bits = __ldcg(p.marks + wi) & (0xfu << sh);
        atomicAnd(p.marks + wi, ~(0xfu << sh));
    }
    bits = __shfl_sync(0xffffffffu, bits, 0);
    const int cgx0 = ttx * TX * R, cgy0 = tty * TY * R;
    const int cgz0 = local_to_global_tz(p, ttz) * TZ * R, clz0 = ttz * TZ * R;
    if (COUNT && lane == 0) atomicAdd(&p.ctrl[CTRL_CELLS], (uint32_t)__popc(bits));
    if (bits == 0u) next_ticket(cursor, lane, ticket);
    while (bits) {
        const int b = word * 32 + (__ffs(bits) - 1);
        bits &= bits - 1;
        if (bits == 0u) next_ticket(cursor, lane, ticket);
        const int cx = b % CX, cy = (b / CX) % CY, cz = b / (CX * CY);
        const int kz = cz * CLZ + (lane >> 3);
        colour_cell<COUNT, VAR>(p, near, cgx0 + cx * CLX + 4 * (lane & 1), cgy0 + cy * CLY + ((lane >> 1) & 3), cgz0 + kz, clz0 + kz, st, n, lane, c);
    }
}

// phase: PHASE_ALL = the whole queue in one launch (frames already on the device); PHASE_GEO / PHASE_COL = the geometry
// items / the colour items only, so that vol_integrate_host can run the geometry half while the HD frame is still being
// copied (only the colour update reads it).
enum { PHASE_ALL = 0, PHASE_GEO = 1, PHASE_COL = 2 };

template <int R, bool COUNT, int VAR>
__global__ void __launch_bounds__(CTA, 4) k_fused(const __grid_constant__ Params p, int phase)
{
    __shared__ Stage s_stage[WARPS_PER_CTA];
    const int lane = threadIdx.x & 31;
    Stage &st = s_stage[threadIdx.x >> 5];
    pdl_wait();
    // queue order, longest kind first: NEAR geometry tiles, colour items, ordinary geometry tiles (the shortest: the tail)
    const uint32_t c_near = __ldcg(&p.ctrl[CTRL_NNEAR]), c_col = __ldcg(&p.ctrl[CTRL_NCOL]), c_geo = __ldcg(&p.ctrl[CTRL_NGEO]);
    const uint32_t n_near = phase == PHASE_COL ? 0u : c_near;
    const uint32_t n_col = n_near + (phase == PHASE_GEO ? 0u : c_col);
    const uint32_t n_items = n_col + (phase == PHASE_COL ? 0u : c_geo);
    uint32_t *cursor = &p.ctrl[phase == PHASE_COL ? CTRL_CURSOR2 : CTRL_CURSOR];
    Counts c = {0, 0, 0, 0};
    int n_staged = 0;
    // the ticket of the next item is requested before the current one is processed (the L2 round trip is hidden).
    // Only one item is reserved ahead: colour items are long, and a deeper reservation unbalances the tail.
    uint32_t ticket = 0;
    next_ticket(cursor, lane, ticket);
    for (;;) {
        const uint32_t it = __shfl_sync(0xffffffffu, ticket, 0);
        if (it >= n_items) break;
        const uint32_t item = it < n_near ? __ldcg(p.work_geo + ((uint32_t)p.n_tiles - 1u - it))
                                          : (it < n_col ? __ldcg(p.work_col + (it - n_near)) : __ldcg(p.work_geo + (it - n_col)));
        if (it >= n_near && it < n_col) colour_item<R, COUNT, VAR>(p, item, st, n_staged, lane, c, cursor, ticket);
        else {
            next_ticket(cursor, lane, ticket);
            geometry_prefetch(p, item, lane);
            geometry_tile<COUNT, VAR>(p, item, lane, c);
        }
    }
    if (n_staged > 0) colour_update_staged<COUNT, VAR>(p, st, 0, n_staged, lane, c);
    if (COUNT) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            c.gr += __shfl_xor_sync(0xffffffffu, c.gr, o); c.gc += __shfl_xor_sync(0xffffffffu, c.gc, o);
            c.cr += __shfl_xor_sync(0xffffffffu, c.cr, o); c.cc += __shfl_xor_sync(0xffffffffu, c.cc, o);
        }
        if (lane == 0) {
            if (c.gr) atomicAdd(&p.counters[0], c.gr);
            if (c.gc) atomicAdd(&p.counters[1], c.gc);
            if (c.cr) atomicAdd(&p.counters[2], c.cr);
            if (c.cc) atomicAdd(&p.counters[3], c.cc);
        }
    }
}

}  // namespace vf
