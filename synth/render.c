/*
 * synth/render.c -- analytic ray caster for the seeded synthetic RGB-D frames.
 *
 * HARNESS CODE.  This file holds none of the method's arithmetic (no TSDF, no
 * colour update, no voxel projection): it only renders the *inputs* -- a
 * z-depth image and an RGB8 image of a small analytic scene seen by a pinhole
 * camera -- which are then fed, byte for byte, to both the CPU oracle
 * (oracle/) and the CUDA path (paper_1602_06645_b200/).  The scenes stand in
 * for the paper's handheld Kinect + HD-camera scans, which
 * are not available; recipe in DESIGN.md "Synthetic inputs".
 *
 * Camera convention: x right, y down, z forward; pixel (x,y) <-> ray
 * ((x-cx)/fx, (y-cy)/fy, 1); pixel centres at integer coordinates.
 * Depth = z-depth (camera-frame z of the nearest hit), 0 for a miss.
 *
 * Build: gcc -O2 -fopenmp -ffp-contract=off -shared -fPIC render.c -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

enum { PRIM_SPHERE = 0, PRIM_BOX = 1, PRIM_PLANE = 2, PRIM_CYLINDER = 3, PRIM_TORUS = 4 };
enum { TEX_CONST = 0, TEX_CHECKER = 1, TEX_NOISE = 2, TEX_STRIPES = 3 };

/* One primitive = 16 doubles:
 *  [0] type  [1] texture  [2] seed
 *  [3..5] centre c
 *  [6..8] size: sphere (R,-,-); box half sizes (hx,hy,hz); plane normal n (unit,
 *         the plane is n.(p-c)=0); cylinder (R, half height, -) axis = world z;
 *         torus (R major, r minor, -) axis = world z
 *  [9] texture scale (checker: cells per radian / per metre; noise: base
 *      frequency 1/m; stripes: period in metres)
 *  [10..12] base colour (0..255)  [13..15] spare
 */
#define PRIM_STRIDE 16

static uint32_t mix32(uint32_t x)
{
    x ^= x >> 16; x *= 0x7feb352dU;
    x ^= x >> 15; x *= 0x846ca68bU;
    x ^= x >> 16;
    return x;
}
static uint32_t hash3(uint32_t seed, int32_t a, int32_t b, int32_t c)
{
    uint32_t h = mix32(seed ^ 0x9e3779b9U);
    h = mix32(h ^ (uint32_t)a);
    h = mix32(h ^ ((uint32_t)b * 0x85ebca6bU));
    h = mix32(h ^ ((uint32_t)c * 0xc2b2ae35U));
    return h;
}

/* gradient noise on the integer lattice, value in about [-1,1] */
static double grad_dot(uint32_t h, double x, double y, double z)
{
    static const double g[12][3] = {
        {1,1,0},{-1,1,0},{1,-1,0},{-1,-1,0},{1,0,1},{-1,0,1},
        {1,0,-1},{-1,0,-1},{0,1,1},{0,-1,1},{0,1,-1},{0,-1,-1}};
    const double *v = g[h % 12U];
    return v[0] * x + v[1] * y + v[2] * z;
}
static double fade(double t) { return t * t * t * (t * (t * 6.0 - 15.0) + 10.0); }
static double gnoise(uint32_t seed, double x, double y, double z)
{
    double fx = floor(x), fy = floor(y), fz = floor(z);
    int32_t ix = (int32_t)fx, iy = (int32_t)fy, iz = (int32_t)fz;
    double tx = x - fx, ty = y - fy, tz = z - fz;
    double u = fade(tx), v = fade(ty), w = fade(tz);
    double c[2][2][2];
    for (int a = 0; a < 2; ++a)
        for (int b = 0; b < 2; ++b)
            for (int d = 0; d < 2; ++d)
                c[a][b][d] = grad_dot(hash3(seed, ix + a, iy + b, iz + d), tx - a, ty - b, tz - d);
    double x00 = c[0][0][0] + u * (c[1][0][0] - c[0][0][0]);
    double x10 = c[0][1][0] + u * (c[1][1][0] - c[0][1][0]);
    double x01 = c[0][0][1] + u * (c[1][0][1] - c[0][0][1]);
    double x11 = c[0][1][1] + u * (c[1][1][1] - c[0][1][1]);
    double y0 = x00 + v * (x10 - x00), y1 = x01 + v * (x11 - x01);
    return y0 + w * (y1 - y0);
}

static double clamp255(double v) { return v < 0.0 ? 0.0 : (v > 255.0 ? 255.0 : v); }

/* which "face" of a primitive the (object-space) hit point q with normal n lies on */
static int face_id(int type, const double q[3], const double n[3])
{
    if (type == PRIM_BOX || type == PRIM_PLANE) {
        double ax = fabs(n[0]), ay = fabs(n[1]), az = fabs(n[2]);
        if (ax >= ay && ax >= az) return n[0] > 0 ? 0 : 1;
        if (ay >= az) return n[1] > 0 ? 2 : 3;
        return n[2] > 0 ? 4 : 5;
    }
    /* curved: 8 longitude patches x 4 latitude bands */
    double lon = atan2(q[1], q[0]), len = sqrt(q[0]*q[0] + q[1]*q[1] + q[2]*q[2]);
    double lat = len > 0 ? asin(q[2] / len) : 0.0;
    int a = (int)floor((lon + M_PI) / (2.0 * M_PI) * 8.0); if (a > 7) a = 7; if (a < 0) a = 0;
    int b = (int)floor((lat + M_PI / 2) / M_PI * 4.0);      if (b > 3) b = 3; if (b < 0) b = 0;
    return 8 + b * 8 + a;
}

static void shade(const double *pr, const double p[3], const double n[3], uint8_t out[3])
{
    int type = (int)pr[0], tex = (int)pr[1];
    uint32_t seed = (uint32_t)pr[2];
    double q[3] = { p[0] - pr[3], p[1] - pr[4], p[2] - pr[5] };
    double scale = pr[9];
    double col[3] = { pr[10], pr[11], pr[12] };
    if (tex == TEX_CHECKER) {
        int32_t a, b, f = 0;
        if (type == PRIM_SPHERE) {
            double len = sqrt(q[0]*q[0] + q[1]*q[1] + q[2]*q[2]);
            double lat = asin(q[1] / len), lon = atan2(q[0], -q[2]); /* pole along camera-frame y */
            a = (int32_t)floor(lat * scale); b = (int32_t)floor(lon * scale);
        } else {
            f = face_id(type, q, n);
            double uu = (f < 2) ? q[1] : q[0], vv = (f < 4) ? q[2] : q[1];
            a = (int32_t)floor(uu * scale); b = (int32_t)floor(vv * scale);
        }
        uint32_t h = hash3(seed, a, b, f);
        col[0] = 32 + (h & 0xff) * 223.0 / 255.0;
        col[1] = 32 + ((h >> 8) & 0xff) * 223.0 / 255.0;
        col[2] = 32 + ((h >> 16) & 0xff) * 223.0 / 255.0;
    } else if (tex == TEX_NOISE) {
        for (int ch = 0; ch < 3; ++ch) {
            double s = 0.0, amp = 1.0, fr = scale;
            for (int o = 0; o < 3; ++o) {
                s += amp * gnoise(seed + 101U * (uint32_t)ch + 7U * (uint32_t)o, p[0] * fr, p[1] * fr, p[2] * fr);
                amp *= 0.5; fr *= 2.0;
            }
            col[ch] = clamp255(pr[10 + ch] + 110.0 * s);
        }
    } else if (tex == TEX_STRIPES) {
        int f = face_id(type, q, n);
        uint32_t h = hash3(seed, f, 17, 3);
        /* stripe direction in the face's tangent plane, hashed per face */
        double ang = (h & 0xffff) / 65536.0 * M_PI;
        double t1[3], t2[3];
        if (fabs(n[0]) < 0.9) { t1[0] = 0; t1[1] = -n[2]; t1[2] = n[1]; }
        else                  { t1[0] = -n[2]; t1[1] = 0; t1[2] = n[0]; }
        double l = sqrt(t1[0]*t1[0] + t1[1]*t1[1] + t1[2]*t1[2]);
        t1[0] /= l; t1[1] /= l; t1[2] /= l;
        t2[0] = n[1]*t1[2] - n[2]*t1[1]; t2[1] = n[2]*t1[0] - n[0]*t1[2]; t2[2] = n[0]*t1[1] - n[1]*t1[0];
        double s = cos(ang) * (q[0]*t1[0] + q[1]*t1[1] + q[2]*t1[2]) + sin(ang) * (q[0]*t2[0] + q[1]*t2[1] + q[2]*t2[2]);
        double period = scale * (1.0 + ((h >> 16) & 0xff) / 255.0);   /* scale .. 2*scale */
        int32_t k = (int32_t)floor(s / period);
        /* text-like: stripes are broken into hashed "glyph" runs along the other direction */
        double s2 = -sin(ang) * (q[0]*t1[0] + q[1]*t1[1] + q[2]*t1[2]) + cos(ang) * (q[0]*t2[0] + q[1]*t2[1] + q[2]*t2[2]);
        int32_t g = (int32_t)floor(s2 / (6.0 * period));
        uint32_t hk = hash3(seed, k, g, f);
        int on = (k & 1) && ((hk & 7U) != 0U);
        uint32_t hc = hash3(seed, f, 5, 9);
        if (on) { col[0] = 20 + (hc & 0x3f); col[1] = 20 + ((hc >> 6) & 0x3f); col[2] = 20 + ((hc >> 12) & 0x3f); }
        else    { col[0] = 190 + ((hc >> 18) & 0x3f); col[1] = 190 + ((hc >> 24) & 0x3f); col[2] = 190 + ((hc >> 3) & 0x3f); }
    }
    for (int ch = 0; ch < 3; ++ch) out[ch] = (uint8_t)floor(clamp255(col[ch]) + 0.5);
}

/* nearest positive hit of ray o + t*d with primitive pr; returns t (<0: none), normal in n */
static double hit(const double *pr, const double o[3], const double d[3], double n[3])
{
    int type = (int)pr[0];
    double oc[3] = { o[0] - pr[3], o[1] - pr[4], o[2] - pr[5] };
    const double tmin = 1e-6;
    if (type == PRIM_SPHERE) {
        double R = pr[6];
        double a = d[0]*d[0] + d[1]*d[1] + d[2]*d[2];
        double b = oc[0]*d[0] + oc[1]*d[1] + oc[2]*d[2];
        double c = oc[0]*oc[0] + oc[1]*oc[1] + oc[2]*oc[2] - R * R;
        double disc = b * b - a * c;
        if (disc < 0) return -1.0;
        double sq = sqrt(disc), t = (-b - sq) / a;
        if (t < tmin) t = (-b + sq) / a;
        if (t < tmin) return -1.0;
        for (int i = 0; i < 3; ++i) n[i] = (oc[i] + t * d[i]) / R;
        return t;
    }
    if (type == PRIM_BOX) {
        double t0 = -1e300, t1 = 1e300; int ax0 = 0; double sg0 = 1;
        for (int i = 0; i < 3; ++i) {
            double h = pr[6 + i];
            if (fabs(d[i]) < 1e-300) { if (fabs(oc[i]) > h) return -1.0; continue; }
            double ta = (-h - oc[i]) / d[i], tb = (h - oc[i]) / d[i], sg = -1;
            if (ta > tb) { double s = ta; ta = tb; tb = s; sg = 1; }
            if (ta > t0) { t0 = ta; ax0 = i; sg0 = sg; }
            if (tb < t1) t1 = tb;
        }
        if (t0 > t1 || t0 < tmin) return -1.0;          /* camera is never inside a box */
        n[0] = n[1] = n[2] = 0; n[ax0] = sg0;
        return t0;
    }
    if (type == PRIM_PLANE) {
        const double *nn = pr + 6;
        double dn = d[0]*nn[0] + d[1]*nn[1] + d[2]*nn[2];
        if (fabs(dn) < 1e-12) return -1.0;
        double t = -(oc[0]*nn[0] + oc[1]*nn[1] + oc[2]*nn[2]) / dn;
        if (t < tmin) return -1.0;
        n[0] = nn[0]; n[1] = nn[1]; n[2] = nn[2];
        return t;
    }
    if (type == PRIM_CYLINDER) {
        double R = pr[6], H = pr[7], best = -1.0;
        double a = d[0]*d[0] + d[1]*d[1];
        if (a > 1e-300) {
            double b = oc[0]*d[0] + oc[1]*d[1];
            double c = oc[0]*oc[0] + oc[1]*oc[1] - R * R;
            double disc = b * b - a * c;
            if (disc >= 0) {
                double t = (-b - sqrt(disc)) / a;
                double z = oc[2] + t * d[2];
                if (t >= tmin && fabs(z) <= H) {
                    best = t; n[0] = (oc[0] + t * d[0]) / R; n[1] = (oc[1] + t * d[1]) / R; n[2] = 0;
                }
            }
        }
        if (fabs(d[2]) > 1e-300) {
            for (int s = -1; s <= 1; s += 2) {
                double t = (s * H - oc[2]) / d[2];
                double x = oc[0] + t * d[0], y = oc[1] + t * d[1];
                if (t >= tmin && x * x + y * y <= R * R && (best < 0 || t < best)) {
                    best = t; n[0] = 0; n[1] = 0; n[2] = s;
                }
            }
        }
        return best;
    }
    if (type == PRIM_TORUS) {
        double R = pr[6], r = pr[7];
        /* bounding sphere, then sphere tracing of the torus SDF to 1e-7 m */
        double Rb = R + r, dl = sqrt(d[0]*d[0] + d[1]*d[1] + d[2]*d[2]);
        double b = (oc[0]*d[0] + oc[1]*d[1] + oc[2]*d[2]) / dl;
        double c = oc[0]*oc[0] + oc[1]*oc[1] + oc[2]*oc[2] - Rb * Rb;
        double disc = b * b - c;
        if (disc < 0) return -1.0;
        double s = -b - sqrt(disc), send = -b + sqrt(disc);
        if (s < 0) s = 0;
        for (int it = 0; it < 256 && s <= send; ++it) {
            double p[3] = { oc[0] + s * d[0] / dl, oc[1] + s * d[1] / dl, oc[2] + s * d[2] / dl };
            double rho = sqrt(p[0]*p[0] + p[1]*p[1]) - R;
            double sd = sqrt(rho * rho + p[2]*p[2]) - r;
            if (sd < 1e-7) {
                double rr = sqrt(p[0]*p[0] + p[1]*p[1]);
                double cx = rr > 0 ? p[0] / rr * R : R, cy = rr > 0 ? p[1] / rr * R : 0;
                n[0] = (p[0] - cx) / r; n[1] = (p[1] - cy) / r; n[2] = p[2] / r;
                double t = s / dl;
                return t >= tmin ? t : -1.0;
            }
            s += sd;
        }
        return -1.0;
    }
    return -1.0;
}

/*
 * Render one view.
 *   prims      n_prims x 16 doubles (layout above), world frame
 *   K          fx, fy, cx, cy
 *   T_world_cam row-major 4x4, camera coords -> world
 *   depth_out  (nullable) w*h floats, camera-frame z of the nearest hit, 0 = miss
 *   rgb_out    (nullable) w*h*3 bytes; misses get bg[3]
 */
int synth_render(const double *prims, int n_prims, const double K[4], const double T_world_cam[16],
                 int w, int h, float *depth_out, uint8_t *rgb_out, const uint8_t bg[3])
{
    const double fx = K[0], fy = K[1], cx = K[2], cy = K[3];
    const double *T = T_world_cam;
    const double o[3] = { T[3], T[7], T[11] };
#pragma omp parallel for schedule(dynamic, 4)
    for (int y = 0; y < h; ++y) {
        for (int x = 0; x < w; ++x) {
            double dc[3] = { (x - cx) / fx, (y - cy) / fy, 1.0 };
            double d[3];
            for (int i = 0; i < 3; ++i) d[i] = T[4*i+0] * dc[0] + T[4*i+1] * dc[1] + T[4*i+2] * dc[2];
            double best = -1.0, bn[3] = {0, 0, 0}; int bi = -1;
            for (int k = 0; k < n_prims; ++k) {
                double n[3];
                double t = hit(prims + (size_t)k * PRIM_STRIDE, o, d, n);
                if (t > 0 && (best < 0 || t < best)) { best = t; bi = k; bn[0] = n[0]; bn[1] = n[1]; bn[2] = n[2]; }
            }
            size_t idx = (size_t)y * (size_t)w + (size_t)x;
            if (depth_out) depth_out[idx] = best > 0 ? (float)best : 0.0f;   /* ray dir has camera z = 1 */
            if (rgb_out) {
                uint8_t *px = rgb_out + 3 * idx;
                if (bi < 0) { px[0] = bg[0]; px[1] = bg[1]; px[2] = bg[2]; }
                else {
                    double p[3] = { o[0] + best * d[0], o[1] + best * d[1], o[2] + best * d[2] };
                    shade(prims + (size_t)bi * PRIM_STRIDE, p, bn, px);
                }
            }
        }
    }
    return 0;
}
