/*
 * synth_core.c -- seeded synthetic input generator (scene ray-caster).
 *
 * This file produces INPUTS only (fisheye images of procedural scenes). It is
 * shared by the tests, the oracle runs and bench.py, and contains none of the
 * plane-sweep method (no plane set, no warp, no matching cost, no WTA, no
 * filters).  The one thing it has to know about the paper is what camera took
 * the picture: to render a fisheye image it casts one ray per (sub)pixel, and
 * the ray of a pixel is that of the unified projective model (PAPER.md:149-160,
 * Eq. 1) with the radial/tangential term BASELINE.json configs[2] adds.  That
 * ray function is written here independently (own code, own Newton loop); it
 * is a camera *simulator*, not part of either implementation under test, and
 * tests/test_synth.py cross-checks it against oracle/ as an extra pin.
 *
 * Everything is a pure function of (seed, scene, camera, pose): a counter-based
 * integer hash supplies every random number, so there is no RNG state.
 *
 * Scene model: a list of axis-aligned boxes in the world frame (x right,
 * y down, z forward).  Ground, facades, cars, and "a fronto-parallel plane"
 * are all boxes (possibly huge / thin).  Each box carries a procedural
 * value-noise texture evaluated on the face that was hit.
 */
#include <math.h>
#include <stdint.h>
#include <stddef.h>

#define SYNTH_TEX_STRIDE 6 /* base, contrast, cell0, cell1, cell2 (0 = unused), id */

/* ---- counter-based hash ------------------------------------------------- */
static inline uint32_t mix32(uint32_t h) {
    h ^= h >> 16; h *= 0x7feb352dU;
    h ^= h >> 15; h *= 0x846ca68bU;
    h ^= h >> 16;
    return h;
}
static inline uint32_t hash4(uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
    uint32_t h = mix32(a + 0x9e3779b9U);
    h = mix32(h ^ (b + 0x85ebca6bU + (h << 6) + (h >> 2)));
    h = mix32(h ^ (c + 0xc2b2ae35U + (h << 6) + (h >> 2)));
    h = mix32(h ^ (d + 0x27d4eb2fU + (h << 6) + (h >> 2)));
    return h;
}
static inline double u01(uint32_t h) { return ((double)h + 0.5) * (1.0 / 4294967296.0); }

uint32_t synth_hash4(uint32_t a, uint32_t b, uint32_t c, uint32_t d) { return hash4(a, b, c, d); }

/* ---- value noise -------------------------------------------------------- */
static inline double smooth(double t) { return t * t * (3.0 - 2.0 * t); }

static double vnoise(uint32_t seed, uint32_t id, double x, double y) {
    double fx = floor(x), fy = floor(y);
    int32_t ix = (int32_t)fx, iy = (int32_t)fy;
    double tx = smooth(x - fx), ty = smooth(y - fy);
    double v00 = u01(hash4(seed, id, (uint32_t)ix, (uint32_t)iy));
    double v10 = u01(hash4(seed, id, (uint32_t)(ix + 1), (uint32_t)iy));
    double v01 = u01(hash4(seed, id, (uint32_t)ix, (uint32_t)(iy + 1)));
    double v11 = u01(hash4(seed, id, (uint32_t)(ix + 1), (uint32_t)(iy + 1)));
    double a = v00 + tx * (v10 - v00);
    double b = v01 + tx * (v11 - v01);
    return a + ty * (b - a);
}

/* texture value in [0,1] at face coordinates (s,t) [metres] */
static double texture(uint32_t seed, const double* tex, int face, double s, double t) {
    double base = tex[0], contrast = tex[1];
    uint32_t id = (uint32_t)tex[5] * 8u + (uint32_t)face;
    double acc = 0.0, wsum = 0.0, w = 1.0;
    for (int o = 0; o < 3; ++o) {
        double cell = tex[2 + o];
        if (cell <= 0.0) break;
        acc += w * (vnoise(seed, id + 4096u * (uint32_t)o, s / cell, t / cell) - 0.5);
        wsum += w;
        w *= 0.5;
    }
    double v = base + (wsum > 0.0 ? contrast * acc / wsum * 2.0 : 0.0);
    return v < 0.0 ? 0.0 : (v > 1.0 ? 1.0 : v);
}

/* ---- camera simulator: pixel -> unit ray -------------------------------- */
/* cam = fx fy cx cy xi k1 k2 p1 p2 theta_max */
static int pixel_ray(const double* cam, double u, double v, double* r) {
    double fx = cam[0], fy = cam[1], cx = cam[2], cy = cam[3], xi = cam[4];
    double k1 = cam[5], k2 = cam[6], p1 = cam[7], p2 = cam[8], tmax = cam[9];
    double xd = (u - cx) / fx, yd = (v - cy) / fy;
    /* invert  m_d = m_u (1 + k1 r^2 + k2 r^4) + tangential  by Newton in 2-D */
    double x = xd, y = yd;
    if (k1 != 0.0 || k2 != 0.0 || p1 != 0.0 || p2 != 0.0) {
        int ok = 0;
        for (int it = 0; it < 50; ++it) {
            double r2 = x * x + y * y;
            double rad = 1.0 + k1 * r2 + k2 * r2 * r2;
            double drad = k1 + 2.0 * k2 * r2; /* d rad / d r2 */
            double gx = x * rad + 2.0 * p1 * x * y + p2 * (r2 + 2.0 * x * x) - xd;
            double gy = y * rad + p1 * (r2 + 2.0 * y * y) + 2.0 * p2 * x * y - yd;
            double jxx = rad + 2.0 * x * x * drad + 2.0 * p1 * y + 6.0 * p2 * x;
            double jxy = 2.0 * x * y * drad + 2.0 * p1 * x + 2.0 * p2 * y;
            double jyx = jxy;
            double jyy = rad + 2.0 * y * y * drad + 6.0 * p1 * y + 2.0 * p2 * x;
            double det = jxx * jyy - jxy * jyx;
            if (!(fabs(det) > 1e-12)) return 0;
            double dx = (jyy * gx - jxy * gy) / det;
            double dy = (jxx * gy - jyx * gx) / det;
            x -= dx; y -= dy;
            if (fabs(dx) + fabs(dy) < 1e-15) { ok = 1; break; }
        }
        if (!ok) return 0;
        /* the radial map must still be increasing at the solution */
        double r2 = x * x + y * y;
        if (1.0 + 3.0 * k1 * r2 + 5.0 * k2 * r2 * r2 <= 0.0) return 0;
    }
    double rho2 = x * x + y * y;
    double rad = 1.0 + (1.0 - xi * xi) * rho2;
    if (rad < 0.0) return 0;
    double eta = (xi + sqrt(rad)) / (rho2 + 1.0);
    double rx = eta * x, ry = eta * y, rz = eta - xi;
    double n = sqrt(rx * rx + ry * ry + rz * rz);
    rx /= n; ry /= n; rz /= n;
    double theta = atan2(sqrt(rx * rx + ry * ry), rz);
    if (theta > tmax) return 0;
    r[0] = rx; r[1] = ry; r[2] = rz;
    return 1;
}

int synth_pixel_ray(const double* cam, double u, double v, double* r) { return pixel_ray(cam, u, v, r); }

/* ---- ray / box ---------------------------------------------------------- */
/* returns t of nearest hit (>tmin) or -1; face = 0..5 (axis*2 + side) */
static double hit_box(const double* o, const double* d, const double* b, int* face) {
    double t0 = 1e-6, t1 = 1e30;
    int f0 = -1, f1 = -1;
    for (int a = 0; a < 3; ++a) {
        double lo = b[a], hi = b[3 + a];
        if (fabs(d[a]) < 1e-300) {
            if (o[a] < lo || o[a] > hi) return -1.0;
            continue;
        }
        double inv = 1.0 / d[a];
        double ta = (lo - o[a]) * inv, tb = (hi - o[a]) * inv;
        int fa = a * 2, fb = a * 2 + 1;
        if (ta > tb) { double tt = ta; ta = tb; tb = tt; int ff = fa; fa = fb; fb = ff; }
        if (ta > t0) { t0 = ta; f0 = fa; }
        if (tb < t1) { t1 = tb; f1 = fb; }
        if (t0 > t1) return -1.0;
    }
    if (f0 >= 0) { *face = f0; return t0; }      /* entering from outside */
    if (f1 >= 0 && t1 < 1e29) { *face = f1; return t1; } /* origin inside the box */
    return -1.0;
}

static double shade(uint32_t seed, const double* o, const double* d, int nbox, const double* boxes,
                    const double* tex, double sky, double* t_out) {
    double best = 1e30; int bi = -1, bf = 0;
    for (int i = 0; i < nbox; ++i) {
        int f; double t = hit_box(o, d, boxes + 6 * i, &f);
        if (t > 0.0 && t < best) { best = t; bi = i; bf = f; }
    }
    if (bi < 0) { *t_out = 0.0; return sky; }
    *t_out = best;
    double p[3] = { o[0] + best * d[0], o[1] + best * d[1], o[2] + best * d[2] };
    int axis = bf >> 1;
    double s = p[(axis + 1) % 3], t = p[(axis + 2) % 3];
    return texture(seed, tex + SYNTH_TEX_STRIDE * bi, bf, s, t);
}

/*
 * Render one camera.
 *   cam      : 10 doubles (see pixel_ray)
 *   R_wc[9]  : camera->world rotation (row-major), C_w[3]: camera centre in the world
 *   boxes    : nbox x 6 (min xyz, max xyz), tex: nbox x SYNTH_TEX_STRIDE
 *   S        : supersampling per axis (sub-sample positions (i+0.5)/S - 0.5 around the pixel centre)
 *   sky      : intensity of rays that hit nothing; out-of-FOV pixels get 0
 *   noise_sigma / noise_seed : additive Gaussian noise (Box-Muller on the hash), then clamp to [0,1]
 *   img      : H*W floats in [0,1];  range_gt (nullable): range along the centre ray, 0 = none
 */
int synth_render(const double* cam, int W, int H, const double* R_wc, const double* C_w,
                 int nbox, const double* boxes, const double* tex, uint32_t seed,
                 int S, double sky, double noise_sigma, uint32_t noise_seed,
                 float* img, float* range_gt) {
    if (S < 1) S = 1;
    #pragma omp parallel for schedule(dynamic, 4)
    for (int v = 0; v < H; ++v) {
        for (int u = 0; u < W; ++u) {
            double r[3], dw[3], t;
            size_t idx = (size_t)v * W + u;
            if (!pixel_ray(cam, (double)u, (double)v, r)) {
                img[idx] = 0.0f;
                if (range_gt) range_gt[idx] = 0.0f;
                continue;
            }
            for (int a = 0; a < 3; ++a) dw[a] = R_wc[3 * a] * r[0] + R_wc[3 * a + 1] * r[1] + R_wc[3 * a + 2] * r[2];
            (void)shade(seed, C_w, dw, nbox, boxes, tex, sky, &t);
            if (range_gt) range_gt[idx] = (float)t;
            double acc = 0.0; int cnt = 0;
            for (int j = 0; j < S; ++j) for (int i = 0; i < S; ++i) {
                double uu = u + (i + 0.5) / S - 0.5, vv = v + (j + 0.5) / S - 0.5;
                if (!pixel_ray(cam, uu, vv, r)) continue;
                for (int a = 0; a < 3; ++a) dw[a] = R_wc[3 * a] * r[0] + R_wc[3 * a + 1] * r[1] + R_wc[3 * a + 2] * r[2];
                acc += shade(seed, C_w, dw, nbox, boxes, tex, sky, &t);
                ++cnt;
            }
            double val = cnt ? acc / cnt : 0.0;
            if (noise_sigma > 0.0) {
                double a1 = u01(hash4(noise_seed, 0x6e6f6973U, (uint32_t)u, (uint32_t)v));
                double a2 = u01(hash4(noise_seed, 0x65323334U, (uint32_t)u, (uint32_t)v));
                val += noise_sigma * sqrt(-2.0 * log(a1)) * cos(6.283185307179586 * a2);
            }
            val = val < 0.0 ? 0.0 : (val > 1.0 ? 1.0 : val);
            img[idx] = (float)val;
        }
    }
    return 0;
}
