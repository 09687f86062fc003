/*
 * fsw_oracle.c -- CPU ORACLE (test infrastructure, see fsw_oracle.h).
 *
 * Plain double-precision restatement of fisheye plane-sweeping stereo,
 * PAPER.md section III-A (lines 69-99) and Eq. 1 (lines 149-160).  Step labels
 * O1..O10 are those of SURVEY.md section 8(c); readings of silent / ambiguous
 * passages (Q1..Q24) are listed in DESIGN.md.  No blocking, fusion or
 * reordering beyond the definitions: every (plane, view) gets its own warped
 * image, every window is summed directly in two passes, every pixel scans its
 * full cost vector.  OpenMP only splits independent rows.
 */
#include "fsw_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define EPS_DEN 1e-9   /* O1: projection denominator test, relative to rho */
#define EPS_Q 1e-9     /* O4: ray/plane incidence n.r must exceed this */
#define MARGIN_PX 1e-3 /* O10 fragility margins */
#define MARGIN_ANG 1e-5
#define MARGIN_REL 1e-6

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

static double dot3(const double* a, const double* b) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }

/* ------------------------------------------------------------------------- */
/* O1  camera: unified projective model, PAPER.md:149 (projection, by name),  */
/*     PAPER.md:150-160 Eq. 1 (back-projection); distortion per reading Q2     */
/* ------------------------------------------------------------------------- */
static void distort(const orc_camera* c, double x, double y, double* xd, double* yd) {
    double r2 = x * x + y * y;
    double rad = 1.0 + c->k1 * r2 + c->k2 * r2 * r2;
    *xd = x * rad + 2.0 * c->p1 * x * y + c->p2 * (r2 + 2.0 * x * x);
    *yd = y * rad + c->p1 * (r2 + 2.0 * y * y) + 2.0 * c->p2 * x * y;
}

/* detailed projection: also reports the angular margin to the FOV cut-off */
static int project_detail(const orc_camera* c, const double X[3], double uv[2], double* fov_margin) {
    double rho = sqrt(dot3(X, X));
    if (fov_margin) *fov_margin = 1e30;
    if (!(rho > 0.0)) return 0;
    double den = X[2] + c->xi * rho; /* sphere point shifted by xi along z */
    if (fov_margin) {
        double th = atan2(sqrt(X[0] * X[0] + X[1] * X[1]), X[2]);
        *fov_margin = fabs(th - c->theta_max);
        double dm = fabs(den / rho - EPS_DEN);
        if (dm < *fov_margin) *fov_margin = dm;
    }
    if (den <= EPS_DEN * rho) return 0;
    if (X[2] < cos(c->theta_max) * rho) return 0; /* Q3: outside the field of view */
    double mx = X[0] / den, my = X[1] / den;
    double xd, yd;
    distort(c, mx, my, &xd, &yd);
    uv[0] = c->fx * xd + c->cx;
    uv[1] = c->fy * yd + c->cy;
    return 1;
}

int orc_project(const orc_camera* c, const double X[3], double uv[2]) { return project_detail(c, X, uv, 0); }

/* invert the distortion on the normalised plane */
static int undistort(const orc_camera* c, double xd, double yd, double* xu, double* yu) {
    if (c->k1 == 0.0 && c->k2 == 0.0 && c->p1 == 0.0 && c->p2 == 0.0) { *xu = xd; *yu = yd; return 1; }
    if (c->p1 == 0.0 && c->p2 == 0.0) {
        /* radial only: scalar Newton on rho (1 + k1 rho^2 + k2 rho^4) = rho_d */
        double rd = sqrt(xd * xd + yd * yd);
        if (rd == 0.0) { *xu = 0.0; *yu = 0.0; return 1; }
        double r = rd;
        int ok = 0;
        for (int it = 0; it < 100; ++it) {
            double r2 = r * r;
            double g = r * (1.0 + c->k1 * r2 + c->k2 * r2 * r2) - rd;
            double dg = 1.0 + 3.0 * c->k1 * r2 + 5.0 * c->k2 * r2 * r2;
            if (!(dg > 1e-12)) return 0; /* past the turning point: not invertible */
            double step = g / dg;
            r -= step;
            if (!(r > 0.0) || !isfinite(r)) return 0;
            if (fabs(step) < 1e-14) { ok = 1; break; }
        }
        if (!ok) return 0;
        double r2 = r * r;
        if (!(1.0 + 3.0 * c->k1 * r2 + 5.0 * c->k2 * r2 * r2 > 0.0)) return 0;
        *xu = xd * (r / rd);
        *yu = yd * (r / rd);
        return 1;
    }
    /* general: 2-D Newton */
    double x = xd, y = yd;
    for (int it = 0; it < 100; ++it) {
        double r2 = x * x + y * y;
        double rad = 1.0 + c->k1 * r2 + c->k2 * r2 * r2;
        double drad = c->k1 + 2.0 * c->k2 * r2;
        double gx, gy;
        distort(c, x, y, &gx, &gy);
        gx -= xd; gy -= yd;
        double jxx = rad + 2.0 * x * x * drad + 2.0 * c->p1 * y + 6.0 * c->p2 * x;
        double jxy = 2.0 * x * y * drad + 2.0 * c->p1 * x + 2.0 * c->p2 * y;
        double jyy = rad + 2.0 * y * y * drad + 6.0 * c->p1 * y + 2.0 * c->p2 * x;
        double det = jxx * jyy - jxy * jxy;
        if (!(det > 1e-12)) return 0;
        double dx = (jyy * gx - jxy * gy) / det;
        double dy = (jxx * gy - jxy * gx) / det;
        x -= dx; y -= dy;
        if (!isfinite(x) || !isfinite(y)) return 0;
        if (fabs(dx) + fabs(dy) < 1e-14) { *xu = x; *yu = y; return 1; }
    }
    return 0;
}

int orc_back_project(const orc_camera* c, double u, double v, double r[3]) {
    double xd = (u - c->cx) / c->fx, yd = (v - c->cy) / c->fy;
    double x, y;
    if (!undistort(c, xd, yd, &x, &y)) return 0;
    /* Eq. 1 */
    double rho2 = x * x + y * y;
    double rad = 1.0 + (1.0 - c->xi * c->xi) * rho2;
    if (rad < 0.0) return 0;
    double eta = (c->xi + sqrt(rad)) / (rho2 + 1.0);
    double rx = eta * x, ry = eta * y, rz = eta - c->xi;
    double n = sqrt(rx * rx + ry * ry + rz * rz); /* = 1 up to rounding (Q1); normalising is harmless */
    rx /= n; ry /= n; rz /= n;
    if (atan2(sqrt(rx * rx + ry * ry), rz) > c->theta_max) return 0; /* Q3 */
    r[0] = rx; r[1] = ry; r[2] = rz;
    return 1;
}

double orc_pixel_theta(const orc_camera* c, double u, double v) {
    orc_camera w = *c;
    w.theta_max = 4.0; /* > pi: no cut-off */
    double r[3];
    if (!orc_back_project(&w, u, v, r)) return -1.0;
    return atan2(sqrt(r[0] * r[0] + r[1] * r[1]), r[2]);
}

/* ------------------------------------------------------------------------- */
/* O3  relative pose: X_v = R_v X_ref + T_v with R_v = R_v^c R_ref^cT,          */
/*     T_v = t_v - R_v t_ref  ("known relative poses" PAPER.md:70) */
/* ------------------------------------------------------------------------- */
void orc_relative_pose(const orc_camera* ref, const orc_camera* view, double R[9], double T[3]) {
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {
            double s = 0.0;
            for (int k = 0; k < 3; ++k) s += view->R[3 * i + k] * ref->R[3 * j + k];
            R[3 * i + j] = s;
        }
    for (int i = 0; i < 3; ++i) T[i] = view->t[i] - (R[3 * i] * ref->t[0] + R[3 * i + 1] * ref->t[1] + R[3 * i + 2] * ref->t[2]);
}

/* ------------------------------------------------------------------------- */
/* O2  plane table (Q6, Q7): plane k of family f is n_f.X=d_k  */
/* ------------------------------------------------------------------------- */
int orc_plane_table(const orc_family* fams, int n_fams, double* s, double* d, int32_t* fam, double* nrm) {
    int P = 0;
    for (int f = 0; f < n_fams; ++f) {
        const orc_family* F = &fams[f];
        double nn = sqrt(dot3(F->normal, F->normal));
        if (nrm) for (int a = 0; a < 3; ++a) nrm[3 * f + a] = F->normal[a] / nn;
        double s0 = F->spacing == ORC_INVERSE ? 1.0 / F->d_first : F->d_first;
        double s1 = F->spacing == ORC_INVERSE ? 1.0 / F->d_last : F->d_last;
        for (int k = 0; k < F->n_planes; ++k) {
            double sk = F->n_planes > 1 ? s0 + (double)k * (s1 - s0) / (double)(F->n_planes - 1) : s0;
            if (s) s[P] = sk;
            if (d) d[P] = F->spacing == ORC_INVERSE ? 1.0 / sk : sk;
            if (fam) fam[P] = f;
            ++P;
        }
    }
    return P;
}

/* ------------------------------------------------------------------------- */
/* O4  plane-induced mapping for one pixel ("Each position of a   */
/*     plane defines a homography mapping pixels from the reference image into */
/*     other images"), here through the fisheye model instead of a pinhole K.  */
/* ------------------------------------------------------------------------- */
static int warp_ray(const double r[3], const orc_camera* view, const double R[9], const double T[3],
                    const double n[3], double d, double range_max, double uv[2], int* near_edge) {
    double q = dot3(n, r); /* incidence of the ray on the plane normal */
    int near = fabs(q - EPS_Q) < MARGIN_REL;
    if (near_edge) *near_edge = near;
    if (q <= EPS_Q) return 0; /* parallel or facing away */
    double t = d / q;         /* range along the unit ray to the plane */
    if (fabs(t - range_max) <= MARGIN_REL * range_max) near = 1;
    if (near_edge) *near_edge = near;
    if (t > range_max) return 0; /* Q17 */
    double X[3] = { t * r[0], t * r[1], t * r[2] };
    double Xv[3];
    for (int i = 0; i < 3; ++i) Xv[i] = R[3 * i] * X[0] + R[3 * i + 1] * X[1] + R[3 * i + 2] * X[2] + T[i];
    double margin;
    int ok = project_detail(view, Xv, uv, &margin);
    if (margin < MARGIN_ANG) near = 1;
    if (near_edge) *near_edge = near;
    if (!ok) return 0;
    /* bilinear footprint must lie inside the view image (Q4): 0 <= u' < W-1, 0 <= v' < H-1 */
    double W1 = (double)(view->width - 1), H1 = (double)(view->height - 1);
    if (fabs(uv[0]) < MARGIN_PX || fabs(uv[0] - W1) < MARGIN_PX || fabs(uv[1]) < MARGIN_PX || fabs(uv[1] - H1) < MARGIN_PX) near = 1;
    if (near_edge) *near_edge = near;
    if (!(uv[0] >= 0.0 && uv[0] < W1 && uv[1] >= 0.0 && uv[1] < H1)) return 0;
    return 1;
}

int orc_warp_pixel(const orc_camera* ref, const orc_camera* view, const double n[3], double d,
                   double range_max, double u, double v, double uv[2]) {
    double r[3], R[9], T[3], nn[3];
    if (!orc_back_project(ref, u, v, r)) return 0;
    orc_relative_pose(ref, view, R, T);
    double len = sqrt(dot3(n, n));
    for (int a = 0; a < 3; ++a) nn[a] = n[a] / len;
    return warp_ray(r, view, R, T, nn, d, range_max, uv, 0);
}

double orc_bilinear(const double* img, int W, int H, double u, double v) {
    (void)H;
    int i0 = (int)floor(u), j0 = (int)floor(v);
    double fu = u - i0, fv = v - j0;
    const double* p = img + (size_t)j0 * W + i0;
    double top = (1.0 - fu) * p[0] + fu * p[1];
    double bot = (1.0 - fu) * p[W] + fu * p[W + 1];
    return (1.0 - fv) * top + fv * bot;
}

/* ------------------------------------------------------------------------- */
/* O5  matching cost: "negative ZNCC ... cost of 1 <-> ZNCC -1, cost of 0 <->  */
/*     ZNCC 1"  =>  cost = (1 - ZNCC)/2.  Two-pass; Q10 floor.   */
/* ------------------------------------------------------------------------- */
double orc_zncc_cost(const double* a, const double* b, int n, double var_floor) {
    double ma = 0.0, mb = 0.0;
    for (int i = 0; i < n; ++i) { ma += a[i]; mb += b[i]; }
    ma /= n; mb /= n;
    double cov = 0.0, va = 0.0, vb = 0.0;
    for (int i = 0; i < n; ++i) {
        double da = a[i] - ma, db = b[i] - mb;
        cov += da * db; va += da * da; vb += db * db;
    }
    cov /= n; va /= n; vb /= n;
    double den = sqrt(va * vb);
    if (den < var_floor) den = var_floor;
    double zncc = cov / den;
    double cost = 0.5 * (1.0 - zncc);
    if (cost < 0.0) cost = 0.0;
    if (cost > 1.0) cost = 1.0;
    return cost;
}

static void roi_of(const orc_params* prm, int W, int H, int* x0, int* y0, int* x1, int* y1) {
    if (prm->roi_w > 0 && prm->roi_h > 0) {
        *x0 = prm->roi_x0; *y0 = prm->roi_y0; *x1 = prm->roi_x0 + prm->roi_w; *y1 = prm->roi_y0 + prm->roi_h;
    } else { *x0 = 0; *y0 = 0; *x1 = W; *y1 = H; }
    if (*x0 < 0) *x0 = 0;
    if (*y0 < 0) *y0 = 0;
    if (*x1 > W) *x1 = W;
    if (*y1 > H) *y1 = H;
}

/* ------------------------------------------------------------------------- */
/* O4-O6  cost volume                                                          */
/* ------------------------------------------------------------------------- */
int orc_sweep(const orc_camera* cams, int n_cams, int ref_index, const orc_family* fams, int n_fams,
              const orc_params* prm, const double* const* images, double* cost, int64_t* n_eval,
              uint8_t* fragile_geom) {
    if (n_cams < 2 || ref_index < 0 || ref_index >= n_cams) return -1;
    int w = prm->window;
    if (w < 1 || (w & 1) == 0 || w > 31) return -1;
    const orc_camera* ref = &cams[ref_index];
    int W = ref->width, H = ref->height, h = w / 2, N = w * w;
    size_t npx = (size_t)W * H;
    int x0, y0, x1, y1;
    roi_of(prm, W, H, &x0, &y0, &x1, &y1);

    int P = orc_plane_table(fams, n_fams, 0, 0, 0, 0);
    double* pd = (double*)malloc(sizeof(double) * P);
    int32_t* pf = (int32_t*)malloc(sizeof(int32_t) * P);
    double* nrm = (double*)malloc(sizeof(double) * 3 * n_fams);
    orc_plane_table(fams, n_fams, 0, pd, pf, nrm);

    /* S1: reference rays, once per pixel */
    double* ray = (double*)malloc(sizeof(double) * 3 * npx);
    uint8_t* ray_ok = (uint8_t*)malloc(npx);
    uint8_t* ray_near = (uint8_t*)calloc(npx, 1);
    #pragma omp parallel for schedule(static)
    for (int y = 0; y < H; ++y)
        for (int x = 0; x < W; ++x) {
            size_t i = (size_t)y * W + x;
            ray_ok[i] = (uint8_t)orc_back_project(ref, (double)x, (double)y, ray + 3 * i);
            double th = orc_pixel_theta(ref, (double)x, (double)y);
            if (th >= 0.0 && fabs(th - ref->theta_max) < MARGIN_ANG) ray_near[i] = 1;
        }

    double* B = (double*)malloc(sizeof(double) * npx);    /* plane-warped view image, NaN = NONE */
    uint8_t* Bnear = (uint8_t*)malloc(npx);
    /* per-view costs of the current plane, +inf where the view is invalid: [view slot][pixel] */
    int n_views = n_cams - 1;
    double* vcost = (double*)malloc(sizeof(double) * npx * (size_t)n_views);
    if (fragile_geom) memset(fragile_geom, 0, npx);
    int64_t evals = 0;

    for (int k = 0; k < P; ++k) {
        const double* n = nrm + 3 * pf[k];
        for (size_t i = 0; i < npx * (size_t)n_views; ++i) vcost[i] = INFINITY;
        int slot = -1;
        for (int v = 0; v < n_cams; ++v) {
            if (v == ref_index) continue;
            ++slot;
            double* vc = vcost + (size_t)slot * npx;
            const orc_camera* view = &cams[v];
            double R[9], T[3];
            orc_relative_pose(ref, view, R, T);
            const double* img = images[v];
            /* O4: the plane-warped image B_kv(q) for every reference pixel q */
            #pragma omp parallel for schedule(static)
            for (int y = 0; y < H; ++y)
                for (int x = 0; x < W; ++x) {
                    size_t i = (size_t)y * W + x;
                    B[i] = NAN; Bnear[i] = ray_near[i];
                    if (!ray_ok[i]) continue;
                    double uv[2]; int near = 0;
                    int ok = warp_ray(ray + 3 * i, view, R, T, n, pd[k], prm->range_max, uv, &near);
                    if (near) Bnear[i] = 1;
                    if (ok) B[i] = orc_bilinear(img, view->width, view->height, uv[0], uv[1]);
                }
            /* O5: direct window cost at every ROI pixel p */
            const double* A = images[ref_index];
            #pragma omp parallel for schedule(dynamic, 4) reduction(+ : evals)
            for (int y = y0; y < y1; ++y) {
                double wa[31 * 31], wb[31 * 31];
                for (int x = x0; x < x1; ++x) {
                    size_t i = (size_t)y * W + x;
                    if (y - h < 0 || y + h >= H || x - h < 0 || x + h >= W) continue; /* window leaves the image */
                    int ok = 1, near = 0, m = 0;
                    for (int dy = -h; dy <= h; ++dy)
                        for (int dx = -h; dx <= h; ++dx) {
                            size_t j = (size_t)(y + dy) * W + (x + dx);
                            if (Bnear[j]) near = 1;
                            if (!ray_ok[j] || isnan(B[j])) ok = 0;
                            wa[m] = A[j]; wb[m] = B[j]; ++m;
                        }
                    if (near && fragile_geom) fragile_geom[i] = 1;
                    if (!ok) continue; /* view invalid for this (p,k) */
                    vc[i] = orc_zncc_cost(wa, wb, N, prm->var_floor);
                    evals += 1;
                }
            }
        }
        /* O6: mean over the valid views in fixed view order (Q11), +inf if none; with best_k > 0 the mean of the
         * best_k lowest valid per-view costs instead (Q26), summed in ascending order of cost */
        double* ck = cost + (size_t)k * npx;
        for (size_t i = 0; i < npx; ++i) {
            double c[64];
            int m = 0;
            for (int sl = 0; sl < n_views; ++sl)
                if (isfinite(vcost[(size_t)sl * npx + i])) c[m++] = vcost[(size_t)sl * npx + i];
            if (m == 0) { ck[i] = INFINITY; continue; }
            int use = m;
            if (prm->best_k > 0 && prm->best_k < m) {
                for (int a = 1; a < m; ++a) { /* insertion sort, ascending */
                    double t = c[a];
                    int b = a - 1;
                    while (b >= 0 && c[b] > t) { c[b + 1] = c[b]; --b; }
                    c[b + 1] = t;
                }
                use = prm->best_k;
            }
            double sum = 0.0;
            for (int a = 0; a < use; ++a) sum += c[a];
            ck[i] = sum / (double)use;
        }
    }
    if (n_eval) *n_eval = evals;
    free(pd); free(pf); free(nrm); free(ray); free(ray_ok); free(ray_near); free(B); free(Bnear); free(vcost);
    return P;
}

/* brute force for one pixel: every window sample warped from scratch */
int orc_pixel_costs(const orc_camera* cams, int n_cams, int ref_index, const orc_family* fams, int n_fams,
                    const orc_params* prm, const double* const* images, int px, int py, double* cost_out) {
    const orc_camera* ref = &cams[ref_index];
    int W = ref->width, H = ref->height, w = prm->window, h = w / 2, N = w * w;
    int P = orc_plane_table(fams, n_fams, 0, 0, 0, 0);
    double* pd = (double*)malloc(sizeof(double) * P);
    int32_t* pf = (int32_t*)malloc(sizeof(int32_t) * P);
    double* nrm = (double*)malloc(sizeof(double) * 3 * n_fams);
    orc_plane_table(fams, n_fams, 0, pd, pf, nrm);
    for (int k = 0; k < P; ++k) {
        double cv[64]; int cnt = 0;
        for (int v = 0; v < n_cams; ++v) {
            if (v == ref_index) continue;
            double wa[31 * 31], wb[31 * 31];
            int ok = 1, m = 0;
            for (int dy = -h; dy <= h && ok; ++dy)
                for (int dx = -h; dx <= h; ++dx) {
                    int x = px + dx, y = py + dy;
                    double uv[2];
                    if (x < 0 || x >= W || y < 0 || y >= H) { ok = 0; break; }
                    if (!orc_warp_pixel(ref, &cams[v], nrm + 3 * pf[k], pd[k], prm->range_max, (double)x, (double)y, uv)) { ok = 0; break; }
                    wa[m] = images[ref_index][(size_t)y * W + x];
                    wb[m] = orc_bilinear(images[v], cams[v].width, cams[v].height, uv[0], uv[1]);
                    ++m;
                }
            if (!ok) continue;
            cv[cnt++] = orc_zncc_cost(wa, wb, N, prm->var_floor);
        }
        int use = cnt;
        if (prm->best_k > 0 && prm->best_k < cnt) {
            for (int a = 1; a < cnt; ++a) {
                double t = cv[a];
                int b = a - 1;
                while (b >= 0 && cv[b] > t) { cv[b + 1] = cv[b]; --b; }
                cv[b + 1] = t;
            }
            use = prm->best_k;
        }
        double sum = 0.0;
        for (int a = 0; a < use; ++a) sum += cv[a];
        cost_out[k] = cnt ? sum / use : INFINITY;
    }
    free(pd); free(pf); free(nrm);
    return P;
}

/* ------------------------------------------------------------------------- */
/* O7-O8  winner-take-all, second best, sub-plane parabola, depth              */
/*   "best depth candidate", "first and second best cost values" PAPER.md:99   */
/* ------------------------------------------------------------------------- */
int orc_wta(const orc_camera* ref, const orc_family* fams, int n_fams, const orc_params* prm,
            const double* cost, double* depth, double* c1, double* c2, double* c2raw, int32_t* kbest,
            double* delta, double* pden, uint8_t* raw_valid) {
    int W = ref->width, H = ref->height;
    size_t npx = (size_t)W * H;
    int P = orc_plane_table(fams, n_fams, 0, 0, 0, 0);
    double* ps = (double*)malloc(sizeof(double) * P);
    int32_t* pf = (int32_t*)malloc(sizeof(int32_t) * P);
    double* nrm = (double*)malloc(sizeof(double) * 3 * n_fams);
    orc_plane_table(fams, n_fams, ps, 0, pf, nrm);

    #pragma omp parallel for schedule(static)
    for (int y = 0; y < H; ++y)
        for (int x = 0; x < W; ++x) {
            size_t i = (size_t)y * W + x;
            depth[i] = 0.0; c1[i] = INFINITY; c2[i] = INFINITY; kbest[i] = -1; raw_valid[i] = 0;
            if (c2raw) c2raw[i] = INFINITY;
            if (delta) delta[i] = 0.0;
            if (pden) pden[i] = 0.0;
            /* O7: argmin with lowest-index tie-break */
            int kb = -1; double cb = INFINITY;
            for (int k = 0; k < P; ++k) {
                double c = cost[(size_t)k * npx + i];
                if (c < cb) { cb = c; kb = k; }
            }
            if (kb < 0) continue; /* raw-invalid: no finite cost */
            /* second best: smallest cost among planes of another family or >= 2 indices away (Q12) */
            double cs = INFINITY, csraw = INFINITY;
            for (int k = 0; k < P; ++k) {
                double c = cost[(size_t)k * npx + i];
                if (k != kb && c < csraw) csraw = c;
                if (pf[k] != pf[kb] || abs(k - kb) >= 2) { if (c < cs) cs = c; }
            }
            if (!isfinite(cs)) cs = 1.0;
            /* O8: parabola through (k-1,k,k+1) in the spacing variable s, same family only (Q15) */
            double dl = 0.0, den = 0.0;
            int f = pf[kb];
            if (prm->subpixel && kb > 0 && kb + 1 < P && pf[kb - 1] == f && pf[kb + 1] == f) {
                double cm = cost[(size_t)(kb - 1) * npx + i], cp = cost[(size_t)(kb + 1) * npx + i];
                if (isfinite(cm) && isfinite(cp)) {
                    den = cm - 2.0 * cb + cp;
                    if (den > 1e-12) {
                        dl = 0.5 * (cm - cp) / den;
                        if (dl < -0.5) dl = -0.5;
                        if (dl > 0.5) dl = 0.5;
                    } else den = 0.0;
                }
            }
            double s = ps[kb];
            if (dl != 0.0) s += dl * (ps[kb + 1] - ps[kb]); /* uniform spacing inside a family */
            double d = fams[f].spacing == ORC_INVERSE ? 1.0 / s : s;
            double r[3];
            if (!orc_back_project(ref, (double)x, (double)y, r)) continue;
            double q = dot3(nrm + 3 * f, r);
            double range = d / q; /* Q16: Euclidean range along the unit ray */
            depth[i] = prm->depth_kind == ORC_DEPTH_Z ? range * r[2] : range;
            c1[i] = cb; c2[i] = cs; kbest[i] = kb; raw_valid[i] = 1;
            if (c2raw) c2raw[i] = csraw;
            if (delta) delta[i] = dl;
            if (pden) pden[i] = den;
        }
    free(ps); free(pf); free(nrm);
    return 0;
}

/* ------------------------------------------------------------------------- */
/* S9 filters then S11 mask; order per Q20         */
/* ------------------------------------------------------------------------- */
int orc_filter_mask(int W, int H, const orc_params* prm, const uint8_t* mask, const uint8_t* raw_valid,
                    const double* c1, const double* c2, double* depth, uint8_t* reason, uint8_t* fragile) {
    for (int y = 0; y < H; ++y)
        for (int x = 0; x < W; ++x) {
            size_t i = (size_t)y * W + x;
            uint8_t why = ORC_OK;
            if (!raw_valid[i]) why = ORC_NO_PLANE;
            else {
                double alpha = y < prm->horizon_row ? prm->alpha_upper : prm->alpha_lower; /* Q14 */
                double floor1 = c1[i] > 1e-6 ? c1[i] : 1e-6;
                if ((prm->filters & ORC_FILTER_COST) && c1[i] > alpha) why = ORC_COST_FILTER;
                else if ((prm->filters & ORC_FILTER_RATIO) && c2[i] < prm->beta * floor1) why = ORC_RATIO_FILTER; /* Q13 */
                else if (mask && mask[i]) why = ORC_MASKED;
                if (fragile) {
                    if ((prm->filters & ORC_FILTER_COST) && fabs(c1[i] - alpha) < 2e-4) fragile[i] = 1;
                    if ((prm->filters & ORC_FILTER_RATIO) && fabs(c2[i] - prm->beta * floor1) < 3e-4) fragile[i] = 1;
                }
            }
            reason[i] = why;
            if (why != ORC_OK) depth[i] = 0.0;
        }
    return 0;
}

/* Third filter of PAPER.md:99, reading Q25: see fsw_oracle.h. */
int orc_filter_continuity(const double* in, int W, int H, int window, double gamma, double delta,
                          const uint8_t* mask, double* out, uint8_t* reason) {
    if (window < 3 || window % 2 == 0) return -1;
    const int hw = window / 2;
    const double denom = (double)(window * window - 1);
    for (int y = 0; y < H; ++y)
        for (int x = 0; x < W; ++x) {
            size_t i = (size_t)y * W + x;
            double dc = in[i];
            uint8_t why = ORC_OK;
            if (!(dc > 0.0)) why = ORC_NO_PLANE;
            else {
                int consistent = 0;
                for (int dy = -hw; dy <= hw; ++dy)
                    for (int dx = -hw; dx <= hw; ++dx) {
                        if (dx == 0 && dy == 0) continue;
                        int xx = x + dx, yy = y + dy;
                        if (xx < 0 || yy < 0 || xx >= W || yy >= H) continue; /* outside: not consistent */
                        double dn = in[(size_t)yy * W + xx];
                        if (dn > 0.0 && fabs(dn - dc) < gamma) ++consistent;
                    }
                if ((double)consistent / denom < delta) why = ORC_CONTINUITY;
                else if (mask && mask[i]) why = ORC_MASKED;
            }
            reason[i] = why;
            out[i] = why == ORC_OK ? dc : 0.0;
        }
    return 0;
}

/* ------------------------------------------------------------------------- */
/* S10 multi-resolution (Q4, Q18, Q19)                         */
/* ------------------------------------------------------------------------- */
int orc_downsample2(const double* img, int W, int H, double* out) {
    int W2 = W / 2, H2 = H / 2;
    for (int y = 0; y < H2; ++y)
        for (int x = 0; x < W2; ++x) {
            const double* p = img + (size_t)(2 * y) * W + 2 * x;
            out[(size_t)y * W2 + x] = 0.25 * (p[0] + p[1] + p[W] + p[W + 1]);
        }
    return 0;
}

void orc_camera_half(const orc_camera* c, orc_camera* out) {
    *out = *c;
    out->width = c->width / 2; out->height = c->height / 2;
    out->fx = c->fx / 2.0; out->fy = c->fy / 2.0;
    out->cx = (c->cx - 0.5) / 2.0; out->cy = (c->cy - 0.5) / 2.0; /* low-res centre i <-> full-res 2i+0.5 */
}

int orc_merge(int W, int H, int crop_x0, int crop_y0, int crop_w, int crop_h,
              const double* depth_lo, const double* c1_lo, const double* c2_lo, const int32_t* k_lo,
              const uint8_t* rv_lo, const double* depth_hi, const double* c1_hi, const double* c2_hi,
              const int32_t* k_hi, const uint8_t* rv_hi, double* depth, double* c1, double* c2, int32_t* kbest,
              uint8_t* raw_valid) {
    int W2 = W / 2, H2 = H / 2;
    for (int y = 0; y < H; ++y)
        for (int x = 0; x < W; ++x) {
            size_t i = (size_t)y * W + x;
            int in_crop = x >= crop_x0 && x < crop_x0 + crop_w && y >= crop_y0 && y < crop_y0 + crop_h;
            if (in_crop && rv_hi[i]) { /* full resolution wins where it has any valid plane */
                depth[i] = depth_hi[i]; c1[i] = c1_hi[i]; c2[i] = c2_hi[i]; kbest[i] = k_hi[i] | (1 << 14); raw_valid[i] = 1;
                continue;
            }
            int xl = x >> 1, yl = y >> 1; /* nearest-neighbour upsample (Q18) */
            if (xl < W2 && yl < H2 && rv_lo[(size_t)yl * W2 + xl]) {
                size_t j = (size_t)yl * W2 + xl;
                depth[i] = depth_lo[j]; c1[i] = c1_lo[j]; c2[i] = c2_lo[j]; kbest[i] = k_lo[j]; raw_valid[i] = 1;
            } else {
                depth[i] = 0.0; c1[i] = INFINITY; c2[i] = INFINITY; kbest[i] = -1; raw_valid[i] = 0;
            }
        }
    return 0;
}
