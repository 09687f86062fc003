/*
 * fsw_oracle.h -- CPU ORACLE for fisheye plane-sweeping stereo (TEST INFRASTRUCTURE).
 *
 * A plain, slow, double-precision restatement of what the hot path computes,
 * written from /root/reference/PAPER.md (arXiv 1809.06132, section III-A and
 * Eq. 1) with the readings listed in DESIGN.md ("Readings of the paper").  It
 * exists to check the CUDA path and to be timed as the CPU baseline.  Only
 * tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may use it.  It shares no code with paper_1809_06132_b200/
 * (the CUDA path) and neither includes the other.
 *
 * Method = exhaustive search, so the oracle is the plain definition: for every
 * plane and view build the plane-warped image, score every window directly
 * (two-pass ZNCC), average over views, scan all planes per pixel.
 *
 * Parity pins (tests/test_oracle_*.py, -m "not gpu"): see DESIGN.md "Oracle pins".
 * parity unpinned: absolute cost / depth values on the procedural scenes, the
 * effect of beta, and behaviour exactly at FOV edges (pinned only by the
 * invariants and by oracle<->CUDA parity).
 */
#ifndef FSW_ORACLE_H
#define FSW_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define ORC_INVERSE 0 /* planes uniform in 1/d */
#define ORC_LINEAR 1  /* planes uniform in d   */

#define ORC_FILTER_COST 1
#define ORC_FILTER_RATIO 2

#define ORC_DEPTH_RANGE 0 /* Euclidean range along the unit ray */
#define ORC_DEPTH_Z 1

/* reason codes of the per-pixel decision chain (first that fires) */
#define ORC_OK 0
#define ORC_NO_PLANE 1
#define ORC_COST_FILTER 2
#define ORC_RATIO_FILTER 3
#define ORC_MASKED 4
#define ORC_CONTINUITY 5

typedef struct {
    int32_t width, height;
    double fx, fy, cx, cy; /* pixels; pixel centres at integer coordinates */
    double xi;             /* mirror parameter of the unified model */
    double k1, k2, p1, p2; /* radial / tangential distortion on the normalised plane */
    double theta_max;      /* half field of view, radians */
    double R[9];           /* rig->camera rotation, row-major: X_cam = R X_rig + t */
    double t[3];
} orc_camera;

typedef struct {
    double normal[3]; /* in the reference-camera frame; normalised by the oracle */
    int32_t n_planes;
    int32_t spacing;  /* ORC_INVERSE / ORC_LINEAR */
    double d_first, d_last; /* offsets n.X = d of the first and last plane, metres */
} orc_family;

typedef struct {
    int32_t window;   /* odd side w of the matching window */
    int32_t subpixel; /* 1 = 3-point parabola in the spacing variable */
    int32_t filters;  /* ORC_FILTER_* bits */
    int32_t depth_kind;
    int32_t roi_x0, roi_y0, roi_w, roi_h; /* output region on the reference raster; roi_w<=0 = full image */
    int32_t horizon_row;
    double alpha_upper, alpha_lower; /* best-cost thresholds above / below horizon_row */
    double beta;                     /* keep iff c2 >= beta*max(c1,1e-6) */
    double var_floor;                /* eps_v: floor of sqrt(var_a var_b) */
    double range_max;                /* NONE if the ray/plane range exceeds this */
    int32_t best_k;                  /* view aggregation (reading Q26; "occlusion-robust best-k"): 0 = mean
                                        over all valid views (Q11); k > 0 = mean of the k lowest per-view costs among
                                        the valid views (all of them if fewer than k are valid) */
} orc_params;

/* O1: unified projective model.  Return 1 = valid, 0 = NONE. */
int orc_project(const orc_camera* c, const double X[3], double uv[2]);
int orc_back_project(const orc_camera* c, double u, double v, double r[3]);
/* angle between the optical axis and the pixel ray (for fragility margins), <0 if NONE */
double orc_pixel_theta(const orc_camera* c, double u, double v);

/* O3: relative pose reference -> view from the rig->camera extrinsics: X_v = R X_ref + T */
void orc_relative_pose(const orc_camera* ref, const orc_camera* view, double R[9], double T[3]);

/* O2: plane table.  s[k] = spacing variable, d[k] = offset, fam[k] = family index.  Returns P. */
int orc_plane_table(const orc_family* fams, int n_fams, double* s, double* d, int32_t* fam, double* nrm /*n_fams*3*/);

/* O4 for one pixel: plane-induced mapping reference pixel -> view pixel.  Return 1 valid / 0 NONE. */
int orc_warp_pixel(const orc_camera* ref, const orc_camera* view, const double n[3], double d,
                   double range_max, double u, double v, double uv[2]);

/* bilinear sample; the caller guarantees 0<=u<W-1, 0<=v<H-1 */
double orc_bilinear(const double* img, int W, int H, double u, double v);

/* O5: matching cost of two equal-size windows: (1 - ZNCC)/2 clamped to [0,1] */
double orc_zncc_cost(const double* a, const double* b, int n, double var_floor);

/*
 * O4-O6: cost volume over the reference raster.
 *   images[c]    : camera c's image as doubles, row-major height x width
 *   cost         : out, P*H*W, +inf where no view is valid (and outside the ROI)
 *   n_eval       : out, number of (pixel, plane, view) with a finite cost
 *   fragile_geom : out (nullable), H*W, 1 where some validity decision feeding this pixel was within its margin
 */
int orc_sweep(const orc_camera* cams, int n_cams, int ref_index, const orc_family* fams, int n_fams,
              const orc_params* prm, const double* const* images, double* cost, int64_t* n_eval,
              uint8_t* fragile_geom);

/* brute force for ONE pixel: recompute every window sample from scratch (no shared warped image). cost_out[P]. */
int orc_pixel_costs(const orc_camera* cams, int n_cams, int ref_index, const orc_family* fams, int n_fams,
                    const orc_params* prm, const double* const* images, int px, int py, double* cost_out);

/*
 * O7-O8: winner-take-all, non-adjacent second best, parabola, depth.
 * Outputs are H*W; outside the ROI / raw-invalid: depth 0, c1=c2=+inf, kbest=-1.
 *   c2raw : plain second-smallest cost (debug / tie detection), +inf if none
 *   delta : sub-plane offset in [-0.5,0.5]; pden: parabola denominator (0 if not refined)
 */
int orc_wta(const orc_camera* ref, const orc_family* fams, int n_fams, const orc_params* prm,
            const double* cost, double* depth, double* c1, double* c2, double* c2raw, int32_t* kbest,
            double* delta, double* pden, uint8_t* raw_valid);

/* S9 + S11: cost filter, ratio filter, mask.  reason[] gets ORC_* codes; depth is zeroed where reason != 0.
 * fragile (nullable) |= 1 where a threshold margin is below its epsilon. */
int orc_filter_mask(int W, int H, const orc_params* prm, const uint8_t* mask /*nullable*/, const uint8_t* raw_valid,
                    const double* c1, const double* c2, double* depth, uint8_t* reason, uint8_t* fragile);

/* S10(a): 2x2 box downsample of an image and of a camera (f/2, c' = (c-0.5)/2) */
/* Local depth-continuity filter, the third filter of PAPER.md:99 ("we compare its depth value against the depths of its
 * neighboring pixels in a local window ... smaller than a threshold gamma ... ratio of the consistent pixels ...
 * smaller than delta"; gamma = 0.5 m, delta = 0.3).  Reading Q25: window x window neighbourhood without
 * the centre; a neighbour is consistent iff it is valid (depth > 0), inside the image and |d_n - d_c| < gamma; the
 * centre is invalidated iff consistent / (window^2 - 1) < delta (exactly delta is kept).  Reads `in` only (never a
 * partially filtered state), then applies the mask (nullable).  out: depth (0 = invalid), reason: 0 kept,
 * ORC_NO_PLANE where the input was invalid, ORC_CONTINUITY, ORC_MASKED. */
int orc_filter_continuity(const double* in, int W, int H, int window, double gamma, double delta,
                          const uint8_t* mask /*nullable*/, double* out, uint8_t* reason);

int orc_downsample2(const double* img, int W, int H, double* out);
void orc_camera_half(const orc_camera* c, orc_camera* out);

/* S10(c)-(e): nearest-neighbour upsample of the low pass and merge with the crop pass.
 * kbest_out gets bit 14 set where the crop pass supplied the value. */
int orc_merge(int W, int H, int crop_x0, int crop_y0, int crop_w, int crop_h,
              const double* depth_lo, const double* c1_lo, const double* c2_lo, const int32_t* k_lo,
              const uint8_t* rv_lo, const double* depth_hi, const double* c1_hi, const double* c2_hi,
              const int32_t* k_hi, const uint8_t* rv_hi, double* depth, double* c1, double* c2, int32_t* kbest,
              uint8_t* raw_valid);

int orc_num_threads(void);

#ifdef __cplusplus
}
#endif
#endif
