/*
 * fsw_internal.h -- device-side argument blocks shared by the host API (fsw_api.cu) and the kernels.
 * Not part of the public ABI (that is include/fsw.h).  Notation follows SURVEY.md section 8(a): S1..S12.
 */
#ifndef FSW_INTERNAL_H
#define FSW_INTERNAL_H

#include <cuda_runtime.h>
#include <stdint.h>

#include "fsw.h"

#define FSW_MAX_VIEWS (FSW_MAX_CAMERAS - 1)

/* thresholds of the geometric validity decisions (the oracle states the same values; they are the paper-silent
 * readings Q3/Q17 of DESIGN.md) */
#define FSW_EPS_DEN 1e-9f /* projection denominator must exceed this times rho */
#define FSW_EPS_Q 1e-9f   /* ray/plane incidence n.r must exceed this */

/* distortion mode of a camera */
#define FSW_DIST_NONE 0
#define FSW_DIST_K1 1   /* k1 only */
#define FSW_DIST_FULL 2 /* k1,k2,p1,p2 */

/* how a view image is stored on the device */
#define FSW_PIX_FOOT_U8 0 /* footprint-packed: word(x,y) = I(x,y) | I(x+1,y)<<8 | I(x,y+1)<<16 | I(x+1,y+1)<<24 */
#define FSW_PIX_F32 1     /* plain float32, pitch in elements */

struct FswDevCam {
    float fx, fy, cx, cy, xi;
    float k1, k2, p1, p2;
    float cos_fov; /* cos(fov_max/2) */
    int32_t W, H;
    int32_t dist_mode;
};

struct FswDevView {
    FswDevCam cam;
    float R[9]; /* reference -> view: X_v = R X_ref + T */
    float T[3];
    int32_t ident_R;  /* 1 if R is exactly the identity */
    int32_t pix_mode; /* FSW_PIX_* */
    const void* img;
    int64_t pitch_elems; /* row pitch in elements (uint32 words or floats) */
};

struct FswDevFamily {
    float n[3];
    int32_t first, count; /* global index of the first plane, number of planes */
    int32_t spacing;
    float s0, ds; /* spacing variable of plane j in the family: s0 + j*ds */
};

struct FswSweepArgs {
    /* S1: reference camera and image */
    FswDevCam ref;
    const void* ref_img;
    int64_t ref_pitch_bytes;
    int32_t ref_dtype; /* FSW_U8 / FSW_F32 */
    /* S3/S4: matching views, fixed order */
    int32_t n_views;
    FswDevView views[FSW_MAX_VIEWS];
    /* S2: planes */
    int32_t n_fams;
    int32_t n_planes;
    FswDevFamily fam[FSW_MAX_FAMILIES];
    float inv_d[FSW_MAX_PLANES]; /* 1/d_k of every global plane */
    /* parameters */
    int32_t roi_x0, roi_y0, roi_x1, roi_y1; /* clipped to the image, half-open */
    int32_t subpixel, filters, depth_kind, horizon_row;
    float alpha_upper, alpha_lower, beta;
    float floor2;        /* (var_floor * N^2)^2, the floor applied to (N^2 var_a)(N^2 var_b) */
    float inv_range_max; /* 1/range_max */
    float* debug_cost;   /* [P][H][W] or null */
    /* S10 merge input (crop pass of the multi-resolution call): half-resolution raw maps, or null */
    const float* lo_depth;
    const float* lo_c1;
    const float* lo_c2;
    const int16_t* lo_k;
    int32_t lo_W, lo_H;
    int32_t index_flag; /* OR-ed into the plane index this pass writes (FSW_INDEX_FROM_CROP or 0) */
    /* S11 */
    const uint8_t* mask;
    int64_t mask_pitch;
    /* S12 outputs (device) */
    float* out_depth;   int64_t out_depth_pitch;
    float* out_c1;      int64_t out_c1_pitch;
    float* out_c2;      int64_t out_c2_pitch;
    int16_t* out_k;     int64_t out_k_pitch;
    uint8_t* out_reason; int64_t out_reason_pitch;
    /* counters: [0] n_eval, [1] n_raw_valid, [2] n_valid ([1],[2] only if count_pixels) */
    unsigned long long* counters;
    int32_t count_pixels;
};

/* launchers implemented in the .cu files; all enqueue on `stream` and return the launch status */
cudaError_t fsw_launch_sweep(const FswSweepArgs& args, int window, cudaStream_t stream);
cudaError_t fsw_sweep_prepare(int window); /* sets the dynamic shared memory attribute of that instantiation */

struct FswPackArgs {
    int32_t n;
    const uint8_t* src[FSW_MAX_CAMERAS];
    int64_t src_pitch[FSW_MAX_CAMERAS];
    uint32_t* dst[FSW_MAX_CAMERAS];
    int32_t W[FSW_MAX_CAMERAS], H[FSW_MAX_CAMERAS];
    unsigned long long* counters_to_zero; /* nullable: the first thread clears 4 counters */
};
cudaError_t fsw_launch_pack_footprints(const FswPackArgs& args, cudaStream_t stream);

struct FswDownArgs {
    int32_t n;
    const void* src[FSW_MAX_CAMERAS];
    int64_t src_pitch[FSW_MAX_CAMERAS];
    int32_t dtype[FSW_MAX_CAMERAS];
    float* dst[FSW_MAX_CAMERAS]; /* [H/2][W/2] dense */
    int32_t W[FSW_MAX_CAMERAS], H[FSW_MAX_CAMERAS];
    unsigned long long* counters_to_zero;
};
cudaError_t fsw_launch_downsample(const FswDownArgs& args, cudaStream_t stream);

cudaError_t fsw_launch_ffma_peak(float* sink, int blocks, int iters, cudaStream_t stream);

#endif
