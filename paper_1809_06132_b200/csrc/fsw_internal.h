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

/* internal depth_kind of the half-resolution pass under plane-consistent upsampling: write the refined plane offset */
#define FSW_DEPTH_PLANE_OFFSET 2

/* Footprint image of a matching view (S4): four numbers per pixel (x,y),
 *   .x = I(x,y), .y = I(x+1,y) - I(x,y), .z = I(x,y+1), .w = I(x+1,y+1) - I(x,y+1)
 * so that one load fetches everything a bilinear sample needs:
 *   top = .x + au*.y, bot = .z + au*.w, b = top + av*(bot - top).
 * Stored as four floats (128-bit load), or -- when every view of the call is an 8-bit image -- as four bfloat16
 * (64-bit load: integers up to 256 and their differences are exact in bfloat16; half the cache footprint).
 * Built per frame set by pack_footprints_kernel (fsw_aux.cu) from 8-bit or float images; dense, pitch = W. */

struct FswDevCam {
    float fx, fy, cx, cy, xi;
    float k1, k2, p1, p2;
    float cos_fov;     /* cos(fov_max/2) */
    float cos_fov_xi;  /* cos(fov_max/2) + xi: the FOV test on cos(theta) + xi */
    int32_t W, H;
    int32_t Wm1, Hm1;  /* W - 1, H - 1: a bilinear footprint starts at 0 <= floor(u) < W - 1, 0 <= floor(v) < H - 1 */
    int32_t dist_mode;
};

struct FswDevView {
    FswDevCam cam;
    float R[9]; /* reference -> view: X_v = R X_ref + T */
    float T[3];
    int32_t ident_R;  /* 1 if R is exactly the identity */
};

struct FswDevFamily {
    float n[3];
    int32_t first, count; /* global index of the first plane, number of planes */
    int32_t spacing;
    float s0, ds; /* spacing variable of plane j in the family: s0 + j*ds */
};

/* the buffers of one synchronized frame set */
struct FswSetPtrs {
    /* S1: reference image */
    const void* ref_img;
    int64_t ref_pitch_bytes;
    int32_t ref_dtype; /* FSW_U8 / FSW_F32 */
    int32_t pad_;
    /* S4: footprint images of the matching views, fixed view order, pitch = view width */
    const void* foot[FSW_MAX_VIEWS];
    float* debug_cost; /* [P][H][W] or null */
    /* S10 merge input (crop pass of the multi-resolution call): half-resolution raw maps, or null */
    const float* lo_depth;
    const float* lo_c1;
    const float* lo_c2;
    const int16_t* lo_k;
    const uint8_t* lo_reason; /* filter-before-merge order: verdicts of the half-resolution pass, else null */
    /* S11 */
    const uint8_t* mask;
    int64_t mask_pitch;
    /* S12 outputs (device) */
    float* out_depth;   int64_t out_depth_pitch;
    float* out_c1;      int64_t out_c1_pitch;
    float* out_c2;      int64_t out_c2_pitch;
    int16_t* out_k;     int64_t out_k_pitch;
    uint8_t* out_reason; int64_t out_reason_pitch;
};

#define FSW_VARIANT_PROGRAMMATIC 0x100 /* flag added to a kernel variant: programmatic dependent launch */

struct FswSweepArgs {
    FswDevCam ref;
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
    float floor2;        /* (var_floor * N)^2, the floor applied to (N var_a)(N var_b) */
    float inv_range_max; /* 1/range_max */
    float inv_count[FSW_MAX_CAMERAS]; /* 1/c for c valid views (S6: mean over the valid views) */
    float ref_rd2_max;   /* squared distorted normalised radius beyond which no reference pixel is inside the FOV
                            (+inf when the bound does not apply): tiles entirely beyond it skip S1 */
    int32_t lo_W, lo_H;
    int32_t foot_f16;   /* 1: the footprint images hold four bfloat16 per pixel, 0: four floats */
    int32_t best_k;       /* 0: mean over the valid views; 1, 2: mean of the lowest one / two per-view costs (run-time
                             view loop only) */
    int32_t filter_first; /* crop pass of a multi-resolution call in the filter-before-merge order */
    /* plane-consistent upsampling (crop pass): the half-resolution pass wrote plane offsets d* instead of ranges;
     * normals and first plane index of ITS families */
    int32_t upsample_plane, n_lo_fams;
    float lo_fam_n[FSW_MAX_FAMILIES][3];
    int32_t lo_fam_first[FSW_MAX_FAMILIES];
    int32_t views_inside; /* 1: the field of view of every view lies inside its image (no border test needed) */
    int32_t index_flag; /* OR-ed into the plane index this pass writes (FSW_INDEX_FROM_CROP or 0) */
    /* frame sets: set0 inline for the single-set calls, `sets` (device array) for batches */
    int32_t n_sets;
    FswSetPtrs set0;
    const FswSetPtrs* sets;
    /* work queue: items = n_sets * n_tiles, item i -> set i % n_sets, tile tile_order[i / n_sets] */
    const int32_t* tile_order; /* device, n_tiles entries: tile index ty * n_tiles_x + tx, heaviest first */
    int32_t n_tiles_x, n_tiles;
    int32_t slot_first, slot_count; /* split launches: the (tile, set) slots of the queue order the launch covers */
    unsigned int* queue; /* zero before the launch; CTAs claim items beyond gridDim.x from it */
    /* plane split (single frame sets do not fill the persistent grid: 176 live tiles of a 1280 x 1024 frame for 148
     * CTAs): with split = 1 a (set, tile) slot is two work items, item half 0 sweeps the planes [0, split_k) in
     * ascending order, half 1 the planes [split_k, P) in descending order; the half that finishes first leaves its
     * winner-take-all state in split_state ([n_sets][6][H][W] floats), the other one merges it into its registers
     * and runs S8-S12.  split_ticket: one word per (set, tile), zero before and after the launch. */
    int32_t split, split_k;
    int32_t split_whole;    /* the first split_whole (tile, set) slots of the queue are swept whole, the rest in halves */
    int32_t split_adjacent; /* planes split_k - 1 and split_k belong to the same family */
    float* split_state;
    unsigned int* split_ticket;
    /* counters: [0] n_eval, [1] n_raw_valid, [2] n_valid ([1],[2] only if count_pixels) */
    unsigned long long* counters;
    int32_t count_pixels;
};

/* geometry of the sweep kernel's tiles; fsw_api.cu needs it for the tile order and the grid */
struct FswSweepGeometry {
    int32_t tile_w, tile_h, threads, ctas_per_sm;
    size_t smem_bytes;
};

/* launchers implemented in the .cu files; all enqueue on `stream` and return the launch status */
#define FSW_PACK_MAX 64 /* images per pack launch */
struct FswPackArgs {
    int32_t n; /* images to pack in this launch (views of one or several frame sets), all W x H */
    int32_t W, H;
    const void* src[FSW_PACK_MAX];
    int64_t src_pitch[FSW_PACK_MAX]; /* bytes */
    int32_t dtype[FSW_PACK_MAX];
    void* dst[FSW_PACK_MAX];         /* dense [H][W] footprints */
    int32_t f16;                     /* 1: four bfloat16 per footprint (8 bytes), 0: four floats (16 bytes) */
    unsigned int* words_to_zero;     /* nullable: the first threads clear n_words_to_zero 32-bit words (queue, counters) */
    int32_t n_words_to_zero;
};
cudaError_t fsw_launch_pack_footprints(const FswPackArgs& args, cudaStream_t stream);

struct FswDownArgs {
    int32_t n; /* images of this launch (the cameras of one or several frame sets), at most FSW_PACK_MAX */
    const void* src[FSW_PACK_MAX];
    int64_t src_pitch[FSW_PACK_MAX];
    int32_t dtype[FSW_PACK_MAX];
    float* dst[FSW_PACK_MAX]; /* [H/2][W/2] dense */
    int32_t W[FSW_PACK_MAX], H[FSW_PACK_MAX];
};
cudaError_t fsw_launch_downsample(const FswDownArgs& args, cudaStream_t stream);

struct FswContinuityArgs {
    const float* in; int64_t in_pitch;     /* bytes */
    float* out; int64_t out_pitch;
    const uint8_t* mask; int64_t mask_pitch;
    uint8_t* reason; int64_t reason_pitch;
    int32_t W, H, window;
    double gamma, delta;
};
cudaError_t fsw_launch_continuity(const FswContinuityArgs& args, cudaStream_t stream);

#endif
