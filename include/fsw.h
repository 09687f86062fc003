/*
 * fsw.h -- C ABI of the B200-native fisheye plane-sweeping stereo library (libfsw.so).
 *
 * What it computes: the depth-map estimation stage of arXiv 1809.06132
 * ("Real-time dense mapping for self-driving vehicles using fisheye cameras"),
 * PAPER.md section III-A (lines 69-99): plane-sweeping stereo run directly on
 * the fisheye images through the unified projective camera model (PAPER.md:149,
 * back-projection = Eq. 1), ZNCC matching cost over a w x w
 * window, accumulation over >2 cameras, best depth
 * candidate with first / second best cost, the best-cost and
 * uniqueness-ratio filters, the two-scale strategy
 * and the dynamic-object mask.  Readings of passages the paper
 * leaves open are listed in DESIGN.md.
 *
 * Conventions
 *  - Camera frame: x right, y down, z forward.  Pixel centres at integer
 *    coordinates: I(u,v) for integer u,v is the stored sample; u in [0,W-1].
 *  - Extrinsics are rig->camera: X_cam = R * X_rig + t (R row-major).
 *  - All functions return an int32 status (FSW_OK = 0, negative = error) and
 *    never throw.  fsw_last_error() returns a thread-local message for the last
 *    failing call of the calling thread.
 *  - Geometric failures (pixel outside the field of view, ray parallel to a
 *    plane, projection outside a view image) are VALUES, not errors: they make a
 *    view / plane / pixel invalid.  An invalid depth is exactly 0.0f.
 *  - Every struct starts with `struct_size` (= sizeof the struct as compiled by
 *    the caller) so the ABI can grow.
 *  - "device" pointers are CUDA device memory of the context's device; "host"
 *    pointers are ordinary process memory.  The library never takes ownership of
 *    a caller buffer.
 *  - There is no CPU fallback: without a CUDA device fsw_context_create fails
 *    with FSW_E_CUDA.
 */
#ifndef FSW_H
#define FSW_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define FSW_VERSION_MAJOR 0
#define FSW_VERSION_MINOR 3

/* status codes */
#define FSW_OK 0
#define FSW_E_INVALID_ARG (-1) /* null pointer, bad size, bad enum, struct_size mismatch */
#define FSW_E_CONFIG (-2)      /* arguments are well-formed but describe an impossible rig / plane set */
#define FSW_E_CUDA (-3)        /* a CUDA runtime call failed (message holds cudaGetErrorString) */
#define FSW_E_NOMEM (-4)
#define FSW_E_UNSUPPORTED (-5)

/* limits */
#define FSW_MAX_CAMERAS 8
#define FSW_MAX_PLANES 1024
#define FSW_MAX_FAMILIES 8
#define FSW_MAX_WINDOW 15
#define FSW_MAX_BATCH 256 /* frame sets per fsw_compute_depth_batch call */
#define FSW_STATIC_SCRATCH_BYTES (24u << 20) /* device scratch of fsw_compute_depth_static: 24 MiB per GPU, see there */

/* pixel types of input images */
#define FSW_U8 0  /* uint8 grey levels 0..255 ("gray scale images") */
#define FSW_F32 1 /* float32 intensities, any scale */

/* plane spacing inside a family */
#define FSW_INVERSE 0 /* uniform in 1/d */
#define FSW_LINEAR 1  /* uniform in d   */

/* filters_enabled bits */
#define FSW_FILTER_COST 1  /* invalidate if best cost > alpha(row)            */
#define FSW_FILTER_RATIO 2 /* invalidate if second best < beta * max(best,1e-6) */

/* depth_kind */
#define FSW_DEPTH_RANGE 0 /* Euclidean range along the unit ray (PAPER.md:161-162 integrates along the ray) */
#define FSW_DEPTH_Z 1     /* range * r_z: negative for a ray more than 90 degrees off the optical axis; validity is
                             valid_reason, not the sign (an invalid pixel holds 0) */

/* reason codes written to fsw_depth_out.valid_reason (0 = valid) */
#define FSW_REASON_OK 0
#define FSW_REASON_NO_PLANE 1     /* no plane has a finite cost (outside FOV / ROI / every view invalid) */
#define FSW_REASON_COST_FILTER 2
#define FSW_REASON_RATIO_FILTER 3
#define FSW_REASON_MASKED 4
#define FSW_REASON_CONTINUITY 5   /* fsw_filter_continuity: too few consistent neighbours */

/* bit set in plane_index where the full-resolution crop pass supplied the value (multi-resolution call) */
#define FSW_INDEX_FROM_CROP (1 << 14)

typedef struct fsw_rig fsw_rig;
typedef struct fsw_planeset fsw_planeset;
typedef struct fsw_context fsw_context;

/* One fisheye camera: unified projective (Mei) model.
 * projection: X -> X/|X| on the unit sphere -> m = (X_x, X_y) / (X_z + xi |X|)
 *             -> m_d = m (1 + k1 r^2 + k2 r^4) + tangential(p1,p2), r^2 = |m|^2
 *             -> (u,v) = (fx m_d.x + cx, fy m_d.y + cy);
 * back-projection: undistort, then Eq. 1.  Rays / points further than
 * fov_max_deg/2 from the optical axis are outside the camera (invalid). */
typedef struct fsw_camera {
    uint32_t struct_size;
    int32_t width, height;
    double fx, fy, cx, cy;
    double xi;             /* mirror parameter, 0 <= xi <= 3 */
    double k1, k2, p1, p2; /* distortion on the normalised plane (0 = none) */
    double fov_max_deg;    /* full field of view in degrees, (0, 360] */
    double R[9];           /* rig->camera rotation, row-major, orthonormal within 1e-5 */
    double t[3];           /* rig->camera translation, metres */
} fsw_camera;

/* One family of sweep planes n.X = d_k in the REFERENCE-camera frame (PAPER.md:74:
 * fronto-parallel to the reference image plane, and parallel to the ground).
 * Plane k (0 <= k < n_planes): s_k = s_first + k (s_last - s_first)/(n_planes-1),
 * s = 1/d (FSW_INVERSE) or d (FSW_LINEAR).  Global plane index = families
 * concatenated in call order. */
typedef struct fsw_plane_family {
    uint32_t struct_size;
    double normal[3]; /* need not be unit length; normalised by the library */
    int32_t n_planes; /* >= 1 */
    int32_t spacing;  /* FSW_INVERSE / FSW_LINEAR */
    double d_first, d_last; /* metres; > 0 */
} fsw_plane_family;

typedef struct fsw_rect {
    int32_t x0, y0, w, h;
} fsw_rect;

typedef struct fsw_sweep_params {
    uint32_t struct_size;
    int32_t window;          /* odd, 3..FSW_MAX_WINDOW: side of the ZNCC window (9 full-res, 7 half-res) */
    int32_t subpixel;        /* 1 = three-point parabola over the plane index in the spacing variable */
    int32_t filters_enabled; /* FSW_FILTER_* bits */
    int32_t depth_kind;      /* FSW_DEPTH_RANGE / FSW_DEPTH_Z */
    fsw_rect roi;            /* output region on the reference raster; w <= 0 or h <= 0 = whole image */
    int32_t horizon_row;     /* rows < horizon_row use alpha_upper, others alpha_lower (0.05 / 0.3) */
    float alpha_upper, alpha_lower;
    float beta;      /* keep iff second >= beta * max(best, 1e-6) */
    float var_floor; /* floor of sqrt(var_a var_b) in the ZNCC denominator, in intensity units squared */
    float range_max; /* a ray/plane intersection further than this (metres along the ray) is invalid */
    float* debug_cost_volume; /* device, nullable: [P][H][W] float32, view-averaged cost, +inf = undefined */
    /* Variants (readings Q26, Q27, Q28); 0 = the default behaviour described above.
     * best_k: occlusion-robust view aggregation: the cost of a plane is the mean of the best_k lowest
     *   per-view costs among the valid views (of all valid ones if fewer than best_k are valid) instead of the mean
     *   over all valid views.  Supported: 0 (off), 1, 2; other values give FSW_E_UNSUPPORTED.
     * filter_before_merge (read from params_crop by the multi-resolution calls): each scale is filtered on its own
     *   -- the half-resolution pass with the thresholds of params_low, whose horizon_row counts half-resolution rows
     *   -- and inside the crop the full-resolution estimate wins where it SURVIVED its filters, else a surviving
     *   upsampled estimate fills in; an invalid pixel reports the reason of the estimate the default order would have
     *   taken.
     * upsample_plane (read from params_crop by the multi-resolution calls; the alternative of reading Q18): a
     *   full-resolution pixel that takes the half-resolution estimate does not copy its range but intersects ITS OWN
     *   ray with the refined plane the half-resolution pixel chose (depth = d* / (n.r), times r_z for FSW_DEPTH_Z);
     *   where its ray lies outside the field of view or does not face that plane the pixel is invalid
     *   (FSW_REASON_NO_PLANE).  Costs and index are copied. */
    int32_t best_k;
    int32_t filter_before_merge;
    int32_t upsample_plane;
    int32_t reserved_;
} fsw_sweep_params;

/* one input image: row-major, pitch in BYTES */
typedef struct fsw_image {
    const void* data; /* device pointer (host pointer for fsw_compute_depth*_host) */
    size_t pitch_bytes;
    int32_t dtype; /* FSW_U8 / FSW_F32 */
} fsw_image;

/* output maps, all at the reference camera's full resolution, row-major, pitches in BYTES.
 * depth is required; every other pointer may be NULL. */
typedef struct fsw_depth_out {
    uint32_t struct_size;
    float* depth;        size_t depth_pitch;        /* metres, 0.0f = invalid */
    float* best_cost;    size_t best_cost_pitch;    /* c1, +inf where no plane */
    float* second_cost;  size_t second_cost_pitch;  /* c2 (non-adjacent second best), +inf where no plane */
    int16_t* plane_index; size_t plane_index_pitch; /* winning global plane index, -1 where no plane */
    uint8_t* valid_reason; size_t valid_reason_pitch; /* FSW_REASON_* */
} fsw_depth_out;

typedef struct fsw_counters {
    uint32_t struct_size;
    int64_t n_eval;      /* (pixel, plane, view) triples with a finite matching cost in the last call */
    int64_t n_raw_valid; /* pixels with at least one finite plane cost (before filters / mask) */
    int64_t n_valid;     /* pixels valid after filters and mask */
    int64_t n_launches;  /* CUDA kernels launched by the last call */
    double sweep_ms;     /* device time of the sweep kernel(s) of the last call, CUDA events on the call's stream;
                            -1 unless fsw_context_set_timing(ctx, 1) was in effect */
    int64_t n_split_launches; /* sweep launches of the last call that split their tiles (fsw_context_set_split) */
} fsw_counters;

/* ---- version / errors ---------------------------------------------------- */
int32_t fsw_version(int32_t* major, int32_t* minor);
const char* fsw_last_error(void);

/* ---- rig (host-only, no CUDA needed) ------------------------------------- */
/* cams: host array of n_cams cameras (copied).  2 <= n_cams <= FSW_MAX_CAMERAS; ref_index selects the reference
 * camera; every other camera is a matching view, used in array order.
 * Errors: FSW_E_INVALID_ARG (null, n_cams, ref_index, struct_size), FSW_E_CONFIG (fx,fy <= 0; principal point outside
 * the image; R not orthonormal; xi outside [0,3]; fov outside (0,360]; distortion not invertible inside the FOV). */
int32_t fsw_rig_create(const fsw_camera* cams, int32_t n_cams, int32_t ref_index, fsw_rig** out);
int32_t fsw_rig_destroy(fsw_rig* rig);
/* A rig made of a subset of the cameras of `rig` (the paper evaluates camera configurations with
 * fewer matching views, "3 cameras ... save about 17 % of run time"): cam_indices lists n_cams distinct cameras of
 * `rig` in the order the new rig shall have them; it must contain the reference camera of `rig`, which stays the
 * reference.  The new rig is independent of the old one (destroy both).
 * Errors: FSW_E_INVALID_ARG (null, n_cams outside 2..FSW_MAX_CAMERAS, index out of range or repeated, reference camera
 * missing). */
int32_t fsw_rig_subset(const fsw_rig* rig, const int32_t* cam_indices, int32_t n_cams, fsw_rig** out);
/* relative pose reference -> camera `cam`: X_cam = R X_ref + T (R row-major, 9 doubles; T 3 doubles) */
int32_t fsw_rig_relative_pose(const fsw_rig* rig, int32_t cam, double* R, double* T);
/* a rig-frame direction (e.g. "down" = (0,1,0)) expressed in the reference-camera frame (the ground
 * plane normal comes from the extrinsic calibration) */
int32_t fsw_ground_normal_in_ref(const fsw_rig* rig, const double* dir_rig, double* out);

/* ---- plane set (host-only) ------------------------------------------------ */
/* Errors: FSW_E_INVALID_ARG (null, n_fams outside 1..FSW_MAX_FAMILIES, spacing enum), FSW_E_CONFIG (n_planes < 1,
 * d <= 0, zero normal, total planes > FSW_MAX_PLANES). */
int32_t fsw_planeset_create(const fsw_plane_family* fams, int32_t n_fams, fsw_planeset** out);
int32_t fsw_planeset_destroy(fsw_planeset* ps);
int32_t fsw_planeset_size(const fsw_planeset* ps, int32_t* n_planes);
/* copies out the plane table: s[k] spacing variable, d[k] offset, family[k]; any pointer may be NULL */
int32_t fsw_planeset_table(const fsw_planeset* ps, double* s, double* d, int32_t* family);

/* ---- context (needs a CUDA device) ---------------------------------------- */
/* Owns device-side scratch (footprint images of the views, half-resolution images and maps, tile schedule, work
 * queue, counters).  Scratch is allocated lazily and reused, so one context serves one stream at a time.  All work of
 * a call is ordered on the stream given to it: whatever follows the call on that stream sees its results.  The
 * library launches on no other stream ("no hidden streams"). */
int32_t fsw_context_create(const fsw_rig* rig, int32_t cuda_device, fsw_context** out);
int32_t fsw_context_destroy(fsw_context* ctx);

/* ---- depth for one synchronized frame set ------------------- */
/* images: host array of n_cams fsw_image descriptors in rig order, each `data` a DEVICE pointer to an image of that
 * camera's width x height.  mask: device, nullable, uint8 [H][W] of the reference camera, non-zero = invalidate
 * (PAPER.md:66).  out: device output maps.  Asynchronous: work is enqueued on cuda_stream (a cudaStream_t; NULL =
 * default stream) and the call returns; the caller keeps every buffer alive until the stream reaches this work.
 * Errors: FSW_E_INVALID_ARG (nulls, window even / out of range, pitches too small, dtype enum),
 * FSW_E_CUDA (launch or allocation failure). */
int32_t fsw_compute_depth(fsw_context* ctx, const fsw_planeset* planes, const fsw_sweep_params* params,
                          const fsw_image* images, const uint8_t* mask, size_t mask_pitch,
                          const fsw_depth_out* out, void* cuda_stream);

/* ---- depth for a batch of independent frame sets ---------------------------- */
/* The same computation as fsw_compute_depth for n_sets synchronized frame sets of the same rig (one
 * frame set per timestamp; the sets are independent given the rig and the plane set), enqueued as ONE sweep launch
 * whose persistent thread blocks draw (frame set, tile) work items from a common queue, so that the tiles of one
 * frame set fill the tail of another.  Results are identical to n_sets separate fsw_compute_depth calls.
 * images: host array of n_sets * n_cams descriptors, set-major (images[s * n_cams + c]), device pointers.
 * masks: host array of n_sets device pointers (each nullable), or NULL for no masks; one mask_pitch for all.
 * outs: host array of n_sets output descriptors (device pointers; the sets must not alias each other).
 * 1 <= n_sets <= FSW_MAX_BATCH.  The context's footprint scratch grows to n_sets frame sets (8 bytes per view
 * pixel for 8-bit views, 16 for float views).  params->debug_cost_volume must be NULL unless n_sets == 1.  Asynchronous like fsw_compute_depth.
 * fsw_get_last_counters then reports totals over the batch. */
int32_t fsw_compute_depth_batch(fsw_context* ctx, const fsw_planeset* planes, const fsw_sweep_params* params,
                                int32_t n_sets, const fsw_image* images, const uint8_t* const* masks, size_t mask_pitch,
                                const fsw_depth_out* outs, void* cuda_stream);

/* Two-scale strategy of PAPER.md:88-90: every image is 2x2-box downsampled and swept over the whole field of view
 * with planes_low / params_low (intrinsics f/2, c' = (c-0.5)/2); the result is upsampled (nearest neighbour); the
 * full-resolution images are swept inside `crop` with planes_crop / params_crop; inside the crop the full-resolution
 * estimate wins where it has any finite plane cost, elsewhere the upsampled one is used; then the filters (thresholds
 * of params_crop) and the mask.  plane_index carries FSW_INDEX_FROM_CROP where the crop pass supplied the value. */
int32_t fsw_compute_depth_multires(fsw_context* ctx, const fsw_planeset* planes_low, const fsw_planeset* planes_crop,
                                   const fsw_sweep_params* params_low, const fsw_sweep_params* params_crop,
                                   fsw_rect crop, const fsw_image* images, const uint8_t* mask, size_t mask_pitch,
                                   const fsw_depth_out* out, void* cuda_stream);

/* The two-scale strategy for n_sets independent frame sets of the rig (arguments as in fsw_compute_depth_batch): one
 * downsample launch, ONE half-resolution sweep launch and ONE crop sweep launch for the whole batch, so that the
 * (frame set, tile) queue of the sweep kernel also serves the paper's production path (the multi-scale
 * estimator is what runs in the vehicle).  Results are identical to n_sets separate fsw_compute_depth_multires calls.
 * The context's half-resolution scratch grows to n_sets frame sets. */
int32_t fsw_compute_depth_multires_batch(fsw_context* ctx, const fsw_planeset* planes_low, const fsw_planeset* planes_crop,
                                         const fsw_sweep_params* params_low, const fsw_sweep_params* params_crop,
                                         fsw_rect crop, int32_t n_sets, const fsw_image* images,
                                         const uint8_t* const* masks, size_t mask_pitch, const fsw_depth_out* outs,
                                         void* cuda_stream);

/* ---- depth for one frame set without any allocation ------------------------- */
/* fsw_compute_depth (same arguments, same maps bit for bit, steps S1-S12) for callers that may not
 * allocate device memory: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  The
 * call allocates nothing on the device and nothing pinned (no cudaMalloc, cudaFree, cudaMallocHost): its scratch --
 * the work-queue word, the tile schedule and the footprint images of the matching views (8 bytes per view pixel for
 * 8-bit views, 16 for float views) -- lives in one static device array of FSW_STATIC_SCRATCH_BYTES (24 MiB) inside
 * the library, which every GPU that loads the library holds until the process exits.  The caller passes inputs and
 * outputs as for fsw_compute_depth (device pointers).
 * Limit: 256 + 4 x tiles + the footprint images, each rounded up to 256 bytes, must fit the array -- e.g. two 8-bit
 * views of 1280 x 1024 (21 MB) or four of 1024 x 544 (17.8 MB) do, two float views of 1280 x 1024 do not.  A rig
 * beyond it gets FSW_E_UNSUPPORTED with the sizes in fsw_last_error() and nothing is launched.
 * Sharing: there is ONE array per GPU and every call on that GPU uses it, whatever the context or stream.  Calls that
 * can overlap on the GPU (different streams, or different host threads on different streams) race on it; serialise
 * them on one stream or with events.  The array keeps the last call's contents: the queue word is cleared by the
 * call's own first launch, the footprints and the tile schedule are rewritten by every call (the schedule by a small
 * kernel that takes it as launch parameters, not by a copy: a call is kernel launches only).
 * The sweep runs as one launch of the unsplit kernel (the plane split of fsw_context_set_split needs 48 bytes of
 * state per pixel and is not used), so a single large frame set costs what it costs with FSW_SPLIT_OFF (about a
 * quarter more than the default at 1280 x 1024).  The context's statistics (fsw_get_last_counters) are not updated.  The first call on a
 * device resolves the array's device address (cudaGetSymbolAddress) and the first call with a window size sets the
 * kernels' shared-memory attribute: make one warm-up call before capturing into a graph.  Asynchronous on
 * cuda_stream.  Errors: as fsw_compute_depth, plus FSW_E_UNSUPPORTED (scratch limit, more than 16384 tiles). */
int32_t fsw_compute_depth_static(fsw_context* ctx, const fsw_planeset* planes, const fsw_sweep_params* params,
                                 const fsw_image* images, const uint8_t* mask, size_t mask_pitch,
                                 const fsw_depth_out* out, void* cuda_stream);

/* Same calls with HOST buffers: images[i].data, mask and every pointer of `out` are host memory (pinned memory
 * makes the copies asynchronous).  The library stages them through context-owned device buffers on cuda_stream:
 * host->device copies, the kernels, device->host copies, then synchronizes the stream before returning. */
int32_t fsw_compute_depth_host(fsw_context* ctx, const fsw_planeset* planes, const fsw_sweep_params* params,
                               const fsw_image* images, const uint8_t* mask, size_t mask_pitch,
                               const fsw_depth_out* out, void* cuda_stream);
int32_t fsw_compute_depth_batch_host(fsw_context* ctx, const fsw_planeset* planes, const fsw_sweep_params* params,
                                     int32_t n_sets, const fsw_image* images, const uint8_t* const* masks,
                                     size_t mask_pitch, const fsw_depth_out* outs, void* cuda_stream);
int32_t fsw_compute_depth_multires_host(fsw_context* ctx, const fsw_planeset* planes_low,
                                        const fsw_planeset* planes_crop, const fsw_sweep_params* params_low,
                                        const fsw_sweep_params* params_crop, fsw_rect crop, const fsw_image* images,
                                        const uint8_t* mask, size_t mask_pitch, const fsw_depth_out* out,
                                        void* cuda_stream);
int32_t fsw_compute_depth_multires_batch_host(fsw_context* ctx, const fsw_planeset* planes_low,
                                              const fsw_planeset* planes_crop, const fsw_sweep_params* params_low,
                                              const fsw_sweep_params* params_crop, fsw_rect crop, int32_t n_sets,
                                              const fsw_image* images, const uint8_t* const* masks, size_t mask_pitch,
                                              const fsw_depth_out* outs, void* cuda_stream);

/* on != 0: the *_host calls of this context enqueue their host-to-device copies, kernels and device-to-host copies on
 * the caller's stream and return WITHOUT synchronizing it.  The caller then owns the ordering: the host images, masks
 * and outputs must stay untouched (and should be pinned, or the copies are not asynchronous) until the stream has
 * reached the end of the call.  The staging buffers belong to the context, so calls issued on different streams need
 * different contexts; with two contexts on two streams the copies of one frame-set batch overlap the sweep of the
 * other (bench.py's end-to-end figure does exactly that).  Off by default.  Errors: FSW_E_INVALID_ARG (null). */
int32_t fsw_context_set_host_async(fsw_context* ctx, int32_t on);

/* Load balancing of calls with few frame sets (S0).  The sweep kernel runs one persistent CTA per SM over a queue of
 * (frame set, tile) items, heaviest first by a host estimate of the work of every tile; a single 1280 x 1024 frame set
 * has 176 tiles with work for 148 SMs, and its heaviest tile takes longer than the mean load of an SM.  With the plane
 * split a tile becomes two work items that sweep one half of the planes each (the planes are
 * independent hypotheses) and merge their winner-take-all states; the maps are bit-identical to the unsplit ones.
 * FSW_SPLIT_AUTO (default): when the tiles with work are fewer than three per SM, the heavy tiles at the head of the
 * queue are swept whole and the light ones behind them in halves, how many being chosen to minimise the estimated
 * makespan.  The two groups are two launches on the caller's stream, the second one a programmatic dependent of the
 * first (its thread blocks take the SMs the first launch's blocks leave; it completes after the first); no other
 * stream is involved, and under stream capture the pair is captured like any two launches.
 * FSW_SPLIT_OFF: never; FSW_SPLIT_ON: every tile in halves, one launch.
 * Calls with fewer than two planes are never split.  The context owns 48 bytes of scratch per reference pixel and
 * frame set of a split call.  Errors: FSW_E_INVALID_ARG for a null context or an unknown mode. */
#define FSW_SPLIT_AUTO 0
#define FSW_SPLIT_OFF 1
#define FSW_SPLIT_ON 2
int32_t fsw_context_set_split(fsw_context* ctx, int32_t mode);

/* The schedule FSW_SPLIT_AUTO gives a call (S0; host only, no device needed): the queue order of the tiles of the
 * reference image and how many (tile, frame set) slots at its head are swept whole.  n_blocks: thread blocks of the
 * persistent grid (the SM count of the device a context would run on).  tile_order / tile_weight (HOST, capacity
 * entries each, may be NULL with capacity 0): tile index ty * n_tiles_x + tx and estimated work, in plane passes, of
 * the first min(capacity, n_tiles) tiles of the queue.  The estimate orders the queue and sizes the split; it decides
 * nothing about the maps.  Errors: FSW_E_INVALID_ARG. */
typedef struct fsw_schedule_plan {
    uint32_t struct_size;
    int32_t tile_w, tile_h;   /* tile size of the window's kernel geometry */
    int32_t n_tiles_x, n_tiles;
    int32_t n_live;           /* tiles with work (inside the region of interest and the image circle) */
    int32_t by_weight;        /* 1: heaviest tile first (short queues); 0: nearest to the principal point first */
    int64_t n_whole_slots;    /* slots at the head of the queue swept whole; n_tiles * n_sets = no split */
    int64_t n_halved_slots;   /* the rest: two work items each */
} fsw_schedule_plan;
int32_t fsw_plan_schedule(const fsw_rig* rig, const fsw_planeset* planes, const fsw_sweep_params* params, int32_t n_sets,
                          int32_t n_blocks, int32_t capacity, int32_t* tile_order, float* tile_weight,
                          fsw_schedule_plan* out);

/* Part of the statistics call below (SURVEY.md 8(b) "stats ... for benches only"): on != 0 makes every following
 * compute call bracket its sweep kernel launches (the dominant kernels, S1-S12) with a pair of CUDA events on the
 * call's stream so that fsw_get_last_counters can report their device time (the roofline record of bench.py needs the
 * duration of that kernel alone, measured on the stream it is launched on).  Off by default (two event records per
 * call); it changes no result. */
int32_t fsw_context_set_timing(fsw_context* ctx, int32_t on);

/* Counters of the most recent compute call on this context.  Synchronizes the stream that call used. */
int32_t fsw_get_last_counters(fsw_context* ctx, fsw_counters* out);

/* ---- local depth-continuity filter ------------------------------------------ */
/* The third filter of PAPER.md:99: a pixel's depth is held against the depths around it in a local window; a
 * neighbour whose depth differs by less than gamma counts as consistent with the centre, and the centre is rejected
 * when the consistent share of the window falls below delta (the paper states gamma = 0.5 m and delta = 0.3).  The
 * mask follows.
 * Reading Q25: window x window neighbourhood (odd, 3..FSW_MAX_WINDOW; SPEC.md proposes 5) without the
 * centre; a neighbour is consistent iff it is valid (depth > 0), inside the image and |d_n - d_c| < gamma (compared in
 * double precision); the centre is invalidated iff consistent / (window^2 - 1) < delta, decided in double precision
 * with gamma and delta as given (they are doubles in this ABI: delta = 0.3 with a 9 x 9 window keeps a centre with
 * exactly 24 consistent neighbours of 80, which a float 0.3f > 0.3 would reject).  Only depth_in is read (never a
 * partially filtered state), so depth_out must not overlap depth_in.
 * depth_in / depth_out: device, float32, reference-camera size of the context's rig, pitches in BYTES, 0.0f = invalid.
 * Call fsw_compute_depth* WITHOUT a mask and pass the mask here (nullable): the mask comes after the filters.
 * reason_out (device, nullable, uint8): FSW_REASON_OK, FSW_REASON_NO_PLANE where depth_in was invalid,
 * FSW_REASON_CONTINUITY, FSW_REASON_MASKED.  Asynchronous on cuda_stream.
 * Errors: FSW_E_INVALID_ARG (null pointers, even / out-of-range window, gamma <= 0, delta outside [0,1], pitches too
 * small, overlapping depth buffers), FSW_E_CUDA. */
int32_t fsw_filter_continuity(fsw_context* ctx, const float* depth_in, size_t depth_in_pitch, int32_t window,
                              double gamma, double delta, const uint8_t* mask, size_t mask_pitch,
                              float* depth_out, size_t depth_out_pitch, uint8_t* reason_out, size_t reason_pitch,
                              void* cuda_stream);

/* ---- TSDF consumer of the depth maps (section III-C) ------------------------ */
/* A local map of fixed size around the vehicle (60 m x 60 m x 3 m) as a dense torus of 8^3-voxel blocks on
 * the device: every voxel holds the running average D(X) of the truncated signed distance (in units of mu, |D| <= 1)
 * and its observation count w(X) (Eq. 2); every block a state and the number of frames that updated
 * it.  Readings where the paper is silent are DESIGN.md T1-T6 (blocks of 8^3 voxels, voxel centres at (index + 0.5)
 * voxel_size, the depth map stores range along the ray and eta is taken against |X_d|, nearest-pixel depth lookup, the
 * box is snapped to whole blocks).  World coordinates are metres in any fixed frame; poses are world -> camera. */
typedef struct fsw_tsdf fsw_tsdf;

typedef struct fsw_tsdf_params {
    uint32_t struct_size;
    float voxel_size;  /* metres (the paper uses 0.05) */
    float mu;          /* truncation distance, metres (unstated in the paper; SPEC.md proposes 0.2) */
    int32_t w_max;     /* cap of the observation count ("capped to a fixed maximum value") */
    float box_size[3]; /* extent of the local map, metres; rounded up to whole blocks of 8 voxels */
} fsw_tsdf_params;

typedef struct fsw_tsdf_stats {
    uint32_t struct_size;
    int64_t n_new_blocks;     /* blocks allocated by the last fsw_tsdf_integrate */
    int64_t n_visible_blocks; /* allocated blocks of the local map during the last fsw_tsdf_integrate */
    int64_t n_voxels_updated; /* voxels that Eq. 2 updated in the last fsw_tsdf_integrate */
    int64_t n_points;         /* points found by the last fsw_tsdf_extract_points (may exceed its capacity) */
    int64_t n_blocks_freed;   /* blocks that left the box in the last fsw_tsdf_recentre */
    int64_t n_frames;         /* depth maps integrated so far */
} fsw_tsdf_stats;

/* Allocates the local map centred at centre[3] (metres; the box is snapped so that the block that contains the centre
 * is the middle block).  Errors: FSW_E_INVALID_ARG, FSW_E_CONFIG (more than 2^26 blocks), FSW_E_CUDA, FSW_E_NOMEM.
 * The TSDF calls keep their own thread-local error text: fsw_tsdf_last_error. */
int32_t fsw_tsdf_create(int32_t cuda_device, const fsw_tsdf_params* params, const double* centre, fsw_tsdf** out);
int32_t fsw_tsdf_destroy(fsw_tsdf* vol);
const char* fsw_tsdf_last_error(void);
/* integer block coordinate of the box's first block and the number of blocks per axis (host ints, 3 each) */
int32_t fsw_tsdf_box(const fsw_tsdf* vol, int32_t* block_origin, int32_t* blocks);
/* Moves the box to a new centre ("we only allocate new voxel blocks within this region and swap old blocks that are
 * no longer in this region"): blocks whose world coordinate leaves the box are freed (their content is
 * dropped, nothing is archived), the others keep their content.  Asynchronous on cuda_stream. */
int32_t fsw_tsdf_recentre(fsw_tsdf* vol, const double* centre, void* cuda_stream);
/* One depth map: allocation along [d - mu, d + mu] of the Eq. 1 ray of every valid pixel, the list
 * of the frame's blocks, Eq. 2 for every voxel of those blocks.  cam: intrinsics, distortion and
 * field of view of the depth camera (its R, t are ignored); R (9, row-major), t (3): world -> camera, X_d = R X + t,
 * host doubles; depth: DEVICE, float32 [height][width] of that camera, pitch in bytes, range along the pixel ray in
 * metres, <= 0 = invalid (the maps fsw_compute_depth* writes with FSW_DEPTH_RANGE).  Asynchronous on cuda_stream; the
 * depth map must stay alive until the stream reaches this work. */
int32_t fsw_tsdf_integrate(fsw_tsdf* vol, const fsw_camera* cam, const double* R, const double* t, const float* depth,
                           size_t depth_pitch, void* cuda_stream);
/* Points of the map: zero crossings of D between axis neighbours that both carry weight, in blocks with at least
 * min_block_observations updates ("we only consider voxel blocks with at least 3 observations"), placed
 * by linear interpolation; points: DEVICE, capacity x 3 floats (x, y, z in metres RELATIVE TO THE BOX ORIGIN =
 * block_origin x 8 x voxel_size), in no particular order; the count is in fsw_tsdf_get_stats. */
int32_t fsw_tsdf_extract_points(fsw_tsdf* vol, int32_t min_block_observations, float* points, int32_t capacity, void* cuda_stream);
/* synchronizes the stream of the last TSDF call */
int32_t fsw_tsdf_get_stats(fsw_tsdf* vol, fsw_tsdf_stats* out);
/* Dense copy of the local map in box order, for inspection and tests: tsdf / weight DEVICE float32
 * [blocks_z*8][blocks_y*8][blocks_x*8], observations int32 / allocated uint8 [blocks_z][blocks_y][blocks_x]. */
int32_t fsw_tsdf_download(fsw_tsdf* vol, float* tsdf, float* weight, int32_t* observations, uint8_t* allocated, void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* FSW_H */
