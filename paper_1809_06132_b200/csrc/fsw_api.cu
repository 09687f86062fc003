/*
 * fsw_api.cu -- the C ABI of include/fsw.h: handle lifecycle, argument validation, host precompute (S0 of
 * relative poses, plane tables, half-resolution intrinsics) and kernel launches.
 * The host never touches pixels: every step S1..S12 runs in the kernels of fsw_sweep.cuh / fsw_aux.cu.
 */
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>
#include <algorithm>
#include <array>
#include <functional>
#include <mutex>
#include <queue>
#include <vector>

#include "fsw_internal.h"

/* fsw_sweep_dispatch.cu: the sweep-kernel instantiations, one object per (window, view count) */
cudaError_t fsw_launch_sweep(int window, const FswSweepArgs& args, int variant, int grid, cudaStream_t stream);
cudaError_t fsw_prepare_sweep(int window, int n_views);
FswSweepGeometry fsw_sweep_geometry(int window, int n_views);

namespace {

thread_local char g_err[512] = "";

int32_t fail(int32_t code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

int32_t cuda_fail(cudaError_t e, const char* what) {
    return fail(FSW_E_CUDA, "%s: %s", what, cudaGetErrorString(e));
}

#define FSW_CUDA(call)                                        \
    do {                                                      \
        cudaError_t e__ = (call);                             \
        if (e__ != cudaSuccess) return cuda_fail(e__, #call); \
    } while (0)

struct DeviceGuard {
    int prev = -1;
    bool changed = false;
    cudaError_t enter(int dev) {
        cudaError_t e = cudaGetDevice(&prev);
        if (e != cudaSuccess) return e;
        if (prev != dev) {
            e = cudaSetDevice(dev);
            changed = (e == cudaSuccess);
        }
        return e;
    }
    ~DeviceGuard() {
        if (changed) cudaSetDevice(prev);
    }
};

struct DevBuf {
    void* p = nullptr;
    size_t bytes = 0;
    cudaError_t reserve(size_t n) {
        if (n <= bytes) return cudaSuccess;
        if (p) cudaFree(p);
        p = nullptr;
        bytes = 0;
        cudaError_t e = cudaMalloc(&p, n);
        if (e == cudaSuccess) bytes = n;
        return e;
    }
    void release() {
        if (p) cudaFree(p);
        p = nullptr;
        bytes = 0;
    }
};

}  // namespace

struct fsw_rig {
    int32_t n_cams, ref_index;
    fsw_camera cams[FSW_MAX_CAMERAS];
    double Rrel[FSW_MAX_CAMERAS][9]; /* reference -> camera c */
    double Trel[FSW_MAX_CAMERAS][3];
};

struct fsw_planeset {
    int32_t n_fams, n_planes;
    fsw_plane_family fams[FSW_MAX_FAMILIES]; /* normals normalised */
    int32_t first[FSW_MAX_FAMILIES];
    std::vector<double> s, d;
    std::vector<int32_t> family;
};

/* scheduling order of the tiles of one (image size, tile shape, principal point) combination, on the device */
struct TileOrder {
    uint64_t key;               /* hash of everything the tile weights depend on (tile_order_key) */
    int32_t n_tiles_x, n_tiles;
    int32_t n_live;             /* tiles with work; they come first, heaviest first */
    std::vector<float> weight;  /* estimated work of the tiles in queue order, in plane passes */
    std::vector<int32_t> order_w, order_d; /* host copies of the two orders (dev, dev_dist) */
    std::vector<std::array<int64_t, 3>> whole_for; /* cache of split_whole_for: (n_sets, slots) -> whole slots */
    DevBuf dev;      /* heaviest first: the order of calls with few frame sets (the split regime) */
    DevBuf dev_dist; /* nearest to the principal point first: the order of long queues */
};

/* words of the control block: [0], [1] work queues of the sweep launches, [2..9] four 64-bit counters */
#define FSW_CTRL_WORDS 10
#define FSW_QUEUE_WORDS 2 /* [0] queue of the (first) sweep launch, [1] queue of the launch of the halved tiles */

struct fsw_context {
    fsw_rig rig;
    int32_t device;
    int32_t n_sm = 0;
    std::vector<DevBuf> foot;      /* footprint images of the views: [set slot][camera] */
    std::vector<DevBuf> half;      /* half-resolution float images: [set slot][camera] */
    std::vector<DevBuf> half_foot; /* ... and their footprint images */
    std::vector<DevBuf> lo_depth, lo_c1, lo_c2, lo_k, lo_reason; /* maps of the half-resolution pass: [set slot] */
    DevBuf ctrl;                   /* FSW_CTRL_WORDS x uint32 */
    DevBuf sets_dev, sets_dev2;    /* FswSetPtrs of a batch (second table: the crop pass of a multi-resolution batch) */
    /* host side of the set table: a ring of pinned buffers, each guarded by an event recorded after its upload, so
     * that the upload is a true asynchronous copy (a pageable source would make cudaMemcpyAsync wait for the stream) */
    static constexpr int N_SET_STAGE = 4;
    FswSetPtrs* sets_pinned[N_SET_STAGE] = {nullptr, nullptr, nullptr, nullptr};
    size_t sets_pinned_cap[N_SET_STAGE] = {0, 0, 0, 0};
    cudaEvent_t sets_ev[N_SET_STAGE] = {nullptr, nullptr, nullptr, nullptr};
    int sets_next = 0;
    DevBuf split_state;            /* plane split: [set][half][6][H][W] floats */
    DevBuf split_ticket;           /* plane split: one word per (set, tile), zero between launches */
    int32_t split_mode = FSW_SPLIT_AUTO;
    bool host_async = false;       /* the *_host calls return without synchronizing their stream */
    int64_t last_split = 0;        /* sweep launches of the last call that split their tiles */
    std::vector<TileOrder*> orders;
    /* staging for the *_host calls: [set slot] */
    std::vector<DevBuf> st_img, st_mask, st_depth, st_c1, st_c2, st_k, st_reason;
    cudaStream_t last_stream = nullptr;
    int64_t last_launches = 0;
    bool timing = false, timed = false;
    cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr}; /* [0,1] around the (crop) sweep, [2,3] around the low sweep */
    int n_timed = 0;
    bool prepared[FSW_MAX_WINDOW + 1] = {false};
    unsigned int* queue() { return (unsigned int*)ctrl.p; }
    unsigned long long* counters() { return (unsigned long long*)((unsigned int*)ctrl.p + 2); }
};

namespace {

/* ---- host precompute (S0) ------------------------------------------------------------------------------------ */
void relative_pose(const fsw_camera& ref, const fsw_camera& view, double* R, double* T) {
    /* "known relative poses" of PAPER.md:70 from the rig->camera extrinsics: where the reference camera sits in the
     * view's frame.  Its optical centre is at o = -R_ref^T t_ref in the rig; seen from the view that is T = R_v o + t_v.
     * Its axes are the rows of R_ref; column j of the relative rotation is the view's image of axis j. */
    double o[3];
    for (int j = 0; j < 3; ++j) o[j] = -(ref.R[j] * ref.t[0] + ref.R[3 + j] * ref.t[1] + ref.R[6 + j] * ref.t[2]);
    for (int i = 0; i < 3; ++i) {
        const double* rv = &view.R[3 * i];
        T[i] = rv[0] * o[0] + rv[1] * o[1] + rv[2] * o[2] + view.t[i];
        for (int j = 0; j < 3; ++j) {
            const double* axis = &ref.R[3 * j];
            R[3 * i + j] = rv[0] * axis[0] + rv[1] * axis[1] + rv[2] * axis[2];
        }
    }
}

int32_t check_camera(const fsw_camera& c, int idx) {
    if (c.struct_size != sizeof(fsw_camera)) return fail(FSW_E_INVALID_ARG, "camera %d: struct_size %u != %zu", idx, c.struct_size, sizeof(fsw_camera));
    if (c.width < 2 || c.height < 2 || c.width > 32768 || c.height > 32768) return fail(FSW_E_CONFIG, "camera %d: image size %dx%d", idx, c.width, c.height);
    if (!(c.fx > 0.0) || !(c.fy > 0.0)) return fail(FSW_E_CONFIG, "camera %d: focal lengths must be positive", idx);
    if (!(c.cx >= 0.0 && c.cx <= c.width - 1 && c.cy >= 0.0 && c.cy <= c.height - 1))
        return fail(FSW_E_CONFIG, "camera %d: principal point (%g,%g) outside the image", idx, c.cx, c.cy);
    if (!(c.xi >= 0.0 && c.xi <= 3.0)) return fail(FSW_E_CONFIG, "camera %d: xi=%g outside [0,3]", idx, c.xi);
    if (!(c.fov_max_deg > 0.0 && c.fov_max_deg <= 360.0)) return fail(FSW_E_CONFIG, "camera %d: fov_max_deg=%g outside (0,360]", idx, c.fov_max_deg);
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {
            double s = 0.0;
            for (int k = 0; k < 3; ++k) s += c.R[3 * i + k] * c.R[3 * j + k];
            if (std::fabs(s - (i == j ? 1.0 : 0.0)) > 1e-5) return fail(FSW_E_CONFIG, "camera %d: R is not orthonormal", idx);
        }
    double det = c.R[0] * (c.R[4] * c.R[8] - c.R[5] * c.R[7]) - c.R[1] * (c.R[3] * c.R[8] - c.R[5] * c.R[6]) +
                 c.R[2] * (c.R[3] * c.R[7] - c.R[4] * c.R[6]);
    if (!(det > 0.0)) return fail(FSW_E_CONFIG, "camera %d: R is a reflection", idx);
    for (int i = 0; i < 3; ++i)
        if (!std::isfinite(c.t[i])) return fail(FSW_E_CONFIG, "camera %d: t is not finite", idx);
    /* the distortion must be invertible over the field of view: d/drho [rho (1 + k1 rho^2 + k2 rho^4)] > 0 up to
     * the normalised radius of the FOV edge (radial part; the tangential part is assumed small) */
    if (c.k1 != 0.0 || c.k2 != 0.0 || c.p1 != 0.0 || c.p2 != 0.0) {
        double th = 0.5 * c.fov_max_deg * M_PI / 180.0;
        double den = std::cos(th) + c.xi;
        if (!(den > 1e-6)) return fail(FSW_E_CONFIG, "camera %d: distortion given but the FOV edge maps to infinity on the normalised plane", idx);
        double rmax = std::sin(th) / den;
        for (int i = 0; i <= 256; ++i) {
            double r = rmax * i / 256.0, r2 = r * r;
            if (!(1.0 + 3.0 * c.k1 * r2 + 5.0 * c.k2 * r2 * r2 > 1e-3))
                return fail(FSW_E_CONFIG, "camera %d: radial distortion is not monotone inside the field of view", idx);
        }
    }
    return FSW_OK;
}

FswDevCam dev_cam(const fsw_camera& c, bool half) {
    FswDevCam d;
    double fx = c.fx, fy = c.fy, cx = c.cx, cy = c.cy;
    int W = c.width, H = c.height;
    if (half) { /* S10(a): 2x2 box downsample => f/2, c' = (c - 0.5)/2: low-res centre i <-> full-res 2i + 0.5 */
        fx *= 0.5; fy *= 0.5; cx = (cx - 0.5) * 0.5; cy = (cy - 0.5) * 0.5; W /= 2; H /= 2;
    }
    d.fx = (float)fx; d.fy = (float)fy; d.cx = (float)cx; d.cy = (float)cy; d.xi = (float)c.xi;
    d.k1 = (float)c.k1; d.k2 = (float)c.k2; d.p1 = (float)c.p1; d.p2 = (float)c.p2;
    d.cos_fov = (float)std::cos(0.5 * c.fov_max_deg * M_PI / 180.0);
    d.cos_fov_xi = (float)(std::cos(0.5 * c.fov_max_deg * M_PI / 180.0) + c.xi);
    d.W = W; d.H = H;
    d.Wm1 = W - 1; d.Hm1 = H - 1;
    if (c.k1 == 0.0 && c.k2 == 0.0 && c.p1 == 0.0 && c.p2 == 0.0) d.dist_mode = FSW_DIST_NONE;
    else if (c.k2 == 0.0 && c.p1 == 0.0 && c.p2 == 0.0) d.dist_mode = FSW_DIST_K1;
    else d.dist_mode = FSW_DIST_FULL;
    return d;
}

/* Squared distorted normalised radius of the edge of the field of view, with a 2 % margin: a reference pixel whose
 * normalised coordinates lie beyond it cannot be inside the FOV, so tiles entirely beyond it skip S1.  Only when
 * the bound is provable: radial-only distortion, monotone over the FOV (checked at rig creation), finite edge. */
float ref_rd2_bound(const fsw_camera& c) {
    if (c.p1 != 0.0 || c.p2 != 0.0) return INFINITY;
    const double th = 0.5 * c.fov_max_deg * M_PI / 180.0;
    const double den = std::cos(th) + c.xi;
    if (!(den > 1e-3)) return INFINITY;
    const double ru = std::sin(th) / den;
    if (c.xi > 1.0 && std::cos(th) < -1.0 / c.xi) return INFINITY; /* rho_u(theta) is no longer monotone there */
    const double r2 = ru * ru;
    const double rd = ru * (1.0 + c.k1 * r2 + c.k2 * r2 * r2) * 1.02;
    if (!(rd > 0.0) || !std::isfinite(rd)) return INFINITY;
    return (float)(rd * rd);
}

int32_t check_params(const fsw_sweep_params* p, const char* name) {
    if (!p) return fail(FSW_E_INVALID_ARG, "%s is null", name);
    if (p->struct_size != sizeof(fsw_sweep_params)) return fail(FSW_E_INVALID_ARG, "%s: struct_size %u != %zu", name, p->struct_size, sizeof(fsw_sweep_params));
    if (p->window < 3 || p->window > FSW_MAX_WINDOW || (p->window & 1) == 0) return fail(FSW_E_INVALID_ARG, "%s: window=%d must be odd in 3..%d", name, p->window, FSW_MAX_WINDOW);
    if (p->depth_kind != FSW_DEPTH_RANGE && p->depth_kind != FSW_DEPTH_Z) return fail(FSW_E_INVALID_ARG, "%s: depth_kind=%d", name, p->depth_kind);
    if (p->filters_enabled & ~(FSW_FILTER_COST | FSW_FILTER_RATIO)) return fail(FSW_E_INVALID_ARG, "%s: unknown filter bits 0x%x", name, p->filters_enabled);
    if (!(p->range_max > 0.f)) return fail(FSW_E_INVALID_ARG, "%s: range_max must be positive", name);
    if (!(p->var_floor >= 0.f)) return fail(FSW_E_INVALID_ARG, "%s: var_floor must be >= 0", name);
    if (!std::isfinite(p->alpha_upper) || !std::isfinite(p->alpha_lower) || !std::isfinite(p->beta)) return fail(FSW_E_INVALID_ARG, "%s: thresholds must be finite", name);
    if (p->best_k < 0) return fail(FSW_E_INVALID_ARG, "%s: best_k=%d must be >= 0", name, p->best_k);
    if (p->best_k > 2) return fail(FSW_E_UNSUPPORTED, "%s: best_k=%d: the kernels aggregate the best one or two views (or all)", name, p->best_k);
    return FSW_OK;
}

int32_t check_images(const fsw_rig& rig, const fsw_image* images) {
    if (!images) return fail(FSW_E_INVALID_ARG, "images is null");
    for (int c = 0; c < rig.n_cams; ++c) {
        const fsw_image& im = images[c];
        if (!im.data) return fail(FSW_E_INVALID_ARG, "images[%d].data is null", c);
        if (im.dtype != FSW_U8 && im.dtype != FSW_F32) return fail(FSW_E_INVALID_ARG, "images[%d].dtype=%d", c, im.dtype);
        size_t es = im.dtype == FSW_U8 ? 1 : 4;
        if (im.pitch_bytes < es * (size_t)rig.cams[c].width) return fail(FSW_E_INVALID_ARG, "images[%d].pitch_bytes=%zu < row size", c, im.pitch_bytes);
        if (im.dtype == FSW_F32 && (im.pitch_bytes % 4 != 0 || ((uintptr_t)im.data) % 4 != 0)) return fail(FSW_E_INVALID_ARG, "images[%d]: float image must be 4-byte aligned", c);
    }
    return FSW_OK;
}

int32_t check_out(const fsw_rig& rig, const fsw_depth_out* out, const uint8_t* mask, size_t mask_pitch) {
    if (!out) return fail(FSW_E_INVALID_ARG, "out is null");
    if (out->struct_size != sizeof(fsw_depth_out)) return fail(FSW_E_INVALID_ARG, "out: struct_size %u != %zu", out->struct_size, sizeof(fsw_depth_out));
    const size_t W = (size_t)rig.cams[rig.ref_index].width;
    if (!out->depth) return fail(FSW_E_INVALID_ARG, "out->depth is required");
    if (out->depth_pitch < 4 * W || out->depth_pitch % 4) return fail(FSW_E_INVALID_ARG, "out->depth_pitch=%zu", out->depth_pitch);
    if (out->best_cost && (out->best_cost_pitch < 4 * W || out->best_cost_pitch % 4)) return fail(FSW_E_INVALID_ARG, "out->best_cost_pitch=%zu", out->best_cost_pitch);
    if (out->second_cost && (out->second_cost_pitch < 4 * W || out->second_cost_pitch % 4)) return fail(FSW_E_INVALID_ARG, "out->second_cost_pitch=%zu", out->second_cost_pitch);
    if (out->plane_index && (out->plane_index_pitch < 2 * W || out->plane_index_pitch % 2)) return fail(FSW_E_INVALID_ARG, "out->plane_index_pitch=%zu", out->plane_index_pitch);
    if (out->valid_reason && out->valid_reason_pitch < W) return fail(FSW_E_INVALID_ARG, "out->valid_reason_pitch=%zu", out->valid_reason_pitch);
    if (mask && mask_pitch < W) return fail(FSW_E_INVALID_ARG, "mask_pitch=%zu < width", mask_pitch);
    return FSW_OK;
}

bool view_fov_inside_image(const fsw_camera& c, bool half);

/* fills the part of the argument block that depends on rig, planes and parameters */
int32_t fill_args(FswSweepArgs& a, const fsw_rig& rig, const fsw_planeset& ps, const fsw_sweep_params& p, bool half) {
    std::memset(&a, 0, sizeof(a));
    const fsw_camera& ref = rig.cams[rig.ref_index];
    a.ref = dev_cam(ref, half);
    a.ref_rd2_max = ref_rd2_bound(ref); /* normalised coordinates: the same at both resolutions */
    a.n_views = 0;
    bool inside = true;
    for (int c = 0; c < rig.n_cams; ++c) {
        if (c == rig.ref_index) continue;
        FswDevView& v = a.views[a.n_views++];
        v.cam = dev_cam(rig.cams[c], half);
        bool ident = true;
        for (int i = 0; i < 9; ++i) {
            v.R[i] = (float)rig.Rrel[c][i];
            if (rig.Rrel[c][i] != ((i % 4 == 0) ? 1.0 : 0.0)) ident = false;
        }
        for (int i = 0; i < 3; ++i) v.T[i] = (float)rig.Trel[c][i];
        v.ident_R = ident ? 1 : 0;
        inside = inside && view_fov_inside_image(rig.cams[c], half);
    }
    a.views_inside = inside ? 1 : 0;
    a.n_fams = ps.n_fams;
    a.n_planes = ps.n_planes;
    for (int f = 0; f < ps.n_fams; ++f) {
        const fsw_plane_family& F = ps.fams[f];
        FswDevFamily& D = a.fam[f];
        for (int i = 0; i < 3; ++i) D.n[i] = (float)F.normal[i];
        D.first = ps.first[f];
        D.count = F.n_planes;
        D.spacing = F.spacing;
        double s0 = F.spacing == FSW_INVERSE ? 1.0 / F.d_first : F.d_first;
        double s1 = F.spacing == FSW_INVERSE ? 1.0 / F.d_last : F.d_last;
        D.s0 = (float)s0;
        D.ds = F.n_planes > 1 ? (float)((s1 - s0) / (double)(F.n_planes - 1)) : 0.f;
    }
    for (int k = 0; k < ps.n_planes; ++k) a.inv_d[k] = (float)(1.0 / ps.d[k]);
    const int W = a.ref.W, H = a.ref.H;
    int x0 = 0, y0 = 0, x1 = W, y1 = H;
    if (p.roi.w > 0 && p.roi.h > 0) {
        x0 = p.roi.x0; y0 = p.roi.y0; x1 = p.roi.x0 + p.roi.w; y1 = p.roi.y0 + p.roi.h;
    }
    a.roi_x0 = x0 < 0 ? 0 : x0; a.roi_y0 = y0 < 0 ? 0 : y0;
    a.roi_x1 = x1 > W ? W : x1; a.roi_y1 = y1 > H ? H : y1;
    a.subpixel = p.subpixel ? 1 : 0;
    a.filters = p.filters_enabled;
    a.depth_kind = p.depth_kind;
    a.horizon_row = p.horizon_row;
    a.alpha_upper = p.alpha_upper; a.alpha_lower = p.alpha_lower; a.beta = p.beta;
    /* the kernel compares (N var_a)(N var_b) with (var_floor N)^2, N = window^2 */
    const double fl = (double)p.var_floor * (double)p.window * (double)p.window;
    a.floor2 = (float)(fl * fl);
    if (!(a.floor2 > 0.f)) a.floor2 = 1e-30f; /* keeps the reciprocal square root finite on flat windows */
    a.inv_range_max = 1.f / p.range_max;
    a.best_k = p.best_k < a.n_views ? p.best_k : 0; /* the best k of k views or fewer is the plain mean */
    for (int c = 0; c < FSW_MAX_CAMERAS; ++c) a.inv_count[c] = c > 0 ? 1.f / (float)c : 0.f;
    a.n_sets = 1;
    return FSW_OK;
}

cudaError_t prepare_window(fsw_context* ctx, int w) {
    if (ctx->prepared[w]) return cudaSuccess;
    cudaError_t e = fsw_prepare_sweep(w, ctx->rig.n_cams - 1);
    if (e == cudaSuccess) ctx->prepared[w] = true;
    return e;
}

FswSweepGeometry window_geometry(int w, int n_views) { return fsw_sweep_geometry(w, n_views); }

/* picks the kernel variant the views allow (see fsw_sweep.cuh) */
int pick_variant(const FswSweepArgs& a, int foot_f16) {
    bool ident = true, simple = true;
    for (int v = 0; v < a.n_views; ++v) {
        ident = ident && a.views[v].ident_R;
        simple = simple && a.views[v].cam.dist_mode != FSW_DIST_FULL;
        simple = simple && (a.views[v].cam.cos_fov_xi >= 1e-3f); /* lets the kernel drop the denominator test */
    }
    const int mode = !simple ? 0 : (ident ? 1 : 2);
    if (mode != 0 && foot_f16 && a.views_inside) return 5 + mode; /* 6, 7: no test against the image borders */
    return mode + (foot_f16 ? 3 : 0);
}

/* Does the whole field of view of the camera fall inside its raster, with half a pixel to spare on every side?  Then
 * a projection that passes the field-of-view test has its bilinear footprint inside the image (S3) and the kernel
 * drops the border test.  Only where the edge of the field of view is a provable bound of the distorted radius
 * (ref_rd2_bound: radial distortion only, monotone, 2 % margin included). */
bool view_fov_inside_image(const fsw_camera& c, bool half) {
    const float rd2 = ref_rd2_bound(c);
    if (!std::isfinite(rd2)) return false;
    const double rd = std::sqrt((double)rd2);
    const FswDevCam d = dev_cam(c, half);
    const double rx = (double)d.fx * rd, ry = (double)d.fy * rd;
    return (double)d.cx - rx >= 0.5 && (double)d.cx + rx <= (double)d.W - 1.5 &&
           (double)d.cy - ry >= 0.5 && (double)d.cy + ry <= (double)d.H - 1.5;
}

/* FNV-1a over the bytes of the inputs of tile_weights */
uint64_t tile_order_key(const FswSweepArgs& a, const FswSweepGeometry& g) {
    uint64_t h = 1469598103934665603ull;
    auto mix = [&](const void* p, size_t n) {
        const unsigned char* b = static_cast<const unsigned char*>(p);
        for (size_t i = 0; i < n; ++i) { h ^= b[i]; h *= 1099511628211ull; }
    };
    mix(&a.ref, sizeof(a.ref)); mix(&a.ref_rd2_max, sizeof(float)); mix(&g.tile_w, sizeof(int)); mix(&g.tile_h, sizeof(int));
    mix(&a.n_fams, sizeof(int)); mix(a.fam, sizeof(FswDevFamily) * (size_t)a.n_fams);
    mix(&a.n_planes, sizeof(int)); mix(a.inv_d, sizeof(float) * (size_t)a.n_planes);
    mix(&a.inv_range_max, sizeof(float));
    const int32_t roi[4] = { a.roi_x0, a.roi_y0, a.roi_x1, a.roi_y1 };
    mix(roi, sizeof(roi));
    return h;
}

/* Estimated work of every tile, in plane passes (host model of what the kernel skips: tiles outside the region of
 * interest or the image circle, planes no ray of the tile faces or reaches within range_max, rows without rays).
 * Twelve sample points per tile, rays by the closed-form inverse of the unified model without the distortion: the
 * figures only order the queue and size the plane split, they decide nothing about the result. */
void tile_weights(const FswSweepArgs& a, const FswSweepGeometry& g, int hw, int ntx, int nty, std::vector<float>& w) {
    w.assign((size_t)ntx * nty, 0.f);
    const FswDevCam& c = a.ref;
    constexpr int NPX = 4, NPY = 3;
    for (int ty = 0; ty < nty; ++ty)
        for (int tx = 0; tx < ntx; ++tx) {
            const int x0 = tx * g.tile_w, y0 = ty * g.tile_h;
            if (!(x0 < a.roi_x1 && x0 + g.tile_w > a.roi_x0 && y0 < a.roi_y1 && y0 + g.tile_h > a.roi_y0)) continue;
            const float nx = std::max(std::max((float)(x0 - hw) - c.cx, c.cx - (float)(x0 + g.tile_w - 1 + hw)), 0.f) / c.fx;
            const float ny = std::max(std::max((float)(y0 - hw) - c.cy, c.cy - (float)(y0 + g.tile_h - 1 + hw)), 0.f) / c.fy;
            if (!(nx * nx + ny * ny <= a.ref_rd2_max)) continue; /* the kernel's own test: nothing to do */
            float ray[NPX * NPY][3];
            int n_pts = 0;
            for (int j = 0; j < NPY; ++j)
                for (int i = 0; i < NPX; ++i) {
                    const float px = (float)x0 + ((float)i + 0.5f) * (float)g.tile_w / NPX - 0.5f;
                    const float py = (float)y0 + ((float)j + 0.5f) * (float)g.tile_h / NPY - 0.5f;
                    if (px < (float)a.roi_x0 || px > (float)(a.roi_x1 - 1) || py < (float)a.roi_y0 || py > (float)(a.roi_y1 - 1)) continue;
                    const float mx = (px - c.cx) / c.fx, my = (py - c.cy) / c.fy, r2 = mx * mx + my * my;
                    if (r2 > a.ref_rd2_max) continue;
                    const float disc = 1.f + (1.f - c.xi * c.xi) * r2;
                    if (disc < 0.f) continue;
                    const float zf = (c.xi + std::sqrt(disc)) / (r2 + 1.f);
                    if (zf - c.xi < c.cos_fov) continue;
                    ray[n_pts][0] = zf * mx; ray[n_pts][1] = zf * my; ray[n_pts][2] = zf - c.xi;
                    ++n_pts;
                }
            float sum = 0.f;
            for (int f = 0; f < a.n_fams; ++f) {
                const FswDevFamily& F = a.fam[f];
                float q[NPX * NPY];
                for (int p = 0; p < n_pts; ++p) q[p] = F.n[0] * ray[p][0] + F.n[1] * ray[p][1] + F.n[2] * ray[p][2];
                for (int k = F.first; k < F.first + F.count; ++k) {
                    int cnt = 0;
                    for (int p = 0; p < n_pts; ++p) cnt += (q[p] > FSW_EPS_Q && q[p] * a.inv_d[k] >= a.inv_range_max) ? 1 : 0;
                    if (cnt) sum += 0.5f + 0.5f * (float)cnt / (float)(NPX * NPY);
                }
            }
            /* S1 and the epilogue are worth about two plane passes; a live tile that sweeps nothing still runs S1 */
            w[(size_t)ty * ntx + tx] = sum > 0.f ? sum + 2.f : 0.5f;
        }
}

/* Scheduling orders of the tiles (S0), tiles without work last in both.  (1) Heaviest first by the estimate of
 * tile_weights (longest processing time first), nearest to the principal point first among equals: for calls whose
 * queue is only a wave or two long, where the order decides the makespan (a single 1280 x 1024 frame set: 1.52 ->
 * 1.48 ms against the other order).  (2) Nearest to the principal point first, lower image half before the upper half
 * at equal distance: for long queues, where the tail is made of cheap tiles either way and blocks that run together
 * read neighbouring parts of the views (eight C5 frame sets per launch: 1.150 ms per map against 1.163 with (1)). */
void plan_tiles(const FswSweepArgs& a, const FswSweepGeometry& g, int hw, TileOrder* t) {
    const FswDevCam& ref = a.ref;
    t->key = tile_order_key(a, g);
    t->n_tiles_x = (ref.W + g.tile_w - 1) / g.tile_w;
    const int nty = (ref.H + g.tile_h - 1) / g.tile_h;
    t->n_tiles = t->n_tiles_x * nty;
    std::vector<float> w;
    tile_weights(a, g, hw, t->n_tiles_x, nty, w);
    std::vector<std::pair<std::pair<float, float>, int32_t>> by_w((size_t)t->n_tiles), by_d((size_t)t->n_tiles);
    for (int ty = 0; ty < nty; ++ty)
        for (int tx = 0; tx < t->n_tiles_x; ++tx) {
            const float dx = ((float)tx + 0.5f) * g.tile_w - 0.5f - ref.cx, dy = ((float)ty + 0.5f) * g.tile_h - 0.5f - ref.cy;
            const float r = std::sqrt(dx * dx + dy * dy);
            const int32_t id = ty * t->n_tiles_x + tx;
            by_w[(size_t)id] = std::make_pair(std::make_pair(-w[(size_t)id], r), id);
            by_d[(size_t)id] = std::make_pair(std::make_pair(w[(size_t)id] > 0.f ? 0.f : 1.f, r - (dy > 0.f ? 0.25f * g.tile_h : 0.f)), id);
        }
    std::stable_sort(by_w.begin(), by_w.end());
    std::stable_sort(by_d.begin(), by_d.end());
    std::vector<int32_t>& order_w = t->order_w;
    std::vector<int32_t>& order_d = t->order_d;
    order_w.resize((size_t)t->n_tiles); order_d.resize((size_t)t->n_tiles);
    t->weight.resize((size_t)t->n_tiles);
    t->n_live = 0;
    for (int i = 0; i < t->n_tiles; ++i) {
        order_w[(size_t)i] = by_w[(size_t)i].second;
        order_d[(size_t)i] = by_d[(size_t)i].second;
        t->weight[(size_t)i] = w[(size_t)order_w[(size_t)i]];
        if (t->weight[(size_t)i] > 0.f) t->n_live = i + 1;
    }
}

int32_t get_tile_order(fsw_context* ctx, const FswSweepArgs& a, const FswSweepGeometry& g, int hw, TileOrder** out) {
    const uint64_t key = tile_order_key(a, g);
    for (TileOrder* t : ctx->orders)
        if (t->key == key) {
            *out = t;
            return FSW_OK;
        }
    TileOrder* t = new (std::nothrow) TileOrder;
    if (!t) return fail(FSW_E_NOMEM, "tile order: out of memory");
    plan_tiles(a, g, hw, t);
    const size_t bytes = sizeof(int32_t) * (size_t)t->n_tiles;
    cudaError_t e = t->dev.reserve(bytes);
    if (e == cudaSuccess) e = t->dev_dist.reserve(bytes);
    if (e == cudaSuccess) e = cudaMemcpy(t->dev.p, t->order_w.data(), bytes, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(t->dev_dist.p, t->order_d.data(), bytes, cudaMemcpyHostToDevice);
    if (e != cudaSuccess) {
        t->dev.release();
        t->dev_dist.release();
        delete t;
        return cuda_fail(e, "tile order upload");
    }
    ctx->orders.push_back(t);
    *out = t;
    return FSW_OK;
}

/* Plane split: how many (tile, set) slots of the queue order are swept whole (by the unsplit kernel) before the
 * rest goes in halves.  List scheduling of the estimated weights on `slots` blocks, whole tiles first; a half costs
 * 0.6 of its tile (two halves repeat S1, score the plane across the cut and merge) plus a constant.  The smallest
 * makespan wins; every tile whole (= no split) is one of the candidates. */
int64_t split_whole_for(TileOrder* t, int n_sets, long long slots) {
    for (const auto& c : t->whole_for)
        if (c[0] == n_sets && c[1] == slots) return c[2];
    const int n_live = t->n_live;
    std::vector<double> load((size_t)slots);
    auto makespan = [&](int n_whole) {
        std::fill(load.begin(), load.end(), 0.0);
        std::priority_queue<double, std::vector<double>, std::greater<double>> pq(std::greater<double>(), load);
        auto put = [&](double w) { double l = pq.top(); pq.pop(); pq.push(l + w); };
        for (int i = 0; i < n_whole; ++i)
            for (int s = 0; s < n_sets; ++s) put((double)t->weight[(size_t)i]);
        for (int i = n_whole; i < n_live; ++i)
            for (int s = 0; s < 2 * n_sets; ++s) put(0.6 * (double)t->weight[(size_t)i] + 0.5);
        double m = 0.0;
        while (!pq.empty()) { m = std::max(m, pq.top()); pq.pop(); }
        return m;
    };
    int best = n_live;
    double best_m = makespan(n_live);
    for (int n_whole = n_live - 1; n_whole >= 0; --n_whole) {
        const double m = makespan(n_whole);
        if (m < best_m * 0.999) { best_m = m; best = n_whole; }
    }
    const int64_t whole = best == n_live ? (int64_t)t->n_tiles * n_sets : (int64_t)best * n_sets;
    t->whole_for.push_back({ (int64_t)n_sets, (int64_t)slots, whole });
    return whole;
}

/* enqueues the sweep kernel for a.n_sets frame sets (a.set0 / a.sets filled by the caller); the queue word must be
 * zero when the kernel starts (the pack launch before it clears it) */
int32_t launch_sweep(fsw_context* ctx, FswSweepArgs& a, int w, cudaStream_t s) {
    const FswSweepGeometry g = window_geometry(w, a.n_views);
    TileOrder* order = nullptr;
    int32_t rc = get_tile_order(ctx, a, g, w / 2, &order);
    if (rc != FSW_OK) return rc;
    const long long slots = (long long)ctx->n_sm * g.ctas_per_sm;
    const bool short_queue = (long long)order->n_live * a.n_sets < 3 * slots;
    a.tile_order = (const int32_t*)(short_queue ? order->dev.p : order->dev_dist.p);
    a.n_tiles_x = order->n_tiles_x;
    a.n_tiles = order->n_tiles;
    a.queue = ctx->queue();
    a.counters = ctx->counters();
    const int total_slots = a.n_tiles * a.n_sets;
    /* Plane split (fsw_context_set_split): few frame sets leave the persistent grid unbalanced -- a 1280 x 1024 frame
     * has 176 tiles with work for 148 CTAs, and the heaviest tile alone takes longer than the mean load of a CTA.
     * Then the light tiles at the end of the queue become two work items each, with half of the planes (by expected
     * work: a family facing away from the optical axis is reached by about (1 + n_z)/2 of the rays), and the halves
     * merge their winner-take-all states (fsw_sweep.cuh).  The heavy tiles at the head of the queue stay whole, in
     * the unsplit kernel; how many is decided by split_whole_for on the estimated tile weights. */
    a.split = 0;
    long long split_whole = total_slots;
    if (ctx->split_mode != FSW_SPLIT_OFF && a.n_planes >= 2) {
        if (ctx->split_mode == FSW_SPLIT_ON) split_whole = 0;
        else if (short_queue) split_whole = split_whole_for(order, a.n_sets, slots);
    }
    if (split_whole < total_slots) {
        double total = 0.0, acc = 0.0;
        std::vector<double> wk((size_t)a.n_planes);
        for (int f = 0; f < a.n_fams; ++f)
            for (int j = 0; j < a.fam[f].count; ++j) {
                wk[(size_t)a.fam[f].first + j] = std::max(0.1, 0.5 * (1.0 + (double)a.fam[f].n[2]));
                total += wk[(size_t)a.fam[f].first + j];
            }
        int kb = 1;
        for (int k = 0; k < a.n_planes - 1; ++k) {
            acc += wk[(size_t)k];
            kb = k + 1;
            if (acc >= 0.5 * total) break;
        }
        int fa = 0, fb = 0;
        for (int f = 0; f < a.n_fams; ++f) {
            if (kb - 1 >= a.fam[f].first) fa = f;
            if (kb >= a.fam[f].first) fb = f;
        }
        const size_t mapsz = (size_t)a.ref.W * a.ref.H;
        FSW_CUDA(ctx->split_state.reserve((size_t)a.n_sets * 2 * 6 * mapsz * sizeof(float)));
        const size_t tbytes = (size_t)a.n_sets * a.n_tiles * sizeof(unsigned int);
        if (tbytes > ctx->split_ticket.bytes) {
            FSW_CUDA(ctx->split_ticket.reserve(tbytes));
            FSW_CUDA(cudaMemsetAsync(ctx->split_ticket.p, 0, ctx->split_ticket.bytes, s));
        }
        a.split = 1;
        a.split_k = kb;
        a.split_whole = 0; /* the whole tiles go to the unsplit kernel */
        a.split_adjacent = fa == fb ? 1 : 0;
        a.split_state = (float*)ctx->split_state.p;
        a.split_ticket = (unsigned int*)ctx->split_ticket.p;
    }
    ctx->last_split += a.split;
    auto grid_for = [&](long long items) { return (int)(items < slots ? items : slots); };
    a.slot_first = 0;
    a.slot_count = total_slots;
    cudaError_t e;
    if (!a.split) {
        e = fsw_launch_sweep(w, a, pick_variant(a, a.foot_f16), grid_for(total_slots), s);
    } else if (split_whole == 0) {
        e = fsw_launch_sweep(w, a, pick_variant(a, a.foot_f16) + 8, grid_for(2LL * total_slots), s);
    } else {
        /* Two launches on the caller's stream: the whole tiles in the unsplit instantiation (the split one is about
         * 15 % slower on a whole tile), then the halved tiles as a PROGRAMMATIC DEPENDENT launch: every block of the
         * first kernel executes griddepcontrol.launch_dependents when it starts, so the blocks of the second one
         * become resident as the first one's blocks run out of whole tiles and exit -- the overlap of a second
         * stream without one.  The two kernels touch disjoint tiles and have a queue word each; a block of the second
         * kernel waits for the first grid (griddepcontrol.wait) before it exits, so whatever follows in the stream
         * sees both complete. */
        FswSweepArgs whole = a, halves = a;
        whole.split = 0;
        whole.n_tiles = (int32_t)(split_whole / a.n_sets); /* the unsplit kernel sweeps the first n_tiles * n_sets slots */
        halves.slot_first = (int32_t)split_whole;
        halves.slot_count = (int32_t)(total_slots - split_whole);
        halves.queue = ctx->queue() + 1;
        e = fsw_launch_sweep(w, whole, pick_variant(whole, whole.foot_f16), grid_for(split_whole), s);
        if (e == cudaSuccess) {
            e = fsw_launch_sweep(w, halves, (pick_variant(halves, halves.foot_f16) + 8) | FSW_VARIANT_PROGRAMMATIC,
                                 grid_for(2LL * halves.slot_count), s);
            ctx->last_launches++;
        }
    }
    if (e != cudaSuccess) return cuda_fail(e, "sweep kernel launch");
    ctx->last_launches++;
    return FSW_OK;
}

/* S4 staging: builds the footprint image of every matching view of n_sets frame sets (images[set * n_cams + cam]) in
 * context scratch and records the pointers in sets[]; the first pack launch also clears the work queue (and the
 * counters if asked).  half = the images are the context's half-resolution float images. */
int32_t stage_views(fsw_context* ctx, const fsw_image* images, int n_sets, bool half, FswSetPtrs* sets,
                    cudaStream_t stream, bool zero_counters, int32_t* foot_f16) {
    const fsw_rig& rig = ctx->rig;
    /* 8-byte bfloat16 footprints when every view of the call is an 8-bit image (exact), 16-byte float ones otherwise */
    int f16 = half ? 0 : 1;
    for (int s = 0; s < n_sets && f16; ++s)
        for (int c = 0; c < rig.n_cams; ++c)
            if (c != rig.ref_index && images[(size_t)s * rig.n_cams + c].dtype != FSW_U8) f16 = 0;
    *foot_f16 = f16;
    std::vector<DevBuf>& foots = half ? ctx->half_foot : ctx->foot;
    if (foots.size() < (size_t)n_sets * FSW_MAX_CAMERAS) foots.resize((size_t)n_sets * FSW_MAX_CAMERAS);
    bool first = true;
    /* one launch per camera size (all views of a rig usually share one) and per FSW_PACK_MAX images */
    std::vector<bool> done((size_t)rig.n_cams, false);
    for (int c0 = 0; c0 < rig.n_cams; ++c0) {
        if (c0 == rig.ref_index || done[c0]) continue;
        const int W = half ? rig.cams[c0].width / 2 : rig.cams[c0].width;
        const int H = half ? rig.cams[c0].height / 2 : rig.cams[c0].height;
        FswPackArgs pk;
        std::memset(&pk, 0, sizeof(pk));
        pk.W = W; pk.H = H; pk.f16 = f16;
        auto flush = [&]() -> int32_t {
            if (pk.n == 0) return FSW_OK;
            if (first) {
                pk.words_to_zero = (unsigned int*)ctx->ctrl.p;
                pk.n_words_to_zero = zero_counters ? FSW_CTRL_WORDS : FSW_QUEUE_WORDS;
                first = false;
            } else {
                pk.words_to_zero = nullptr;
                pk.n_words_to_zero = 0;
            }
            FSW_CUDA(fsw_launch_pack_footprints(pk, stream));
            ctx->last_launches++;
            pk.n = 0;
            return FSW_OK;
        };
        for (int c = c0; c < rig.n_cams; ++c) {
            if (c == rig.ref_index || done[c]) continue;
            const int Wc = half ? rig.cams[c].width / 2 : rig.cams[c].width;
            const int Hc = half ? rig.cams[c].height / 2 : rig.cams[c].height;
            if (Wc != W || Hc != H) continue;
            done[c] = true;
            int vi = c < rig.ref_index ? c : c - 1; /* view index = camera order without the reference */
            for (int s = 0; s < n_sets; ++s) {
                DevBuf& fb = foots[(size_t)s * FSW_MAX_CAMERAS + c];
                FSW_CUDA(fb.reserve((size_t)W * H * sizeof(float4)));
                if (half) {
                    pk.src[pk.n] = ctx->half[(size_t)s * FSW_MAX_CAMERAS + c].p; pk.src_pitch[pk.n] = (int64_t)W * 4; pk.dtype[pk.n] = FSW_F32;
                } else {
                    const fsw_image& im = images[(size_t)s * rig.n_cams + c];
                    pk.src[pk.n] = im.data; pk.src_pitch[pk.n] = (int64_t)im.pitch_bytes; pk.dtype[pk.n] = im.dtype;
                }
                pk.dst[pk.n] = fb.p;
                sets[s].foot[vi] = fb.p;
                pk.n++;
                if (pk.n == FSW_PACK_MAX) {
                    int32_t rc = flush();
                    if (rc != FSW_OK) return rc;
                }
            }
        }
        int32_t rc = flush();
        if (rc != FSW_OK) return rc;
    }
    if (first) /* cannot happen (a rig has at least one view), but never start a sweep with a dirty queue */
        FSW_CUDA(cudaMemsetAsync(ctx->ctrl.p, 0, (zero_counters ? FSW_CTRL_WORDS : FSW_QUEUE_WORDS) * sizeof(unsigned int), stream));
    return FSW_OK;
}

/* the set table of a batch goes to the device through the next pinned staging slot of the context; a slot is reused
 * only after the copy that last read it has completed (its event), which a ring of four makes the common case */
int32_t upload_sets(fsw_context* ctx, const FswSetPtrs* sets, int n_sets, cudaStream_t stream, int table = 0) {
    const size_t bytes = sizeof(FswSetPtrs) * (size_t)n_sets;
    DevBuf& dev = table ? ctx->sets_dev2 : ctx->sets_dev;
    FSW_CUDA(dev.reserve(bytes));
    const int slot = ctx->sets_next;
    ctx->sets_next = (slot + 1) % fsw_context::N_SET_STAGE;
    if (!ctx->sets_ev[slot]) FSW_CUDA(cudaEventCreateWithFlags(&ctx->sets_ev[slot], cudaEventDisableTiming));
    else FSW_CUDA(cudaEventSynchronize(ctx->sets_ev[slot]));
    if (ctx->sets_pinned_cap[slot] < bytes) {
        if (ctx->sets_pinned[slot]) cudaFreeHost(ctx->sets_pinned[slot]);
        ctx->sets_pinned[slot] = nullptr;
        ctx->sets_pinned_cap[slot] = 0;
        FSW_CUDA(cudaMallocHost((void**)&ctx->sets_pinned[slot], bytes));
        ctx->sets_pinned_cap[slot] = bytes;
    }
    std::memcpy(ctx->sets_pinned[slot], sets, bytes);
    FSW_CUDA(cudaMemcpyAsync(dev.p, ctx->sets_pinned[slot], bytes, cudaMemcpyHostToDevice, stream));
    FSW_CUDA(cudaEventRecord(ctx->sets_ev[slot], stream));
    return FSW_OK;
}

void set_outputs(FswSetPtrs& a, const fsw_depth_out* out, const uint8_t* mask, size_t mask_pitch) {
    a.mask = mask; a.mask_pitch = (int64_t)mask_pitch;
    a.out_depth = out->depth; a.out_depth_pitch = (int64_t)out->depth_pitch;
    a.out_c1 = out->best_cost; a.out_c1_pitch = (int64_t)out->best_cost_pitch;
    a.out_c2 = out->second_cost; a.out_c2_pitch = (int64_t)out->second_cost_pitch;
    a.out_k = out->plane_index; a.out_k_pitch = (int64_t)out->plane_index_pitch;
    a.out_reason = out->valid_reason; a.out_reason_pitch = (int64_t)out->valid_reason_pitch;
}

}  // namespace

/* ================================================================================================================ */
extern "C" {

int32_t fsw_version(int32_t* major, int32_t* minor) {
    if (major) *major = FSW_VERSION_MAJOR;
    if (minor) *minor = FSW_VERSION_MINOR;
    return FSW_OK;
}

const char* fsw_last_error(void) { return g_err; }

int32_t fsw_rig_create(const fsw_camera* cams, int32_t n_cams, int32_t ref_index, fsw_rig** out) {
    if (!cams || !out) return fail(FSW_E_INVALID_ARG, "fsw_rig_create: null argument");
    *out = nullptr;
    if (n_cams < 2 || n_cams > FSW_MAX_CAMERAS) return fail(FSW_E_INVALID_ARG, "fsw_rig_create: n_cams=%d must be in 2..%d", n_cams, FSW_MAX_CAMERAS);
    if (ref_index < 0 || ref_index >= n_cams) return fail(FSW_E_INVALID_ARG, "fsw_rig_create: ref_index=%d out of range", ref_index);
    for (int c = 0; c < n_cams; ++c) {
        int32_t rc = check_camera(cams[c], c);
        if (rc != FSW_OK) return rc;
    }
    fsw_rig* rig = new (std::nothrow) fsw_rig;
    if (!rig) return fail(FSW_E_NOMEM, "fsw_rig_create: out of memory");
    rig->n_cams = n_cams;
    rig->ref_index = ref_index;
    for (int c = 0; c < n_cams; ++c) {
        rig->cams[c] = cams[c];
        relative_pose(cams[ref_index], cams[c], rig->Rrel[c], rig->Trel[c]);
    }
    /* the reference relative pose is exactly the identity */
    for (int i = 0; i < 9; ++i) rig->Rrel[ref_index][i] = (i % 4 == 0) ? 1.0 : 0.0;
    for (int i = 0; i < 3; ++i) rig->Trel[ref_index][i] = 0.0;
    *out = rig;
    return FSW_OK;
}

int32_t fsw_rig_subset(const fsw_rig* rig, const int32_t* cam_indices, int32_t n_cams, fsw_rig** out) {
    if (!rig || !cam_indices || !out) return fail(FSW_E_INVALID_ARG, "fsw_rig_subset: null argument");
    *out = nullptr;
    if (n_cams < 2 || n_cams > FSW_MAX_CAMERAS) return fail(FSW_E_INVALID_ARG, "fsw_rig_subset: n_cams=%d must be in 2..%d", n_cams, FSW_MAX_CAMERAS);
    fsw_camera cams[FSW_MAX_CAMERAS];
    int ref = -1;
    for (int i = 0; i < n_cams; ++i) {
        const int c = cam_indices[i];
        if (c < 0 || c >= rig->n_cams) return fail(FSW_E_INVALID_ARG, "fsw_rig_subset: camera index %d out of range", c);
        for (int j = 0; j < i; ++j)
            if (cam_indices[j] == c) return fail(FSW_E_INVALID_ARG, "fsw_rig_subset: camera %d listed twice", c);
        if (c == rig->ref_index) ref = i;
        cams[i] = rig->cams[c];
    }
    if (ref < 0) return fail(FSW_E_INVALID_ARG, "fsw_rig_subset: the reference camera (%d) must be part of the subset", rig->ref_index);
    return fsw_rig_create(cams, n_cams, ref, out);
}

int32_t fsw_rig_destroy(fsw_rig* rig) {
    delete rig;
    return FSW_OK;
}

int32_t fsw_rig_relative_pose(const fsw_rig* rig, int32_t cam, double* R, double* T) {
    if (!rig || !R || !T) return fail(FSW_E_INVALID_ARG, "fsw_rig_relative_pose: null argument");
    if (cam < 0 || cam >= rig->n_cams) return fail(FSW_E_INVALID_ARG, "fsw_rig_relative_pose: cam=%d out of range", cam);
    std::memcpy(R, rig->Rrel[cam], sizeof(double) * 9);
    std::memcpy(T, rig->Trel[cam], sizeof(double) * 3);
    return FSW_OK;
}

int32_t fsw_ground_normal_in_ref(const fsw_rig* rig, const double* dir_rig, double* out) {
    if (!rig || !dir_rig || !out) return fail(FSW_E_INVALID_ARG, "fsw_ground_normal_in_ref: null argument");
    const double* R = rig->cams[rig->ref_index].R;
    double n = std::sqrt(dir_rig[0] * dir_rig[0] + dir_rig[1] * dir_rig[1] + dir_rig[2] * dir_rig[2]);
    if (!(n > 0.0)) return fail(FSW_E_CONFIG, "fsw_ground_normal_in_ref: zero direction");
    for (int i = 0; i < 3; ++i) out[i] = (R[3 * i] * dir_rig[0] + R[3 * i + 1] * dir_rig[1] + R[3 * i + 2] * dir_rig[2]) / n;
    return FSW_OK;
}

int32_t fsw_planeset_create(const fsw_plane_family* fams, int32_t n_fams, fsw_planeset** out) {
    if (!fams || !out) return fail(FSW_E_INVALID_ARG, "fsw_planeset_create: null argument");
    *out = nullptr;
    if (n_fams < 1 || n_fams > FSW_MAX_FAMILIES) return fail(FSW_E_INVALID_ARG, "fsw_planeset_create: n_fams=%d must be in 1..%d", n_fams, FSW_MAX_FAMILIES);
    int64_t total = 0;
    for (int f = 0; f < n_fams; ++f) {
        const fsw_plane_family& F = fams[f];
        if (F.struct_size != sizeof(fsw_plane_family)) return fail(FSW_E_INVALID_ARG, "family %d: struct_size %u != %zu", f, F.struct_size, sizeof(fsw_plane_family));
        if (F.spacing != FSW_INVERSE && F.spacing != FSW_LINEAR) return fail(FSW_E_INVALID_ARG, "family %d: spacing=%d", f, F.spacing);
        if (F.n_planes < 1) return fail(FSW_E_CONFIG, "family %d: n_planes=%d", f, F.n_planes);
        if (!(F.d_first > 0.0) || !(F.d_last > 0.0) || !std::isfinite(F.d_first) || !std::isfinite(F.d_last)) return fail(FSW_E_CONFIG, "family %d: plane offsets must be positive and finite", f);
        double n = std::sqrt(F.normal[0] * F.normal[0] + F.normal[1] * F.normal[1] + F.normal[2] * F.normal[2]);
        if (!(n > 1e-12) || !std::isfinite(n)) return fail(FSW_E_CONFIG, "family %d: zero normal", f);
        total += F.n_planes;
    }
    if (total > FSW_MAX_PLANES) return fail(FSW_E_CONFIG, "fsw_planeset_create: %lld planes > %d", (long long)total, FSW_MAX_PLANES);
    fsw_planeset* ps = new (std::nothrow) fsw_planeset;
    if (!ps) return fail(FSW_E_NOMEM, "fsw_planeset_create: out of memory");
    ps->n_fams = n_fams;
    ps->n_planes = (int32_t)total;
    int k0 = 0;
    for (int f = 0; f < n_fams; ++f) {
        fsw_plane_family F = fams[f];
        double n = std::sqrt(F.normal[0] * F.normal[0] + F.normal[1] * F.normal[1] + F.normal[2] * F.normal[2]);
        for (int i = 0; i < 3; ++i) F.normal[i] /= n;
        ps->fams[f] = F;
        ps->first[f] = k0;
        /* the planes divide [first, last] evenly in the spacing variable (1/d or d): plane k is the point with
         * barycentric weights (n-1-k, k)/(n-1) of the two end planes */
        const bool inv = F.spacing == FSW_INVERSE;
        const double end0 = inv ? 1.0 / F.d_first : F.d_first, end1 = inv ? 1.0 / F.d_last : F.d_last;
        const int last = F.n_planes - 1;
        for (int k = 0; k <= last; ++k) {
            const double sk = last > 0 ? ((double)(last - k) * end0 + (double)k * end1) / (double)last : end0;
            ps->s.push_back(sk);
            ps->d.push_back(inv ? 1.0 / sk : sk);
            ps->family.push_back(f);
        }
        k0 += F.n_planes;
    }
    *out = ps;
    return FSW_OK;
}

int32_t fsw_planeset_destroy(fsw_planeset* ps) {
    delete ps;
    return FSW_OK;
}

int32_t fsw_planeset_size(const fsw_planeset* ps, int32_t* n_planes) {
    if (!ps || !n_planes) return fail(FSW_E_INVALID_ARG, "fsw_planeset_size: null argument");
    *n_planes = ps->n_planes;
    return FSW_OK;
}

int32_t fsw_planeset_table(const fsw_planeset* ps, double* s, double* d, int32_t* family) {
    if (!ps) return fail(FSW_E_INVALID_ARG, "fsw_planeset_table: null argument");
    for (int k = 0; k < ps->n_planes; ++k) {
        if (s) s[k] = ps->s[k];
        if (d) d[k] = ps->d[k];
        if (family) family[k] = ps->family[k];
    }
    return FSW_OK;
}

int32_t fsw_context_create(const fsw_rig* rig, int32_t cuda_device, fsw_context** out) {
    if (!rig || !out) return fail(FSW_E_INVALID_ARG, "fsw_context_create: null argument");
    *out = nullptr;
    int n_dev = 0;
    cudaError_t e = cudaGetDeviceCount(&n_dev);
    if (e != cudaSuccess) return cuda_fail(e, "fsw_context_create: no usable CUDA device (there is no CPU fallback)");
    if (cuda_device < 0 || cuda_device >= n_dev) return fail(FSW_E_INVALID_ARG, "fsw_context_create: cuda_device=%d of %d", cuda_device, n_dev);
    cudaDeviceProp prop;
    FSW_CUDA(cudaGetDeviceProperties(&prop, cuda_device));
    if (prop.major < 10) return fail(FSW_E_UNSUPPORTED, "fsw_context_create: device %d is sm_%d%d; this library holds sm_100a code only", cuda_device, prop.major, prop.minor);
    fsw_context* ctx = new (std::nothrow) fsw_context;
    if (!ctx) return fail(FSW_E_NOMEM, "fsw_context_create: out of memory");
    ctx->rig = *rig;
    ctx->device = cuda_device;
    ctx->n_sm = prop.multiProcessorCount;
    DeviceGuard g;
    e = g.enter(cuda_device);
    if (e == cudaSuccess) e = ctx->ctrl.reserve(FSW_CTRL_WORDS * sizeof(unsigned int));
    if (e == cudaSuccess) e = cudaMemset(ctx->ctrl.p, 0, FSW_CTRL_WORDS * sizeof(unsigned int));
    if (e != cudaSuccess) {
        delete ctx;
        return cuda_fail(e, "fsw_context_create");
    }
    *out = ctx;
    return FSW_OK;
}

int32_t fsw_context_destroy(fsw_context* ctx) {
    if (!ctx) return FSW_OK;
    DeviceGuard g;
    g.enter(ctx->device);
    for (std::vector<DevBuf>* v : {&ctx->foot, &ctx->half, &ctx->half_foot, &ctx->lo_depth, &ctx->lo_c1, &ctx->lo_c2, &ctx->lo_k, &ctx->lo_reason,
                                   &ctx->st_img, &ctx->st_mask, &ctx->st_depth, &ctx->st_c1, &ctx->st_c2, &ctx->st_k, &ctx->st_reason})
        for (DevBuf& b : *v) b.release();
    ctx->ctrl.release(); ctx->sets_dev.release(); ctx->sets_dev2.release();
    for (int i = 0; i < fsw_context::N_SET_STAGE; ++i) {
        if (ctx->sets_pinned[i]) cudaFreeHost(ctx->sets_pinned[i]);
        if (ctx->sets_ev[i]) cudaEventDestroy(ctx->sets_ev[i]);
    }
    ctx->split_state.release(); ctx->split_ticket.release();
    for (TileOrder* t : ctx->orders) {
        t->dev.release();
        t->dev_dist.release();
        delete t;
    }
    for (int i = 0; i < 4; ++i)
        if (ctx->ev[i]) cudaEventDestroy(ctx->ev[i]);
    delete ctx;
    return FSW_OK;
}

/* the single-resolution path for n_sets frame sets: pack launch(es) + one sweep launch */
static int32_t run_sets(fsw_context* ctx, const fsw_planeset* planes, const fsw_sweep_params* params, int32_t n_sets,
                        const fsw_image* images, const uint8_t* const* masks, size_t mask_pitch,
                        const fsw_depth_out* outs, void* cuda_stream, const char* who) {
    if (!ctx || !planes) return fail(FSW_E_INVALID_ARG, "%s: null context or plane set", who);
    if (n_sets < 1 || n_sets > FSW_MAX_BATCH) return fail(FSW_E_INVALID_ARG, "%s: n_sets=%d must be in 1..%d", who, n_sets, FSW_MAX_BATCH);
    int32_t rc;
    if ((rc = check_params(params, "params")) != FSW_OK) return rc;
    if (!images || !outs) return fail(FSW_E_INVALID_ARG, "%s: null images or outputs", who);
    const fsw_rig& rig = ctx->rig;
    for (int s = 0; s < n_sets; ++s) {
        if ((rc = check_images(rig, images + (size_t)s * rig.n_cams)) != FSW_OK) return rc;
        if ((rc = check_out(rig, &outs[s], masks ? masks[s] : nullptr, mask_pitch)) != FSW_OK) return rc;
    }
    if (params->debug_cost_volume && n_sets > 1) return fail(FSW_E_UNSUPPORTED, "%s: debug_cost_volume needs n_sets == 1", who);
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    DeviceGuard g;
    FSW_CUDA(g.enter(ctx->device));
    FSW_CUDA(prepare_window(ctx, params->window));
    ctx->last_stream = stream;
    ctx->last_launches = 0;
    ctx->last_split = 0;

    FswSweepArgs a;
    fill_args(a, rig, *planes, *params, false);
    std::vector<FswSetPtrs> sets((size_t)n_sets);
    std::memset(sets.data(), 0, sizeof(FswSetPtrs) * (size_t)n_sets);
    for (int s = 0; s < n_sets; ++s) {
        const fsw_image& ri = images[(size_t)s * rig.n_cams + rig.ref_index];
        sets[s].ref_img = ri.data; sets[s].ref_pitch_bytes = (int64_t)ri.pitch_bytes; sets[s].ref_dtype = ri.dtype;
        sets[s].debug_cost = params->debug_cost_volume;
        set_outputs(sets[s], &outs[s], masks ? masks[s] : nullptr, mask_pitch);
    }
    if ((rc = stage_views(ctx, images, n_sets, false, sets.data(), stream, true, &a.foot_f16)) != FSW_OK) return rc;
    a.n_sets = n_sets;
    a.set0 = sets[0];
    if (n_sets > 1) {
        if ((rc = upload_sets(ctx, sets.data(), n_sets, stream)) != FSW_OK) return rc;
        a.sets = (const FswSetPtrs*)ctx->sets_dev.p;
    }
    a.count_pixels = 1;
    ctx->n_timed = 0;
    if (ctx->timing) FSW_CUDA(cudaEventRecord(ctx->ev[0], stream));
    if ((rc = launch_sweep(ctx, a, params->window, stream)) != FSW_OK) return rc;
    if (ctx->timing) { FSW_CUDA(cudaEventRecord(ctx->ev[1], stream)); ctx->n_timed = 1; }
    return FSW_OK;
}

int32_t fsw_compute_depth(fsw_context* ctx, const fsw_planeset* planes, const fsw_sweep_params* params,
                          const fsw_image* images, const uint8_t* mask, size_t mask_pitch,
                          const fsw_depth_out* out, void* cuda_stream) {
    const uint8_t* masks[1] = {mask};
    return run_sets(ctx, planes, params, 1, images, mask ? masks : nullptr, mask_pitch, out, cuda_stream, "fsw_compute_depth");
}

int32_t fsw_compute_depth_batch(fsw_context* ctx, const fsw_planeset* planes, const fsw_sweep_params* params,
                                int32_t n_sets, const fsw_image* images, const uint8_t* const* masks, size_t mask_pitch,
                                const fsw_depth_out* outs, void* cuda_stream) {
    return run_sets(ctx, planes, params, n_sets, images, masks, mask_pitch, outs, cuda_stream, "fsw_compute_depth_batch");
}

/* the two-scale path (S10) for n_sets frame sets: one downsample launch per FSW_PACK_MAX images, the half-resolution
 * sweep of all sets in one launch, the crop sweep of all sets in one launch */
static int32_t run_multires(fsw_context* ctx, const fsw_planeset* planes_low, const fsw_planeset* planes_crop,
                            const fsw_sweep_params* params_low, const fsw_sweep_params* params_crop, fsw_rect crop,
                            int32_t n_sets, const fsw_image* images, const uint8_t* const* masks, size_t mask_pitch,
                            const fsw_depth_out* outs, void* cuda_stream, const char* who) {
    if (!ctx || !planes_low || !planes_crop) return fail(FSW_E_INVALID_ARG, "%s: null context or plane set", who);
    if (n_sets < 1 || n_sets > FSW_MAX_BATCH) return fail(FSW_E_INVALID_ARG, "%s: n_sets=%d must be in 1..%d", who, n_sets, FSW_MAX_BATCH);
    if (!images || !outs) return fail(FSW_E_INVALID_ARG, "%s: null images or outputs", who);
    int32_t rc;
    if ((rc = check_params(params_low, "params_low")) != FSW_OK) return rc;
    if ((rc = check_params(params_crop, "params_crop")) != FSW_OK) return rc;
    const fsw_rig& rig = ctx->rig;
    for (int s = 0; s < n_sets; ++s) {
        if ((rc = check_images(rig, images + (size_t)s * rig.n_cams)) != FSW_OK) return rc;
        if ((rc = check_out(rig, &outs[s], masks ? masks[s] : nullptr, mask_pitch)) != FSW_OK) return rc;
    }
    const fsw_camera& ref = rig.cams[rig.ref_index];
    if (crop.w <= 0 || crop.h <= 0 || crop.x0 < 0 || crop.y0 < 0 || crop.x0 + crop.w > ref.width || crop.y0 + crop.h > ref.height)
        return fail(FSW_E_INVALID_ARG, "%s: crop (%d,%d,%d,%d) not inside the reference image", who, crop.x0, crop.y0, crop.w, crop.h);
    if (params_low->debug_cost_volume || params_crop->debug_cost_volume)
        return fail(FSW_E_UNSUPPORTED, "%s: debug_cost_volume is only available in fsw_compute_depth", who);
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    DeviceGuard g;
    FSW_CUDA(g.enter(ctx->device));
    FSW_CUDA(prepare_window(ctx, params_low->window));
    FSW_CUDA(prepare_window(ctx, params_crop->window));
    ctx->last_stream = stream;
    ctx->last_launches = 0;
    ctx->last_split = 0;
    const size_t ns = (size_t)n_sets;
    if (ctx->half.size() < ns * FSW_MAX_CAMERAS) ctx->half.resize(ns * FSW_MAX_CAMERAS);
    for (std::vector<DevBuf>* v : {&ctx->lo_depth, &ctx->lo_c1, &ctx->lo_c2, &ctx->lo_k, &ctx->lo_reason})
        if (v->size() < ns) v->resize(ns);
    const bool filter_first = params_crop->filter_before_merge != 0;

    /* S10(a): 2x2 box downsample of every image of every set */
    FswDownArgs dn;
    std::memset(&dn, 0, sizeof(dn));
    for (int s = 0; s < n_sets; ++s)
        for (int c = 0; c < rig.n_cams; ++c) {
            const int W = rig.cams[c].width, H = rig.cams[c].height;
            const fsw_image& im = images[(size_t)s * rig.n_cams + c];
            DevBuf& hb = ctx->half[(size_t)s * FSW_MAX_CAMERAS + c];
            FSW_CUDA(hb.reserve((size_t)(W / 2) * (H / 2) * 4));
            dn.src[dn.n] = im.data; dn.src_pitch[dn.n] = (int64_t)im.pitch_bytes; dn.dtype[dn.n] = im.dtype;
            dn.dst[dn.n] = (float*)hb.p; dn.W[dn.n] = W; dn.H[dn.n] = H;
            if (++dn.n == FSW_PACK_MAX || (s == n_sets - 1 && c == rig.n_cams - 1)) {
                FSW_CUDA(fsw_launch_downsample(dn, stream));
                ctx->last_launches++;
                dn.n = 0;
            }
        }

    /* S10(b): half-resolution sweep over the whole field of view, raw maps into context scratch */
    const int LW = ref.width / 2, LH = ref.height / 2;
    FswSweepArgs a;
    fsw_sweep_params pl = *params_low;
    /* filters run after the merge (reading Q20), unless the caller asks for the other order (Q27): then the
     * half-resolution pass applies its own and hands its verdicts to the crop pass */
    if (!filter_first) pl.filters_enabled = 0;
    const bool up_plane = params_crop->upsample_plane != 0;
    fill_args(a, rig, *planes_low, pl, true);
    if (up_plane) a.depth_kind = FSW_DEPTH_PLANE_OFFSET; /* the crop pass turns offsets into depths of its own rays */
    std::vector<FswSetPtrs> sets(ns);
    std::memset(sets.data(), 0, sizeof(FswSetPtrs) * ns);
    for (int s = 0; s < n_sets; ++s) {
        FSW_CUDA(ctx->lo_depth[s].reserve((size_t)LW * LH * 4));
        FSW_CUDA(ctx->lo_c1[s].reserve((size_t)LW * LH * 4));
        FSW_CUDA(ctx->lo_c2[s].reserve((size_t)LW * LH * 4));
        FSW_CUDA(ctx->lo_k[s].reserve((size_t)LW * LH * 2));
        FswSetPtrs& lo = sets[s];
        lo.ref_img = ctx->half[(size_t)s * FSW_MAX_CAMERAS + rig.ref_index].p; lo.ref_pitch_bytes = (int64_t)LW * 4; lo.ref_dtype = FSW_F32;
        lo.out_depth = (float*)ctx->lo_depth[s].p; lo.out_depth_pitch = (int64_t)LW * 4;
        lo.out_c1 = (float*)ctx->lo_c1[s].p; lo.out_c1_pitch = (int64_t)LW * 4;
        lo.out_c2 = (float*)ctx->lo_c2[s].p; lo.out_c2_pitch = (int64_t)LW * 4;
        lo.out_k = (int16_t*)ctx->lo_k[s].p; lo.out_k_pitch = (int64_t)LW * 2;
        if (filter_first) {
            FSW_CUDA(ctx->lo_reason[s].reserve((size_t)LW * LH));
            lo.out_reason = (uint8_t*)ctx->lo_reason[s].p; lo.out_reason_pitch = (int64_t)LW;
        }
    }
    if ((rc = stage_views(ctx, nullptr, n_sets, true, sets.data(), stream, true, &a.foot_f16)) != FSW_OK) return rc;
    a.n_sets = n_sets;
    a.set0 = sets[0];
    if (n_sets > 1) {
        if ((rc = upload_sets(ctx, sets.data(), n_sets, stream, 0)) != FSW_OK) return rc;
        a.sets = (const FswSetPtrs*)ctx->sets_dev.p;
    }
    a.count_pixels = 0;
    ctx->n_timed = 0;
    if (ctx->timing) FSW_CUDA(cudaEventRecord(ctx->ev[2], stream));
    if ((rc = launch_sweep(ctx, a, params_low->window, stream)) != FSW_OK) return rc;
    if (ctx->timing) FSW_CUDA(cudaEventRecord(ctx->ev[3], stream));

    /* S10(d)-(e) + S9 + S11: full-resolution sweep inside the crop, merged with the upsampled maps in its epilogue */
    fsw_sweep_params pc = *params_crop;
    pc.roi = crop;
    fill_args(a, rig, *planes_crop, pc, false);
    std::memset(sets.data(), 0, sizeof(FswSetPtrs) * ns);
    for (int s = 0; s < n_sets; ++s) {
        FswSetPtrs& hi = sets[s];
        const fsw_image& ri = images[(size_t)s * rig.n_cams + rig.ref_index];
        hi.ref_img = ri.data; hi.ref_pitch_bytes = (int64_t)ri.pitch_bytes; hi.ref_dtype = ri.dtype;
        set_outputs(hi, &outs[s], masks ? masks[s] : nullptr, mask_pitch);
        hi.lo_depth = (const float*)ctx->lo_depth[s].p; hi.lo_c1 = (const float*)ctx->lo_c1[s].p;
        hi.lo_c2 = (const float*)ctx->lo_c2[s].p; hi.lo_k = (const int16_t*)ctx->lo_k[s].p;
        hi.lo_reason = filter_first ? (const uint8_t*)ctx->lo_reason[s].p : nullptr;
    }
    if ((rc = stage_views(ctx, images, n_sets, false, sets.data(), stream, false, &a.foot_f16)) != FSW_OK) return rc;
    a.n_sets = n_sets;
    a.set0 = sets[0];
    if (n_sets > 1) {
        /* second table of the call: the low sweep may still be reading the first one */
        if ((rc = upload_sets(ctx, sets.data(), n_sets, stream, 1)) != FSW_OK) return rc;
        a.sets = (const FswSetPtrs*)ctx->sets_dev2.p;
    }
    a.lo_W = LW; a.lo_H = LH;
    a.filter_first = filter_first ? 1 : 0;
    a.upsample_plane = up_plane ? 1 : 0;
    a.n_lo_fams = planes_low->n_fams;
    for (int f = 0; f < planes_low->n_fams; ++f) {
        for (int i = 0; i < 3; ++i) a.lo_fam_n[f][i] = (float)planes_low->fams[f].normal[i];
        a.lo_fam_first[f] = planes_low->first[f];
    }
    a.index_flag = FSW_INDEX_FROM_CROP;
    a.count_pixels = 1;
    if (ctx->timing) FSW_CUDA(cudaEventRecord(ctx->ev[0], stream));
    if ((rc = launch_sweep(ctx, a, params_crop->window, stream)) != FSW_OK) return rc;
    if (ctx->timing) { FSW_CUDA(cudaEventRecord(ctx->ev[1], stream)); ctx->n_timed = 2; }
    return FSW_OK;
}

int32_t fsw_compute_depth_multires(fsw_context* ctx, const fsw_planeset* planes_low, const fsw_planeset* planes_crop,
                                   const fsw_sweep_params* params_low, const fsw_sweep_params* params_crop,
                                   fsw_rect crop, const fsw_image* images, const uint8_t* mask, size_t mask_pitch,
                                   const fsw_depth_out* out, void* cuda_stream) {
    const uint8_t* masks[1] = {mask};
    return run_multires(ctx, planes_low, planes_crop, params_low, params_crop, crop, 1, images, mask ? masks : nullptr,
                        mask_pitch, out, cuda_stream, "fsw_compute_depth_multires");
}

int32_t fsw_compute_depth_multires_batch(fsw_context* ctx, const fsw_planeset* planes_low, const fsw_planeset* planes_crop,
                                         const fsw_sweep_params* params_low, const fsw_sweep_params* params_crop,
                                         fsw_rect crop, int32_t n_sets, const fsw_image* images,
                                         const uint8_t* const* masks, size_t mask_pitch, const fsw_depth_out* outs,
                                         void* cuda_stream) {
    return run_multires(ctx, planes_low, planes_crop, params_low, params_crop, crop, n_sets, images, masks, mask_pitch,
                        outs, cuda_stream, "fsw_compute_depth_multires_batch");
}

/* ---- host-buffer variants ------------------------------------------------------------------------------------- */
static int32_t run_host(fsw_context* ctx, bool multires, const fsw_planeset* p0, const fsw_planeset* p1,
                        const fsw_sweep_params* q0, const fsw_sweep_params* q1, fsw_rect crop, int32_t n_sets,
                        const fsw_image* images, const uint8_t* const* masks, size_t mask_pitch,
                        const fsw_depth_out* outs, void* cuda_stream) {
    if (!ctx) return fail(FSW_E_INVALID_ARG, "null context");
    if (n_sets < 1 || n_sets > FSW_MAX_BATCH) return fail(FSW_E_INVALID_ARG, "n_sets=%d must be in 1..%d", n_sets, FSW_MAX_BATCH);
    if (!images || !outs) return fail(FSW_E_INVALID_ARG, "null images or outputs");
    int32_t rc;
    const fsw_rig& rig = ctx->rig;
    for (int s = 0; s < n_sets; ++s) {
        if ((rc = check_images(rig, images + (size_t)s * rig.n_cams)) != FSW_OK) return rc;
        if ((rc = check_out(rig, &outs[s], masks ? masks[s] : nullptr, mask_pitch)) != FSW_OK) return rc;
    }
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    DeviceGuard g;
    FSW_CUDA(g.enter(ctx->device));
    const int W = rig.cams[rig.ref_index].width, H = rig.cams[rig.ref_index].height;
    const size_t ns = (size_t)n_sets;
    if (ctx->st_img.size() < ns * FSW_MAX_CAMERAS) ctx->st_img.resize(ns * FSW_MAX_CAMERAS);
    for (std::vector<DevBuf>* v : {&ctx->st_mask, &ctx->st_depth, &ctx->st_c1, &ctx->st_c2, &ctx->st_k, &ctx->st_reason})
        if (v->size() < ns) v->resize(ns);
    std::vector<fsw_image> dimg(ns * rig.n_cams);
    std::vector<const uint8_t*> dmask(ns, nullptr);
    std::vector<fsw_depth_out> dout(ns);
    for (int s = 0; s < n_sets; ++s) {
        for (int c = 0; c < rig.n_cams; ++c) {
            const fsw_image& im = images[(size_t)s * rig.n_cams + c];
            const size_t es = im.dtype == FSW_U8 ? 1 : 4;
            const size_t row = es * (size_t)rig.cams[c].width;
            DevBuf& b = ctx->st_img[(size_t)s * FSW_MAX_CAMERAS + c];
            FSW_CUDA(b.reserve(row * rig.cams[c].height));
            FSW_CUDA(cudaMemcpy2DAsync(b.p, row, im.data, im.pitch_bytes, row, rig.cams[c].height, cudaMemcpyHostToDevice, stream));
            fsw_image& d = dimg[(size_t)s * rig.n_cams + c];
            d.data = b.p; d.pitch_bytes = row; d.dtype = im.dtype;
        }
        if (masks && masks[s]) {
            FSW_CUDA(ctx->st_mask[s].reserve((size_t)W * H));
            FSW_CUDA(cudaMemcpy2DAsync(ctx->st_mask[s].p, W, masks[s], mask_pitch, W, H, cudaMemcpyHostToDevice, stream));
            dmask[s] = (const uint8_t*)ctx->st_mask[s].p;
        }
        fsw_depth_out& o = dout[s];
        std::memset(&o, 0, sizeof(o));
        o.struct_size = sizeof(o);
        FSW_CUDA(ctx->st_depth[s].reserve((size_t)W * H * 4));
        o.depth = (float*)ctx->st_depth[s].p; o.depth_pitch = (size_t)W * 4;
        if (outs[s].best_cost) { FSW_CUDA(ctx->st_c1[s].reserve((size_t)W * H * 4)); o.best_cost = (float*)ctx->st_c1[s].p; o.best_cost_pitch = (size_t)W * 4; }
        if (outs[s].second_cost) { FSW_CUDA(ctx->st_c2[s].reserve((size_t)W * H * 4)); o.second_cost = (float*)ctx->st_c2[s].p; o.second_cost_pitch = (size_t)W * 4; }
        if (outs[s].plane_index) { FSW_CUDA(ctx->st_k[s].reserve((size_t)W * H * 2)); o.plane_index = (int16_t*)ctx->st_k[s].p; o.plane_index_pitch = (size_t)W * 2; }
        if (outs[s].valid_reason) { FSW_CUDA(ctx->st_reason[s].reserve((size_t)W * H)); o.valid_reason = (uint8_t*)ctx->st_reason[s].p; o.valid_reason_pitch = (size_t)W; }
    }
    bool any_mask = false;
    for (int s = 0; s < n_sets; ++s) any_mask = any_mask || dmask[s] != nullptr;
    if (multires) rc = run_multires(ctx, p0, p1, q0, q1, crop, n_sets, dimg.data(), any_mask ? dmask.data() : nullptr, (size_t)W, dout.data(), cuda_stream, "fsw_compute_depth_multires_host");
    else rc = run_sets(ctx, p0, q0, n_sets, dimg.data(), any_mask ? dmask.data() : nullptr, (size_t)W, dout.data(), cuda_stream, "fsw_compute_depth_host");
    if (rc != FSW_OK) return rc;
    for (int s = 0; s < n_sets; ++s) {
        const fsw_depth_out& o = dout[s];
        const fsw_depth_out* out = &outs[s];
        FSW_CUDA(cudaMemcpy2DAsync(out->depth, out->depth_pitch, o.depth, o.depth_pitch, (size_t)W * 4, H, cudaMemcpyDeviceToHost, stream));
        if (out->best_cost) FSW_CUDA(cudaMemcpy2DAsync(out->best_cost, out->best_cost_pitch, o.best_cost, o.best_cost_pitch, (size_t)W * 4, H, cudaMemcpyDeviceToHost, stream));
        if (out->second_cost) FSW_CUDA(cudaMemcpy2DAsync(out->second_cost, out->second_cost_pitch, o.second_cost, o.second_cost_pitch, (size_t)W * 4, H, cudaMemcpyDeviceToHost, stream));
        if (out->plane_index) FSW_CUDA(cudaMemcpy2DAsync(out->plane_index, out->plane_index_pitch, o.plane_index, o.plane_index_pitch, (size_t)W * 2, H, cudaMemcpyDeviceToHost, stream));
        if (out->valid_reason) FSW_CUDA(cudaMemcpy2DAsync(out->valid_reason, out->valid_reason_pitch, o.valid_reason, o.valid_reason_pitch, (size_t)W, H, cudaMemcpyDeviceToHost, stream));
    }
    if (!ctx->host_async) FSW_CUDA(cudaStreamSynchronize(stream));
    return FSW_OK;
}

int32_t fsw_compute_depth_host(fsw_context* ctx, const fsw_planeset* planes, const fsw_sweep_params* params,
                               const fsw_image* images, const uint8_t* mask, size_t mask_pitch,
                               const fsw_depth_out* out, void* cuda_stream) {
    fsw_rect none = {0, 0, 0, 0};
    const uint8_t* masks[1] = {mask};
    return run_host(ctx, false, planes, nullptr, params, nullptr, none, 1, images, mask ? masks : nullptr, mask_pitch, out, cuda_stream);
}

int32_t fsw_compute_depth_batch_host(fsw_context* ctx, const fsw_planeset* planes, const fsw_sweep_params* params,
                                     int32_t n_sets, const fsw_image* images, const uint8_t* const* masks,
                                     size_t mask_pitch, const fsw_depth_out* outs, void* cuda_stream) {
    fsw_rect none = {0, 0, 0, 0};
    return run_host(ctx, false, planes, nullptr, params, nullptr, none, n_sets, images, masks, mask_pitch, outs, cuda_stream);
}

int32_t fsw_compute_depth_multires_host(fsw_context* ctx, const fsw_planeset* planes_low,
                                        const fsw_planeset* planes_crop, const fsw_sweep_params* params_low,
                                        const fsw_sweep_params* params_crop, fsw_rect crop, const fsw_image* images,
                                        const uint8_t* mask, size_t mask_pitch, const fsw_depth_out* out,
                                        void* cuda_stream) {
    const uint8_t* masks[1] = {mask};
    return run_host(ctx, true, planes_low, planes_crop, params_low, params_crop, crop, 1, images, mask ? masks : nullptr, mask_pitch, out, cuda_stream);
}

int32_t fsw_compute_depth_multires_batch_host(fsw_context* ctx, const fsw_planeset* planes_low,
                                              const fsw_planeset* planes_crop, const fsw_sweep_params* params_low,
                                              const fsw_sweep_params* params_crop, fsw_rect crop, int32_t n_sets,
                                              const fsw_image* images, const uint8_t* const* masks, size_t mask_pitch,
                                              const fsw_depth_out* outs, void* cuda_stream) {
    return run_host(ctx, true, planes_low, planes_crop, params_low, params_crop, crop, n_sets, images, masks, mask_pitch, outs, cuda_stream);
}

int32_t fsw_filter_continuity(fsw_context* ctx, const float* depth_in, size_t depth_in_pitch, int32_t window,
                              double gamma, double delta, const uint8_t* mask, size_t mask_pitch,
                              float* depth_out, size_t depth_out_pitch, uint8_t* reason_out, size_t reason_pitch,
                              void* cuda_stream) {
    if (!ctx || !depth_in || !depth_out) return fail(FSW_E_INVALID_ARG, "fsw_filter_continuity: null context or depth buffer");
    if (window < 3 || window > FSW_MAX_WINDOW || window % 2 == 0)
        return fail(FSW_E_INVALID_ARG, "fsw_filter_continuity: window=%d must be odd and in 3..%d", window, FSW_MAX_WINDOW);
    if (!(gamma > 0.0) || !(delta >= 0.0 && delta <= 1.0))
        return fail(FSW_E_INVALID_ARG, "fsw_filter_continuity: gamma=%g must be > 0 and delta=%g in [0,1]", gamma, delta);
    const fsw_camera& ref = ctx->rig.cams[ctx->rig.ref_index];
    const int W = ref.width, H = ref.height;
    if (depth_in_pitch < (size_t)W * 4 || depth_out_pitch < (size_t)W * 4 || (mask && mask_pitch < (size_t)W) ||
        (reason_out && reason_pitch < (size_t)W))
        return fail(FSW_E_INVALID_ARG, "fsw_filter_continuity: a pitch is smaller than one row of %d pixels", W);
    const char* i0 = (const char*)depth_in; const char* i1 = i0 + depth_in_pitch * (size_t)H;
    const char* o0 = (const char*)depth_out; const char* o1 = o0 + depth_out_pitch * (size_t)H;
    if (i0 < o1 && o0 < i1) return fail(FSW_E_INVALID_ARG, "fsw_filter_continuity: depth_out overlaps depth_in");
    DeviceGuard g;
    FSW_CUDA(g.enter(ctx->device));
    FswContinuityArgs a;
    a.in = depth_in; a.in_pitch = (int64_t)depth_in_pitch;
    a.out = depth_out; a.out_pitch = (int64_t)depth_out_pitch;
    a.mask = mask; a.mask_pitch = (int64_t)mask_pitch;
    a.reason = reason_out; a.reason_pitch = (int64_t)reason_pitch;
    a.W = W; a.H = H; a.window = window;
    a.gamma = gamma; a.delta = delta;
    FSW_CUDA(fsw_launch_continuity(a, (cudaStream_t)cuda_stream));
    return FSW_OK;
}

int32_t fsw_context_set_host_async(fsw_context* ctx, int32_t on) {
    if (!ctx) return fail(FSW_E_INVALID_ARG, "fsw_context_set_host_async: null context");
    ctx->host_async = on != 0;
    return FSW_OK;
}

int32_t fsw_plan_schedule(const fsw_rig* rig, const fsw_planeset* planes, const fsw_sweep_params* params, int32_t n_sets,
                          int32_t n_blocks, int32_t capacity, int32_t* tile_order, float* tile_weight,
                          fsw_schedule_plan* out) {
    if (!rig || !planes || !out) return fail(FSW_E_INVALID_ARG, "fsw_plan_schedule: null argument");
    if (out->struct_size != sizeof(fsw_schedule_plan))
        return fail(FSW_E_INVALID_ARG, "fsw_plan_schedule: struct_size %u != %zu", out->struct_size, sizeof(fsw_schedule_plan));
    int32_t rc = check_params(params, "params");
    if (rc != FSW_OK) return rc;
    if (n_sets < 1 || n_sets > FSW_MAX_BATCH || n_blocks < 1 || capacity < 0 || (capacity > 0 && (!tile_order || !tile_weight)))
        return fail(FSW_E_INVALID_ARG, "fsw_plan_schedule: n_sets=%d n_blocks=%d capacity=%d", n_sets, n_blocks, capacity);
    FswSweepArgs a;
    fill_args(a, *rig, *planes, *params, false);
    const FswSweepGeometry g = window_geometry(params->window, a.n_views);
    TileOrder t;
    plan_tiles(a, g, params->window / 2, &t);
    const long long slots = (long long)n_blocks * g.ctas_per_sm;
    const bool short_queue = (long long)t.n_live * n_sets < 3 * slots;
    out->tile_w = g.tile_w; out->tile_h = g.tile_h;
    out->n_tiles_x = t.n_tiles_x; out->n_tiles = t.n_tiles; out->n_live = t.n_live;
    out->by_weight = short_queue ? 1 : 0;
    const long long total_slots = (long long)t.n_tiles * n_sets;
    out->n_whole_slots = (short_queue && a.n_planes >= 2) ? split_whole_for(&t, n_sets, slots) : total_slots;
    out->n_halved_slots = total_slots - out->n_whole_slots;
    const std::vector<int32_t>& order = short_queue ? t.order_w : t.order_d;
    std::vector<float> w_by_tile((size_t)t.n_tiles);
    for (int i = 0; i < t.n_tiles; ++i) w_by_tile[(size_t)t.order_w[(size_t)i]] = t.weight[(size_t)i];
    for (int i = 0; i < t.n_tiles && i < capacity; ++i) {
        tile_order[i] = order[(size_t)i];
        tile_weight[i] = w_by_tile[(size_t)order[(size_t)i]];
    }
    return FSW_OK;
}

int32_t fsw_context_set_split(fsw_context* ctx, int32_t mode) {
    if (!ctx) return fail(FSW_E_INVALID_ARG, "fsw_context_set_split: null context");
    if (mode != FSW_SPLIT_AUTO && mode != FSW_SPLIT_OFF && mode != FSW_SPLIT_ON)
        return fail(FSW_E_INVALID_ARG, "fsw_context_set_split: mode %d", mode);
    ctx->split_mode = mode;
    return FSW_OK;
}

int32_t fsw_context_set_timing(fsw_context* ctx, int32_t on) {
    if (!ctx) return fail(FSW_E_INVALID_ARG, "fsw_context_set_timing: null context");
    DeviceGuard g;
    FSW_CUDA(g.enter(ctx->device));
    if (on && !ctx->ev[0])
        for (int i = 0; i < 4; ++i) FSW_CUDA(cudaEventCreate(&ctx->ev[i]));
    ctx->timing = on != 0;
    if (!on) ctx->n_timed = 0;
    return FSW_OK;
}

int32_t fsw_get_last_counters(fsw_context* ctx, fsw_counters* out) {
    if (!ctx || !out) return fail(FSW_E_INVALID_ARG, "fsw_get_last_counters: null argument");
    if (out->struct_size != sizeof(fsw_counters)) return fail(FSW_E_INVALID_ARG, "fsw_get_last_counters: struct_size %u != %zu", out->struct_size, sizeof(fsw_counters));
    DeviceGuard g;
    FSW_CUDA(g.enter(ctx->device));
    FSW_CUDA(cudaStreamSynchronize(ctx->last_stream));
    unsigned long long h[4] = {0, 0, 0, 0};
    FSW_CUDA(cudaMemcpy(h, ctx->counters(), sizeof(h), cudaMemcpyDeviceToHost));
    out->n_eval = (int64_t)h[0];
    out->n_raw_valid = (int64_t)h[1];
    out->n_valid = (int64_t)h[2];
    out->n_split_launches = ctx->last_split;
    out->n_launches = ctx->last_launches;
    out->sweep_ms = -1.0;
    if (ctx->n_timed > 0) {
        float t = 0.f, t2 = 0.f;
        FSW_CUDA(cudaEventElapsedTime(&t, ctx->ev[0], ctx->ev[1]));
        if (ctx->n_timed > 1) FSW_CUDA(cudaEventElapsedTime(&t2, ctx->ev[2], ctx->ev[3]));
        out->sweep_ms = (double)t + (double)t2;
    }
    return FSW_OK;
}

}  /* extern "C" */

/* ================================================================================================================
 * fsw_compute_depth_static: the single-frame-set sweep for callers that may not allocate device memory.
 *
 * Every byte of device scratch the call needs -- the work-queue word, the tile schedule and the footprint images of
 * the matching views (S4 staging) -- lives in ONE file-scope array of FSW_STATIC_SCRATCH_BYTES that is part of the
 * library image: every GPU that loads libfsw.so holds it until the process exits.  In host code the array's name is
 * only a host-side stand-in for the symbol, not a device address; the address the kernels get comes from
 * cudaGetSymbolAddress, resolved once per device with that device current (static_scratch_for_device).
 * ================================================================================================================ */
static __device__ __align__(256) unsigned char g_fsw_static_scratch[FSW_STATIC_SCRATCH_BYTES];

/* the tile schedule reaches the array through kernel parameters (no copy from pageable host memory, so that even a
 * call that changes the schedule is a pure sequence of kernel launches); device code of this file names the array
 * directly */
struct FswWordChunk {
    int32_t n, first; /* w[0..n) go to words first .. first + n - 1 of the schedule */
    int32_t w[960];
};
static __global__ void static_schedule_kernel(const __grid_constant__ FswWordChunk c, uint32_t schedule_offset_bytes) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < c.n) reinterpret_cast<int32_t*>(g_fsw_static_scratch + schedule_offset_bytes)[c.first + i] = c.w[i];
}

namespace {

constexpr int FSW_STATIC_MAX_DEVICES = 64;
constexpr size_t FSW_STATIC_ALIGN = 256;
constexpr size_t FSW_STATIC_MAX_TILES = 16384; /* tile schedule entries: 64 KiB of the array */

struct StaticScratchDev {
    unsigned char* base = nullptr; /* device address of g_fsw_static_scratch on this device */
};
StaticScratchDev g_static_dev[FSW_STATIC_MAX_DEVICES];
std::mutex g_static_mutex;

size_t align_up(size_t n) { return (n + FSW_STATIC_ALIGN - 1) / FSW_STATIC_ALIGN * FSW_STATIC_ALIGN; }

/* set-up, once per device, `device` current: the device address of the static array */
int32_t static_scratch_for_device(int device, StaticScratchDev** out) {
    if (device < 0 || device >= FSW_STATIC_MAX_DEVICES) return fail(FSW_E_UNSUPPORTED, "fsw_compute_depth_static: device %d beyond %d", device, FSW_STATIC_MAX_DEVICES);
    StaticScratchDev& d = g_static_dev[device];
    if (!d.base) {
        unsigned char* p = nullptr;
        cudaError_t e = cudaGetSymbolAddress((void**)&p, g_fsw_static_scratch);
        if (e != cudaSuccess) return cuda_fail(e, "fsw_compute_depth_static: cudaGetSymbolAddress of the static scratch array");
        if (!p || ((uintptr_t)p % FSW_STATIC_ALIGN) != 0) return fail(FSW_E_CUDA, "fsw_compute_depth_static: the static scratch array has no aligned device address");
        d.base = p;
    }
    *out = &d;
    return FSW_OK;
}

}  // namespace

extern "C" {

int32_t fsw_compute_depth_static(fsw_context* ctx, const fsw_planeset* planes, const fsw_sweep_params* params,
                                 const fsw_image* images, const uint8_t* mask, size_t mask_pitch,
                                 const fsw_depth_out* out, void* cuda_stream) {
    const char* who = "fsw_compute_depth_static";
    if (!ctx || !planes) return fail(FSW_E_INVALID_ARG, "%s: null context or plane set", who);
    int32_t rc;
    if ((rc = check_params(params, "params")) != FSW_OK) return rc;
    if (!images || !out) return fail(FSW_E_INVALID_ARG, "%s: null images or outputs", who);
    const fsw_rig& rig = ctx->rig;
    if ((rc = check_images(rig, images)) != FSW_OK) return rc;
    if ((rc = check_out(rig, out, mask, mask_pitch)) != FSW_OK) return rc;

    /* layout of the array: [0, 256) queue words; the tile schedule; one footprint image per view, each 256-aligned */
    int f16 = 1;
    for (int c = 0; c < rig.n_cams; ++c)
        if (c != rig.ref_index && images[c].dtype != FSW_U8) f16 = 0;
    FswSweepArgs a;
    fill_args(a, rig, *planes, *params, false);
    a.foot_f16 = f16;
    const FswSweepGeometry g = window_geometry(params->window, a.n_views);
    const int ntx = (a.ref.W + g.tile_w - 1) / g.tile_w, nty = (a.ref.H + g.tile_h - 1) / g.tile_h;
    const size_t n_tiles = (size_t)ntx * (size_t)nty;
    if (n_tiles > FSW_STATIC_MAX_TILES)
        return fail(FSW_E_UNSUPPORTED, "%s: %zu tiles of %d x %d pixels, the static tile schedule holds %zu", who, n_tiles, g.tile_w, g.tile_h, FSW_STATIC_MAX_TILES);
    const size_t off_order = FSW_STATIC_ALIGN;
    size_t need = off_order + align_up(sizeof(int32_t) * n_tiles);
    size_t off_foot[FSW_MAX_CAMERAS];
    for (int c = 0; c < rig.n_cams; ++c) {
        off_foot[c] = need;
        if (c == rig.ref_index) continue;
        need += align_up((size_t)rig.cams[c].width * (size_t)rig.cams[c].height * (f16 ? 8u : 16u));
    }
    if (need > (size_t)FSW_STATIC_SCRATCH_BYTES)
        return fail(FSW_E_UNSUPPORTED, "%s: this rig needs %zu bytes of scratch (%d bytes per view pixel), the static array holds %zu: use fsw_compute_depth",
                    who, need, f16 ? 8 : 16, (size_t)FSW_STATIC_SCRATCH_BYTES);

    cudaStream_t stream = (cudaStream_t)cuda_stream;
    DeviceGuard dg;
    FSW_CUDA(dg.enter(ctx->device));
    std::lock_guard<std::mutex> lock(g_static_mutex);
    StaticScratchDev* sd = nullptr;
    if ((rc = static_scratch_for_device(ctx->device, &sd)) != FSW_OK) return rc;
    FSW_CUDA(prepare_window(ctx, params->window)); /* function attributes only */
    unsigned char* const base = sd->base;

    /* S0: tile schedule, written on every call (one small launch): a captured graph that replays an older call may
     * have put another schedule into the array since, which the host cannot know */
    const long long slots = (long long)ctx->n_sm * g.ctas_per_sm;
    TileOrder plan;
    plan_tiles(a, g, params->window / 2, &plan);
    const bool short_queue = (long long)plan.n_live < 3 * slots;
    {
        const std::vector<int32_t>& src = short_queue ? plan.order_w : plan.order_d;
        FswWordChunk chunk;
        for (size_t first = 0; first < n_tiles; first += 960) {
            chunk.n = (int32_t)std::min<size_t>(960, n_tiles - first);
            chunk.first = (int32_t)first;
            std::memcpy(chunk.w, src.data() + first, sizeof(int32_t) * (size_t)chunk.n);
            static_schedule_kernel<<<(chunk.n + 255) / 256, 256, 0, stream>>>(chunk, (uint32_t)off_order);
            FSW_CUDA(cudaGetLastError());
        }
    }

    /* S4 staging into the array: one pack launch per view size; the first one clears the queue word */
    FswSetPtrs set;
    std::memset(&set, 0, sizeof(set));
    const fsw_image& ri = images[rig.ref_index];
    set.ref_img = ri.data; set.ref_pitch_bytes = (int64_t)ri.pitch_bytes; set.ref_dtype = ri.dtype;
    set.debug_cost = params->debug_cost_volume;
    set_outputs(set, out, mask, mask_pitch);
    bool first = true;
    bool done[FSW_MAX_CAMERAS] = {false};
    for (int c0 = 0; c0 < rig.n_cams; ++c0) {
        if (c0 == rig.ref_index || done[c0]) continue;
        FswPackArgs pk;
        std::memset(&pk, 0, sizeof(pk));
        pk.W = rig.cams[c0].width; pk.H = rig.cams[c0].height; pk.f16 = f16;
        for (int c = c0; c < rig.n_cams; ++c) {
            if (c == rig.ref_index || done[c] || rig.cams[c].width != pk.W || rig.cams[c].height != pk.H) continue;
            done[c] = true;
            const int vi = c < rig.ref_index ? c : c - 1;
            pk.src[pk.n] = images[c].data; pk.src_pitch[pk.n] = (int64_t)images[c].pitch_bytes; pk.dtype[pk.n] = images[c].dtype;
            pk.dst[pk.n] = base + off_foot[c];
            set.foot[vi] = base + off_foot[c];
            pk.n++;
        }
        if (first) { pk.words_to_zero = (unsigned int*)base; pk.n_words_to_zero = FSW_QUEUE_WORDS; first = false; }
        FSW_CUDA(fsw_launch_pack_footprints(pk, stream));
    }

    /* the unsplit sweep kernel over every tile (the plane split would need 48 bytes of state per pixel) */
    a.n_sets = 1;
    a.set0 = set;
    a.tile_order = (const int32_t*)(base + off_order);
    a.n_tiles_x = ntx; a.n_tiles = (int32_t)n_tiles;
    a.queue = (unsigned int*)base;
    a.counters = nullptr;
    a.count_pixels = 0;
    a.split = 0;
    a.slot_first = 0; a.slot_count = (int32_t)n_tiles;
    const long long items = (long long)n_tiles;
    cudaError_t e = fsw_launch_sweep(params->window, a, pick_variant(a, a.foot_f16), (int)(items < slots ? items : slots), stream);
    if (e != cudaSuccess) return cuda_fail(e, "sweep kernel launch");
    return FSW_OK;
}

}  /* extern "C" */
