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
#include <vector>

#include "fsw_internal.h"

/* per-window launchers, one object file each (fsw_sweep_inst.cu) */
#define FSW_DECL_WIN(w)                                                               \
    cudaError_t fsw_launch_sweep_w##w(const FswSweepArgs& args, int variant, cudaStream_t stream); \
    cudaError_t fsw_prepare_sweep_w##w();
FSW_DECL_WIN(3) FSW_DECL_WIN(5) FSW_DECL_WIN(7) FSW_DECL_WIN(9) FSW_DECL_WIN(11) FSW_DECL_WIN(13) FSW_DECL_WIN(15)
#undef FSW_DECL_WIN

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

struct fsw_context {
    fsw_rig rig;
    int32_t device;
    DevBuf foot[FSW_MAX_CAMERAS];  /* footprint-packed 8-bit views */
    DevBuf half[FSW_MAX_CAMERAS];  /* half-resolution float images */
    DevBuf lo_depth, lo_c1, lo_c2, lo_k;
    DevBuf counters;               /* 4 x uint64 */
    /* staging for the *_host calls */
    DevBuf st_img[FSW_MAX_CAMERAS], st_mask, st_depth, st_c1, st_c2, st_k, st_reason;
    cudaStream_t last_stream = nullptr;
    int64_t last_launches = 0;
    bool timing = false, timed = false;
    cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr}; /* [0,1] around the (crop) sweep, [2,3] around the low sweep */
    int n_timed = 0;
    bool prepared[FSW_MAX_WINDOW + 1] = {false};
};

namespace {

/* ---- host precompute (S0) ------------------------------------------------------------------------------------ */
void relative_pose(const fsw_camera& ref, const fsw_camera& view, double* R, double* T) {
    /* X_v = R_v^c (R_ref^c)^T X_ref + (t_v - R t_ref): "known relative poses" of PAPER.md:70 from rig->camera extrinsics */
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {
            double s = 0.0;
            for (int k = 0; k < 3; ++k) s += view.R[3 * i + k] * ref.R[3 * j + k];
            R[3 * i + j] = s;
        }
    for (int i = 0; i < 3; ++i)
        T[i] = view.t[i] - (R[3 * i] * ref.t[0] + R[3 * i + 1] * ref.t[1] + R[3 * i + 2] * ref.t[2]);
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
    d.W = W; d.H = H;
    if (c.k1 == 0.0 && c.k2 == 0.0 && c.p1 == 0.0 && c.p2 == 0.0) d.dist_mode = FSW_DIST_NONE;
    else if (c.k2 == 0.0 && c.p1 == 0.0 && c.p2 == 0.0) d.dist_mode = FSW_DIST_K1;
    else d.dist_mode = FSW_DIST_FULL;
    return d;
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

/* fills the part of the argument block that depends on rig, planes and parameters */
int32_t fill_args(FswSweepArgs& a, const fsw_rig& rig, const fsw_planeset& ps, const fsw_sweep_params& p, bool half) {
    std::memset(&a, 0, sizeof(a));
    const fsw_camera& ref = rig.cams[rig.ref_index];
    a.ref = dev_cam(ref, half);
    a.n_views = 0;
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
    }
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
    const double n2 = (double)p.window * p.window * (double)p.window * p.window;
    const double fl = (double)p.var_floor * n2;
    a.floor2 = (float)(fl * fl);
    if (!(a.floor2 > 0.f)) a.floor2 = 1e-30f; /* keeps the reciprocal square root finite on flat windows */
    a.inv_range_max = 1.f / p.range_max;
    a.debug_cost = p.debug_cost_volume;
    return FSW_OK;
}

cudaError_t prepare_window(fsw_context* ctx, int w) {
    if (ctx->prepared[w]) return cudaSuccess;
    cudaError_t e = cudaErrorInvalidValue;
    switch (w) {
        case 3: e = fsw_prepare_sweep_w3(); break;
        case 5: e = fsw_prepare_sweep_w5(); break;
        case 7: e = fsw_prepare_sweep_w7(); break;
        case 9: e = fsw_prepare_sweep_w9(); break;
        case 11: e = fsw_prepare_sweep_w11(); break;
        case 13: e = fsw_prepare_sweep_w13(); break;
        case 15: e = fsw_prepare_sweep_w15(); break;
    }
    if (e == cudaSuccess) ctx->prepared[w] = true;
    return e;
}

/* picks the kernel variant the views allow (see fsw_sweep.cuh) */
int pick_variant(const FswSweepArgs& a) {
    bool ident = true, k1only = true, all_u8 = true, all_f32 = true;
    for (int v = 0; v < a.n_views; ++v) {
        ident = ident && a.views[v].ident_R;
        k1only = k1only && a.views[v].cam.dist_mode != FSW_DIST_FULL;
        k1only = k1only && (a.views[v].cam.cos_fov + a.views[v].cam.xi >= 1e-3f); /* lets the kernel drop the den test */
        all_u8 = all_u8 && a.views[v].pix_mode == FSW_PIX_FOOT_U8;
        all_f32 = all_f32 && a.views[v].pix_mode == FSW_PIX_F32;
    }
    if (ident && k1only && all_u8) return 1;
    if (ident && k1only && all_f32) return 2;
    return 0;
}

cudaError_t launch_window(const FswSweepArgs& a, int w, cudaStream_t s) {
    const int var = pick_variant(a);
    switch (w) {
        case 3: return fsw_launch_sweep_w3(a, var, s);
        case 5: return fsw_launch_sweep_w5(a, var, s);
        case 7: return fsw_launch_sweep_w7(a, var, s);
        case 9: return fsw_launch_sweep_w9(a, var, s);
        case 11: return fsw_launch_sweep_w11(a, var, s);
        case 13: return fsw_launch_sweep_w13(a, var, s);
        case 15: return fsw_launch_sweep_w15(a, var, s);
    }
    return cudaErrorInvalidValue;
}

/* makes the device representation of every matching view: 8-bit images are footprint-packed into context scratch
 * (one launch for all of them), float images are used in place */
int32_t stage_views(fsw_context* ctx, const fsw_image* images, FswSweepArgs& a, cudaStream_t stream, bool zero_counters,
                    bool* zeroed) {
    const fsw_rig& rig = ctx->rig;
    FswPackArgs pk;
    std::memset(&pk, 0, sizeof(pk));
    int vi = 0;
    for (int c = 0; c < rig.n_cams; ++c) {
        if (c == rig.ref_index) continue;
        FswDevView& v = a.views[vi++];
        const int W = rig.cams[c].width, H = rig.cams[c].height;
        if (images[c].dtype == FSW_U8) {
            FSW_CUDA(ctx->foot[c].reserve((size_t)W * H * 4));
            pk.src[pk.n] = (const uint8_t*)images[c].data;
            pk.src_pitch[pk.n] = (int64_t)images[c].pitch_bytes;
            pk.dst[pk.n] = (uint32_t*)ctx->foot[c].p;
            pk.W[pk.n] = W; pk.H[pk.n] = H;
            pk.n++;
            v.pix_mode = FSW_PIX_FOOT_U8;
            v.img = ctx->foot[c].p;
            v.pitch_elems = W;
        } else {
            v.pix_mode = FSW_PIX_F32;
            v.img = images[c].data;
            v.pitch_elems = (int64_t)(images[c].pitch_bytes / 4);
        }
    }
    *zeroed = false;
    if (pk.n > 0) {
        pk.counters_to_zero = zero_counters ? (unsigned long long*)ctx->counters.p : nullptr;
        FSW_CUDA(fsw_launch_pack_footprints(pk, stream));
        ctx->last_launches++;
        *zeroed = zero_counters;
    }
    return FSW_OK;
}

void set_outputs(FswSweepArgs& a, const fsw_depth_out* out, const uint8_t* mask, size_t mask_pitch) {
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
        double s0 = F.spacing == FSW_INVERSE ? 1.0 / F.d_first : F.d_first;
        double s1 = F.spacing == FSW_INVERSE ? 1.0 / F.d_last : F.d_last;
        for (int k = 0; k < F.n_planes; ++k) {
            double sk = F.n_planes > 1 ? s0 + (double)k * (s1 - s0) / (double)(F.n_planes - 1) : s0;
            ps->s.push_back(sk);
            ps->d.push_back(F.spacing == FSW_INVERSE ? 1.0 / sk : sk);
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
    DeviceGuard g;
    e = g.enter(cuda_device);
    if (e == cudaSuccess) e = ctx->counters.reserve(4 * sizeof(unsigned long long));
    if (e == cudaSuccess) e = cudaMemset(ctx->counters.p, 0, 4 * sizeof(unsigned long long));
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
    for (int c = 0; c < FSW_MAX_CAMERAS; ++c) {
        ctx->foot[c].release(); ctx->half[c].release(); ctx->st_img[c].release();
    }
    ctx->lo_depth.release(); ctx->lo_c1.release(); ctx->lo_c2.release(); ctx->lo_k.release(); ctx->counters.release();
    for (int i = 0; i < 4; ++i)
        if (ctx->ev[i]) cudaEventDestroy(ctx->ev[i]);
    ctx->st_mask.release(); ctx->st_depth.release(); ctx->st_c1.release(); ctx->st_c2.release(); ctx->st_k.release(); ctx->st_reason.release();
    delete ctx;
    return FSW_OK;
}

int32_t fsw_compute_depth(fsw_context* ctx, const fsw_planeset* planes, const fsw_sweep_params* params,
                          const fsw_image* images, const uint8_t* mask, size_t mask_pitch,
                          const fsw_depth_out* out, void* cuda_stream) {
    if (!ctx || !planes) return fail(FSW_E_INVALID_ARG, "fsw_compute_depth: null context or plane set");
    int32_t rc;
    if ((rc = check_params(params, "params")) != FSW_OK) return rc;
    if ((rc = check_images(ctx->rig, images)) != FSW_OK) return rc;
    if ((rc = check_out(ctx->rig, out, mask, mask_pitch)) != FSW_OK) return rc;
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    DeviceGuard g;
    FSW_CUDA(g.enter(ctx->device));
    FSW_CUDA(prepare_window(ctx, params->window));
    ctx->last_stream = stream;
    ctx->last_launches = 0;

    FswSweepArgs a;
    fill_args(a, ctx->rig, *planes, *params, false);
    const fsw_image& ri = images[ctx->rig.ref_index];
    a.ref_img = ri.data; a.ref_pitch_bytes = (int64_t)ri.pitch_bytes; a.ref_dtype = ri.dtype;
    bool zeroed = false;
    if ((rc = stage_views(ctx, images, a, stream, true, &zeroed)) != FSW_OK) return rc;
    if (!zeroed) FSW_CUDA(cudaMemsetAsync(ctx->counters.p, 0, 4 * sizeof(unsigned long long), stream));
    set_outputs(a, out, mask, mask_pitch);
    a.counters = (unsigned long long*)ctx->counters.p;
    a.count_pixels = 1;
    ctx->n_timed = 0;
    if (ctx->timing) FSW_CUDA(cudaEventRecord(ctx->ev[0], stream));
    FSW_CUDA(launch_window(a, params->window, stream));
    if (ctx->timing) { FSW_CUDA(cudaEventRecord(ctx->ev[1], stream)); ctx->n_timed = 1; }
    ctx->last_launches++;
    return FSW_OK;
}

int32_t fsw_compute_depth_multires(fsw_context* ctx, const fsw_planeset* planes_low, const fsw_planeset* planes_crop,
                                   const fsw_sweep_params* params_low, const fsw_sweep_params* params_crop,
                                   fsw_rect crop, const fsw_image* images, const uint8_t* mask, size_t mask_pitch,
                                   const fsw_depth_out* out, void* cuda_stream) {
    if (!ctx || !planes_low || !planes_crop) return fail(FSW_E_INVALID_ARG, "fsw_compute_depth_multires: null context or plane set");
    int32_t rc;
    if ((rc = check_params(params_low, "params_low")) != FSW_OK) return rc;
    if ((rc = check_params(params_crop, "params_crop")) != FSW_OK) return rc;
    if ((rc = check_images(ctx->rig, images)) != FSW_OK) return rc;
    if ((rc = check_out(ctx->rig, out, mask, mask_pitch)) != FSW_OK) return rc;
    const fsw_rig& rig = ctx->rig;
    const fsw_camera& ref = rig.cams[rig.ref_index];
    if (crop.w <= 0 || crop.h <= 0 || crop.x0 < 0 || crop.y0 < 0 || crop.x0 + crop.w > ref.width || crop.y0 + crop.h > ref.height)
        return fail(FSW_E_INVALID_ARG, "fsw_compute_depth_multires: crop (%d,%d,%d,%d) not inside the reference image", crop.x0, crop.y0, crop.w, crop.h);
    if (params_low->debug_cost_volume || params_crop->debug_cost_volume)
        return fail(FSW_E_UNSUPPORTED, "fsw_compute_depth_multires: debug_cost_volume is only available in fsw_compute_depth");
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    DeviceGuard g;
    FSW_CUDA(g.enter(ctx->device));
    FSW_CUDA(prepare_window(ctx, params_low->window));
    FSW_CUDA(prepare_window(ctx, params_crop->window));
    ctx->last_stream = stream;
    ctx->last_launches = 0;

    /* S10(a): 2x2 box downsample of every image */
    FswDownArgs dn;
    std::memset(&dn, 0, sizeof(dn));
    dn.n = rig.n_cams;
    for (int c = 0; c < rig.n_cams; ++c) {
        const int W = rig.cams[c].width, H = rig.cams[c].height;
        FSW_CUDA(ctx->half[c].reserve((size_t)(W / 2) * (H / 2) * 4));
        dn.src[c] = images[c].data; dn.src_pitch[c] = (int64_t)images[c].pitch_bytes; dn.dtype[c] = images[c].dtype;
        dn.dst[c] = (float*)ctx->half[c].p; dn.W[c] = W; dn.H[c] = H;
    }
    dn.counters_to_zero = (unsigned long long*)ctx->counters.p;
    FSW_CUDA(fsw_launch_downsample(dn, stream));
    ctx->last_launches++;

    /* S10(b): half-resolution sweep over the whole field of view, raw maps into context scratch */
    const int LW = ref.width / 2, LH = ref.height / 2;
    FSW_CUDA(ctx->lo_depth.reserve((size_t)LW * LH * 4));
    FSW_CUDA(ctx->lo_c1.reserve((size_t)LW * LH * 4));
    FSW_CUDA(ctx->lo_c2.reserve((size_t)LW * LH * 4));
    FSW_CUDA(ctx->lo_k.reserve((size_t)LW * LH * 2));
    FswSweepArgs a;
    fsw_sweep_params pl = *params_low;
    pl.filters_enabled = 0; /* filters run after the merge (reading Q20) */
    fill_args(a, rig, *planes_low, pl, true);
    a.ref_img = ctx->half[rig.ref_index].p; a.ref_pitch_bytes = (int64_t)LW * 4; a.ref_dtype = FSW_F32;
    {
        int vi = 0;
        for (int c = 0; c < rig.n_cams; ++c) {
            if (c == rig.ref_index) continue;
            FswDevView& v = a.views[vi++];
            v.pix_mode = FSW_PIX_F32; v.img = ctx->half[c].p; v.pitch_elems = rig.cams[c].width / 2;
        }
    }
    a.out_depth = (float*)ctx->lo_depth.p; a.out_depth_pitch = (int64_t)LW * 4;
    a.out_c1 = (float*)ctx->lo_c1.p; a.out_c1_pitch = (int64_t)LW * 4;
    a.out_c2 = (float*)ctx->lo_c2.p; a.out_c2_pitch = (int64_t)LW * 4;
    a.out_k = (int16_t*)ctx->lo_k.p; a.out_k_pitch = (int64_t)LW * 2;
    a.counters = (unsigned long long*)ctx->counters.p;
    a.count_pixels = 0;
    ctx->n_timed = 0;
    if (ctx->timing) FSW_CUDA(cudaEventRecord(ctx->ev[2], stream));
    FSW_CUDA(launch_window(a, params_low->window, stream));
    if (ctx->timing) FSW_CUDA(cudaEventRecord(ctx->ev[3], stream));
    ctx->last_launches++;

    /* S10(d)-(e) + S9 + S11: full-resolution sweep inside the crop, merged with the upsampled maps in its epilogue */
    fsw_sweep_params pc = *params_crop;
    pc.roi = crop;
    fill_args(a, rig, *planes_crop, pc, false);
    const fsw_image& ri = images[rig.ref_index];
    a.ref_img = ri.data; a.ref_pitch_bytes = (int64_t)ri.pitch_bytes; a.ref_dtype = ri.dtype;
    bool zeroed = false;
    if ((rc = stage_views(ctx, images, a, stream, false, &zeroed)) != FSW_OK) return rc;
    set_outputs(a, out, mask, mask_pitch);
    a.lo_depth = (const float*)ctx->lo_depth.p; a.lo_c1 = (const float*)ctx->lo_c1.p; a.lo_c2 = (const float*)ctx->lo_c2.p;
    a.lo_k = (const int16_t*)ctx->lo_k.p; a.lo_W = LW; a.lo_H = LH;
    a.index_flag = FSW_INDEX_FROM_CROP;
    a.counters = (unsigned long long*)ctx->counters.p;
    a.count_pixels = 1;
    if (ctx->timing) FSW_CUDA(cudaEventRecord(ctx->ev[0], stream));
    FSW_CUDA(launch_window(a, params_crop->window, stream));
    if (ctx->timing) { FSW_CUDA(cudaEventRecord(ctx->ev[1], stream)); ctx->n_timed = 2; }
    ctx->last_launches++;
    return FSW_OK;
}

/* ---- host-buffer variants ------------------------------------------------------------------------------------- */
static int32_t run_host(fsw_context* ctx, bool multires, const fsw_planeset* p0, const fsw_planeset* p1,
                        const fsw_sweep_params* q0, const fsw_sweep_params* q1, fsw_rect crop, const fsw_image* images,
                        const uint8_t* mask, size_t mask_pitch, const fsw_depth_out* out, void* cuda_stream) {
    if (!ctx) return fail(FSW_E_INVALID_ARG, "null context");
    int32_t rc;
    if ((rc = check_images(ctx->rig, images)) != FSW_OK) return rc;
    if ((rc = check_out(ctx->rig, out, mask, mask_pitch)) != FSW_OK) return rc;
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    DeviceGuard g;
    FSW_CUDA(g.enter(ctx->device));
    const fsw_rig& rig = ctx->rig;
    const int W = rig.cams[rig.ref_index].width, H = rig.cams[rig.ref_index].height;
    fsw_image dimg[FSW_MAX_CAMERAS];
    for (int c = 0; c < rig.n_cams; ++c) {
        const size_t es = images[c].dtype == FSW_U8 ? 1 : 4;
        const size_t row = es * (size_t)rig.cams[c].width;
        FSW_CUDA(ctx->st_img[c].reserve(row * rig.cams[c].height));
        FSW_CUDA(cudaMemcpy2DAsync(ctx->st_img[c].p, row, images[c].data, images[c].pitch_bytes, row, rig.cams[c].height, cudaMemcpyHostToDevice, stream));
        dimg[c].data = ctx->st_img[c].p; dimg[c].pitch_bytes = row; dimg[c].dtype = images[c].dtype;
    }
    const uint8_t* dmask = nullptr;
    if (mask) {
        FSW_CUDA(ctx->st_mask.reserve((size_t)W * H));
        FSW_CUDA(cudaMemcpy2DAsync(ctx->st_mask.p, W, mask, mask_pitch, W, H, cudaMemcpyHostToDevice, stream));
        dmask = (const uint8_t*)ctx->st_mask.p;
    }
    fsw_depth_out dout;
    std::memset(&dout, 0, sizeof(dout));
    dout.struct_size = sizeof(dout);
    FSW_CUDA(ctx->st_depth.reserve((size_t)W * H * 4));
    dout.depth = (float*)ctx->st_depth.p; dout.depth_pitch = (size_t)W * 4;
    if (out->best_cost) { FSW_CUDA(ctx->st_c1.reserve((size_t)W * H * 4)); dout.best_cost = (float*)ctx->st_c1.p; dout.best_cost_pitch = (size_t)W * 4; }
    if (out->second_cost) { FSW_CUDA(ctx->st_c2.reserve((size_t)W * H * 4)); dout.second_cost = (float*)ctx->st_c2.p; dout.second_cost_pitch = (size_t)W * 4; }
    if (out->plane_index) { FSW_CUDA(ctx->st_k.reserve((size_t)W * H * 2)); dout.plane_index = (int16_t*)ctx->st_k.p; dout.plane_index_pitch = (size_t)W * 2; }
    if (out->valid_reason) { FSW_CUDA(ctx->st_reason.reserve((size_t)W * H)); dout.valid_reason = (uint8_t*)ctx->st_reason.p; dout.valid_reason_pitch = (size_t)W; }
    if (multires) rc = fsw_compute_depth_multires(ctx, p0, p1, q0, q1, crop, dimg, dmask, (size_t)W, &dout, cuda_stream);
    else rc = fsw_compute_depth(ctx, p0, q0, dimg, dmask, (size_t)W, &dout, cuda_stream);
    if (rc != FSW_OK) return rc;
    FSW_CUDA(cudaMemcpy2DAsync(out->depth, out->depth_pitch, dout.depth, dout.depth_pitch, (size_t)W * 4, H, cudaMemcpyDeviceToHost, stream));
    if (out->best_cost) FSW_CUDA(cudaMemcpy2DAsync(out->best_cost, out->best_cost_pitch, dout.best_cost, dout.best_cost_pitch, (size_t)W * 4, H, cudaMemcpyDeviceToHost, stream));
    if (out->second_cost) FSW_CUDA(cudaMemcpy2DAsync(out->second_cost, out->second_cost_pitch, dout.second_cost, dout.second_cost_pitch, (size_t)W * 4, H, cudaMemcpyDeviceToHost, stream));
    if (out->plane_index) FSW_CUDA(cudaMemcpy2DAsync(out->plane_index, out->plane_index_pitch, dout.plane_index, dout.plane_index_pitch, (size_t)W * 2, H, cudaMemcpyDeviceToHost, stream));
    if (out->valid_reason) FSW_CUDA(cudaMemcpy2DAsync(out->valid_reason, out->valid_reason_pitch, dout.valid_reason, dout.valid_reason_pitch, (size_t)W, H, cudaMemcpyDeviceToHost, stream));
    FSW_CUDA(cudaStreamSynchronize(stream));
    return FSW_OK;
}

int32_t fsw_compute_depth_host(fsw_context* ctx, const fsw_planeset* planes, const fsw_sweep_params* params,
                               const fsw_image* images, const uint8_t* mask, size_t mask_pitch,
                               const fsw_depth_out* out, void* cuda_stream) {
    fsw_rect none = {0, 0, 0, 0};
    return run_host(ctx, false, planes, nullptr, params, nullptr, none, images, mask, mask_pitch, out, cuda_stream);
}

int32_t fsw_compute_depth_multires_host(fsw_context* ctx, const fsw_planeset* planes_low,
                                        const fsw_planeset* planes_crop, const fsw_sweep_params* params_low,
                                        const fsw_sweep_params* params_crop, fsw_rect crop, const fsw_image* images,
                                        const uint8_t* mask, size_t mask_pitch, const fsw_depth_out* out,
                                        void* cuda_stream) {
    return run_host(ctx, true, planes_low, planes_crop, params_low, params_crop, crop, images, mask, mask_pitch, out, cuda_stream);
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
    FSW_CUDA(cudaMemcpy(h, ctx->counters.p, sizeof(h), cudaMemcpyDeviceToHost));
    out->n_eval = (int64_t)h[0];
    out->n_raw_valid = (int64_t)h[1];
    out->n_valid = (int64_t)h[2];
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

int32_t fsw_measure_fp32_peak(int32_t cuda_device, void* cuda_stream, double* tflops, double* ms) {
    if (!tflops || !ms) return fail(FSW_E_INVALID_ARG, "fsw_measure_fp32_peak: null argument");
    DeviceGuard g;
    FSW_CUDA(g.enter(cuda_device));
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    cudaDeviceProp prop;
    FSW_CUDA(cudaGetDeviceProperties(&prop, cuda_device));
    float* sink = nullptr;
    FSW_CUDA(cudaMalloc(&sink, 4));
    const int blocks = prop.multiProcessorCount * 8, iters = 4096;
    cudaEvent_t e0, e1;
    FSW_CUDA(cudaEventCreate(&e0));
    FSW_CUDA(cudaEventCreate(&e1));
    double best = 1e30;
    cudaError_t err = cudaSuccess;
    for (int rep = 0; rep < 4 && err == cudaSuccess; ++rep) {
        cudaEventRecord(e0, stream);
        err = fsw_launch_ffma_peak(sink, blocks, iters, stream);
        cudaEventRecord(e1, stream);
        if (err == cudaSuccess) err = cudaEventSynchronize(e1);
        float t = 0.f;
        if (err == cudaSuccess) err = cudaEventElapsedTime(&t, e0, e1);
        if (rep > 0 && t < best) best = t;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(sink);
    if (err != cudaSuccess) return cuda_fail(err, "fsw_measure_fp32_peak");
    const double flops = 2.0 * 8.0 * 16.0 * (double)iters * 256.0 * (double)blocks;
    *ms = best;
    *tflops = flops / (best * 1e-3) / 1e12;
    return FSW_OK;
}

}  /* extern "C" */
