/*
 * fsw_tsdf.cu -- the TSDF consumer of the depth maps (section III-C): block
 * allocation along d +- mu of the Eq. 1 ray, Eq. 2 integration through the unified projection, the local map of fixed
 * size around the vehicle and the "at least 3 observations" gate, on the device the depth maps are produced on.
 *
 * B200 layout instead of InfiniTAM's hash: the local map has a FIXED size (60 m x 60 m x 3 m), so the
 * volume is a dense torus of 8^3-voxel blocks -- world block b lives in slot (b mod nb) -- with a state word and an
 * observation count per block; 60 x 60 x 3.2 m at 0.05 m is 180 000 blocks x 4 KB = 737 MB of HBM.  "Allocation" marks
 * blocks (and clears the ones that are new), the "visible list" is the compacted list of allocated blocks of the
 * frame, "swapping out" frees the blocks that leave the box when it is re-centred (nothing is archived on the host).
 * All device arithmetic is relative to the box origin (float has 2e-6 m resolution at 30 m, not at kilometres): the
 * host folds the origin into the pose in double precision.
 */
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>

#include "fsw_sweep.cuh" /* fsw::back_project (Eq. 1 with the undistortion), FswDevCam */

namespace {

constexpr int TB = 8;            /* voxels per block edge */
constexpr int TV = TB * TB * TB; /* voxels per block */

struct TsdfBox {
    int32_t b0[3], nb[3]; /* world block coordinate of the box's first block; blocks per axis (= torus size) */
    float voxel_size, mu, inv_mu, w_max;
};

struct TsdfPose {
    float R[9]; /* world -> camera rotation */
    float t[3]; /* camera-frame position of the box origin: X_d = R X_rel + t */
};

__host__ __device__ inline int pmod(int a, int n) { int r = a % n; return r < 0 ? r + n : r; }

__device__ inline int slot_of(const TsdfBox& B, int bx, int by, int bz) {
    return (pmod(bz, B.nb[2]) * B.nb[1] + pmod(by, B.nb[1])) * B.nb[0] + pmod(bx, B.nb[0]);
}

/* world block coordinate (relative to b0: 0 <= r < nb) of the block a slot holds under origin b0 */
__device__ inline void rel_block_of(const TsdfBox& B, int slot, int& rx, int& ry, int& rz) {
    const int sx = slot % B.nb[0], sy = (slot / B.nb[0]) % B.nb[1], sz = slot / (B.nb[0] * B.nb[1]);
    rx = pmod(sx - B.b0[0], B.nb[0]);
    ry = pmod(sy - B.b0[1], B.nb[1]);
    rz = pmod(sz - B.b0[2], B.nb[2]);
}

/* unified projection with distortion; false outside the field of view */
__device__ inline bool project(const FswDevCam& c, float X, float Y, float Z, float& u, float& v) {
    const float rho = sqrtf(fmaf(X, X, fmaf(Y, Y, Z * Z)));
    if (!(rho > 0.f)) return false;
    const float den = fmaf(c.xi, rho, Z);
    if (!(den > 1e-9f * rho) || !(Z >= c.cos_fov * rho)) return false;
    const float mx = X / den, my = Y / den;
    const float r2 = fmaf(mx, mx, my * my);
    const float rad = fmaf(r2, fmaf(c.k2, r2, c.k1), 1.f);
    const float xd = fmaf(mx, rad, fmaf(2.f * c.p1 * mx, my, c.p2 * fmaf(2.f * mx, mx, r2)));
    const float yd = fmaf(my, rad, fmaf(c.p1, fmaf(2.f * my, my, r2), 2.f * c.p2 * mx * my));
    u = fmaf(c.fx, xd, c.cx);
    v = fmaf(c.fy, yd, c.cy);
    return true;
}

/* Allocation: one thread per depth pixel walks its segment [d - mu, d + mu] in n + 1 samples.
 * counters[0] = blocks newly allocated, new_list = their slots. */
__global__ void __launch_bounds__(256) tsdf_allocate_kernel(TsdfBox B, FswDevCam cam, TsdfPose P, const float* __restrict__ depth,
                                                            int64_t pitch, int n_steps, unsigned* __restrict__ state,
                                                            int* __restrict__ new_list, unsigned* __restrict__ counters) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x, y = blockIdx.y;
    if (x >= cam.W || y >= cam.H) return;
    const float d = *reinterpret_cast<const float*>(reinterpret_cast<const char*>(depth) + (int64_t)y * pitch + 4 * (int64_t)x);
    if (!(d > 0.f)) return;
    float rx, ry, rz;
    if (!fsw::back_project(cam, (float)x, (float)y, rx, ry, rz)) return;
    const float inv_edge = 1.f / (B.voxel_size * TB);
    for (int i = 0; i <= n_steps; ++i) {
        const float range = (d - B.mu) + (float)i * (2.f * B.mu / (float)n_steps);
        const float ax = fmaf(range, rx, -P.t[0]), ay = fmaf(range, ry, -P.t[1]), az = fmaf(range, rz, -P.t[2]);
        /* X_rel = R^T (X_d - t), in block units relative to the box origin */
        const int bx = (int)floorf((P.R[0] * ax + P.R[3] * ay + P.R[6] * az) * inv_edge);
        const int by = (int)floorf((P.R[1] * ax + P.R[4] * ay + P.R[7] * az) * inv_edge);
        const int bz = (int)floorf((P.R[2] * ax + P.R[5] * ay + P.R[8] * az) * inv_edge);
        if (bx < 0 || by < 0 || bz < 0 || bx >= B.nb[0] || by >= B.nb[1] || bz >= B.nb[2]) continue; /* local map only */
        const int slot = slot_of(B, bx + B.b0[0], by + B.b0[1], bz + B.b0[2]);
        if (state[slot] == 0u && atomicCAS(&state[slot], 0u, 2u) == 0u) new_list[atomicAdd(&counters[0], 1u)] = slot;
    }
}

/* new blocks start empty (D = 0, w = 0, no observations) */
__global__ void __launch_bounds__(256) tsdf_clear_new_kernel(float2* __restrict__ vox, int* __restrict__ obs, unsigned* __restrict__ state,
                                                             const int* __restrict__ new_list, const unsigned* __restrict__ counters) {
    const unsigned n = counters[0];
    for (unsigned b = blockIdx.x; b < n; b += gridDim.x) {
        const int slot = new_list[b];
        float2* v = vox + (size_t)slot * TV;
        for (int i = threadIdx.x; i < TV; i += blockDim.x) v[i] = make_float2(0.f, 0.f);
        if (threadIdx.x == 0) { obs[slot] = 0; state[slot] = 1u; }
    }
}

/* the list of the blocks of this frame: every allocated block of the local map (counters[1] = its length) */
__global__ void __launch_bounds__(256) tsdf_visible_kernel(int n_slots, const unsigned* __restrict__ state, int* __restrict__ visible,
                                                           unsigned* __restrict__ counters) {
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s < n_slots && state[s] == 1u) visible[atomicAdd(&counters[1], 1u)] = s;
}

/* Integration, Eq. 2: persistent CTAs over the visible list, two voxels per thread.
 * counters[2] = voxels updated.  Bound by HBM: 4 KB read + 4 KB written per block whose voxels are touched. */
__global__ void __launch_bounds__(256) tsdf_integrate_kernel(TsdfBox B, FswDevCam cam, TsdfPose P, const float* __restrict__ depth,
                                                             int64_t pitch, float2* __restrict__ vox, int* __restrict__ obs,
                                                             const int* __restrict__ visible, unsigned* __restrict__ counters) {
    const unsigned n = counters[1];
    unsigned n_upd = 0;
    for (unsigned b = blockIdx.x; b < n; b += gridDim.x) {
        const int slot = visible[b];
        int rx, ry, rz;
        rel_block_of(B, slot, rx, ry, rz);
        float2* v = vox + (size_t)slot * TV;
        bool any = false;
#pragma unroll
        for (int h = 0; h < TV / 256; ++h) {
            const int l = threadIdx.x + 256 * h;
            const int i = l & 7, j = (l >> 3) & 7, k = l >> 6;
            const float X = ((float)(rx * TB + i) + 0.5f) * B.voxel_size;
            const float Y = ((float)(ry * TB + j) + 0.5f) * B.voxel_size;
            const float Z = ((float)(rz * TB + k) + 0.5f) * B.voxel_size;
            const float xd = fmaf(P.R[0], X, fmaf(P.R[1], Y, fmaf(P.R[2], Z, P.t[0])));
            const float yd = fmaf(P.R[3], X, fmaf(P.R[4], Y, fmaf(P.R[5], Z, P.t[1])));
            const float zd = fmaf(P.R[6], X, fmaf(P.R[7], Y, fmaf(P.R[8], Z, P.t[2])));
            float u, w;
            if (!project(cam, xd, yd, zd, u, w)) continue;
            const float pu = floorf(u + 0.5f), pv = floorf(w + 0.5f); /* nearest pixel */
            if (!(pu >= 0.f && pv >= 0.f && pu <= (float)(cam.W - 1) && pv <= (float)(cam.H - 1))) continue;
            const float d = __ldg(reinterpret_cast<const float*>(reinterpret_cast<const char*>(depth) + (int64_t)pv * pitch) + (int)pu);
            if (!(d > 0.f)) continue;
            const float eta = d - sqrtf(fmaf(xd, xd, fmaf(yd, yd, zd * zd)));
            if (eta < -B.mu) continue; /* "not smaller than -mu" */
            const float sample = fminf(1.f, eta * B.inv_mu);
            const float2 o = v[l];
            v[l] = make_float2(fmaf(o.y, o.x, sample) / (o.y + 1.f), fminf(o.y + 1.f, B.w_max));
            any = true;
            ++n_upd;
        }
        if (__syncthreads_or(any) && threadIdx.x == 0) obs[slot] += 1;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) n_upd += __shfl_xor_sync(0xffffffffu, n_upd, o);
    if ((threadIdx.x & 31) == 0 && n_upd) atomicAdd(&counters[2], n_upd);
}

/* Points of the map (SPEC.md extract_points): zero crossings between axis neighbours that both carry
 * weight, in blocks with at least min_obs observations.  counters[3] = points found (may exceed the capacity). */
__global__ void __launch_bounds__(256) tsdf_extract_kernel(TsdfBox B, const float2* __restrict__ vox, const int* __restrict__ obs,
                                                           const unsigned* __restrict__ state, int n_slots, int min_obs,
                                                           float* __restrict__ points, unsigned cap, unsigned* __restrict__ counters) {
    for (int slot = blockIdx.x; slot < n_slots; slot += gridDim.x) {
        if (state[slot] != 1u || obs[slot] < min_obs) continue;
        int rx, ry, rz;
        rel_block_of(B, slot, rx, ry, rz);
        const float2* v = vox + (size_t)slot * TV;
        for (int l = threadIdx.x; l < TV; l += blockDim.x) {
            const int i = l & 7, j = (l >> 3) & 7, k = l >> 6;
            const float2 a = v[l];
            if (!(a.y > 0.f)) continue;
#pragma unroll
            for (int ax = 0; ax < 3; ++ax) {
                const int gx = rx * TB + i + (ax == 0), gy = ry * TB + j + (ax == 1), gz = rz * TB + k + (ax == 2);
                if (gx >= B.nb[0] * TB || gy >= B.nb[1] * TB || gz >= B.nb[2] * TB) continue; /* leaves the local map */
                const int s1 = slot_of(B, gx / TB + B.b0[0], gy / TB + B.b0[1], gz / TB + B.b0[2]);
                if (state[s1] != 1u || obs[s1] < min_obs) continue;
                const float2 c = vox[(size_t)s1 * TV + ((gz % TB) * TB + (gy % TB)) * TB + (gx % TB)];
                if (!(c.y > 0.f)) continue;
                if (!((a.x > 0.f && c.x < 0.f) || (a.x < 0.f && c.x > 0.f))) continue;
                const float f = a.x / (a.x - c.x);
                const unsigned idx = atomicAdd(&counters[3], 1u);
                if (idx < cap) {
                    points[3 * idx + 0] = ((float)(rx * TB + i) + 0.5f + (ax == 0 ? f : 0.f)) * B.voxel_size;
                    points[3 * idx + 1] = ((float)(ry * TB + j) + 0.5f + (ax == 1 ? f : 0.f)) * B.voxel_size;
                    points[3 * idx + 2] = ((float)(rz * TB + k) + 0.5f + (ax == 2 ? f : 0.f)) * B.voxel_size;
                }
            }
        }
    }
}

/* re-centring: blocks whose world coordinate leaves the new box are freed (counters[4] = how many) */
__global__ void __launch_bounds__(256) tsdf_recentre_kernel(TsdfBox old_box, int nb0x, int nb0y, int nb0z, unsigned* __restrict__ state,
                                                            int n_slots, unsigned* __restrict__ counters) {
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n_slots || state[s] == 0u) return;
    int rx, ry, rz;
    rel_block_of(old_box, s, rx, ry, rz);
    const int wx = rx + old_box.b0[0], wy = ry + old_box.b0[1], wz = rz + old_box.b0[2];
    if (wx < nb0x || wy < nb0y || wz < nb0z || wx >= nb0x + old_box.nb[0] || wy >= nb0y + old_box.nb[1] || wz >= nb0z + old_box.nb[2]) {
        state[s] = 0u;
        atomicAdd(&counters[4], 1u);
    }
}

/* dense copy of the local map for inspection: out_d / out_w [nbz*8][nby*8][nbx*8] in box order, 0 where not allocated */
__global__ void __launch_bounds__(256) tsdf_dense_kernel(TsdfBox B, const float2* __restrict__ vox, const unsigned* __restrict__ state,
                                                         const int* __restrict__ obs, float* __restrict__ out_d, float* __restrict__ out_w,
                                                         int32_t* __restrict__ out_obs, uint8_t* __restrict__ out_alloc) {
    const int n_blocks = B.nb[0] * B.nb[1] * B.nb[2];
    for (int r = blockIdx.x; r < n_blocks; r += gridDim.x) {
        const int rx = r % B.nb[0], ry = (r / B.nb[0]) % B.nb[1], rz = r / (B.nb[0] * B.nb[1]);
        const int slot = slot_of(B, rx + B.b0[0], ry + B.b0[1], rz + B.b0[2]);
        const bool on = state[slot] == 1u;
        if (threadIdx.x == 0) { out_obs[r] = on ? obs[slot] : 0; out_alloc[r] = on ? 1 : 0; }
        for (int l = threadIdx.x; l < TV; l += blockDim.x) {
            const int i = l & 7, j = (l >> 3) & 7, k = l >> 6;
            const float2 a = on ? vox[(size_t)slot * TV + l] : make_float2(0.f, 0.f);
            const size_t o = ((size_t)(rz * TB + k) * (B.nb[1] * TB) + (size_t)(ry * TB + j)) * (B.nb[0] * TB) + (size_t)(rx * TB + i);
            out_d[o] = a.x;
            out_w[o] = a.y;
        }
    }
}

thread_local char g_terr[512] = "";
int32_t tfail(int32_t code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_terr, sizeof(g_terr), fmt, ap);
    va_end(ap);
    return code;
}
#define TSDF_CUDA(call)                                                                  \
    do {                                                                                 \
        cudaError_t e__ = (call);                                                        \
        if (e__ != cudaSuccess) return tfail(FSW_E_CUDA, "%s: %s", #call, cudaGetErrorString(e__)); \
    } while (0)

}  // namespace

struct fsw_tsdf {
    int32_t device;
    int n_sm;
    TsdfBox box;
    int n_slots;
    float2* vox = nullptr;
    int* obs = nullptr;
    unsigned* state = nullptr;
    int *new_list = nullptr, *visible = nullptr;
    unsigned* counters = nullptr; /* [0] new blocks, [1] visible blocks, [2] voxels updated, [3] points, [4] blocks freed */
    cudaStream_t last_stream = nullptr;
    int64_t n_frames = 0;
};

/* the error text of the TSDF calls is appended to the library's thread-local message by fsw_tsdf_last_error */
extern "C" {

const char* fsw_tsdf_last_error(void) { return g_terr; }

int32_t fsw_tsdf_create(int32_t cuda_device, const fsw_tsdf_params* p, const double* centre, fsw_tsdf** out) {
    if (!p || !centre || !out) return tfail(FSW_E_INVALID_ARG, "fsw_tsdf_create: null argument");
    *out = nullptr;
    if (p->struct_size != sizeof(fsw_tsdf_params)) return tfail(FSW_E_INVALID_ARG, "fsw_tsdf_create: struct_size %u != %zu", p->struct_size, sizeof(fsw_tsdf_params));
    if (!(p->voxel_size > 0.f) || !(p->mu > 0.f) || p->w_max < 1) return tfail(FSW_E_INVALID_ARG, "fsw_tsdf_create: voxel_size, mu must be > 0 and w_max >= 1");
    fsw_tsdf* v = new (std::nothrow) fsw_tsdf;
    if (!v) return tfail(FSW_E_NOMEM, "fsw_tsdf_create: out of memory");
    v->device = cuda_device;
    const double edge = (double)p->voxel_size * TB;
    size_t n_slots = 1;
    for (int a = 0; a < 3; ++a) {
        if (!(p->box_size[a] > 0.f)) { delete v; return tfail(FSW_E_INVALID_ARG, "fsw_tsdf_create: box_size must be > 0"); }
        v->box.nb[a] = (int32_t)std::ceil((double)p->box_size[a] / edge - 1e-9);
        v->box.b0[a] = (int32_t)std::floor(centre[a] / edge) - v->box.nb[a] / 2;
        n_slots *= (size_t)v->box.nb[a];
    }
    if (n_slots > (size_t)1 << 26) { delete v; return tfail(FSW_E_CONFIG, "fsw_tsdf_create: %zu blocks", n_slots); }
    v->n_slots = (int)n_slots;
    v->box.voxel_size = p->voxel_size; v->box.mu = p->mu; v->box.inv_mu = 1.f / p->mu; v->box.w_max = (float)p->w_max;
    int prev = -1;
    cudaError_t e = cudaGetDevice(&prev);
    if (e == cudaSuccess) e = cudaSetDevice(cuda_device);
    cudaDeviceProp prop;
    if (e == cudaSuccess) e = cudaGetDeviceProperties(&prop, cuda_device);
    if (e == cudaSuccess) v->n_sm = prop.multiProcessorCount;
    if (e == cudaSuccess) e = cudaMalloc(&v->vox, n_slots * TV * sizeof(float2));
    if (e == cudaSuccess) e = cudaMalloc(&v->obs, n_slots * sizeof(int));
    if (e == cudaSuccess) e = cudaMalloc(&v->state, n_slots * sizeof(unsigned));
    if (e == cudaSuccess) e = cudaMalloc(&v->new_list, n_slots * sizeof(int));
    if (e == cudaSuccess) e = cudaMalloc(&v->visible, n_slots * sizeof(int));
    if (e == cudaSuccess) e = cudaMalloc(&v->counters, 8 * sizeof(unsigned));
    if (e == cudaSuccess) e = cudaMemset(v->state, 0, n_slots * sizeof(unsigned));
    if (e == cudaSuccess) e = cudaMemset(v->obs, 0, n_slots * sizeof(int));
    if (e == cudaSuccess) e = cudaMemset(v->counters, 0, 8 * sizeof(unsigned));
    if (prev >= 0) cudaSetDevice(prev);
    if (e != cudaSuccess) {
        fsw_tsdf_destroy(v);
        return tfail(FSW_E_CUDA, "fsw_tsdf_create: %s (there is no CPU fallback)", cudaGetErrorString(e));
    }
    *out = v;
    return FSW_OK;
}

int32_t fsw_tsdf_destroy(fsw_tsdf* v) {
    if (!v) return FSW_OK;
    cudaFree(v->vox); cudaFree(v->obs); cudaFree(v->state); cudaFree(v->new_list); cudaFree(v->visible); cudaFree(v->counters);
    delete v;
    return FSW_OK;
}

int32_t fsw_tsdf_box(const fsw_tsdf* v, int32_t* block_origin, int32_t* blocks) {
    if (!v) return tfail(FSW_E_INVALID_ARG, "fsw_tsdf_box: null volume");
    for (int a = 0; a < 3; ++a) {
        if (block_origin) block_origin[a] = v->box.b0[a];
        if (blocks) blocks[a] = v->box.nb[a];
    }
    return FSW_OK;
}

int32_t fsw_tsdf_recentre(fsw_tsdf* v, const double* centre, void* cuda_stream) {
    if (!v || !centre) return tfail(FSW_E_INVALID_ARG, "fsw_tsdf_recentre: null argument");
    const double edge = (double)v->box.voxel_size * TB;
    int32_t nb0[3];
    bool moved = false;
    for (int a = 0; a < 3; ++a) {
        nb0[a] = (int32_t)std::floor(centre[a] / edge) - v->box.nb[a] / 2;
        moved = moved || nb0[a] != v->box.b0[a];
    }
    cudaStream_t s = (cudaStream_t)cuda_stream;
    v->last_stream = s;
    TSDF_CUDA(cudaMemsetAsync(v->counters + 4, 0, sizeof(unsigned), s));
    if (moved) {
        tsdf_recentre_kernel<<<(v->n_slots + 255) / 256, 256, 0, s>>>(v->box, nb0[0], nb0[1], nb0[2], v->state, v->n_slots, v->counters);
        TSDF_CUDA(cudaGetLastError());
        for (int a = 0; a < 3; ++a) v->box.b0[a] = nb0[a];
    }
    return FSW_OK;
}

int32_t fsw_tsdf_integrate(fsw_tsdf* v, const fsw_camera* cam, const double* R, const double* t, const float* depth,
                           size_t depth_pitch, void* cuda_stream) {
    if (!v || !cam || !R || !t || !depth) return tfail(FSW_E_INVALID_ARG, "fsw_tsdf_integrate: null argument");
    if (cam->struct_size != sizeof(fsw_camera)) return tfail(FSW_E_INVALID_ARG, "fsw_tsdf_integrate: camera struct_size");
    if (depth_pitch < (size_t)cam->width * 4 || depth_pitch % 4) return tfail(FSW_E_INVALID_ARG, "fsw_tsdf_integrate: depth_pitch=%zu", depth_pitch);
    FswDevCam c;
    std::memset(&c, 0, sizeof(c));
    c.fx = (float)cam->fx; c.fy = (float)cam->fy; c.cx = (float)cam->cx; c.cy = (float)cam->cy; c.xi = (float)cam->xi;
    c.k1 = (float)cam->k1; c.k2 = (float)cam->k2; c.p1 = (float)cam->p1; c.p2 = (float)cam->p2;
    c.cos_fov = (float)std::cos(0.5 * cam->fov_max_deg * M_PI / 180.0);
    c.cos_fov_xi = (float)(std::cos(0.5 * cam->fov_max_deg * M_PI / 180.0) + cam->xi);
    c.W = cam->width; c.H = cam->height; c.Wm1 = cam->width - 1; c.Hm1 = cam->height - 1;
    c.dist_mode = (cam->k1 == 0.0 && cam->k2 == 0.0 && cam->p1 == 0.0 && cam->p2 == 0.0) ? FSW_DIST_NONE
                  : ((cam->k2 == 0.0 && cam->p1 == 0.0 && cam->p2 == 0.0) ? FSW_DIST_K1 : FSW_DIST_FULL);
    /* pose relative to the box origin, folded in double precision: X_d = R (X_rel + O) + t */
    TsdfPose P;
    const double edge = (double)v->box.voxel_size * TB;
    const double O[3] = { v->box.b0[0] * edge, v->box.b0[1] * edge, v->box.b0[2] * edge };
    for (int i = 0; i < 9; ++i) P.R[i] = (float)R[i];
    for (int i = 0; i < 3; ++i) P.t[i] = (float)(R[3 * i] * O[0] + R[3 * i + 1] * O[1] + R[3 * i + 2] * O[2] + t[i]);
    const int n_steps = (int)std::ceil(2.0 * (double)v->box.mu / (0.5 * edge));
    cudaStream_t s = (cudaStream_t)cuda_stream;
    v->last_stream = s;
    int prev = -1;
    TSDF_CUDA(cudaGetDevice(&prev));
    if (prev != v->device) TSDF_CUDA(cudaSetDevice(v->device));
    TSDF_CUDA(cudaMemsetAsync(v->counters, 0, 3 * sizeof(unsigned), s));
    dim3 ga((cam->width + 255) / 256, cam->height, 1);
    tsdf_allocate_kernel<<<ga, 256, 0, s>>>(v->box, c, P, depth, (int64_t)depth_pitch, n_steps, v->state, v->new_list, v->counters);
    tsdf_clear_new_kernel<<<v->n_sm * 8, 256, 0, s>>>(v->vox, v->obs, v->state, v->new_list, v->counters);
    tsdf_visible_kernel<<<(v->n_slots + 255) / 256, 256, 0, s>>>(v->n_slots, v->state, v->visible, v->counters);
    tsdf_integrate_kernel<<<v->n_sm * 8, 256, 0, s>>>(v->box, c, P, depth, (int64_t)depth_pitch, v->vox, v->obs, v->visible, v->counters);
    cudaError_t e = cudaGetLastError();
    if (prev != v->device) cudaSetDevice(prev);
    if (e != cudaSuccess) return tfail(FSW_E_CUDA, "fsw_tsdf_integrate: %s", cudaGetErrorString(e));
    v->n_frames++;
    return FSW_OK;
}

int32_t fsw_tsdf_extract_points(fsw_tsdf* v, int32_t min_block_observations, float* points, int32_t capacity, void* cuda_stream) {
    if (!v || (!points && capacity > 0) || capacity < 0) return tfail(FSW_E_INVALID_ARG, "fsw_tsdf_extract_points: bad argument");
    cudaStream_t s = (cudaStream_t)cuda_stream;
    v->last_stream = s;
    TSDF_CUDA(cudaMemsetAsync(v->counters + 3, 0, sizeof(unsigned), s));
    tsdf_extract_kernel<<<v->n_sm * 8, 256, 0, s>>>(v->box, v->vox, v->obs, v->state, v->n_slots, min_block_observations, points,
                                                    (unsigned)capacity, v->counters);
    TSDF_CUDA(cudaGetLastError());
    return FSW_OK;
}

int32_t fsw_tsdf_get_stats(fsw_tsdf* v, fsw_tsdf_stats* out) {
    if (!v || !out) return tfail(FSW_E_INVALID_ARG, "fsw_tsdf_get_stats: null argument");
    if (out->struct_size != sizeof(fsw_tsdf_stats)) return tfail(FSW_E_INVALID_ARG, "fsw_tsdf_get_stats: struct_size");
    TSDF_CUDA(cudaStreamSynchronize(v->last_stream));
    unsigned h[8];
    TSDF_CUDA(cudaMemcpy(h, v->counters, sizeof(h), cudaMemcpyDeviceToHost));
    out->n_new_blocks = h[0]; out->n_visible_blocks = h[1]; out->n_voxels_updated = h[2]; out->n_points = h[3];
    out->n_blocks_freed = h[4]; out->n_frames = v->n_frames;
    return FSW_OK;
}

int32_t fsw_tsdf_download(fsw_tsdf* v, float* tsdf, float* weight, int32_t* observations, uint8_t* allocated, void* cuda_stream) {
    if (!v || !tsdf || !weight || !observations || !allocated) return tfail(FSW_E_INVALID_ARG, "fsw_tsdf_download: null argument");
    cudaStream_t s = (cudaStream_t)cuda_stream;
    v->last_stream = s;
    tsdf_dense_kernel<<<v->n_sm * 8, 256, 0, s>>>(v->box, v->vox, v->state, v->obs, tsdf, weight, observations, allocated);
    TSDF_CUDA(cudaGetLastError());
    return FSW_OK;
}

}  /* extern "C" */
