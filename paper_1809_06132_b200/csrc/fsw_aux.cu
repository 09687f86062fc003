/*
 * fsw_aux.cu -- the small kernels around the sweep:
 *   - footprint packing of the view images (one 64- or 128-bit load then fetches a whole bilinear footprint, S4),
 *   - the 2x2 box downsample of the two-scale strategy (PAPER.md:88-90, S10(a)),
 *   - an FFMA-chain kernel that measures the FP32 throughput used as the "alu" roofline denominator.
 */
#include "fsw_internal.h"

namespace {

__device__ __forceinline__ float load_px(const void* base, int64_t pitch, int dtype, int x, int y) {
    const char* row = reinterpret_cast<const char*>(base) + (int64_t)y * pitch;
    return dtype == FSW_U8 ? (float)__ldg(reinterpret_cast<const uint8_t*>(row) + x)
                           : __ldg(reinterpret_cast<const float*>(row) + x);
}

/* (value, difference) as two bfloat16 in one word: value in the low half */
__device__ __forceinline__ unsigned pack_bf16(float v, float d) {
    return (__float_as_uint(v) >> 16) | (__float_as_uint(d) & 0xffff0000u);
}

/* foot(x,y) = (I(x,y), I(x+1,y) - I(x,y), I(x,y+1), I(x+1,y+1) - I(x,y+1)), indices clamped at the right / bottom
 * border (a valid bilinear footprint never starts in the last column / row, so the clamped entries are never used).
 * Two outputs per thread; a warp writes 1 KB of consecutive footprints. */
__global__ void __launch_bounds__(256) pack_footprints_kernel(const __grid_constant__ FswPackArgs a) {
    const int img = blockIdx.z;
    if (a.words_to_zero != nullptr && img == 0 && blockIdx.x == 0 && blockIdx.y == 0 && (int)threadIdx.x < a.n_words_to_zero)
        a.words_to_zero[threadIdx.x] = 0u;
    const int W = a.W, H = a.H;
    const int x2 = (blockIdx.x * blockDim.x + threadIdx.x) * 2;
    const int y = blockIdx.y;
    if (y >= H || x2 >= W) return;
    const int y1 = min(y + 1, H - 1);
    const int dt = a.dtype[img];
    float t[3], b[3];
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        int x = min(x2 + i, W - 1);
        t[i] = load_px(a.src[img], a.src_pitch[img], dt, x, y);
        b[i] = load_px(a.src[img], a.src_pitch[img], dt, x, y1);
    }
    if (a.f16) { /* integers up to 256 are exact in bfloat16 = the upper half of the float */
        uint2* dst = reinterpret_cast<uint2*>(a.dst[img]) + (int64_t)y * W + x2;
        const uint2 f0 = make_uint2(pack_bf16(t[0], t[1] - t[0]), pack_bf16(b[0], b[1] - b[0]));
        const uint2 f1 = make_uint2(pack_bf16(t[1], t[2] - t[1]), pack_bf16(b[1], b[2] - b[1]));
        if (x2 + 1 < W && (W & 1) == 0) *reinterpret_cast<uint4*>(dst) = make_uint4(f0.x, f0.y, f1.x, f1.y);
        else {
            dst[0] = f0;
            if (x2 + 1 < W) dst[1] = f1;
        }
    } else {
        float4* dst = reinterpret_cast<float4*>(a.dst[img]) + (int64_t)y * W + x2;
        dst[0] = make_float4(t[0], t[1] - t[0], b[0], b[1] - b[0]);
        if (x2 + 1 < W) dst[1] = make_float4(t[1], t[2] - t[1], b[1], b[2] - b[1]);
    }
}

/* out(x,y) = 0.25 * (I(2x,2y) + I(2x+1,2y) + I(2x,2y+1) + I(2x+1,2y+1)) as float32 */
__global__ void __launch_bounds__(256) downsample_kernel(const __grid_constant__ FswDownArgs a) {
    const int cam = blockIdx.z;
    const int W2 = a.W[cam] / 2, H2 = a.H[cam] / 2;
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y;
    if (x >= W2 || y >= H2) return;
    float s;
    if (a.dtype[cam] == FSW_U8) {
        const uint8_t* r0 = reinterpret_cast<const uint8_t*>(a.src[cam]) + (int64_t)(2 * y) * a.src_pitch[cam] + 2 * x;
        const uint8_t* r1 = r0 + a.src_pitch[cam];
        s = (float)((int)r0[0] + (int)r0[1] + (int)r1[0] + (int)r1[1]);
    } else {
        const float* r0 = reinterpret_cast<const float*>(reinterpret_cast<const char*>(a.src[cam]) + (int64_t)(2 * y) * a.src_pitch[cam]) + 2 * x;
        const float* r1 = reinterpret_cast<const float*>(reinterpret_cast<const char*>(r0) + a.src_pitch[cam]);
        s = (r0[0] + r0[1]) + (r1[0] + r1[1]);
    }
    a.dst[cam][(int64_t)y * W2 + x] = 0.25f * s;
}

/* Local depth-continuity filter (third filter; reading Q25 of DESIGN.md) + mask.  One thread per pixel,
 * a 32 x 16 tile plus its halo staged in shared memory (0 = invalid, also outside the image); the comparisons run in
 * double precision so that the result is a function of the float32 input map alone. */
constexpr int CT_X = 32, CT_Y = 16, CT_HALO = FSW_MAX_WINDOW / 2;
__global__ void __launch_bounds__(CT_X * CT_Y) continuity_kernel(const __grid_constant__ FswContinuityArgs a) {
    __shared__ float tile[CT_Y + 2 * CT_HALO][CT_X + 2 * CT_HALO + 1];
    const int hw = a.window / 2;
    const int x0 = blockIdx.x * CT_X - hw, y0 = blockIdx.y * CT_Y - hw;
    const int tw = CT_X + 2 * hw, th = CT_Y + 2 * hw;
    for (int i = threadIdx.y * CT_X + threadIdx.x; i < tw * th; i += CT_X * CT_Y) {
        const int ty = i / tw, tx = i - ty * tw;
        const int x = x0 + tx, y = y0 + ty;
        float d = 0.f;
        if (x >= 0 && y >= 0 && x < a.W && y < a.H)
            d = __ldg(reinterpret_cast<const float*>(reinterpret_cast<const char*>(a.in) + (int64_t)y * a.in_pitch) + x);
        tile[ty][tx] = d;
    }
    __syncthreads();
    const int x = blockIdx.x * CT_X + threadIdx.x, y = blockIdx.y * CT_Y + threadIdx.y;
    if (x >= a.W || y >= a.H) return;
    const float dcf = tile[threadIdx.y + hw][threadIdx.x + hw];
    int reason = FSW_REASON_OK;
    if (!(dcf > 0.f)) reason = FSW_REASON_NO_PLANE;
    else {
        const double dc = (double)dcf;
        int consistent = 0;
        for (int dy = 0; dy < a.window; ++dy)
            for (int dx = 0; dx < a.window; ++dx) {
                const float dn = tile[threadIdx.y + dy][threadIdx.x + dx];
                if ((dx != hw || dy != hw) && dn > 0.f && fabs((double)dn - dc) < a.gamma) ++consistent;
            }
        if ((double)consistent / (double)(a.window * a.window - 1) < a.delta) reason = FSW_REASON_CONTINUITY;
        else if (a.mask != nullptr && a.mask[(int64_t)y * a.mask_pitch + x]) reason = FSW_REASON_MASKED;
    }
    *(reinterpret_cast<float*>(reinterpret_cast<char*>(a.out) + (int64_t)y * a.out_pitch) + x) = reason == FSW_REASON_OK ? dcf : 0.f;
    if (a.reason != nullptr) a.reason[(int64_t)y * a.reason_pitch + x] = (uint8_t)reason;
}

}  // namespace

cudaError_t fsw_launch_pack_footprints(const FswPackArgs& args, cudaStream_t stream) {
    dim3 grid((args.W + 2 * 256 - 1) / (2 * 256), args.H, args.n);
    pack_footprints_kernel<<<grid, 256, 0, stream>>>(args);
    return cudaGetLastError();
}

cudaError_t fsw_launch_downsample(const FswDownArgs& args, cudaStream_t stream) {
    int maxW = 0, maxH = 0;
    for (int i = 0; i < args.n; ++i) {
        maxW = args.W[i] / 2 > maxW ? args.W[i] / 2 : maxW;
        maxH = args.H[i] / 2 > maxH ? args.H[i] / 2 : maxH;
    }
    dim3 grid((maxW + 255) / 256, maxH, args.n);
    downsample_kernel<<<grid, 256, 0, stream>>>(args);
    return cudaGetLastError();
}

cudaError_t fsw_launch_continuity(const FswContinuityArgs& args, cudaStream_t stream) {
    dim3 grid((args.W + CT_X - 1) / CT_X, (args.H + CT_Y - 1) / CT_Y, 1);
    continuity_kernel<<<grid, dim3(CT_X, CT_Y, 1), 0, stream>>>(args);
    return cudaGetLastError();
}
