/*
 * fsw_sweep.cuh -- the fused fisheye plane-sweep kernel (sm_100a), steps S1..S12 of SURVEY.md section 8(a).
 *
 * One CTA owns a TX x TY tile of reference pixels.  It
 *   S1  back-projects the tile plus a halo of w/2 pixels through the unified model (Eq. 1) into
 *       shared memory (no ray LUT ever touches HBM),
 *   and then, for every sweep plane k and every matching view v,
 *   S2-S4 maps every halo pixel through the plane into the view (ray-homography form X' ~ R r + (n.r / d_k) T),
 *       projects it with the view's fisheye model and samples the view bilinearly,
 *   S5  forms the windowed sums of b, b^2, ab with separable box sums staged in shared memory and scores
 *       cost = (1 - ZNCC)/2,
 *   S6  averages the cost over the views whose window is fully valid,
 *   S7  keeps best cost, non-adjacent second best and the neighbours of the best in registers --
 *       the cost volume is never written unless args.debug_cost is set,
 *   and finally
 *   S8-S12 refines the plane with a parabola, converts to depth, merges with the half-resolution pass if one is
 *       given, applies the cost / ratio filters and the mask and
 *       stores the maps with coalesced row writes.
 *
 * Numerics: everything is FP32, no fast-math.  Intensities are centred on a per-tile constant before any sum
 * (ZNCC is invariant to offsets) so that N*Sum(b^2) - Sum(b)^2 does not cancel catastrophically.
 */
#ifndef FSW_SWEEP_CUH
#define FSW_SWEEP_CUH

#include <math_constants.h>

#include "fsw_internal.h"

namespace fsw {

constexpr int TX = 32;       /* tile width  = one warp of columns */
constexpr int TY = 32;       /* tile height */
constexpr int NT = 256;      /* threads per CTA */
constexpr int RPT = TY / (NT / 32); /* output rows per thread in the vertical pass (4) */
constexpr int RUN = 8;       /* outputs per work item of the horizontal pass */
constexpr int NRUN = TX / RUN;
constexpr int HS = TX + 4;   /* row stride of the row-sum planes: == 4 (mod 8) keeps 128-bit stores conflict free */

template <int WIN>
struct Cfg {
    static constexpr int HW = WIN / 2;
    static constexpr int EW = TX + 2 * HW; /* tile + halo */
    static constexpr int EH = TY + 2 * HW;
    static constexpr int NE = EW * EH;
    static constexpr int NV = RUN + 2 * HW;        /* values one horizontal work item reads */
    static constexpr int NV4 = (NV + 3) / 4;       /* ... as 128-bit loads */
    static constexpr int SB0 = ((EW + 3) / 4) * 4;
    static constexpr int SB1 = (SB0 % 8 == 0) ? SB0 + 4 : SB0; /* == 4 (mod 8): conflict-free 128-bit row loads */
    /* the last run of a row starts at column 24 and reads NV4*4 values */
    static constexpr int SB = (SB1 >= (NRUN - 1) * RUN + NV4 * 4) ? SB1 : SB1 + 8;
    static constexpr int PLANE = EH * SB;          /* floats in one sample plane */
    static constexpr int HPLANE = EH * HS;         /* floats in one row-sum plane */
    static constexpr size_t SMEM = sizeof(float4) * PLANE + sizeof(float) * (2 * PLANE + 4 * HPLANE);
};

__device__ __forceinline__ float rsqrt_approx(float x) {
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float rcp_approx(float x) {
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

/* S1: pixel -> unit ray of the reference camera.  Returns false outside the field of view / not invertible.
 * Unified model back-projection, PAPER.md:150-160 (Eq. 1), after removing the distortion by Newton iterations
 * with a fixed count. */
__device__ inline bool back_project(const FswDevCam& c, float u, float v, float& rx, float& ry, float& rz) {
    float xd = (u - c.cx) / c.fx, yd = (v - c.cy) / c.fy;
    float x = xd, y = yd;
    if (c.dist_mode == FSW_DIST_K1 || (c.dist_mode == FSW_DIST_FULL && c.p1 == 0.f && c.p2 == 0.f)) {
        float rd = sqrtf(xd * xd + yd * yd);
        if (rd > 0.f) {
            float r = rd;
#pragma unroll 1
            for (int it = 0; it < 10; ++it) {
                float r2 = r * r;
                float g = r * (1.f + c.k1 * r2 + c.k2 * r2 * r2) - rd;
                float dg = 1.f + 3.f * c.k1 * r2 + 5.f * c.k2 * r2 * r2;
                if (!(dg > 1e-6f)) return false; /* past the turning point of the radial polynomial */
                r -= g / dg;
                if (!(r > 0.f)) return false;
            }
            float r2 = r * r;
            if (!(1.f + 3.f * c.k1 * r2 + 5.f * c.k2 * r2 * r2 > 0.f)) return false;
            float sc = r / rd;
            x = xd * sc;
            y = yd * sc;
        }
    } else if (c.dist_mode == FSW_DIST_FULL) {
#pragma unroll 1
        for (int it = 0; it < 12; ++it) {
            float r2 = x * x + y * y;
            float rad = 1.f + c.k1 * r2 + c.k2 * r2 * r2;
            float drad = c.k1 + 2.f * c.k2 * r2;
            float gx = x * rad + 2.f * c.p1 * x * y + c.p2 * (r2 + 2.f * x * x) - xd;
            float gy = y * rad + c.p1 * (r2 + 2.f * y * y) + 2.f * c.p2 * x * y - yd;
            float jxx = rad + 2.f * x * x * drad + 2.f * c.p1 * y + 6.f * c.p2 * x;
            float jxy = 2.f * x * y * drad + 2.f * c.p1 * x + 2.f * c.p2 * y;
            float jyy = rad + 2.f * y * y * drad + 6.f * c.p1 * y + 2.f * c.p2 * x;
            float det = jxx * jyy - jxy * jxy;
            if (!(det > 1e-6f)) return false;
            x -= (jyy * gx - jxy * gy) / det;
            y -= (jxx * gy - jxy * gx) / det;
        }
        if (!(isfinite(x) && isfinite(y))) return false;
    }
    float rho2 = x * x + y * y;
    float rad = 1.f + (1.f - c.xi * c.xi) * rho2;
    if (rad < 0.f) return false;
    float eta = (c.xi + sqrtf(rad)) / (rho2 + 1.f);
    rx = eta * x;
    ry = eta * y;
    rz = eta - c.xi;
    float inv = 1.f / sqrtf(rx * rx + ry * ry + rz * rz); /* = 1 up to rounding */
    rx *= inv;
    ry *= inv;
    rz *= inv;
    return rz >= c.cos_fov; /* theta <= fov/2 */
}

/* Per-view constants of the sample phase, copied out of the kernel arguments once per (plane, view). */
struct ViewK {
    float T0, T1, T2;
    float R[9];
    float fx, fy, cx, cy, xi, cos_fov, k1, k2, p1, p2;
    unsigned W1, H1; /* W-1, H-1 */
    const void* img;
    int pitch, pix;
};

__device__ __forceinline__ ViewK load_view(const FswDevView& vw) {
    ViewK k;
    k.T0 = vw.T[0]; k.T1 = vw.T[1]; k.T2 = vw.T[2];
#pragma unroll
    for (int i = 0; i < 9; ++i) k.R[i] = vw.R[i];
    k.fx = vw.cam.fx; k.fy = vw.cam.fy; k.cx = vw.cam.cx; k.cy = vw.cam.cy; k.xi = vw.cam.xi;
    k.cos_fov = vw.cam.cos_fov; k.k1 = vw.cam.k1; k.k2 = vw.cam.k2; k.p1 = vw.cam.p1; k.p2 = vw.cam.p2;
    k.W1 = (unsigned)(vw.cam.W - 1); k.H1 = (unsigned)(vw.cam.H - 1);
    k.img = vw.img; k.pitch = (int)vw.pitch_elems; k.pix = vw.pix_mode;
    return k;
}

/* S2-S4 for one halo pixel: returns the bilinear sample of the view at the plane-induced position minus `centre`,
 * or NaN if the pixel / plane / view combination is invalid ("NONE" of SURVEY 8(b)).
 * IDENT: the view's relative rotation is the identity.  FULLDIST: k2 / p1 / p2 may be non-zero.
 * PIX: FSW_PIX_FOOT_U8, FSW_PIX_F32, or -1 = decided per view at run time.
 * cbias = 2^23 + rint(centre): 8-bit samples are widened by OR-ing them into the mantissa of 2^23, so subtracting
 * cbias both removes that bias and centres the sample, exactly. */
template <bool IDENT, bool FULLDIST, int PIX, bool CHECKDEN>
__device__ __forceinline__ float warp_sample(const float4 ray, const ViewK& k, float nx, float ny, float nz,
                                             float inv_d, float inv_range_max, float centre, float cbias) {
    /* S2: incidence and inverse range; X' ~ R r + (q/d) T */
    float q = fmaf(nx, ray.x, fmaf(ny, ray.y, nz * ray.z));
    float s = q * inv_d;
    bool ok = (q > FSW_EPS_Q) & (s >= inv_range_max); /* an invalid reference ray is stored as 0: q = 0 */
    float X, Y, Z;
    if (IDENT) {
        X = fmaf(s, k.T0, ray.x);
        Y = fmaf(s, k.T1, ray.y);
        Z = fmaf(s, k.T2, ray.z);
    } else {
        X = fmaf(k.R[0], ray.x, fmaf(k.R[1], ray.y, fmaf(k.R[2], ray.z, s * k.T0)));
        Y = fmaf(k.R[3], ray.x, fmaf(k.R[4], ray.y, fmaf(k.R[5], ray.z, s * k.T1)));
        Z = fmaf(k.R[6], ray.x, fmaf(k.R[7], ray.y, fmaf(k.R[8], ray.z, s * k.T2)));
    }
    /* S3: unified projection; one Newton step on each approximate reciprocal */
    float rho2 = fmaf(X, X, fmaf(Y, Y, Z * Z));
#ifdef FSW_REFINE_RECIPROCALS
    float y0 = rsqrt_approx(rho2);
    float t0 = rho2 * y0;
    float rho = fmaf(0.5f * t0, fmaf(-t0, y0, 1.f), t0);
#else
    float rho = rho2 * rsqrt_approx(rho2);
#endif
    float den = fmaf(k.xi, rho, Z);
    ok &= (Z >= k.cos_fov * rho); /* also false for NaN (rho2 == 0) */
    /* with cos(fov/2) + xi >= 1e-3 (checked on the host for the fast variants) the FOV test implies den > eps rho */
    if (CHECKDEN) ok &= (den > FSW_EPS_DEN * rho);
#ifdef FSW_REFINE_RECIPROCALS
    float i0 = rcp_approx(den);
    float iden = fmaf(i0, fmaf(-den, i0, 1.f), i0);
#else
    float iden = rcp_approx(den);
#endif
    float mx = X * iden, my = Y * iden;
    float r2 = fmaf(mx, mx, my * my);
    float xd, yd;
    if (!FULLDIST) {
        float rad = fmaf(k.k1, r2, 1.f);
        xd = mx * rad;
        yd = my * rad;
    } else {
        float rad = fmaf(r2, fmaf(k.k2, r2, k.k1), 1.f);
        xd = fmaf(mx, rad, fmaf(2.f * k.p1 * mx, my, k.p2 * fmaf(2.f * mx, mx, r2)));
        yd = fmaf(my, rad, fmaf(k.p1, fmaf(2.f * my, my, r2), 2.f * k.p2 * mx * my));
    }
    float u = fmaf(k.fx, xd, k.cx);
    float v = fmaf(k.fy, yd, k.cy);
    /* bilinear footprint inside the view image: 0 <= u < W-1, 0 <= v < H-1  <=>  0 <= floor(u) < W-1, ... */
    int ix = __float2int_rd(u), iy = __float2int_rd(v);
    ok &= ((unsigned)ix < k.W1) & ((unsigned)iy < k.H1);
    float b = CUDART_NAN_F;
    if (ok) {
        /* S4: point fetches + FP32 lerp (hardware texture filtering has 8-bit weights: too coarse for 1e-4) */
        float au = u - (__int_as_float(ix + 0x4B400000) - 12582912.f); /* u - floor(u) without a second conversion */
        float av = v - (__int_as_float(iy + 0x4B400000) - 12582912.f);
        int idx = iy * k.pitch + ix;
        float i00, d0, i01, d1;
        if (PIX == FSW_PIX_FOOT_U8 || (PIX < 0 && k.pix == FSW_PIX_FOOT_U8)) {
            uint32_t w = __ldg(reinterpret_cast<const uint32_t*>(k.img) + idx);
            float f00 = __uint_as_float(__byte_perm(w, 0x4B000000u, 0x7540));
            float f10 = __uint_as_float(__byte_perm(w, 0x4B000000u, 0x7541));
            float f01 = __uint_as_float(__byte_perm(w, 0x4B000000u, 0x7542));
            float f11 = __uint_as_float(__byte_perm(w, 0x4B000000u, 0x7543));
            i00 = f00 - cbias; d0 = f10 - f00;
            i01 = f01 - cbias; d1 = f11 - f01;
        } else {
            const float* p = reinterpret_cast<const float*>(k.img) + idx;
            float f00 = __ldg(p), f10 = __ldg(p + 1), f01 = __ldg(p + k.pitch), f11 = __ldg(p + k.pitch + 1);
            i00 = f00 - centre; d0 = f10 - f00;
            i01 = f01 - centre; d1 = f11 - f01;
        }
        float top = fmaf(au, d0, i00);
        float bot = fmaf(au, d1, i01);
        b = fmaf(av, bot - top, top);
    }
    return b;
}

/* Horizontal pass of the separable box sums: one work item = RUN consecutive outputs of one halo row.
 * MODE 0: p = a', q = ray-valid flag      -> planes {sum a', sum a'^2, sum flag}
 * MODE 1: p = b', q = a' (all valid)      -> planes {sum b', sum b'^2, sum a'b'}
 * MODE 2: p = b' (NaN = invalid), q = a'  -> as MODE 1 with invalid samples as 0, plus plane 3 = sum valid */
template <int WIN, int MODE>
__device__ __forceinline__ void hpass(const float* __restrict__ ps, const float* __restrict__ qs, float* __restrict__ hs,
                                      int item) {
    using C = Cfg<WIN>;
    const int row = item / NRUN, run = item % NRUN;
    const float4* p4 = reinterpret_cast<const float4*>(ps + row * C::SB + run * RUN);
    const float4* q4 = reinterpret_cast<const float4*>(qs + row * C::SB + run * RUN);
    float p[C::NV4 * 4], q[C::NV4 * 4];
#pragma unroll
    for (int i = 0; i < C::NV4; ++i) {
        float4 a = p4[i], b = q4[i];
        p[4 * i] = a.x; p[4 * i + 1] = a.y; p[4 * i + 2] = a.z; p[4 * i + 3] = a.w;
        q[4 * i] = b.x; q[4 * i + 1] = b.y; q[4 * i + 2] = b.z; q[4 * i + 3] = b.w;
    }
    float okf[C::NV4 * 4];
    if (MODE == 2) {
#pragma unroll
        for (int i = 0; i < C::NV; ++i) {
            bool ok = (p[i] == p[i]);
            okf[i] = ok ? 1.f : 0.f;
            p[i] = ok ? p[i] : 0.f;
        }
    }
    float pp[C::NV4 * 4], pq[C::NV4 * 4];
#pragma unroll
    for (int i = 0; i < C::NV; ++i) {
        pp[i] = p[i] * p[i];
        pq[i] = (MODE == 0) ? q[i] : p[i] * q[i];
    }
    float s0 = 0.f, s1 = 0.f, s2 = 0.f, s3 = 0.f;
#pragma unroll
    for (int i = 0; i < WIN; ++i) {
        s0 += p[i]; s1 += pp[i]; s2 += pq[i];
        if (MODE == 2) s3 += okf[i];
    }
    float o0[RUN], o1[RUN], o2[RUN], o3[RUN];
    o0[0] = s0; o1[0] = s1; o2[0] = s2; o3[0] = s3;
#pragma unroll
    for (int j = 1; j < RUN; ++j) {
        s0 += p[j + WIN - 1] - p[j - 1];
        s1 += pp[j + WIN - 1] - pp[j - 1];
        s2 += pq[j + WIN - 1] - pq[j - 1];
        if (MODE == 2) s3 += okf[j + WIN - 1] - okf[j - 1];
        o0[j] = s0; o1[j] = s1; o2[j] = s2; o3[j] = s3;
    }
    float4* h0 = reinterpret_cast<float4*>(hs + row * HS + run * RUN);
    float4* h1 = reinterpret_cast<float4*>(hs + C::HPLANE + row * HS + run * RUN);
    float4* h2 = reinterpret_cast<float4*>(hs + 2 * C::HPLANE + row * HS + run * RUN);
    h0[0] = make_float4(o0[0], o0[1], o0[2], o0[3]); h0[1] = make_float4(o0[4], o0[5], o0[6], o0[7]);
    h1[0] = make_float4(o1[0], o1[1], o1[2], o1[3]); h1[1] = make_float4(o1[4], o1[5], o1[6], o1[7]);
    h2[0] = make_float4(o2[0], o2[1], o2[2], o2[3]); h2[1] = make_float4(o2[4], o2[5], o2[6], o2[7]);
    if (MODE == 2) {
        float4* h3 = reinterpret_cast<float4*>(hs + 3 * C::HPLANE + row * HS + run * RUN);
        h3[0] = make_float4(o3[0], o3[1], o3[2], o3[3]); h3[1] = make_float4(o3[4], o3[5], o3[6], o3[7]);
    }
}

/* Vertical pass: column x, output rows r0..r0+RPT-1; sums WIN consecutive row sums of one plane. */
template <int WIN>
__device__ __forceinline__ void vpass(const float* __restrict__ h, int x, int r0, float (&out)[RPT]) {
    float v[RPT + WIN - 1];
#pragma unroll
    for (int i = 0; i < RPT + WIN - 1; ++i) v[i] = h[(r0 + i) * HS + x];
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < WIN; ++i) s += v[i];
    out[0] = s;
#pragma unroll
    for (int j = 1; j < RPT; ++j) {
        s += v[j + WIN - 1] - v[j - 1];
        out[j] = s;
    }
}

/* warp-uniform value that the compiler can also prove uniform (lets it keep loop state in uniform registers) */
__device__ __forceinline__ int uniform_int(int x) { return __shfl_sync(0xffffffffu, x, 0); }

template <int WIN, bool IDENT, bool FULLDIST, int PIX, bool CHECKDEN>
__global__ void __launch_bounds__(NT, 2) sweep_kernel(const __grid_constant__ FswSweepArgs args) {
    using C = Cfg<WIN>;
    constexpr int HW = C::HW;
    constexpr float NWIN = (float)(WIN * WIN);
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float4* rays = reinterpret_cast<float4*>(smem_raw);
    float* a_s = reinterpret_cast<float*>(rays + C::PLANE);
    float* b_s = a_s + C::PLANE;
    float* hs = b_s + C::PLANE;
    __shared__ float red_sum[NT / 32];
    __shared__ int red_cnt[NT / 32];

    const int tid = threadIdx.x, lane = tid & 31, wy = tid >> 5;
    const int x0t = blockIdx.x * TX, y0t = blockIdx.y * TY;
    const int W = args.ref.W, H = args.ref.H;
    const int ox = x0t + lane;     /* this thread's output column */
    const int oy0 = y0t + wy * RPT; /* ... and first output row */

    /* WTA state (S7), per owned output pixel */
    float b1[RPT], s2[RPT], m0[RPT], m1[RPT], cm[RPT], cp[RPT], cprev[RPT];
    int k1[RPT], knext[RPT];
#pragma unroll
    for (int i = 0; i < RPT; ++i) {
        b1[i] = CUDART_INF_F; s2[i] = CUDART_INF_F; m0[i] = CUDART_INF_F; m1[i] = CUDART_INF_F;
        cm[i] = CUDART_INF_F; cp[i] = CUDART_INF_F; cprev[i] = CUDART_INF_F;
        k1[i] = -1; knext[i] = -1;
    }
    unsigned n_eval = 0;

    const bool tile_in_roi = (x0t < args.roi_x1) && (x0t + TX > args.roi_x0) && (y0t < args.roi_y1) && (y0t + TY > args.roi_y0);
    bool tile_active = false;
    unsigned active_mask = 0; /* bit i: output i of this thread can have a finite cost */
    float A1[RPT], A2[RPT];
#pragma unroll
    for (int i = 0; i < RPT; ++i) { A1[i] = 0.f; A2[i] = 0.f; }

    if (tile_in_roi) {
        /* ---- S1: rays and reference intensities of the tile + halo ------------------------------------ */
        float lsum = 0.f;
        int lcnt = 0;
        int my_n = 0; /* halo pixels (not pad entries) this thread samples per plane and view */
        for (int p = tid; p < C::PLANE; p += NT) {
            int row = p / C::SB, col = p - row * C::SB;
            int px = x0t - HW + col, py = y0t - HW + row;
            float4 ry = make_float4(0.f, 0.f, 0.f, 0.f); /* invalid rays (and pad entries) are zero vectors */
            float a = 0.f;
            if (col < C::EW) {
                my_n += 1;
                if (px >= 0 && px < W && py >= 0 && py < H) {
                    float rx, ryy, rz;
                    bool ok = back_project(args.ref, (float)px, (float)py, rx, ryy, rz);
                    if (ok) ry = make_float4(rx, ryy, rz, 1.f);
                    if (args.ref_dtype == FSW_U8)
                        a = (float)__ldg(reinterpret_cast<const uint8_t*>(args.ref_img) + (int64_t)py * args.ref_pitch_bytes + px);
                    else
                        a = __ldg(reinterpret_cast<const float*>(reinterpret_cast<const char*>(args.ref_img) + (int64_t)py * args.ref_pitch_bytes) + px);
                    if (ok) { lsum += a; lcnt += 1; } /* pixels outside the FOV never enter a valid window */
                }
            }
            rays[p] = ry;
            a_s[p] = a;
            b_s[p] = ry.w;
        }
        /* centring constant of the tile: mean reference intensity (rounded to an integer for 8-bit images so
         * that a - centre stays exact) */
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            lsum += __shfl_xor_sync(0xffffffffu, lsum, o);
            lcnt += __shfl_xor_sync(0xffffffffu, lcnt, o);
        }
        if (lane == 0) { red_sum[wy] = lsum; red_cnt[wy] = lcnt; }
        __syncthreads();
        float tsum = 0.f;
        int tcnt = 0;
#pragma unroll
        for (int i = 0; i < NT / 32; ++i) { tsum += red_sum[i]; tcnt += red_cnt[i]; }
        float centre = tcnt > 0 ? tsum / (float)tcnt : 0.f;
        if (args.ref_dtype == FSW_U8) centre = rintf(centre);
        const float cbias = 8388608.f + rintf(centre);
        for (int p = tid; p < C::PLANE; p += NT) a_s[p] -= centre;
        __syncthreads();
        /* window sums of the reference side, once per pixel: A1 = sum a', A2 = N sum a'^2 - (sum a')^2 */
        if (tid < C::EH * NRUN) hpass<WIN, 0>(a_s, b_s, hs, tid);
        __syncthreads();
        {
            float sa[RPT], saa[RPT], sf[RPT];
            vpass<WIN>(hs, lane, wy * RPT, sa);
            vpass<WIN>(hs + C::HPLANE, lane, wy * RPT, saa);
            vpass<WIN>(hs + 2 * C::HPLANE, lane, wy * RPT, sf);
#pragma unroll
            for (int i = 0; i < RPT; ++i) {
                int oy = oy0 + i;
                bool in_roi = ox >= args.roi_x0 && ox < args.roi_x1 && oy >= args.roi_y0 && oy < args.roi_y1;
                bool act = in_roi && (sf[i] == NWIN); /* every window pixel inside the image and the FOV */
                if (act) active_mask |= 1u << i;
                A1[i] = sa[i];
                A2[i] = fmaf(NWIN, saa[i], -sa[i] * sa[i]);
            }
        }
        tile_active = uniform_int(__syncthreads_or(active_mask != 0)) != 0;

        if (tile_active) {
            const float inv_views = 1.f / (float)args.n_views;
            for (int f = 0; f < args.n_fams; ++f) {
                const FswDevFamily& F = args.fam[f];
                const float nx = F.n[0], ny = F.n[1], nz = F.n[2];
                /* family start: planes of another family are never "adjacent" (reading Q12) */
#pragma unroll
                for (int i = 0; i < RPT; ++i) { m1[i] = m0[i]; cprev[i] = CUDART_INF_F; knext[i] = -1; }
                /* does any halo ray face this family's planes? */
                bool faces = false;
                for (int p = tid; p < C::PLANE; p += NT) {
                    float4 ry = rays[p];
                    faces |= (ry.w != 0.f) && (fmaf(nx, ry.x, fmaf(ny, ry.y, nz * ry.z)) > FSW_EPS_Q);
                }
                const bool fam_active = uniform_int(__syncthreads_or(faces)) != 0;
                for (int j = 0; j < F.count; ++j) {
                    const int k = F.first + j;
                    const float inv_d = args.inv_d[k];
                    float acc[RPT];
                    int cnt[RPT];
#pragma unroll
                    for (int i = 0; i < RPT; ++i) { acc[i] = 0.f; cnt[i] = 0; }
                    if (fam_active) {
                        for (int v = 0; v < args.n_views; ++v) {
                            const ViewK vk = load_view(args.views[v]);
                            /* ---- S2-S4: sample the plane-warped view at every halo pixel -------------------- */
                            int nvalid = 0;
#pragma unroll 2
                            for (int p = tid; p < C::PLANE; p += NT) {
                                float b = warp_sample<IDENT, FULLDIST, PIX, CHECKDEN>(rays[p], vk, nx, ny, nz, inv_d,
                                                                                      args.inv_range_max, centre, cbias);
                                nvalid += (b == b) ? 1 : 0;
                                b_s[p] = b;
                            }
                            const int n_all = uniform_int(__syncthreads_count(nvalid == my_n));
                            const bool mixed = n_all != NT;
                            if (mixed) {
                                if (!uniform_int(__syncthreads_or(nvalid > 0))) continue; /* this view sees nothing of the tile */
                            }
                            /* ---- S5: separable box sums and ZNCC ------------------------------------------- */
                            if (tid < C::EH * NRUN) {
                                if (mixed) hpass<WIN, 2>(b_s, a_s, hs, tid);
                                else hpass<WIN, 1>(b_s, a_s, hs, tid);
                            }
                            __syncthreads();
                            float sb[RPT], sbb[RPT], sab[RPT], sv[RPT];
                            vpass<WIN>(hs, lane, wy * RPT, sb);
                            vpass<WIN>(hs + C::HPLANE, lane, wy * RPT, sbb);
                            vpass<WIN>(hs + 2 * C::HPLANE, lane, wy * RPT, sab);
                            if (mixed) vpass<WIN>(hs + 3 * C::HPLANE, lane, wy * RPT, sv);
#pragma unroll
                            for (int i = 0; i < RPT; ++i) {
                                bool okv = (active_mask >> i) & 1u;
                                if (mixed) okv = okv && (sv[i] == NWIN);
                                float cov = fmaf(NWIN, sab[i], -A1[i] * sb[i]);
                                float vb = fmaf(NWIN, sbb[i], -sb[i] * sb[i]);
                                float prod = fmaxf(A2[i] * vb, args.floor2);
                                float z = cov * rsqrt_approx(prod);
                                float cst = __saturatef(fmaf(-0.5f, z, 0.5f));
                                if (okv) { acc[i] += cst; cnt[i] += 1; n_eval += 1; }
                            }
                        }
                    }
                    /* ---- S6 + S7: view mean, streaming winner-take-all ------------------------------------- */
#pragma unroll
                    for (int i = 0; i < RPT; ++i) {
                        float c = CUDART_INF_F;
                        if (cnt[i] == args.n_views) c = acc[i] * inv_views;
                        else if (cnt[i] > 0) c = acc[i] / (float)cnt[i];
                        if (args.debug_cost != nullptr) {
                            int oy = oy0 + i;
                            if (ox < W && oy < H) args.debug_cost[((int64_t)k * H + oy) * W + ox] = c;
                        }
                        if (k == knext[i]) cp[i] = c;            /* neighbour above the running best */
                        else if (k > knext[i]) s2[i] = fminf(s2[i], c); /* eligible second best */
                        if (c < b1[i]) {                         /* strict: lowest index wins ties */
                            s2[i] = m1[i];                       /* best of everything at least two planes back */
                            cm[i] = cprev[i];
                            cp[i] = CUDART_INF_F;
                            b1[i] = c; k1[i] = k; knext[i] = k + 1;
                        }
                        m1[i] = m0[i];
                        m0[i] = fminf(m0[i], c);
                        cprev[i] = c;
                    }
                }
            }
        }
    }
    if (args.debug_cost != nullptr && !tile_active) {
        for (int k = 0; k < args.n_planes; ++k)
#pragma unroll
            for (int i = 0; i < RPT; ++i) {
                int oy = oy0 + i;
                if (ox < W && oy < H) args.debug_cost[((int64_t)k * H + oy) * W + ox] = CUDART_INF_F;
            }
    }

    /* ---- S8-S12: refinement, depth, merge, filters, mask, stores ------------------------------------------- */
    unsigned n_raw = 0, n_ok = 0;
#pragma unroll
    for (int i = 0; i < RPT; ++i) {
        const int oy = oy0 + i;
        if (ox >= W || oy >= H) continue;
        bool raw_valid = k1[i] >= 0;
        float depth = 0.f, c1 = CUDART_INF_F, c2 = CUDART_INF_F;
        int kidx = -1;
        if (raw_valid) {
            int f = 0;
            for (int g = 1; g < args.n_fams; ++g)
                if (k1[i] >= args.fam[g].first) f = g;
            const FswDevFamily& F = args.fam[f];
            float dl = 0.f;
            if (args.subpixel && cm[i] < CUDART_INF_F && cp[i] < CUDART_INF_F) {
                float den = cm[i] - 2.f * b1[i] + cp[i];
                if (den > 1e-12f) dl = fminf(fmaxf(0.5f * (cm[i] - cp[i]) / den, -0.5f), 0.5f);
            }
            float s = fmaf((float)(k1[i] - F.first) + dl, F.ds, F.s0);
            float d = F.spacing == FSW_INVERSE ? 1.f / s : s;
            float4 ry = rays[(wy * RPT + i + HW) * C::SB + lane + HW];
            float q = fmaf(F.n[0], ry.x, fmaf(F.n[1], ry.y, F.n[2] * ry.z));
            float range = d / q;
            depth = args.depth_kind == FSW_DEPTH_Z ? range * ry.z : range;
            c1 = b1[i];
            c2 = s2[i] < CUDART_INF_F ? s2[i] : 1.f;
            kidx = k1[i] | args.index_flag;
        } else if (args.lo_k != nullptr) {
            /* S10(c)-(e): nearest-neighbour upsample of the half-resolution pass */
            int xl = ox >> 1, yl = oy >> 1;
            if (xl < args.lo_W && yl < args.lo_H) {
                int64_t j = (int64_t)yl * args.lo_W + xl;
                int kl = args.lo_k[j];
                if (kl >= 0) {
                    raw_valid = true;
                    depth = args.lo_depth[j]; c1 = args.lo_c1[j]; c2 = args.lo_c2[j]; kidx = kl;
                }
            }
        }
        int reason = FSW_REASON_OK;
        if (!raw_valid) reason = FSW_REASON_NO_PLANE;
        else {
            float alpha = oy < args.horizon_row ? args.alpha_upper : args.alpha_lower;
            if ((args.filters & FSW_FILTER_COST) && c1 > alpha) reason = FSW_REASON_COST_FILTER;
            else if ((args.filters & FSW_FILTER_RATIO) && c2 < args.beta * fmaxf(c1, 1e-6f)) reason = FSW_REASON_RATIO_FILTER;
            else if (args.mask != nullptr && args.mask[(int64_t)oy * args.mask_pitch + ox]) reason = FSW_REASON_MASKED;
        }
        if (reason != FSW_REASON_OK) depth = 0.f;
        n_raw += raw_valid ? 1u : 0u;
        n_ok += reason == FSW_REASON_OK ? 1u : 0u;
        *reinterpret_cast<float*>(reinterpret_cast<char*>(args.out_depth) + (int64_t)oy * args.out_depth_pitch + 4 * (int64_t)ox) = depth;
        if (args.out_c1) *reinterpret_cast<float*>(reinterpret_cast<char*>(args.out_c1) + (int64_t)oy * args.out_c1_pitch + 4 * (int64_t)ox) = c1;
        if (args.out_c2) *reinterpret_cast<float*>(reinterpret_cast<char*>(args.out_c2) + (int64_t)oy * args.out_c2_pitch + 4 * (int64_t)ox) = c2;
        if (args.out_k) *reinterpret_cast<int16_t*>(reinterpret_cast<char*>(args.out_k) + (int64_t)oy * args.out_k_pitch + 2 * (int64_t)ox) = (int16_t)kidx;
        if (args.out_reason) args.out_reason[(int64_t)oy * args.out_reason_pitch + ox] = (uint8_t)reason;
    }
    /* counters */
    if (args.counters != nullptr) {
        unsigned e = n_eval;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            e += __shfl_xor_sync(0xffffffffu, e, o);
            n_raw += __shfl_xor_sync(0xffffffffu, n_raw, o);
            n_ok += __shfl_xor_sync(0xffffffffu, n_ok, o);
        }
        if (lane == 0) {
            if (e) atomicAdd(&args.counters[0], (unsigned long long)e);
            if (n_raw && args.count_pixels) atomicAdd(&args.counters[1], (unsigned long long)n_raw);
            if (n_ok && args.count_pixels) atomicAdd(&args.counters[2], (unsigned long long)n_ok);
        }
    }
}

/* Kernel variants: 0 = generic (any rotation, full distortion polynomial, pixel type decided per view),
 * 1 = identity rotations, k1-only (or no) distortion, cos(fov/2) + xi >= 1e-3, footprint-packed 8-bit views,
 * 2 = the same with float32 views. */
template <int WIN>
cudaError_t launch_sweep_win(const FswSweepArgs& args, int variant, cudaStream_t stream) {
    dim3 grid((args.ref.W + TX - 1) / TX, (args.ref.H + TY - 1) / TY);
    if (variant == 1) sweep_kernel<WIN, true, false, FSW_PIX_FOOT_U8, false><<<grid, NT, Cfg<WIN>::SMEM, stream>>>(args);
    else if (variant == 2) sweep_kernel<WIN, true, false, FSW_PIX_F32, false><<<grid, NT, Cfg<WIN>::SMEM, stream>>>(args);
    else sweep_kernel<WIN, false, true, -1, true><<<grid, NT, Cfg<WIN>::SMEM, stream>>>(args);
    return cudaGetLastError();
}

template <int WIN>
cudaError_t prepare_sweep_win() {
    cudaError_t e = cudaFuncSetAttribute(sweep_kernel<WIN, true, false, FSW_PIX_FOOT_U8, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg<WIN>::SMEM);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(sweep_kernel<WIN, true, false, FSW_PIX_F32, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg<WIN>::SMEM);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(sweep_kernel<WIN, false, true, -1, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg<WIN>::SMEM);
}

}  // namespace fsw
#endif
