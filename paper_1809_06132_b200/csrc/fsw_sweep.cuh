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
    static constexpr size_t SMEM = sizeof(float4) * NE + sizeof(float) * (2 * PLANE + 4 * HPLANE);
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

/* S2-S4 for one halo pixel: returns the bilinear sample of the view at the plane-induced position, or NaN if the
 * pixel / plane / view combination is invalid ("NONE" of SURVEY 8(b)). */
__device__ __forceinline__ float warp_sample(const float4 ray, const FswDevView& vw, float nx, float ny, float nz,
                                             float inv_d, float inv_range_max, float centre) {
    /* S2: incidence and inverse range; X' ~ R r + (q/d) T */
    float q = fmaf(nx, ray.x, fmaf(ny, ray.y, nz * ray.z));
    float s = q * inv_d;
    bool ok = (ray.w != 0.f) & (q > FSW_EPS_Q) & (s >= inv_range_max);
    float X, Y, Z;
    if (vw.ident_R) {
        X = fmaf(s, vw.T[0], ray.x);
        Y = fmaf(s, vw.T[1], ray.y);
        Z = fmaf(s, vw.T[2], ray.z);
    } else {
        X = fmaf(vw.R[0], ray.x, fmaf(vw.R[1], ray.y, fmaf(vw.R[2], ray.z, s * vw.T[0])));
        Y = fmaf(vw.R[3], ray.x, fmaf(vw.R[4], ray.y, fmaf(vw.R[5], ray.z, s * vw.T[1])));
        Z = fmaf(vw.R[6], ray.x, fmaf(vw.R[7], ray.y, fmaf(vw.R[8], ray.z, s * vw.T[2])));
    }
    /* S3: unified projection */
    const FswDevCam& c = vw.cam;
    float rho2 = fmaf(X, X, fmaf(Y, Y, Z * Z));
    float rho = rho2 * rsqrt_approx(rho2);
    float den = fmaf(c.xi, rho, Z);
    ok &= (den > FSW_EPS_DEN * rho) & (Z >= c.cos_fov * rho);
    float iden = rcp_approx(den);
    float mx = X * iden, my = Y * iden;
    float xd = mx, yd = my;
    if (c.dist_mode != FSW_DIST_NONE) {
        float r2 = fmaf(mx, mx, my * my);
        if (c.dist_mode == FSW_DIST_K1) {
            float rad = fmaf(c.k1, r2, 1.f);
            xd = mx * rad;
            yd = my * rad;
        } else {
            float rad = fmaf(r2, fmaf(c.k2, r2, c.k1), 1.f);
            xd = fmaf(mx, rad, fmaf(2.f * c.p1 * mx, my, c.p2 * fmaf(2.f * mx, mx, r2)));
            yd = fmaf(my, rad, fmaf(c.p1, fmaf(2.f * my, my, r2), 2.f * c.p2 * mx * my));
        }
    }
    float u = fmaf(c.fx, xd, c.cx);
    float v = fmaf(c.fy, yd, c.cy);
    /* bilinear footprint inside the view image: 0 <= u < W-1, 0 <= v < H-1 */
    ok &= (u >= 0.f) & (u < (float)(c.W - 1)) & (v >= 0.f) & (v < (float)(c.H - 1));
    float b = CUDART_NAN_F;
    if (ok) {
        /* S4: four point fetches, FP32 lerp (hardware texture filtering has 8-bit weights: too coarse) */
        float fu = floorf(u), fv = floorf(v);
        int ix = (int)fu, iy = (int)fv;
        float au = u - fu, av = v - fv;
        float i00, i10, i01, i11;
        if (vw.pix_mode == FSW_PIX_FOOT_U8) {
            uint32_t w = __ldg(reinterpret_cast<const uint32_t*>(vw.img) + (int64_t)iy * vw.pitch_elems + ix);
            i00 = (float)(w & 0xffu);
            i10 = (float)((w >> 8) & 0xffu);
            i01 = (float)((w >> 16) & 0xffu);
            i11 = (float)(w >> 24);
        } else {
            const float* p = reinterpret_cast<const float*>(vw.img) + (int64_t)iy * vw.pitch_elems + ix;
            i00 = __ldg(p);
            i10 = __ldg(p + 1);
            i01 = __ldg(p + vw.pitch_elems);
            i11 = __ldg(p + vw.pitch_elems + 1);
        }
        float top = fmaf(au, i10 - i00, i00);
        float bot = fmaf(au, i11 - i01, i01);
        b = fmaf(av, bot - top, top) - centre;
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

template <int WIN>
__global__ void __launch_bounds__(NT, 2) sweep_kernel(const __grid_constant__ FswSweepArgs args) {
    using C = Cfg<WIN>;
    constexpr int HW = C::HW;
    constexpr float NWIN = (float)(WIN * WIN);
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float4* rays = reinterpret_cast<float4*>(smem_raw);
    float* a_s = reinterpret_cast<float*>(rays + C::NE);
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
        for (int e = tid; e < C::NE; e += NT) {
            int row = e / C::EW, col = e - row * C::EW;
            int px = x0t - HW + col, py = y0t - HW + row;
            float4 ry = make_float4(0.f, 0.f, 0.f, 0.f);
            float a = 0.f;
            if (px >= 0 && px < W && py >= 0 && py < H) {
                float rx, ryy, rz;
                if (back_project(args.ref, (float)px, (float)py, rx, ryy, rz)) ry = make_float4(rx, ryy, rz, 1.f);
                if (args.ref_dtype == FSW_U8)
                    a = (float)__ldg(reinterpret_cast<const uint8_t*>(args.ref_img) + (int64_t)py * args.ref_pitch_bytes + px);
                else
                    a = __ldg(reinterpret_cast<const float*>(reinterpret_cast<const char*>(args.ref_img) + (int64_t)py * args.ref_pitch_bytes) + px);
                lsum += a;
                lcnt += 1;
            }
            rays[e] = ry;
            a_s[row * C::SB + col] = a;
            b_s[row * C::SB + col] = ry.w;
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
        for (int e = tid; e < C::NE; e += NT) {
            int row = e / C::EW, col = e - row * C::EW;
            a_s[row * C::SB + col] -= centre;
        }
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
        tile_active = __syncthreads_or(active_mask != 0);

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
                for (int e = tid; e < C::NE; e += NT) {
                    float4 ry = rays[e];
                    faces |= (ry.w != 0.f) && (fmaf(nx, ry.x, fmaf(ny, ry.y, nz * ry.z)) > FSW_EPS_Q);
                }
                const bool fam_active = __syncthreads_or(faces);
                for (int j = 0; j < F.count; ++j) {
                    const int k = F.first + j;
                    const float inv_d = args.inv_d[k];
                    float acc[RPT];
                    int cnt[RPT];
#pragma unroll
                    for (int i = 0; i < RPT; ++i) { acc[i] = 0.f; cnt[i] = 0; }
                    if (fam_active) {
                        for (int v = 0; v < args.n_views; ++v) {
                            const FswDevView& vw = args.views[v];
                            /* ---- S2-S4: sample the plane-warped view at every halo pixel -------------------- */
                            bool all_ok = true, any_ok = false;
                            for (int e = tid; e < C::NE; e += NT) {
                                int row = e / C::EW, col = e - row * C::EW;
                                float b = warp_sample(rays[e], vw, nx, ny, nz, inv_d, args.inv_range_max, centre);
                                bool ok = (b == b);
                                all_ok &= ok;
                                any_ok |= ok;
                                b_s[row * C::SB + col] = b;
                            }
                            const int n_all = __syncthreads_count(all_ok);
                            const bool mixed = n_all != NT;
                            if (mixed) {
                                if (!__syncthreads_or(any_ok)) continue; /* this view sees nothing of the tile */
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
            float4 ry = rays[(wy * RPT + i + HW) * C::EW + lane + HW];
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

template <int WIN>
cudaError_t launch_sweep_win(const FswSweepArgs& args, cudaStream_t stream) {
    dim3 grid((args.ref.W + TX - 1) / TX, (args.ref.H + TY - 1) / TY);
    sweep_kernel<WIN><<<grid, NT, Cfg<WIN>::SMEM, stream>>>(args);
    return cudaGetLastError();
}

template <int WIN>
cudaError_t prepare_sweep_win() {
    return cudaFuncSetAttribute(sweep_kernel<WIN>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg<WIN>::SMEM);
}

}  // namespace fsw
#endif
