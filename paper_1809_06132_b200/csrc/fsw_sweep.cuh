/*
 * fsw_sweep.cuh -- the fused fisheye plane-sweep kernel (sm_100a), steps S1..S12 of SURVEY.md section 8(a).
 *
 * Persistent CTAs claim (frame set, tile) items from a queue, heaviest tiles first.  For one TX x TY tile of
 * reference pixels a CTA
 *   S1  back-projects the tile plus a halo of w/2 pixels through the unified model (Eq. 1) into
 *       shared memory (no ray LUT ever touches HBM),
 *   and then, for every sweep plane k,
 *   S2-S4 maps every halo pixel through the plane into ALL matching views in one pass (ray-homography form
 *       X' ~ R r + (n.r / d_k) T; the incidence n.r and the range test are shared by the views), projects it with
 *       each view's fisheye model and samples the view bilinearly from its footprint image (one 128-bit load),
 *   S5  forms the windowed sums of b, b^2, ab with separable sliding box sums staged in shared memory and scores
 *       cost = (1 - ZNCC)/2,
 *   S6  averages the cost over the views whose window is fully valid,
 *   S7  keeps best cost, non-adjacent second best and the neighbours of the best in registers --
 *       the cost volume is never written unless a debug buffer is given,
 *   and finally
 *   S8-S12 refines the plane with a parabola, converts to depth, merges with the half-resolution pass if one is
 *       given, applies the cost / ratio filters and the mask and
 *       stores the maps with coalesced row writes.
 * Planes that no ray of the tile can reach within range_max are skipped without sampling.
 *
 * Two block-wide barriers per plane: sample -> [A] -> horizontal sums -> [B] -> vertical sums, ZNCC, WTA.
 *
 * Numerics: everything is FP32, no fast-math.  Intensities are centred on a per-tile constant before any sum
 * (ZNCC is invariant to offsets) so that Sum(b^2) - Sum(b)^2/N does not cancel catastrophically.
 */
#ifndef FSW_SWEEP_CUH
#define FSW_SWEEP_CUH

#include <math_constants.h>

#include "fsw_internal.h"

namespace fsw {

constexpr int RUN = 8; /* outputs per work item of the horizontal pass */

/* tile geometry: TX x TY outputs, NT threads; thread t owns column t % TX and RPT consecutive rows */
template <int WIN, int TX_, int TY_, int NT_, int MINB_>
struct Geo {
    static constexpr int TX = TX_, TY = TY_, NT = NT_, MINB = MINB_;
    static constexpr int NW = NT / 32;
    static constexpr int NG = NT / TX;       /* row groups */
    static constexpr int RPT = TY / NG;      /* output rows per thread */
    static constexpr int NRUN = TX / RUN;
    static constexpr int HW = WIN / 2;
    static constexpr int EW = TX + 2 * HW;   /* tile + halo */
    static constexpr int EH = TY + 2 * HW;
    static constexpr int NE = EW * EH;       /* halo pixels = samples per plane and view */
    static constexpr int NS = (NE + NT - 1) / NT; /* samples per thread */
    static constexpr int NV = RUN + 2 * HW;        /* values one horizontal work item reads */
    static constexpr int NV4 = (NV + 3) / 4;       /* ... as 128-bit loads */
    /* row stride of the sample planes: covers the last run's 128-bit loads and is == 4 (mod 8) words so that
     * 128-bit accesses of consecutive rows are bank-conflict free */
    static constexpr int SBMIN = ((NRUN - 1) * RUN + NV4 * 4) > EW ? ((NRUN - 1) * RUN + NV4 * 4) : EW;
    static constexpr int SB = (SBMIN + 7) / 8 * 8 + 4 >= SBMIN + 8 ? (SBMIN + 7) / 8 * 8 - 4 : (SBMIN + 7) / 8 * 8 + 4;
    static constexpr int HS = TX + 4;              /* row stride of the row-sum planes, == 4 (mod 8) */
    static constexpr int PLANE = EH * SB;
    static constexpr int HPLANE = EH * HS;
    static constexpr int NHITEM = EH * NRUN;       /* work items of the horizontal pass (per view) */
    static_assert(NT % TX == 0 && TY % NG == 0 && TX % 32 == 0 && TX % RUN == 0, "tile / thread mapping");
    static_assert(SB >= SBMIN && SB % 8 == 4 && HS % 8 == 4, "bank-conflict-free strides");
    static constexpr size_t smem(int vc) {
        return sizeof(float4) * PLANE + sizeof(float) * ((size_t)PLANE * (1 + vc) + (size_t)4 * HPLANE * vc);
    }
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

/* S3-S4 for one halo pixel and one view: bilinear sample of the view at the plane-induced position minus `centre`,
 * or NaN if the pixel / plane / view combination is invalid ("NONE" of SURVEY 8(b)).
 * (rx,ry,rz) is the reference ray, s = (n.r)/d_k the inverse range along it (NaN if the ray misses the plane or the
 * intersection is beyond range_max: the NaN then fails the image-bounds test below, no separate flag is carried).
 * IDENT: the view's relative rotation is the identity.  FULLDIST: k2 / p1 / p2 may be non-zero.
 * CHECKDEN: cos(fov/2) + xi may be < 1e-3, so the projection denominator is tested on its own. */
template <bool IDENT, bool FULLDIST, bool CHECKDEN>
__device__ __forceinline__ float warp_sample(float rx, float ry, float rz, float s, const FswDevView& k,
                                             const float4* __restrict__ foot, float centre) {
    /* S2: X' ~ R r + s T */
    float X, Y, Z;
    if (IDENT) {
        X = fmaf(s, k.T[0], rx);
        Y = fmaf(s, k.T[1], ry);
        Z = fmaf(s, k.T[2], rz);
    } else {
        X = fmaf(k.R[0], rx, fmaf(k.R[1], ry, fmaf(k.R[2], rz, s * k.T[0])));
        Y = fmaf(k.R[3], rx, fmaf(k.R[4], ry, fmaf(k.R[5], rz, s * k.T[1])));
        Z = fmaf(k.R[6], rx, fmaf(k.R[7], ry, fmaf(k.R[8], rz, s * k.T[2])));
    }
    /* S3: unified projection: m = (X,Y) / (Z + xi rho) = (X,Y)/rho / (Z/rho + xi) */
    float rho2 = fmaf(X, X, fmaf(Y, Y, Z * Z));
    float irho = rsqrt_approx(rho2);
    float t = fmaf(Z, irho, k.cam.xi);       /* cos(theta) + xi; NaN for rho2 == 0 */
    bool ok = t >= k.cam.cos_fov_xi;         /* theta <= fov/2; false for NaN */
    if (CHECKDEN) ok = ok && (t > FSW_EPS_DEN);
    float g = irho * rcp_approx(t);
    float mx = X * g, my = Y * g;
    float r2 = fmaf(mx, mx, my * my);
    float xd, yd;
    if (!FULLDIST) {
        float rad = fmaf(k.cam.k1, r2, 1.f);
        xd = mx * rad;
        yd = my * rad;
    } else {
        float rad = fmaf(r2, fmaf(k.cam.k2, r2, k.cam.k1), 1.f);
        xd = fmaf(mx, rad, fmaf(2.f * k.cam.p1 * mx, my, k.cam.p2 * fmaf(2.f * mx, mx, r2)));
        yd = fmaf(my, rad, fmaf(k.cam.p1, fmaf(2.f * my, my, r2), 2.f * k.cam.p2 * mx * my));
    }
    float u = fmaf(k.cam.fx, xd, k.cam.cx);
    float v = fmaf(k.cam.fy, yd, k.cam.cy);
    /* floor without a float->int conversion: adding 1.5 * 2^23 with round-down leaves floor(u) in the low mantissa
     * bits (two's complement for negative values); anything with |u| >= 2^22, infinities and NaN fail the test */
    float tu = __fadd_rd(u, 12582912.f), tv = __fadd_rd(v, 12582912.f);
    int ix = __float_as_int(tu) - 0x4B400000, iy = __float_as_int(tv) - 0x4B400000;
    /* bilinear footprint inside the view image: 0 <= u < W-1, 0 <= v < H-1  <=>  0 <= floor(u) < W-1, ... */
    ok = ok && ((unsigned)ix < (unsigned)(k.cam.W - 1)) && ((unsigned)iy < (unsigned)(k.cam.H - 1));
    float b = CUDART_NAN_F;
    if (ok) {
        /* S4: one point fetch of the footprint + FP32 lerp (hardware texture filtering has 8-bit weights: too
         * coarse for the 1e-4 cost tolerance) */
        float au = u - (tu - 12582912.f);
        float av = v - (tv - 12582912.f);
        float4 f = __ldg(foot + (iy * k.cam.W + ix));
        float top = fmaf(au, f.y, f.x);
        float bot = fmaf(au, f.w, f.z);
        b = fmaf(av, bot - top, top) - centre;
    }
    return b;
}

/* 16 consecutive floats of a sample-plane row as 128-bit loads */
template <class G>
__device__ __forceinline__ void load_run(const float* __restrict__ src, float (&p)[G::NV4 * 4]) {
    const float4* p4 = reinterpret_cast<const float4*>(src);
#pragma unroll
    for (int i = 0; i < G::NV4; ++i) {
        float4 a = p4[i];
        p[4 * i] = a.x; p[4 * i + 1] = a.y; p[4 * i + 2] = a.z; p[4 * i + 3] = a.w;
    }
}

/* Horizontal pass of the separable box sums: one work item = RUN consecutive outputs of one halo row.
 * MODE 0: p = a', q = ray-valid flag      -> planes {sum a', sum a'^2, sum flag}
 * MODE 1: p = b', q = a' (all valid)      -> planes {sum b', sum b'^2, sum a'b'}
 * MODE 2: p = b' (NaN = invalid), q = a'  -> as MODE 1 with invalid samples as 0, plus plane 3 = sum valid */
template <class G, int WIN, int MODE>
__device__ __forceinline__ void hsum(float (&p)[G::NV4 * 4], const float (&q)[G::NV4 * 4], float* __restrict__ hs) {
    constexpr int NV = G::NV;
    float okf[G::NV4 * 4];
    if (MODE == 2) {
#pragma unroll
        for (int i = 0; i < NV; ++i) {
            bool ok = (p[i] == p[i]);
            okf[i] = ok ? 1.f : 0.f;
            p[i] = ok ? p[i] : 0.f;
        }
    }
    float pp[G::NV4 * 4], pq[G::NV4 * 4];
#pragma unroll
    for (int i = 0; i < NV; ++i) {
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
    float4* h0 = reinterpret_cast<float4*>(hs);
    float4* h1 = reinterpret_cast<float4*>(hs + G::HPLANE);
    float4* h2 = reinterpret_cast<float4*>(hs + 2 * G::HPLANE);
    h0[0] = make_float4(o0[0], o0[1], o0[2], o0[3]); h0[1] = make_float4(o0[4], o0[5], o0[6], o0[7]);
    h1[0] = make_float4(o1[0], o1[1], o1[2], o1[3]); h1[1] = make_float4(o1[4], o1[5], o1[6], o1[7]);
    h2[0] = make_float4(o2[0], o2[1], o2[2], o2[3]); h2[1] = make_float4(o2[4], o2[5], o2[6], o2[7]);
    if (MODE == 2) {
        float4* h3 = reinterpret_cast<float4*>(hs + 3 * G::HPLANE);
        h3[0] = make_float4(o3[0], o3[1], o3[2], o3[3]); h3[1] = make_float4(o3[4], o3[5], o3[6], o3[7]);
    }
}

/* Vertical pass: column x, output rows r0..r0+RPT-1; sums WIN consecutive row sums of one plane. */
template <class G, int WIN>
__device__ __forceinline__ void vpass(const float* __restrict__ h, int x, int r0, float (&out)[G::RPT]) {
    constexpr int RPT = G::RPT;
    float v[RPT + WIN - 1];
#pragma unroll
    for (int i = 0; i < RPT + WIN - 1; ++i) v[i] = h[(r0 + i) * G::HS + x];
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

/* streaming winner-take-all state of one output pixel (S7) */
struct Wta {
    float b1, s2, m0, m1, cm, cp, cprev;
    int k1, knext;
    __device__ __forceinline__ void init() {
        b1 = CUDART_INF_F; s2 = CUDART_INF_F; m0 = CUDART_INF_F; m1 = CUDART_INF_F;
        cm = CUDART_INF_F; cp = CUDART_INF_F; cprev = CUDART_INF_F;
        k1 = -1; knext = -1;
    }
    /* family start: planes of another family are never "adjacent" (reading Q12) */
    __device__ __forceinline__ void family_start() { m1 = m0; cprev = CUDART_INF_F; knext = -1; }
    __device__ __forceinline__ void update(float c, int k) {
        if (k == knext) cp = c;                 /* neighbour above the running best */
        else if (k > knext) s2 = fminf(s2, c);  /* eligible second best */
        if (c < b1) {                           /* strict: lowest index wins ties */
            s2 = m1;                            /* best of everything at least two planes back */
            cm = cprev;
            cp = CUDART_INF_F;
            b1 = c; k1 = k; knext = k + 1;
        }
        m1 = m0;
        m0 = fminf(m0, c);
        cprev = c;
    }
};

__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

/* VC = views processed together (1 or 2); args.n_views > VC runs the views in chunks of VC.
 * ONECHUNK: args.n_views <= VC, so that view indices are compile-time constants. */
template <int WIN, int VC, bool ONECHUNK, bool IDENT, bool FULLDIST, bool CHECKDEN, class G>
__global__ void __launch_bounds__(G::NT, G::MINB) sweep_kernel(const __grid_constant__ FswSweepArgs args) {
    constexpr int HW = G::HW, RPT = G::RPT, NT = G::NT, NS = G::NS, TX = G::TX, TY = G::TY;
    constexpr float NWIN = (float)(WIN * WIN);
    constexpr float INV_NWIN = 1.f / NWIN;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float4* rays = reinterpret_cast<float4*>(smem_raw);
    float* a_s = reinterpret_cast<float*>(rays + G::PLANE);
    float* b_s = a_s + G::PLANE;          /* [VC][PLANE] */
    float* hs = b_s + VC * G::PLANE;      /* [VC][4][HPLANE] */
    __shared__ float red_f[G::NW];
    __shared__ int red_i[G::NW];
    __shared__ unsigned s_flags[2][2];    /* [parity][0: AND of "all valid" bits, 1: OR of "any valid" bits] */
    __shared__ unsigned s_item;

    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int col = tid % TX, grp = tid / TX;
    const int W = args.ref.W, H = args.ref.H;
    const int n_items = args.n_tiles * args.n_sets;

    /* this thread's halo pixels: logical index -> offset in the padded sample planes */
    int soff[NS];
#pragma unroll
    for (int i = 0; i < NS; ++i) {
        int idx = tid + i * NT;
        int row = idx / G::EW;
        soff[i] = idx < G::NE ? row * G::SB + (idx - row * G::EW) : -1;
    }

    unsigned item = blockIdx.x;
    while (item < (unsigned)n_items) {
        const int set = (int)(item % (unsigned)args.n_sets);
        const int tile = args.tile_order[item / (unsigned)args.n_sets];
        const FswSetPtrs& S = args.n_sets > 1 ? args.sets[set] : args.set0;
        const int tyi = tile / args.n_tiles_x, txi = tile - tyi * args.n_tiles_x;
        const int x0t = txi * TX, y0t = tyi * TY;
        const int ox = x0t + col;            /* this thread's output column */
        const int oy0 = y0t + grp * RPT;     /* ... and first output row */

        Wta st[RPT];
#pragma unroll
        for (int i = 0; i < RPT; ++i) st[i].init();
        unsigned n_eval = 0;

        bool tile_live = (x0t < args.roi_x1) && (x0t + TX > args.roi_x0) && (y0t < args.roi_y1) && (y0t + TY > args.roi_y0);
        if (tile_live) {
            /* nearest point of the tile + halo to the principal point: beyond the image circle -> nothing to do */
            float nx = fmaxf(fmaxf((float)(x0t - HW) - args.ref.cx, args.ref.cx - (float)(x0t + TX - 1 + HW)), 0.f) / args.ref.fx;
            float ny = fmaxf(fmaxf((float)(y0t - HW) - args.ref.cy, args.ref.cy - (float)(y0t + TY - 1 + HW)), 0.f) / args.ref.fy;
            tile_live = fmaf(nx, nx, ny * ny) <= args.ref_rd2_max;
        }
        bool tile_active = false;
        unsigned active_mask = 0; /* bit i: output i of this thread can have a finite cost */
        float A1n[RPT], A2[RPT];  /* (sum a')/N and sum a'^2 - (sum a')^2/N of the output's window */
#pragma unroll
        for (int i = 0; i < RPT; ++i) { A1n[i] = 0.f; A2[i] = 0.f; }
        float centre = 0.f;

        if (tile_live) {
            /* ---- S1: rays and reference intensities of the tile + halo ------------------------------------ */
            float lsum = 0.f;
            int lcnt = 0;
#pragma unroll 1
            for (int i = 0; i < NS; ++i) {
                int idx = tid + i * NT;
                if (idx >= G::NE) break;
                int row = idx / G::EW, cx_ = idx - row * G::EW;
                int px = x0t - HW + cx_, py = y0t - HW + row;
                float4 ry = make_float4(0.f, 0.f, 0.f, 0.f); /* invalid rays are zero vectors */
                float a = 0.f;
                if (px >= 0 && px < W && py >= 0 && py < H) {
                    float rx, ryy, rz;
                    bool ok = back_project(args.ref, (float)px, (float)py, rx, ryy, rz);
                    if (ok) ry = make_float4(rx, ryy, rz, 1.f);
                    if (S.ref_dtype == FSW_U8)
                        a = (float)__ldg(reinterpret_cast<const uint8_t*>(S.ref_img) + (int64_t)py * S.ref_pitch_bytes + px);
                    else
                        a = __ldg(reinterpret_cast<const float*>(reinterpret_cast<const char*>(S.ref_img) + (int64_t)py * S.ref_pitch_bytes) + px);
                    if (ok) { lsum += a; lcnt += 1; } /* pixels outside the FOV never enter a valid window */
                }
                int o = row * G::SB + cx_;
                rays[o] = ry;
                a_s[o] = a;
                b_s[o] = ry.w;
            }
            /* centring constant of the tile: mean reference intensity (rounded to an integer for 8-bit images so
             * that a - centre stays exact) */
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                lsum += __shfl_xor_sync(0xffffffffu, lsum, o);
                lcnt += __shfl_xor_sync(0xffffffffu, lcnt, o);
            }
            if (lane == 0) { red_f[wid] = lsum; red_i[wid] = lcnt; }
            __syncthreads();
            float tsum = 0.f;
            int tcnt = 0;
#pragma unroll
            for (int i = 0; i < G::NW; ++i) { tsum += red_f[i]; tcnt += red_i[i]; }
            centre = tcnt > 0 ? tsum / (float)tcnt : 0.f;
            if (S.ref_dtype == FSW_U8) centre = rintf(centre);
#pragma unroll
            for (int i = 0; i < NS; ++i)
                if (soff[i] >= 0) a_s[soff[i]] -= centre;
            __syncthreads();
            /* window sums of the reference side, once per pixel */
            for (int it = tid; it < G::NHITEM; it += NT) {
                const int run = it / G::EH, row = it - run * G::EH;
                float p[G::NV4 * 4], q[G::NV4 * 4];
                load_run<G>(a_s + row * G::SB + run * RUN, p);
                load_run<G>(b_s + row * G::SB + run * RUN, q);
                hsum<G, WIN, 0>(p, q, hs + row * G::HS + run * RUN);
            }
            __syncthreads();
            {
                float sa[RPT], saa[RPT], sf[RPT];
                vpass<G, WIN>(hs, col, grp * RPT, sa);
                vpass<G, WIN>(hs + G::HPLANE, col, grp * RPT, saa);
                vpass<G, WIN>(hs + 2 * G::HPLANE, col, grp * RPT, sf);
#pragma unroll
                for (int i = 0; i < RPT; ++i) {
                    int oy = oy0 + i;
                    bool in_roi = ox >= args.roi_x0 && ox < args.roi_x1 && oy >= args.roi_y0 && oy < args.roi_y1;
                    bool act = in_roi && (sf[i] == NWIN); /* every window pixel inside the image and the FOV */
                    if (act) active_mask |= 1u << i;
                    A1n[i] = sa[i] * INV_NWIN;
                    A2[i] = fmaf(-A1n[i], sa[i], saa[i]);
                }
            }
            if (tid == 0) { s_flags[0][0] = ~0u; s_flags[0][1] = 0u; s_flags[1][0] = ~0u; s_flags[1][1] = 0u; }
            tile_active = __syncthreads_or(active_mask != 0) != 0;
        }

        if (tile_active) {
            const float inv_views = 1.f / (float)args.n_views;
            unsigned parity = 0;
#pragma unroll 1
            for (int f = 0; f < args.n_fams; ++f) {
                const FswDevFamily& F = args.fam[f];
                const float fnx = F.n[0], fny = F.n[1], fnz = F.n[2];
#pragma unroll
                for (int i = 0; i < RPT; ++i) st[i].family_start();
                /* incidence q = n.r of every halo ray with this family, NaN where the ray does not face the planes
                 * (or is outside the camera); q_max decides which planes can be reached within range_max */
                float qmax = 0.f;
#pragma unroll
                for (int i = 0; i < NS; ++i) {
                    if (soff[i] < 0) continue;
                    float4 ry = rays[soff[i]];
                    float q = fmaf(fnx, ry.x, fmaf(fny, ry.y, fnz * ry.z));
                    bool faces = q > FSW_EPS_Q; /* an invalid reference ray is the zero vector: q = 0 */
                    rays[soff[i]].w = faces ? q : CUDART_NAN_F;
                    if (faces) qmax = fmaxf(qmax, q);
                }
                qmax = warp_max(qmax);
                __syncthreads(); /* previous users of red_f are done */
                if (lane == 0) red_f[wid] = qmax;
                __syncthreads();
                qmax = 0.f;
#pragma unroll
                for (int i = 0; i < G::NW; ++i) qmax = fmaxf(qmax, red_f[i]);

#pragma unroll 1
                for (int j = 0; j < F.count; ++j) {
                    const int k = F.first + j;
                    const float inv_d = args.inv_d[k];
                    float acc[RPT];
                    int cnt[RPT];
#pragma unroll
                    for (int i = 0; i < RPT; ++i) { acc[i] = 0.f; cnt[i] = 0; }
                    /* S2: the plane is out of reach for the whole tile if even the best-facing ray is beyond range */
                    const bool plane_on = qmax * inv_d >= args.inv_range_max;
                    if (plane_on) {
#pragma unroll 1
                        for (int v0 = 0; v0 < (ONECHUNK ? 1 : args.n_views); v0 += VC) {
                            /* ---- S2-S4: sample the plane-warped views at every halo pixel ------------------- */
                            bool all_ok[VC], any_ok[VC];
#pragma unroll
                            for (int v = 0; v < VC; ++v) { all_ok[v] = true; any_ok[v] = false; }
#pragma unroll
                            for (int i = 0; i < NS; ++i) {
                                if (soff[i] < 0) continue;
                                const float4 ry = rays[soff[i]];
                                float s = ry.w * inv_d;
                                s = (s >= args.inv_range_max) ? s : CUDART_NAN_F;
#pragma unroll
                                for (int v = 0; v < VC; ++v) {
                                    if (!ONECHUNK && v0 + v >= args.n_views) break;
                                    const int vi = ONECHUNK ? v : v0 + v;
                                    float b = warp_sample<IDENT, FULLDIST, CHECKDEN>(ry.x, ry.y, ry.z, s, args.views[vi], S.foot[vi], centre);
                                    b_s[v * G::PLANE + soff[i]] = b;
                                    bool okb = (b == b);
                                    all_ok[v] = all_ok[v] && okb;
                                    any_ok[v] = any_ok[v] || okb;
                                }
                            }
                            unsigned fl_all = 0, fl_any = 0;
#pragma unroll
                            for (int v = 0; v < VC; ++v) {
                                if (__all_sync(0xffffffffu, all_ok[v])) fl_all |= 1u << v;
                                if (__any_sync(0xffffffffu, any_ok[v])) fl_any |= 1u << v;
                            }
                            if (lane == 0) {
                                atomicAnd(&s_flags[parity][0], fl_all);
                                atomicOr(&s_flags[parity][1], fl_any);
                            }
                            __syncthreads(); /* [A] */
                            const unsigned f_all = s_flags[parity][0], f_any = s_flags[parity][1];
                            if (tid == 0) { s_flags[parity ^ 1][0] = ~0u; s_flags[parity ^ 1][1] = 0u; }
                            parity ^= 1;
                            if (f_any == 0) continue; /* no view sees anything of the tile through this plane */
                            /* ---- S5: separable box sums ----------------------------------------------------- */
                            for (int it = tid; it < G::NHITEM; it += NT) {
                                const int run = it / G::EH, row = it - run * G::EH;
                                float q[G::NV4 * 4];
                                load_run<G>(a_s + row * G::SB + run * RUN, q);
#pragma unroll
                                for (int v = 0; v < VC; ++v) {
                                    if (!((f_any >> v) & 1u)) continue;
                                    float p[G::NV4 * 4];
                                    load_run<G>(b_s + v * G::PLANE + row * G::SB + run * RUN, p);
                                    float* dst = hs + v * 4 * G::HPLANE + row * G::HS + run * RUN;
                                    if ((f_all >> v) & 1u) hsum<G, WIN, 1>(p, q, dst);
                                    else hsum<G, WIN, 2>(p, q, dst);
                                }
                            }
                            __syncthreads(); /* [B] */
                            /* ---- ZNCC ----------------------------------------------------------------------- */
#pragma unroll
                            for (int v = 0; v < VC; ++v) {
                                if (!((f_any >> v) & 1u)) continue;
                                const bool mixed = !((f_all >> v) & 1u);
                                const float* hv = hs + v * 4 * G::HPLANE;
                                float sb[RPT], sbb[RPT], sab[RPT], sv[RPT];
                                vpass<G, WIN>(hv, col, grp * RPT, sb);
                                vpass<G, WIN>(hv + G::HPLANE, col, grp * RPT, sbb);
                                vpass<G, WIN>(hv + 2 * G::HPLANE, col, grp * RPT, sab);
                                if (mixed) vpass<G, WIN>(hv + 3 * G::HPLANE, col, grp * RPT, sv);
#pragma unroll
                                for (int i = 0; i < RPT; ++i) {
                                    bool okv = (active_mask >> i) & 1u;
                                    if (mixed) okv = okv && (sv[i] == NWIN);
                                    float cov = fmaf(-A1n[i], sb[i], sab[i]);
                                    float vb = fmaf(-sb[i] * INV_NWIN, sb[i], sbb[i]);
                                    float prod = fmaxf(A2[i] * vb, args.floor2);
                                    float z = cov * rsqrt_approx(prod);
                                    float cst = __saturatef(fmaf(-0.5f, z, 0.5f));
                                    if (okv) { acc[i] += cst; cnt[i] += 1; }
                                }
                            }
                        }
                    }
                    /* ---- S6 + S7: view mean, streaming winner-take-all ------------------------------------- */
#pragma unroll
                    for (int i = 0; i < RPT; ++i) {
                        float c = CUDART_INF_F;
                        if (cnt[i] == args.n_views) c = acc[i] * inv_views;
                        else if (cnt[i] > 0) c = acc[i] / (float)cnt[i];
                        n_eval += cnt[i];
                        if (S.debug_cost != nullptr) {
                            int oy = oy0 + i;
                            if (ox < W && oy < H) S.debug_cost[((int64_t)k * H + oy) * W + ox] = c;
                        }
                        st[i].update(c, k);
                    }
                }
            }
        }
        if (S.debug_cost != nullptr && !tile_active) {
            for (int k = 0; k < args.n_planes; ++k)
#pragma unroll
                for (int i = 0; i < RPT; ++i) {
                    int oy = oy0 + i;
                    if (ox < W && oy < H) S.debug_cost[((int64_t)k * H + oy) * W + ox] = CUDART_INF_F;
                }
        }

        /* ---- S8-S12: refinement, depth, merge, filters, mask, stores --------------------------------------- */
        unsigned n_raw = 0, n_ok = 0;
#pragma unroll
        for (int i = 0; i < RPT; ++i) {
            const int oy = oy0 + i;
            if (ox >= W || oy >= H) continue;
            bool raw_valid = st[i].k1 >= 0;
            float depth = 0.f, c1 = CUDART_INF_F, c2 = CUDART_INF_F;
            int kidx = -1;
            if (raw_valid) {
                int f = 0;
                for (int g = 1; g < args.n_fams; ++g)
                    if (st[i].k1 >= args.fam[g].first) f = g;
                const FswDevFamily& F = args.fam[f];
                float dl = 0.f;
                if (args.subpixel && st[i].cm < CUDART_INF_F && st[i].cp < CUDART_INF_F) {
                    float den = st[i].cm - 2.f * st[i].b1 + st[i].cp;
                    if (den > 1e-12f) dl = fminf(fmaxf(0.5f * (st[i].cm - st[i].cp) / den, -0.5f), 0.5f);
                }
                float s = fmaf((float)(st[i].k1 - F.first) + dl, F.ds, F.s0);
                float d = F.spacing == FSW_INVERSE ? 1.f / s : s;
                float4 ry = rays[(grp * RPT + i + HW) * G::SB + col + HW];
                float q = fmaf(F.n[0], ry.x, fmaf(F.n[1], ry.y, F.n[2] * ry.z));
                float range = d / q;
                depth = args.depth_kind == FSW_DEPTH_Z ? range * ry.z : range;
                c1 = st[i].b1;
                c2 = st[i].s2 < CUDART_INF_F ? st[i].s2 : 1.f;
                kidx = st[i].k1 | args.index_flag;
            } else if (S.lo_k != nullptr) {
                /* S10(c)-(e): nearest-neighbour upsample of the half-resolution pass */
                int xl = ox >> 1, yl = oy >> 1;
                if (xl < args.lo_W && yl < args.lo_H) {
                    int64_t j = (int64_t)yl * args.lo_W + xl;
                    int kl = S.lo_k[j];
                    if (kl >= 0) {
                        raw_valid = true;
                        depth = S.lo_depth[j]; c1 = S.lo_c1[j]; c2 = S.lo_c2[j]; kidx = kl;
                    }
                }
            }
            int reason = FSW_REASON_OK;
            if (!raw_valid) reason = FSW_REASON_NO_PLANE;
            else {
                float alpha = oy < args.horizon_row ? args.alpha_upper : args.alpha_lower;
                if ((args.filters & FSW_FILTER_COST) && c1 > alpha) reason = FSW_REASON_COST_FILTER;
                else if ((args.filters & FSW_FILTER_RATIO) && c2 < args.beta * fmaxf(c1, 1e-6f)) reason = FSW_REASON_RATIO_FILTER;
                else if (S.mask != nullptr && S.mask[(int64_t)oy * S.mask_pitch + ox]) reason = FSW_REASON_MASKED;
            }
            if (reason != FSW_REASON_OK) depth = 0.f;
            n_raw += raw_valid ? 1u : 0u;
            n_ok += reason == FSW_REASON_OK ? 1u : 0u;
            *reinterpret_cast<float*>(reinterpret_cast<char*>(S.out_depth) + (int64_t)oy * S.out_depth_pitch + 4 * (int64_t)ox) = depth;
            if (S.out_c1) *reinterpret_cast<float*>(reinterpret_cast<char*>(S.out_c1) + (int64_t)oy * S.out_c1_pitch + 4 * (int64_t)ox) = c1;
            if (S.out_c2) *reinterpret_cast<float*>(reinterpret_cast<char*>(S.out_c2) + (int64_t)oy * S.out_c2_pitch + 4 * (int64_t)ox) = c2;
            if (S.out_k) *reinterpret_cast<int16_t*>(reinterpret_cast<char*>(S.out_k) + (int64_t)oy * S.out_k_pitch + 2 * (int64_t)ox) = (int16_t)kidx;
            if (S.out_reason) S.out_reason[(int64_t)oy * S.out_reason_pitch + ox] = (uint8_t)reason;
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

        /* ---- next item ----------------------------------------------------------------------------------------- */
        __syncthreads(); /* everyone is done with this tile's shared memory (and with s_item) */
        if (tid == 0) s_item = atomicAdd(args.queue, 1u) + gridDim.x;
        __syncthreads();
        item = s_item;
    }
}

/* The tile shapes: A = 64x32 outputs, 512 threads, one CTA per SM (windows up to 9);
 *                  B = 32x32 outputs, 256 threads (larger windows: the halo planes of A would not fit). */
template <int WIN> struct GeoFor { using type = Geo<WIN, 64, 32, 512, 1>; };
template <> struct GeoFor<11> { using type = Geo<11, 32, 32, 256, 1>; };
template <> struct GeoFor<13> { using type = Geo<13, 32, 32, 256, 1>; };
template <> struct GeoFor<15> { using type = Geo<15, 32, 32, 256, 1>; };

/* Kernel variants: 0 = generic (any rotation, full distortion polynomial, denominator test),
 *                  1 = identity rotations, k1-only (or no) distortion, cos(fov/2) + xi >= 1e-3. */
template <int WIN, int VC, bool ONE>
struct SweepInst {
    using G = typename GeoFor<WIN>::type;
    static cudaError_t launch(const FswSweepArgs& args, int variant, int grid, cudaStream_t stream) {
        const size_t smem = G::smem(VC);
        if (variant == 1) sweep_kernel<WIN, VC, ONE, true, false, false, G><<<grid, G::NT, smem, stream>>>(args);
        else sweep_kernel<WIN, VC, ONE, false, true, true, G><<<grid, G::NT, smem, stream>>>(args);
        return cudaGetLastError();
    }
    static cudaError_t prepare() {
        const int smem = (int)G::smem(VC);
        cudaError_t e = cudaFuncSetAttribute(sweep_kernel<WIN, VC, ONE, true, false, false, G>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return e;
        return cudaFuncSetAttribute(sweep_kernel<WIN, VC, ONE, false, true, true, G>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    }
};

/* n_views == 1 -> VC = 1; n_views == 2 -> VC = 2, one chunk; more views -> chunks of 2 */
template <int WIN>
cudaError_t launch_sweep_win(const FswSweepArgs& args, int variant, int grid, cudaStream_t stream) {
    if (args.n_views == 1) return SweepInst<WIN, 1, true>::launch(args, variant, grid, stream);
    if (args.n_views == 2) return SweepInst<WIN, 2, true>::launch(args, variant, grid, stream);
    return SweepInst<WIN, 2, false>::launch(args, variant, grid, stream);
}

template <int WIN>
cudaError_t prepare_sweep_win() {
    cudaError_t e = SweepInst<WIN, 1, true>::prepare();
    if (e != cudaSuccess) return e;
    e = SweepInst<WIN, 2, true>::prepare();
    if (e != cudaSuccess) return e;
    return SweepInst<WIN, 2, false>::prepare();
}

template <int WIN>
FswSweepGeometry geometry_win(int n_views) {
    using G = typename GeoFor<WIN>::type;
    FswSweepGeometry g;
    g.tile_w = G::TX; g.tile_h = G::TY; g.threads = G::NT; g.ctas_per_sm = G::MINB;
    g.smem_bytes = G::smem(n_views == 1 ? 1 : 2);
    return g;
}

}  // namespace fsw
#endif
