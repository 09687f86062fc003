/*
 * fsw_sweep.cuh -- the fused fisheye plane-sweep kernel (sm_100a), steps S1..S12 of SURVEY.md section 8(a).
 *
 * Persistent CTAs (one per SM, 16 warps) claim (frame set, tile) items from a queue, heaviest tiles first.  For one
 * TX x TY tile of reference pixels a CTA
 *   S1  back-projects the tile plus a halo of w/2 pixels through the unified model (Eq. 1) into
 *       shared memory (no ray LUT ever touches HBM),
 *   and then, for every sweep plane k and every matching view,
 *   S2-S4 maps every halo pixel through the plane into the view (ray-homography form X' ~ R r + (n.r / d_k) T),
 *       projects it with the view's fisheye model and samples the view bilinearly from its footprint image (one
 *       64-bit load for 8-bit views, one 128-bit load for float views),
 *   S5  forms the windowed sums of b, b^2, ab with separable sliding box sums and scores cost = (1 - ZNCC)/2
 *       (PAPER.md:76),
 *   S6  averages the cost over the views whose window is fully valid,
 *   S7  keeps best cost, non-adjacent second best and the neighbours of the best in registers --
 *       the cost volume is never written unless a debug buffer is given,
 *   and finally
 *   S8-S12 refines the plane with a parabola, converts to depth, merges with the half-resolution pass if one is
 *       given, applies the cost / ratio filters and the mask and
 *       stores the maps with coalesced row writes.
 *
 * Work split.  Warp w owns R consecutive halo rows of the tile for the whole tile: it samples them (S2-S4) into its
 * private rows of the sample plane and immediately runs the horizontal box sums over them (a __syncwarp, no block
 * barrier, in between); the reference-side operands a' of its horizontal work item stay in registers for the whole
 * sweep.  After one block barrier every thread does the vertical sums, the ZNCC and the winner-take-all update of its
 * own RPT output pixels; the second barrier of a pass sits right after the last loads of the vertical pass, so its
 * arithmetic overlaps the next pass of faster warps.  For windows up to 9 x 9 a pass covers TWO views of the plane
 * (Geo::FUSE_OK): both are sampled from one load of the ray (shared range test and inverse range), both get their own
 * sample plane and row-sum planes, and the pair shares the two block barriers, the pass flags and the loop control.
 * Row groups that no ray can reach (outside the image circle, above the horizon for ground-parallel planes, beyond
 * range_max) are skipped per warp, whole planes per tile.
 *
 * Numerics: everything is FP32, no fast-math.  Intensities are centred on a per-tile constant before any sum
 * (ZNCC is invariant to offsets) so that Sum(b^2) - Sum(b)^2/N does not cancel catastrophically.
 */
#ifndef FSW_SWEEP_CUH
#define FSW_SWEEP_CUH

#include <math_constants.h>

#include <type_traits>

#include "fsw_internal.h"

namespace fsw {

constexpr int RUN = 8; /* outputs per work item of the horizontal pass */

/* tile geometry: 64 x TY outputs, 512 threads; thread t owns column t % 64 and RPT consecutive rows; warp w owns the
 * R halo rows w*R .. w*R+R-1 in the sample / horizontal phase.  The sample planes have a row stride of SB = EW rounded
 * up to a multiple of 4 and no other padding, so that lane l's i-th halo pixel of the warp's rows sits at the fixed
 * offset l + 32 i from the warp's first row (the up to 3 extra columns of a row are sampled like halo pixels). */
template <int WIN>
struct Geo {
    static constexpr int TX = 64, NT = 512, MINB = 1;
    static constexpr int NW = NT / 32;
    static constexpr int NG = NT / TX;                 /* row groups of the vertical pass */
    static constexpr int R = WIN <= 9 ? 3 : 4;         /* halo rows per warp */
    static constexpr int RPT = WIN <= 9 ? 5 : 6;       /* output rows per thread */
    static constexpr int TY = NG * RPT;
    static constexpr int NRUN = TX / RUN;
    static constexpr int HW = WIN / 2;
    static constexpr int EW = TX + 2 * HW;             /* tile + halo */
    static constexpr int EH = TY + 2 * HW;
    static constexpr int EHA = R * NW;                 /* allocated halo rows */
    static constexpr int NV = RUN + 2 * HW;            /* values one horizontal work item reads */
    static constexpr int NV4 = (NV + 3) / 4;           /* ... as 128-bit loads */
    static constexpr int SBMIN = ((NRUN - 1) * RUN + NV4 * 4) > EW ? ((NRUN - 1) * RUN + NV4 * 4) : EW;
    static constexpr int SB = (SBMIN + 3) / 4 * 4;     /* row stride of the sample planes */
    static constexpr int NS = (R * SB + 31) / 32;      /* sample slots per lane */
    static constexpr int NSFULL = (R * SB) / 32;       /* slots in which every lane has a pixel */
    static constexpr int HS = TX + 4;                  /* row stride of the row-sum planes, == 4 (mod 8) */
    static constexpr int PLANE = EHA * SB;
    static constexpr int HPLANE = EHA * HS;
    static constexpr bool A_IN_REGS = WIN <= 9;        /* keep the a' operands of the horizontal item in registers */
    /* two views per pass: the plane of a' is free after S1 (A_IN_REGS) and holds the samples of the first view; a
     * second set of row-sum planes brings the block to 203 KB of the 227 KB an sm_100 block may use (the footprint
     * gathers then have 28 KB of L1 instead of 88 KB: measured + 4 % on the unfused kernel, against - 12 % from fusing) */
    static constexpr bool FUSE_OK = A_IN_REGS;
    /* the parabola neighbours of the running best in shared memory instead of registers (Wta::update): where the
     * block has the 20 KB to spare */
    static constexpr bool NBR_SMEM = WIN <= 9;
    static_assert(EH <= EHA && TX % 32 == 0 && TX % RUN == 0 && NRUN == 8, "tile / thread mapping");
    static_assert(SB >= SBMIN && SB % 4 == 0 && HS % 8 == 4, "aligned strides");
    static_assert(R * NRUN <= 32, "one horizontal work item per lane");
    static constexpr size_t smem(bool fuse) {
        return sizeof(float4) * PLANE + sizeof(float) * ((size_t)2 * PLANE + (size_t)(fuse ? 8 : 4) * HPLANE) +
               (NBR_SMEM ? 2 : 1) * sizeof(float2) * TX * TY;
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
        /* radial + tangential: fixed-point iteration m <- (m_d - tangential(m)) / radial(m), which contracts wherever
         * the distortion is invertible (checked at rig creation); the residual decides whether it arrived */
#pragma unroll 1
        for (int it = 0; it < 40; ++it) {
            const float r2 = fmaf(x, x, y * y);
            const float radial = fmaf(r2, fmaf(c.k2, r2, c.k1), 1.f);
            const float tx = fmaf(2.f * c.p1 * x, y, c.p2 * fmaf(2.f * x, x, r2));
            const float ty = fmaf(c.p1, fmaf(2.f * y, y, r2), 2.f * c.p2 * x * y);
            if (!(radial > 1e-3f)) return false;
            x = (xd - tx) / radial;
            y = (yd - ty) / radial;
        }
        {
            const float r2 = fmaf(x, x, y * y);
            const float radial = fmaf(r2, fmaf(c.k2, r2, c.k1), 1.f);
            const float ex = fmaf(x, radial, fmaf(2.f * c.p1 * x, y, c.p2 * fmaf(2.f * x, x, r2))) - xd;
            const float ey = fmaf(y, radial, fmaf(c.p1, fmaf(2.f * y, y, r2), 2.f * c.p2 * x * y)) - yd;
            if (!(fabsf(ex) + fabsf(ey) <= 1e-5f * (1.f + fabsf(xd) + fabsf(yd)))) return false; /* not converged / NaN */
        }
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

/* S2-S3 for one halo pixel and one view: where the plane-induced position falls in the view (footprint index and
 * bilinear weights); `ok` is false if the pixel / plane / view combination is invalid ("NONE" of SURVEY 8(b)).
 * (rx,ry,rz) is the reference ray, s = (n.r)/d_k the inverse range along it (NaN if the ray misses the plane or the
 * intersection is beyond range_max: the NaN then fails the field-of-view test below, no separate flag is carried).
 * IDENT: the view's relative rotation is the identity.  FULLDIST: k2 / p1 / p2 may be non-zero.
 * CHECKDEN: cos(fov/2) + xi may be < 1e-3, so the projection denominator is tested on its own.
 * INSIDE: the image circle of every view lies inside its raster with half a pixel to spare (decided on the host,
 *   fsw_api.cu: view_fov_inside_image), so a sample inside the field of view needs no test against the image borders.
 * F16: the footprint images hold four bfloat16 per pixel (8-bit views) instead of four floats. */
struct SampleAddr {
    float au, av;  /* bilinear weights */
    unsigned idx;  /* footprint index iy * W + ix, 0 for an invalid sample */
    bool ok;
};
template <bool IDENT, bool FULLDIST, bool CHECKDEN, bool INSIDE>
__device__ __forceinline__ SampleAddr sample_addr(float rx, float ry, float rz, float s, const FswDevView& k) {
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
    unsigned ix = (unsigned)__float_as_int(tu) - 0x4B400000u, iy = (unsigned)__float_as_int(tv) - 0x4B400000u;
    /* bilinear footprint inside the view image: 0 <= u < W-1, 0 <= v < H-1  <=>  0 <= floor(u) < W-1, ... */
    if (!INSIDE) ok = ok && (ix < (unsigned)k.cam.Wm1) && (iy < (unsigned)k.cam.Hm1);
    SampleAddr a;
    a.au = u - (tu - 12582912.f);
    a.av = v - (tv - 12582912.f);
    a.idx = ok ? iy * (unsigned)k.cam.W + ix : 0u; /* invalid samples fetch footprint 0 instead of branching */
    a.ok = ok;
    return a;
}

/* S4: one point fetch of the footprint + FP32 lerp (hardware texture filtering has 8-bit weights: too coarse for the
 * 1e-4 cost tolerance).  Raw footprint: 8 bytes = four bfloat16 (F16, exact for integers up to 256) or four floats. */
template <bool F16> struct FootRaw { float4 v; };
template <> struct FootRaw<true> { uint2 v; };
template <bool F16>
__device__ __forceinline__ FootRaw<F16> foot_fetch(const void* __restrict__ foot, unsigned idx) {
    FootRaw<F16> r;
    /* the index was already forced to 0 for an invalid sample as a 32-bit value; one wide multiply-add forms the
     * address (written as PTX so that the select is not redone on the 64-bit offset) */
    const char* ptr;
    if constexpr (F16) {
        asm("mad.wide.u32 %0, %1, 8, %2;" : "=l"(ptr) : "r"(idx), "l"(foot));
        r.v = __ldg(reinterpret_cast<const uint2*>(ptr));
    } else {
        asm("mad.wide.u32 %0, %1, 16, %2;" : "=l"(ptr) : "r"(idx), "l"(foot));
        r.v = __ldg(reinterpret_cast<const float4*>(ptr));
    }
    return r;
}
template <bool F16>
__device__ __forceinline__ float foot_lerp(const FootRaw<F16>& r, float au, float av, float centre) {
    float4 f;
    if constexpr (F16) {
        f.x = __uint_as_float(r.v.x << 16); f.y = __uint_as_float(r.v.x & 0xffff0000u);
        f.z = __uint_as_float(r.v.y << 16); f.w = __uint_as_float(r.v.y & 0xffff0000u);
    } else {
        f = r.v;
    }
    float top = fmaf(au, f.y, f.x);
    float bot = fmaf(au, f.w, f.z);
    return fmaf(av, bot - top, top) - centre; /* NaN if au is (an invalid sample) */
}

/* NV4 * 4 consecutive floats of a sample-plane row as 128-bit loads */
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
 * MODE 2: p = b' (NaN = invalid), q = a'  -> as MODE 1 with invalid samples as 0, plus plane 3 = sum valid;
 *         returns whether any of the item's samples is valid
 * The products enter and leave the sliding sums through FMAs (no product array is kept). */
template <class G, int WIN, int MODE>
__device__ __forceinline__ bool hsum(float (&p)[G::NV4 * 4], const float (&q)[G::NV4 * 4], float* __restrict__ hs) {
    constexpr int NV = G::NV;
    float okf[MODE == 2 ? G::NV4 * 4 : 1];
    bool any = true;
    if (MODE == 2) {
        any = false;
#pragma unroll
        for (int i = 0; i < NV; ++i) {
            bool ok = (p[i] == p[i]);
            any = any || ok;
            okf[i] = ok ? 1.f : 0.f;
            p[i] = ok ? p[i] : 0.f;
        }
    }
    float s0 = 0.f, s1 = 0.f, s2 = 0.f, s3 = 0.f;
#pragma unroll
    for (int i = 0; i < WIN; ++i) {
        s0 += p[i];
        s1 = fmaf(p[i], p[i], s1);
        s2 = (MODE == 0) ? s2 + q[i] : fmaf(p[i], q[i], s2);
        if (MODE == 2) s3 += okf[i];
    }
    float4* h0 = reinterpret_cast<float4*>(hs);
    float4* h1 = reinterpret_cast<float4*>(hs + G::HPLANE);
    float4* h2 = reinterpret_cast<float4*>(hs + 2 * G::HPLANE);
    float4* h3 = reinterpret_cast<float4*>(hs + 3 * G::HPLANE);
    float o0[4], o1[4], o2[4], o3[4];
#pragma unroll
    for (int j = 0; j < RUN; ++j) {
        if (j > 0) {
            const int in = j + WIN - 1, out = j - 1;
            s0 += p[in] - p[out];
            s1 = fmaf(-p[out], p[out], fmaf(p[in], p[in], s1));
            s2 = (MODE == 0) ? s2 + (q[in] - q[out]) : fmaf(-p[out], q[out], fmaf(p[in], q[in], s2));
            if (MODE == 2) s3 += okf[in] - okf[out];
        }
        o0[j & 3] = s0; o1[j & 3] = s1; o2[j & 3] = s2; o3[j & 3] = s3;
        if ((j & 3) == 3) {
            h0[j >> 2] = make_float4(o0[0], o0[1], o0[2], o0[3]);
            h1[j >> 2] = make_float4(o1[0], o1[1], o1[2], o1[3]);
            h2[j >> 2] = make_float4(o2[0], o2[1], o2[2], o2[3]);
            if (MODE == 2) h3[j >> 2] = make_float4(o3[0], o3[1], o3[2], o3[3]);
        }
    }
    return any;
}

/* the row sums of one work item cleared (rows that no ray reaches: the sliding vertical sums of the columns must not
 * carry values of an earlier pass, or a cost would depend in its last bit on the order the planes are visited in) */
template <class G>
__device__ __forceinline__ void fill_zero(float* __restrict__ hs) {
    const float4 z = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
    for (int pl = 0; pl < 4; ++pl) {
        float4* h = reinterpret_cast<float4*>(hs + pl * G::HPLANE);
        h[0] = z;
        h[1] = z;
    }
}

/* RUN entries of plane 3 (valid counts of the horizontal windows) of one work item set to c */
template <class G>
__device__ __forceinline__ void fill_count(float* __restrict__ hs, float c) {
    float4* h3 = reinterpret_cast<float4*>(hs + 3 * G::HPLANE);
    h3[0] = make_float4(c, c, c, c);
    h3[1] = make_float4(c, c, c, c);
}

/* Vertical pass: h points at the first of the RPT + WIN - 1 row sums of this thread's column in one plane; sliding
 * sums over WIN consecutive rows */
template <class G, int WIN>
__device__ __forceinline__ void vpass(const float* __restrict__ h, float (&out)[G::RPT]) {
    constexpr int RPT = G::RPT;
    float v[RPT + WIN - 1];
#pragma unroll
    for (int i = 0; i < RPT + WIN - 1; ++i) v[i] = h[i * G::HS];
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

/* streaming winner-take-all state of one output pixel (S7).  b1 = lowest cost so far (lowest index wins ties),
 * m2 = lowest cost of the planes at least two back (eligible as second best when the current plane becomes the
 * best), s2 = second best of the current best, cm / cp = costs of the planes below / above the best, knext = index
 * of the plane above the best while it is still to come in the same family (kept in a register by the unsplit
 * kernel only; the split kernel, shorter of registers, derives it from k1). */
struct Wta {
    float b1, m2, s2, cm, cp, cprev;
    int k1, knext;
    __device__ __forceinline__ void init() {
        b1 = CUDART_INF_F; m2 = CUDART_INF_F; s2 = CUDART_INF_F;
        cm = CUDART_INF_F; cp = CUDART_INF_F; cprev = CUDART_INF_F;
        k1 = -1; knext = -1;
    }
    /* family start: planes of another family are never "adjacent" (reading Q12) */
    __device__ __forceinline__ void family_start() { m2 = b1; cprev = CUDART_INF_F; knext = -1; }
    /* Planes are visited in ascending index order (dir = +1), or -- in the second half of a split tile -- in
     * descending order (dir = -1, desc): then an equal cost wins as well (the later plane has the lower index), and
     * cm / cp hold the neighbour visited before / after the best, i.e. above / below it (swap_neighbours()). */
    /* During the sweep the two neighbours of the best live in shared memory (*nbr = (cm, cp), written by this thread
     * only): they change when a new best arrives or the plane after it is scored, which is rare, and ten registers
     * fewer let the sample phase keep more footprint fetches in flight. */
    /* halo (split tiles only, the iteration after a half's own planes): the plane across the cut is scored only as the
     * parabola neighbour of a winner next to the cut; with an infinite cost the rest of the state stays as it is, m2
     * (the lowest cost except the plane next to the cut) included -- selects instead of a branch around the update */
    template <bool KNEXT>
    __device__ __forceinline__ void update(float c_real, int k, int dir, bool desc, bool fam_first, float2* __restrict__ nbr,
                                           bool halo = false) {
        const float c = halo ? CUDART_INF_F : c_real;
        /* neighbour of the running best on the far side (same family): not eligible as second best */
        const bool isn = KNEXT ? (k == knext) : (!fam_first && (k == k1 + dir));
        const bool nb = desc ? ((c <= b1) && (c < CUDART_INF_F)) : (c < b1); /* lowest index wins ties */
        if (isn) nbr->y = c_real;
        const float t = isn ? s2 : fminf(s2, c);
        s2 = nb ? m2 : t;
        if (nb) *nbr = make_float2(cprev, CUDART_INF_F);
        k1 = nb ? k : k1;
        if (KNEXT) knext = nb ? k + dir : knext;
        m2 = halo ? m2 : b1;
        b1 = fminf(b1, c);
        cprev = c;
    }
    __device__ __forceinline__ void swap_neighbours() { const float t = cm; cm = cp; cp = t; }
};

__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

/* horizontal work item of lane `lane`: local row (0..R-1, or -1 for an idle lane) and run (0..7).  A quarter-warp
 * covers rows {r, r+1} x four runs: its 128-bit stores into the row-sum planes (row stride == 4 mod 8 words) hit
 * eight distinct 16-byte bank groups. */
template <class G>
__device__ __forceinline__ void h_item(int lane, int& row, int& run) {
    const int half = lane >> 4, l = lane & 15;
    row = 2 * half + ((l >> 2) & 1);
    run = (l & 3) + ((l >> 3) << 2);
    if (G::R == 3 && half == 1) { /* third row: eight runs in lanes 16..23, lanes 24..31 idle */
        row = l < 8 ? 2 : -1;
        run = l & 7;
    }
}

/* S2-S4 for the R halo rows of one warp, one plane and NJ views (1 or 2): samples into the warp's rows of b0 (first
 * view) and b1 (second view), NaN = invalid.  The ray, its inverse range s = (n.r)/d_k and the range test are shared by
 * the views.  Returns (warp-uniform) bit j set iff every sample of the rows is valid in view j. */
template <class G, int NJ, bool IDENT, bool FULLDIST, bool CHECKDEN, bool INSIDE, bool F16>
__device__ __forceinline__ unsigned sample_rows(const float4* __restrict__ rays, float* __restrict__ b0, float* __restrict__ b1,
                                                int sbase, bool tail_on, float inv_d, float s_min,
                                                const FswDevView& view0, const FswDevView& view1,
                                                const void* __restrict__ f0, const void* __restrict__ f1, float centre) {
    constexpr int NS = G::NS;
    /* Samples in flight per lane: four with the 8-byte footprints of the specialised variants, two otherwise (the raw
     * footprints stay in registers).  The slots (one halo pixel x NJ views each) run through a software pipeline of
     * DEPTH stages: the addresses and footprint fetches of slot i + DEPTH - 1 are issued before the lerps of slot i, so
     * that a fetch that misses L1 has a whole slot of arithmetic to come back from L2.  An invalid sample carries a
     * NaN weight au (and fetches footprint 0 instead of branching), so its lerp yields the NaN that marks it in the
     * sample plane. */
    constexpr int DEPTH = (((!FULLDIST && F16) ? 4 : 2) / NJ) > 1 ? 3 : 1;
    bool all_ok[NJ];
#pragma unroll
    for (int v = 0; v < NJ; ++v) all_ok[v] = true;
    float au[DEPTH][NJ], av[DEPTH][NJ];
    FootRaw<F16> raw[DEPTH][NJ];
    auto issue = [&](const int i) { /* S2-S3 + the fetch of S4 for slot i */
        const int st = i % DEPTH;
        const float4 ry = rays[sbase + 32 * i];
        float s = ry.w * inv_d;
        s = (s >= s_min) ? s : CUDART_NAN_F;
#pragma unroll
        for (int v = 0; v < NJ; ++v) {
            SampleAddr a = sample_addr<IDENT, FULLDIST, CHECKDEN, INSIDE>(ry.x, ry.y, ry.z, s, v ? view1 : view0);
            const bool on = a.ok && (i < G::NSFULL || tail_on); /* a pixel in this slot */
            au[st][v] = on ? a.au : CUDART_NAN_F; av[st][v] = a.av;
            if (i < G::NSFULL || tail_on) all_ok[v] = all_ok[v] && on;
            raw[st][v] = foot_fetch<F16>(v ? f1 : f0, on ? a.idx : 0u);
        }
    };
    auto finish = [&](const int i) { /* the lerp of S4 for slot i */
        const int st = i % DEPTH;
#pragma unroll
        for (int v = 0; v < NJ; ++v) {
            const float b = foot_lerp<F16>(raw[st][v], au[st][v], av[st][v], centre);
            if (i < G::NSFULL || tail_on) (v ? b1 : b0)[sbase + 32 * i] = b;
        }
    };
#pragma unroll
    for (int i = 0; i < DEPTH - 1; ++i) issue(i);
#pragma unroll
    for (int i = 0; i < NS; ++i) {
        if (i + DEPTH - 1 < NS) issue(i + DEPTH - 1);
        finish(i);
    }
    unsigned m = __all_sync(0xffffffffu, all_ok[0]) ? 1u : 0u;
    if (NJ > 1) m |= __all_sync(0xffffffffu, all_ok[NJ - 1]) ? 2u : 0u;
    return m;
}

/* the fields of a frame set the sweep loop touches, staged in shared memory once per tile */
struct SetHot {
    const void* foot[FSW_MAX_VIEWS];
    float* debug_cost;
};

/* Plane-consistent upsampling (alternative of reading Q18, Q28): the value of a pixel came from the
 * half-resolution pass as a plane offset d*; the pixel's own ray meets that plane at range d* / (n.r).  Out of line: a
 * rarely used variant must not cost the sweep loop registers.  The ray is recomputed (tiles outside the crop never
 * ran S1).  Returns the depth; sets reason = FSW_REASON_NO_PLANE where the ray does not meet the plane. */
static __device__ __noinline__ float plane_upsampled_depth(const FswSweepArgs& args, int ox, int oy, int kidx, float d_star, int& reason) {
    int f = 0;
    for (int g = 1; g < args.n_lo_fams; ++g)
        if (kidx >= args.lo_fam_first[g]) f = g;
    float rx = 0.f, ry = 0.f, rz = 0.f;
    const bool in_fov = back_project(args.ref, (float)ox, (float)oy, rx, ry, rz);
    const float q = fmaf(args.lo_fam_n[f][0], rx, fmaf(args.lo_fam_n[f][1], ry, args.lo_fam_n[f][2] * rz));
    if (in_fov && q > FSW_EPS_Q) {
        const float range = d_star / q;
        return args.depth_kind == FSW_DEPTH_Z ? range * rz : range;
    }
    reason = FSW_REASON_NO_PLANE;
    return d_star;
}

/* NVT = number of views known at compile time (1..4), 0 = read args.n_views at run time (then the view parameters
 * come from a copy in shared memory, not from dynamically indexed kernel parameters). */
template <int WIN, int NVT, bool IDENT, bool FULLDIST, bool CHECKDEN, bool INSIDE, bool F16, bool SPLIT>
__global__ void __launch_bounds__(Geo<WIN>::NT, 1) sweep_kernel(const __grid_constant__ FswSweepArgs args) {
    using G = Geo<WIN>;
    constexpr int HW = G::HW, RPT = G::RPT, NS = G::NS, TX = G::TX, TY = G::TY, R = G::R;
    constexpr float NWIN = (float)(WIN * WIN);
    constexpr float INV_NWIN = 1.f / NWIN;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float4* rays = reinterpret_cast<float4*>(smem_raw);   /* [EHA][SB]: unit ray, .w = validity / incidence */
    /* two views per pass where the shared memory allows it and there is more than one view */
    constexpr bool FUSE = G::FUSE_OK && NVT != 1;
    constexpr int NJ = FUSE ? 2 : 1;
    float* a_s = reinterpret_cast<float*>(rays + G::PLANE); /* [EHA][SB]: centred reference intensities a' (S1) */
    float* b_s = a_s + G::PLANE;                           /* [EHA][SB]: samples b' of the current (plane, view) */
    float* hs = b_s + G::PLANE;                            /* [NJ][4][EHA][HS]: row sums, one set per view of a pass */
    /* sample planes of the views of a pass: with FUSE the plane of a' (dead after S1) takes the first view */
    float* const bs0 = FUSE ? a_s : b_s;
    float* const bs1 = b_s;
    __shared__ float red_f[G::NW];
    __shared__ int red_i[G::NW];
    __shared__ unsigned s_mixed[3][2], s_any[3][2]; /* rotating flags of a pass, per view of the pass */
    __shared__ unsigned s_item;
    __shared__ SetHot s_set;
    __shared__ FswDevView s_views[NVT ? 1 : FSW_MAX_VIEWS]; /* run-time view loop: the view parameters */

    /* the thread index held in a register (asm volatile): values derived from it are recomputed before their uses
     * anyway, but from a register and not from S2R */
    /* (measured: 1.3 % faster at C5 / C3 -- two unrotated views --, 1.2 % slower with four rotated views, 2 % slower
     * with two rotated ones: kept where it pays) */
    constexpr bool PIN = (NVT == 1 || NVT == 2) && IDENT;
    unsigned tid_reg = threadIdx.x;
    if constexpr (PIN) asm volatile("mov.b32 %0, %0;" : "+r"(tid_reg));
    const int tid = (int)tid_reg, lane = tid & 31, wid = tid >> 5;
    const int col = tid % TX, grp = tid / TX;
    /* [TY][TX]: reference-side window statistics of every output: ((sum a')/N, sum a'^2 - (sum a')^2/N) */
    float2* const a_stat = reinterpret_cast<float2*>(hs + NJ * 4 * G::HPLANE) + (grp * RPT) * TX + col;
    /* [TY][TX]: costs of the planes below / above the running best of every output (Wta::update) */
    float2* const nbr_s = a_stat + TX * TY;
    const int W = args.ref.W, H = args.ref.H;
    /* split launches: the first split_whole (tile, set) slots are swept whole, every later one as two halves */
    /* a split launch covers the (tile, set) slots slot_first .. slot_first + slot_count - 1 of the queue order, an
     * unsplit one the first n_tiles * n_sets */
    const int n_items = SPLIT ? 2 * args.slot_count - args.split_whole : args.n_tiles * args.n_sets;
    const int n_views = NVT ? NVT : args.n_views;
    if constexpr (NVT == 0) {
        constexpr int NWORDS = (int)(sizeof(FswDevView) / 4) * FSW_MAX_VIEWS;
        static_assert(sizeof(FswDevView) % 4 == 0 && NWORDS <= G::NT, "one word per thread");
        if (threadIdx.x < NWORDS)
            reinterpret_cast<uint32_t*>(s_views)[threadIdx.x] = reinterpret_cast<const uint32_t*>(args.views)[threadIdx.x];
        /* the first barrier of the first tile orders this against the sweep */
    }

    /* this lane's halo pixels: slot i is element lane + 32 i of the warp's R x SB block of the sample planes; in the
     * last slot only the lanes below `tail` have a pixel */
    const int sbase = wid * R * G::SB + lane;
    constexpr int TAIL = R * G::SB - 32 * G::NSFULL; /* 0 if every slot is full */
    const bool tail_on = lane < TAIL;
    /* this lane's horizontal work item */
    int hrow_l, hrun;
    h_item<G>(lane, hrow_l, hrun);
    const int hrow = wid * R + hrow_l;
    /* PIN: where the item sits in the sample planes (13 bits) and in the row-sum planes (13 bits), and whether the lane
     * has one (sign bit), packed into one register that the compiler has to keep: left to itself it recomputes the
     * three values from the thread index before every use, some 25 instructions per view and pass */
    static_assert(G::PLANE < 8192 && G::HPLANE < 8192, "13-bit offsets");
    bool h_on_v;
    int h_src_v, h_dst_v;
    if constexpr (PIN) {
        unsigned hpack = (hrow_l >= 0 && hrow < G::EH)
                             ? ((unsigned)(hrow * G::SB + hrun * RUN) | ((unsigned)(hrow * G::HS + hrun * RUN) << 13) | 0x80000000u) : 0u;
        asm volatile("mov.b32 %0, %0;" : "+r"(hpack));
        h_on_v = (int)hpack < 0;
        h_src_v = (int)(hpack & 0x1fffu);
        h_dst_v = (int)((hpack >> 13) & 0x1fffu);
    } else {
        h_on_v = hrow_l >= 0 && hrow < G::EH;
        h_src_v = h_on_v ? hrow * G::SB + hrun * RUN : 0;
        h_dst_v = h_on_v ? hrow * G::HS + hrun * RUN : 0;
    }
    const bool h_on = h_on_v;
    const int h_src = h_src_v;
    float* const h_dst = hs + h_dst_v;
    const float* const v_src = hs + (grp * RPT) * G::HS + col; /* first row sum of this thread's vertical pass */

    /* An unsplit launch may be followed in the stream by the launch of the halved tiles as its programmatic dependent
     * (fsw_api.cu: launch_sweep): those blocks take the SMs this grid's blocks leave.  Nothing they read is written
     * here, so the trigger comes first; they wait for this grid before they exit. */
    if constexpr (!SPLIT) asm volatile("griddepcontrol.launch_dependents;");

    unsigned item = blockIdx.x;
    while (item < (unsigned)n_items) {
        /* plane split: the slots beyond split_whole are two items each, half 0 and half 1; own planes [k_lo, k_hi),
         * visited downwards in half 1 */
        const bool halved = SPLIT && item >= (unsigned)args.split_whole;
        const int half = halved ? (int)((item - (unsigned)args.split_whole) & 1u) : 0;
        const unsigned titem = !SPLIT ? item : (unsigned)args.slot_first +
                               (halved ? (unsigned)args.split_whole + ((item - (unsigned)args.split_whole) >> 1) : item);
        const bool desc = halved && half != 0;
        const int dir = desc ? -1 : 1;
        const int k_lo = desc ? args.split_k : 0, k_hi = (halved && !half) ? args.split_k : args.n_planes;
        /* the plane across the cut, evaluated only as the parabola neighbour of a winner next to the cut */
        const int k_halo = (halved && args.split_adjacent) ? (half ? args.split_k - 1 : args.split_k) : -1;
        const int set = (int)(titem % (unsigned)args.n_sets);
        const int tile = args.tile_order[titem / (unsigned)args.n_sets];
        const FswSetPtrs& S = args.n_sets > 1 ? args.sets[set] : args.set0;
        const int tyi = tile / args.n_tiles_x, txi = tile - tyi * args.n_tiles_x;
        const int x0t = txi * TX, y0t = tyi * TY;
        const int ox = x0t + col;            /* this thread's output column */
        const int oy0 = y0t + grp * RPT;     /* ... and first output row */

        Wta st[RPT];
        float2 nbr_r[G::NBR_SMEM ? 1 : RPT]; /* ... or in registers */
        auto nbr_at = [&](const int i) -> float2* { return G::NBR_SMEM ? &nbr_s[i * TX] : &nbr_r[G::NBR_SMEM ? 0 : i]; };
#pragma unroll
        for (int i = 0; i < RPT; ++i) {
            st[i].init();
            *nbr_at(i) = make_float2(CUDART_INF_F, CUDART_INF_F);
        }
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
        float centre = 0.f;
        float areg[G::NV4 * 4];   /* a' operands of this lane's horizontal work item */
#pragma unroll
        for (int i = 0; i < G::NV4 * 4; ++i) areg[i] = 0.f;
        /* state of this warp's rows of plane 3 of either row-sum set: 0 = WIN everywhere, 1 = zero, 2 = counts,
         * 3 = never written (the second set; S1 fills the first one) */
        int p3[2] = {0, 3};
        const bool dbg = S.debug_cost != nullptr;

        if (tile_live) {
            if (tid < FSW_MAX_VIEWS) s_set.foot[tid] = S.foot[tid];
            if (tid == 32) s_set.debug_cost = S.debug_cost;
            /* ---- S1: rays and reference intensities of the tile + halo ------------------------------------ */
            float lsum = 0.f;
            int lcnt = 0;
#pragma unroll 1
            for (int i = 0; i < NS; ++i) {
                const int p = lane + 32 * i;
                if (p >= R * G::SB) break;
                const int lr = p / G::SB, cx_ = p - lr * G::SB, row = wid * R + lr;
                const int px = x0t - HW + cx_, py = y0t - HW + row;
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
                const int o = sbase + 32 * i;
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
                if (i < G::NSFULL || tail_on) a_s[sbase + 32 * i] -= centre;
            __syncwarp();
            /* window sums of the reference side, once per pixel; the a' run stays in registers */
            if (h_on) {
                float q[G::NV4 * 4], p[G::NV4 * 4];
                load_run<G>(a_s + h_src, areg);
                load_run<G>(b_s + h_src, q);
#pragma unroll
                for (int i = 0; i < G::NV4 * 4; ++i) p[i] = areg[i];
                hsum<G, WIN, 0>(p, q, h_dst);
                fill_count<G>(h_dst, (float)WIN);
            }
            __syncthreads();
            {
                float sa[RPT], saa[RPT], sf[RPT];
                vpass<G, WIN>(v_src, sa);
                vpass<G, WIN>(v_src + G::HPLANE, saa);
                vpass<G, WIN>(v_src + 2 * G::HPLANE, sf);
#pragma unroll
                for (int i = 0; i < RPT; ++i) {
                    int oy = oy0 + i;
                    bool in_roi = ox >= args.roi_x0 && ox < args.roi_x1 && oy >= args.roi_y0 && oy < args.roi_y1;
                    bool act = in_roi && (sf[i] == NWIN); /* every window pixel inside the image and the FOV */
                    if (act) active_mask |= 1u << i;
                    const float a1n = sa[i] * INV_NWIN;
                    a_stat[i * TX] = make_float2(a1n, fmaf(-a1n, sa[i], saa[i]));
                }
            }
            if (tid < 6) { s_mixed[tid >> 1][tid & 1] = 0u; s_any[tid >> 1][tid & 1] = 0u; }
            tile_active = __syncthreads_or(active_mask != 0) != 0;
        }

        if (tile_active) {
            const float inv_views = 1.f / (float)n_views;
            unsigned ph = 0; /* rotation of the pass flags */
#pragma unroll 1
            for (int fi = 0; fi < args.n_fams; ++fi) {
                const int f = desc ? args.n_fams - 1 - fi : fi;
                const FswDevFamily& F = args.fam[f];
                /* own planes of this item in the family: j0 <= j < j1 */
                int j0 = 0, j1 = F.count;
                bool has_halo = false;
                if constexpr (SPLIT) {
                    j0 = max(k_lo - F.first, 0);
                    j1 = min(k_hi - F.first, F.count);
                    if (j1 <= j0) continue;
                    has_halo = k_halo >= F.first && k_halo < F.first + F.count; /* then the last family visited */
                }
                const int n_own = j1 - j0;
                const float fnx = F.n[0], fny = F.n[1], fnz = F.n[2];
#pragma unroll
                for (int i = 0; i < RPT; ++i) st[i].family_start();
                /* incidence q = n.r of this lane's halo rays with the family, NaN where the ray does not face the
                 * planes (or is outside the camera); the largest q of the warp's rows / of the tile decides which
                 * planes can be reached within range_max */
                float qmax_w = 0.f;
#pragma unroll
                for (int i = 0; i < NS; ++i) {
                    if (i >= G::NSFULL && !tail_on) continue;
                    float4 ry = rays[sbase + 32 * i];
                    float q = fmaf(fnx, ry.x, fmaf(fny, ry.y, fnz * ry.z));
                    bool faces = q > FSW_EPS_Q; /* an invalid reference ray is the zero vector: q = 0 */
                    rays[sbase + 32 * i].w = faces ? q : CUDART_NAN_F;
                    if (faces) qmax_w = fmaxf(qmax_w, q);
                }
                qmax_w = warp_max(qmax_w);
                __syncthreads(); /* previous users of red_f are done */
                if (lane == 0) red_f[wid] = qmax_w;
                __syncthreads();
                float qmax = 0.f;
#pragma unroll
                for (int i = 0; i < G::NW; ++i) qmax = fmaxf(qmax, red_f[i]);
                /* does any active output of this warp face the family at all?  If not (outside the image circle, above
                 * the horizon for ground-parallel planes) the warp skips the vertical pass and the ZNCC of every plane */
                bool v_act = false;
#pragma unroll
                for (int i = 0; i < RPT; ++i)
                    v_act = v_act || (((active_mask >> i) & 1u) && rays[(grp * RPT + i + HW) * G::SB + col + HW].w > 0.f);
                v_act = __any_sync(0xffffffffu, v_act);

#pragma unroll 1
                for (int it = 0; it < n_own + (has_halo ? 1 : 0); ++it) {
                    const bool halo = SPLIT && it >= n_own;
                    const int k = !SPLIT ? F.first + it : (halo ? k_halo : F.first + (desc ? j1 - 1 - it : j0 + it));
                    const float inv_d = args.inv_d[k];
                    float acc[RPT];
                    unsigned cnt = 0; /* valid views per output, 4 bits each */
#pragma unroll
                    for (int i = 0; i < RPT; ++i) acc[i] = 0.f;
                    /* best-k view aggregation (reading Q26; run-time view loop only): the two lowest per-view costs */
                    float bk1[NVT == 0 ? RPT : 1], bk2[NVT == 0 ? RPT : 1];
                    if constexpr (NVT == 0) {
#pragma unroll
                        for (int i = 0; i < RPT; ++i) { bk1[i] = CUDART_INF_F; bk2[i] = CUDART_INF_F; }
                    }
                    /* S2: the plane is out of reach for the whole tile if even the best-facing ray is beyond range */
                    if (qmax * inv_d >= args.inv_range_max) {
                        const bool rows_on = qmax_w * inv_d >= args.inv_range_max; /* any ray of this warp's rows */
                        /* one pass = NJP (1 or 2) views va, va + 1 of the plane: sample, horizontal sums, barrier [A],
                         * vertical sums (barrier [B] after the last loads), ZNCC into acc / cnt */
                        auto run_pass = [&](auto njp_c, const int va) {
                            constexpr int NJP = decltype(njp_c)::value;
                            const int vb = va + NJP - 1;
                            const FswDevView& vw0 = NVT ? args.views[va] : s_views[va];
                            const FswDevView& vw1 = NVT ? args.views[vb] : s_views[vb];
                            float* const b0 = NJP == 2 ? bs0 : bs1; /* a single view always samples into b_s */
                            /* ---- S2-S4: sample the plane-warped views at this warp's halo rows ----------------- */
                            unsigned okmask = (1u << NJP) - 1u;
                            if (rows_on)
                                okmask = sample_rows<G, NJP, IDENT, FULLDIST, CHECKDEN, INSIDE, F16>(
                                    rays, b0, bs1, sbase, tail_on, inv_d, args.inv_range_max, vw0, vw1,
                                    s_set.foot[va], s_set.foot[vb], centre);
                            __syncwarp();
                            /* ---- S5: horizontal box sums of the same rows, view by view ------------------------ */
#pragma unroll
                            for (int j = 0; j < NJP; ++j) {
                                float* const hd = h_dst + j * 4 * G::HPLANE;
                                const bool all_ok = (okmask >> j) & 1u;
                                bool any_ok = rows_on;
                                if (rows_on) {
                                    bool any_l = false;
                                    if (h_on) {
                                        float p[G::NV4 * 4];
                                        load_run<G>((j ? bs1 : b0) + h_src, p);
                                        if (!G::A_IN_REGS) load_run<G>(a_s + h_src, areg);
                                        if (all_ok) {
                                            hsum<G, WIN, 1>(p, areg, hd);
                                            if (p3[j] != 0) fill_count<G>(hd, (float)WIN);
                                        } else {
                                            any_l = hsum<G, WIN, 2>(p, areg, hd);
                                        }
                                    }
                                    if (!all_ok) any_ok = __any_sync(0xffffffffu, any_l);
                                    p3[j] = all_ok ? 0 : 2;
                                } else {
                                    if (p3[j] != 1 && h_on) fill_zero<G>(hd);
                                    p3[j] = 1;
                                }
                                if (lane == 0) {
                                    if (any_ok) s_any[ph][j] = 1u;
                                    if (!(rows_on && all_ok)) s_mixed[ph][j] = 1u;
                                }
                            }
                            __syncthreads(); /* [A] row sums of the pass are complete */
                            unsigned f_mixed[NJP], f_any[NJP];
                            int last = -1; /* last view of the pass that sees anything of the tile */
#pragma unroll
                            for (int j = 0; j < NJP; ++j) {
                                f_mixed[j] = s_mixed[ph][j];
                                f_any[j] = s_any[ph][j];
                                if (f_any[j]) last = j;
                            }
                            {
                                const unsigned nx = ph >= 1 ? ph - 1 : 2; /* (ph + 2) % 3: the flags after next */
                                if (tid < 2) { s_mixed[nx][tid] = 0u; s_any[nx][tid] = 0u; }
                            }
                            ph = ph == 2 ? 0 : ph + 1;
                            if (last < 0) return; /* no view sees anything of the tile through this plane */
                            /* ---- vertical sums, ZNCC -------------------------------------------------------- */
                            if (!v_act) { /* nothing to score in this warp: only keep the barrier count */
                                __syncthreads();
                                return;
                            }
#pragma unroll
                            for (int j = 0; j < NJP; ++j) {
                                if (!f_any[j]) continue;
                                const float* const vs = v_src + j * 4 * G::HPLANE;
                                float sb[RPT], sbb[RPT], sab[RPT], sv[RPT];
                                vpass<G, WIN>(vs, sb);
                                vpass<G, WIN>(vs + G::HPLANE, sbb);
                                vpass<G, WIN>(vs + 2 * G::HPLANE, sab);
                                if (f_mixed[j]) vpass<G, WIN>(vs + 3 * G::HPLANE, sv);
                                /* [B] everyone has read the row sums: the next pass may overwrite them */
                                if (j == last) __syncthreads();
#pragma unroll
                                for (int i = 0; i < RPT; ++i) {
                                    bool okv = (active_mask >> i) & 1u;
                                    if (f_mixed[j]) okv = okv && (sv[i] == NWIN);
                                    const float2 A = a_stat[i * TX]; /* written by this thread */
                                    float cov = fmaf(-A.x, sb[i], sab[i]);
                                    float vbv = fmaf(-sb[i] * INV_NWIN, sb[i], sbb[i]);
                                    float prod = fmaxf(A.y * vbv, args.floor2);
                                    float z = cov * rsqrt_approx(prod);
                                    float cst = __saturatef(fmaf(-0.5f, z, 0.5f));
                                    acc[i] += okv ? cst : 0.f;
                                    cnt += okv ? (1u << (4 * i)) : 0u;
                                    if constexpr (NVT == 0) {
                                        const float cv = okv ? cst : CUDART_INF_F;
                                        const float hi = fmaxf(bk1[i], cv);
                                        bk1[i] = fminf(bk1[i], cv);
                                        bk2[i] = fminf(bk2[i], hi);
                                    }
                                }
                            }
                        };
                        if constexpr (NVT != 0) {
                            /* compile-time view list: pairs, then a single view if the count is odd */
#pragma unroll
                            for (int va = 0; va < NVT; va += NJ) {
                                if (NVT - va >= 2 && NJ == 2) run_pass(std::integral_constant<int, NJ>{}, va);
                                else run_pass(std::integral_constant<int, 1>{}, va);
                            }
                        } else {
#pragma unroll 1
                            for (int va = 0; va < n_views; va += NJ) {
                                if (NJ == 2 && n_views - va >= 2) run_pass(std::integral_constant<int, NJ>{}, va);
                                else run_pass(std::integral_constant<int, 1>{}, va);
                            }
                        }
                    }
                    /* ---- S6 + S7: view mean, streaming winner-take-all ------------------------------------- */
#pragma unroll
                    for (int i = 0; i < RPT; ++i) {
                        const int ci = (int)((cnt >> (4 * i)) & 15u);
                        float c;
                        if (NVT == 1) c = acc[i];
                        else if (NVT == 2) c = ci == 2 ? 0.5f * acc[i] : acc[i];
                        else c = ci == n_views ? acc[i] * inv_views : acc[i] * args.inv_count[ci];
                        if constexpr (NVT == 0) {
                            if (args.best_k == 1) c = bk1[i];
                            else if (args.best_k == 2) c = ci >= 2 ? 0.5f * (bk1[i] + bk2[i]) : bk1[i];
                        }
                        c = ci > 0 ? c : CUDART_INF_F;
                        n_eval += halo ? 0 : ci;
                        st[i].template update<false>(c, k, dir, desc, it == 0, nbr_at(i), halo);
                    }
                    if (dbg) {
                        float* dc = s_set.debug_cost;
#pragma unroll
                        for (int i = 0; i < RPT; ++i) {
                            const int oy = oy0 + i;
                            if (ox < W && oy < H && !halo) dc[((int64_t)k * H + oy) * W + ox] = st[i].cprev;
                        }
                    }
                }
            }
        }
        if (dbg && !tile_active && half == 0) {
            for (int k = 0; k < args.n_planes; ++k)
#pragma unroll
                for (int i = 0; i < RPT; ++i) {
                    int oy = oy0 + i;
                    if (ox < W && oy < H) S.debug_cost[((int64_t)k * H + oy) * W + ox] = CUDART_INF_F;
                }
        }

        /* ---- plane split: the half of a tile that finishes first leaves its winner-take-all state in global memory,
         * the other one merges it into its registers and goes on.  State per pixel: b1, k1, s2, cm, cp and m2 = the
         * lowest cost of the half's planes except the one next to the cut (visited last). ----------------------- */
        bool do_epilogue = true;
#pragma unroll
        for (int i = 0; i < RPT; ++i) {
            const float2 n = *nbr_at(i);
            st[i].cm = n.x; st[i].cp = n.y;
        }
        if (desc) {
#pragma unroll
            for (int i = 0; i < RPT; ++i) st[i].swap_neighbours();
        }
        if (halved) {
            if (!tile_active) {
                do_epilogue = half == 0; /* nothing was swept: one half writes the invalid / upsampled outputs */
            } else {
                const size_t mapsz = (size_t)H * W;
                float* const mine = args.split_state + ((size_t)set * 2 + half) * 6 * mapsz;
                const float* const other = args.split_state + ((size_t)set * 2 + (1 - half)) * 6 * mapsz;
                const unsigned tslot = (unsigned)set * (unsigned)args.n_tiles + (unsigned)tile;
#pragma unroll
                for (int i = 0; i < RPT; ++i) {
                    const int oy = oy0 + i;
                    if (ox >= W || oy >= H) continue;
                    float* q = mine + (size_t)oy * W + ox;
                    __stcg(q, st[i].b1); __stcg(q + mapsz, __int_as_float(st[i].k1)); __stcg(q + 2 * mapsz, st[i].s2);
                    __stcg(q + 3 * mapsz, st[i].cm); __stcg(q + 4 * mapsz, st[i].cp); __stcg(q + 5 * mapsz, st[i].m2);
                }
                __threadfence();
                __syncthreads();
                if (tid == 0) s_item = atomicAdd(&args.split_ticket[tslot], 1u);
                __syncthreads();
                const unsigned ticket = s_item;
                __syncthreads(); /* s_item is reused for the queue below */
                if (ticket == 0) {
                    do_epilogue = false;
                } else {
                    if (tid == 0) args.split_ticket[tslot] = 0u; /* both halves are through: ready for the next launch */
                    __threadfence();
#pragma unroll
                    for (int i = 0; i < RPT; ++i) {
                        const int oy = oy0 + i;
                        if (ox >= W || oy >= H) continue;
                        const float* q = other + (size_t)oy * W + ox;
                        const float ob1 = __ldcg(q), os2 = __ldcg(q + 2 * mapsz), ocm = __ldcg(q + 3 * mapsz);
                        const float ocp = __ldcg(q + 4 * mapsz), om2 = __ldcg(q + 5 * mapsz);
                        const int ok1 = __float_as_int(__ldcg(q + mapsz));
                        Wta& m = st[i];
                        /* A = planes below the cut (half 0), B = planes from the cut on; the lower index wins a tie */
                        const bool a_wins = half == 0 ? (m.b1 <= ob1) : (ob1 <= m.b1);
                        const bool mine_wins = a_wins == (half == 0);
                        const float lb1 = mine_wins ? ob1 : m.b1, lm2 = mine_wins ? om2 : m.m2;
                        m.b1 = mine_wins ? m.b1 : ob1; m.k1 = mine_wins ? m.k1 : ok1; m.s2 = mine_wins ? m.s2 : os2;
                        m.cm = mine_wins ? m.cm : ocm; m.cp = mine_wins ? m.cp : ocp;
                        /* second best (reading Q12): the loser's planes all count, except the one next to the cut when
                         * the winner sits on the other side of it */
                        const int edge = a_wins ? args.split_k - 1 : args.split_k;
                        const bool at_cut = args.split_adjacent && m.k1 == edge;
                        m.s2 = fminf(m.s2, at_cut ? lm2 : lb1);
                    }
                }
            }
        }

        /* ---- S8-S12: refinement, depth, merge, filters, mask, stores --------------------------------------- */
        unsigned n_raw = 0, n_ok = 0;
#pragma unroll
        for (int i = 0; i < RPT; ++i) {
            const int oy = oy0 + i;
            if (ox >= W || oy >= H || !do_epilogue) continue;
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
                depth = args.depth_kind == FSW_DEPTH_Z ? range * ry.z : (args.depth_kind == FSW_DEPTH_PLANE_OFFSET ? d : range);
                c1 = st[i].b1;
                c2 = st[i].s2 < CUDART_INF_F ? st[i].s2 : 1.f;
                kidx = st[i].k1 | args.index_flag;
            }
            /* S9: verdict of the cost / ratio filters on a (best, second best) pair of this row */
            auto verdict = [&](const float b, const float sec) -> int {
                const float alpha = oy < args.horizon_row ? args.alpha_upper : args.alpha_lower;
                if ((args.filters & FSW_FILTER_COST) && b > alpha) return FSW_REASON_COST_FILTER;
                if ((args.filters & FSW_FILTER_RATIO) && sec < args.beta * fmaxf(b, 1e-6f)) return FSW_REASON_RATIO_FILTER;
                return FSW_REASON_OK;
            };
            int reason;
            if (S.lo_k != nullptr) {
                /* S10(c)-(e): merge with the nearest-neighbour upsampled half-resolution pass */
                const int xl = ox >> 1, yl = oy >> 1;
                const bool lo_in = xl < args.lo_W && yl < args.lo_H;
                const int64_t j = lo_in ? (int64_t)yl * args.lo_W + xl : 0;
                const int kl = lo_in ? (int)S.lo_k[j] : -1;
                if (!args.filter_first) {
                    /* reading Q19 / Q20: full resolution where it has any finite plane, else the upsampled estimate;
                     * the filters see the merged map */
                    if (!raw_valid && kl >= 0) {
                        raw_valid = true;
                        depth = S.lo_depth[j]; c1 = S.lo_c1[j]; c2 = S.lo_c2[j]; kidx = kl;
                    }
                    reason = raw_valid ? verdict(c1, c2) : FSW_REASON_NO_PLANE;
                } else {
                    /* reading Q27: each scale filtered on its own; a surviving full-resolution estimate wins, else a
                     * surviving upsampled one fills in; otherwise the pixel reports the estimate (and the reason) the
                     * default order would have taken */
                    reason = raw_valid ? verdict(c1, c2) : FSW_REASON_NO_PLANE;
                    if (reason != FSW_REASON_OK && kl >= 0) {
                        const int lo_reason = S.lo_reason[j];
                        if (lo_reason == FSW_REASON_OK || !raw_valid) {
                            raw_valid = true;
                            depth = S.lo_depth[j]; c1 = S.lo_c1[j]; c2 = S.lo_c2[j]; kidx = kl;
                            reason = lo_reason;
                        }
                    }
                }
            } else {
                reason = raw_valid ? verdict(c1, c2) : FSW_REASON_NO_PLANE;
            }
            if (args.upsample_plane && (kidx >= 0) && !(kidx & FSW_INDEX_FROM_CROP) && S.lo_k != nullptr)
                depth = plane_upsampled_depth(args, ox, oy, kidx, depth, reason);
            if (reason == FSW_REASON_OK && S.mask != nullptr && S.mask[(int64_t)oy * S.mask_pitch + ox]) reason = FSW_REASON_MASKED;
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
    /* a dependent launch completes after the grid before it (no-op for a plain launch) */
    if constexpr (SPLIT) asm volatile("griddepcontrol.wait;" ::: "memory");
}

/* Kernel variants (fsw_api.cu: pick_variant): projection mode 0..2 (see SweepInst::go) + 3 if the footprints are
 * 8-byte bfloat16; 6, 7 = modes 1, 2 with bfloat16 footprints for views whose image circle lies inside the raster (no
 * border test); + 8 for the plane split (two work items per tile). */
template <int WIN, int NVT>
struct SweepInst {
    using G = Geo<WIN>;
    static constexpr bool FUSE = G::FUSE_OK && NVT != 1;
    /* MODE 0: any rotation, full distortion polynomial, denominator test; 1: identity rotations, k1-only distortion;
     * 2: any rotation, k1-only distortion (the last two need cos(fov/2) + xi >= 1e-3) */
    template <int MODE, bool F16, bool INSIDE, bool SPLIT>
    static cudaError_t go(const FswSweepArgs& args, int grid, cudaStream_t stream, bool prepare_only, bool programmatic) {
        auto kern = sweep_kernel<WIN, NVT, MODE == 1, MODE == 0, MODE == 0, INSIDE, F16, SPLIT>;
        if (prepare_only) return cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)G::smem(FUSE));
        if (!programmatic) {
            kern<<<grid, G::NT, G::smem(FUSE), stream>>>(args);
            return cudaGetLastError();
        }
        /* programmatic dependent launch: the blocks of this grid may become resident as soon as every block of the
         * kernel before it in the stream has executed griddepcontrol.launch_dependents or exited */
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3(G::NT); cfg.dynamicSmemBytes = G::smem(FUSE); cfg.stream = stream;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = attr; cfg.numAttrs = 1;
        return cudaLaunchKernelEx(&cfg, kern, args);
    }
    static constexpr int N_VARIANTS = 16;
    template <bool SPLIT>
    static cudaError_t dispatch8(const FswSweepArgs& args, int variant, int grid, cudaStream_t stream, bool prep, bool pdl) {
        switch (variant) {
            case 0: return go<0, false, false, SPLIT>(args, grid, stream, prep, pdl);
            case 1: return go<1, false, false, SPLIT>(args, grid, stream, prep, pdl);
            case 2: return go<2, false, false, SPLIT>(args, grid, stream, prep, pdl);
            case 3: return go<0, true, false, SPLIT>(args, grid, stream, prep, pdl);
            case 4: return go<1, true, false, SPLIT>(args, grid, stream, prep, pdl);
            case 5: return go<2, true, false, SPLIT>(args, grid, stream, prep, pdl);
            case 6: return go<1, true, true, SPLIT>(args, grid, stream, prep, pdl);
            case 7: return go<2, true, true, SPLIT>(args, grid, stream, prep, pdl);
            default: break;
        }
        return cudaErrorInvalidValue;
    }
    static cudaError_t dispatch(const FswSweepArgs& args, int variant, int grid, cudaStream_t stream, bool prep, bool pdl = false) {
        return variant < 8 ? dispatch8<false>(args, variant, grid, stream, prep, pdl)
                           : dispatch8<true>(args, variant - 8, grid, stream, prep, pdl);
    }
    /* variant + FSW_VARIANT_PROGRAMMATIC: launched as a programmatic dependent of the kernel before it in the stream */
    static cudaError_t launch(const FswSweepArgs& args, int variant, int grid, cudaStream_t stream) {
        return dispatch(args, variant & (FSW_VARIANT_PROGRAMMATIC - 1), grid, stream, false, (variant & FSW_VARIANT_PROGRAMMATIC) != 0);
    }
    static cudaError_t prepare() {
        static const FswSweepArgs dummy = {};
        for (int v = 0; v < N_VARIANTS; ++v) {
            cudaError_t e = dispatch(dummy, v, 0, nullptr, true);
            if (e != cudaSuccess) return e;
        }
        return cudaSuccess;
    }
};

/* Which instantiation serves a call: up to four views (the paper's rig has four matching views) have
 * their view loop unrolled, pairs of views sharing a pass; more views, or three / four views with the large windows
 * that cannot pair them, take the run-time loop (NVT = 0); so do calls with best-k view aggregation (its two extra
 * registers per output stay out of the kernels that serve the default). */
template <int WIN>
constexpr int nvt_for(int n_views, int best_k) {
    if (best_k > 0) return 0;
    return n_views <= 2 ? n_views : ((n_views <= 4 && Geo<WIN>::FUSE_OK) ? n_views : 0);
}

template <int WIN>
FswSweepGeometry geometry_win(int n_views) {
    using G = Geo<WIN>;
    FswSweepGeometry g;
    g.tile_w = G::TX; g.tile_h = G::TY; g.threads = G::NT; g.ctas_per_sm = G::MINB;
    g.smem_bytes = G::smem(G::FUSE_OK && n_views != 1);
    return g;
}

}  // namespace fsw
#endif
