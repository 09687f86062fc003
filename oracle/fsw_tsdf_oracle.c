/*
 * fsw_tsdf_oracle.c -- CPU ORACLE of the TSDF consumer.  TEST INFRASTRUCTURE: only tests/ may use it;
 * it shares no code with paper_1809_06132_b200/ and neither includes the other.
 *
 * What it computes (section III-C "TSDF-based Depth Map Fusion"), plain and slow, in double precision:
 *   allocation   "we iterate through each pixel p with a valid depth value d ... compute its back-projected ray
 *                direction [Eq. 1] ... consider the range from d - mu to d + mu along this ray ... compute the
 *                coordinates of voxel blocks along this line segment ... allocate new voxel blocks",
 *                "we only allocate new voxel blocks within this region" (the local map)
 *   integration  Eq. 2: X_d = R_d X + t_d, projection with the unified model, eta = depth - range,
 *                update iff eta >= -mu:  D <- (w D + min(1, eta/mu)) / (w + 1),  w <- min(w + 1, w_max)
 *   gate         "we only consider voxel blocks with at least 3 observations"
 * Readings where the paper is silent (T1-T6): blocks of 8^3 voxels, voxel centre at (index + 0.5) voxel_size,
 * the segment is sampled at n + 1 equidistant points with n = ceil(2 mu / (block edge / 2)), the depth map stores range
 * along the ray (reading Q16) and eta is taken against |X_d|, nearest-neighbour depth lookup at floor(u + 0.5), a block's
 * observation count goes up by one per frame in which at least one of its voxels was updated, the local box is
 * snapped to whole blocks.
 *
 * The volume is the local box only, dense: nb[3] blocks from the integer block origin b0[3] (world block coordinates);
 * voxel (block b, local i,j,k) lives at D[((bz*nby + by)*nbx + bx)*512 + (k*8 + j)*8 + i].
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#include "fsw_oracle.h"

#define TSDF_BLOCK 8

typedef struct {
    double voxel_size, mu;
    int32_t w_max;
    int32_t b0[3]; /* world block coordinate of the box's first block */
    int32_t nb[3]; /* blocks per axis */
} orc_tsdf_box;

static size_t block_slot(const orc_tsdf_box* B, int bx, int by, int bz) {
    return ((size_t)(bz - B->b0[2]) * B->nb[1] + (size_t)(by - B->b0[1])) * B->nb[0] + (size_t)(bx - B->b0[0]);
}

static int in_box(const orc_tsdf_box* B, int bx, int by, int bz) {
    return bx >= B->b0[0] && bx < B->b0[0] + B->nb[0] && by >= B->b0[1] && by < B->b0[1] + B->nb[1] &&
           bz >= B->b0[2] && bz < B->b0[2] + B->nb[2];
}

/* Allocation.  cam: intrinsics of the depth camera; R, t: world -> camera (X_d = R X + t);
 * depth: H*W ranges along the pixel rays, <= 0 = invalid.  allocated: one byte per block of the box, set to 1 for
 * every block that contains a sample of some pixel's segment (never cleared here).  fragile (nullable): set to 1 for
 * blocks that a sample misses or hits by less than 1e-4 of a block edge.  Returns the number of newly set blocks. */
int64_t orc_tsdf_allocate(const orc_tsdf_box* B, const orc_camera* cam, const double R[9], const double t[3],
                          const double* depth, uint8_t* allocated, uint8_t* fragile) {
    const double edge = B->voxel_size * TSDF_BLOCK;
    const int n = (int)ceil(2.0 * B->mu / (0.5 * edge));
    int64_t fresh = 0;
    for (int y = 0; y < cam->height; ++y)
        for (int x = 0; x < cam->width; ++x) {
            const double d = depth[(size_t)y * cam->width + x];
            if (!(d > 0.0)) continue;
            double r[3];
            if (!orc_back_project(cam, (double)x, (double)y, r)) continue; /* Eq. 1 */
            for (int i = 0; i <= n; ++i) {
                const double range = (d - B->mu) + (double)i * (2.0 * B->mu / (double)n);
                const double Xd[3] = { range * r[0] - t[0], range * r[1] - t[1], range * r[2] - t[2] };
                double X[3], f[3];
                int b[3], near = 0, side[3] = { 0, 0, 0 }; /* side: the neighbour across a face the sample almost touches */
                for (int a = 0; a < 3; ++a) { /* X = R^T (X_d - t) */
                    X[a] = R[a] * Xd[0] + R[3 + a] * Xd[1] + R[6 + a] * Xd[2];
                    f[a] = X[a] / edge;
                    b[a] = (int)floor(f[a]);
                    if (fabs(f[a] - floor(f[a] + 0.5)) < 1e-4) { near = 1; side[a] = (f[a] - floor(f[a]) < 0.5) ? -1 : 1; }
                }
                if (near && fragile) /* the sample's block and the blocks across the near face(s) */
                    for (int m = 0; m < 8; ++m) {
                        const int dx = (m & 1) ? side[0] : 0, dy = (m & 2) ? side[1] : 0, dz = (m & 4) ? side[2] : 0;
                        if (in_box(B, b[0] + dx, b[1] + dy, b[2] + dz)) fragile[block_slot(B, b[0] + dx, b[1] + dy, b[2] + dz)] = 1;
                    }
                if (!in_box(B, b[0], b[1], b[2])) continue; /* only inside the local map */
                uint8_t* a = &allocated[block_slot(B, b[0], b[1], b[2])];
                if (!*a) { *a = 1; ++fresh; }
            }
        }
    return fresh;
}

/* Integration, Eq. 2, over every allocated block.  D, Wt: 512 doubles per block of the box.
 * obs: observation count per block (+1 if any voxel of the block was updated).  fragile (nullable, 512 bytes per
 * block): voxels whose update hangs on a decision closer to its threshold than float arithmetic can resolve (pixel
 * rounding within 1e-3 px, eta + mu within 1e-5 mu ... of 0, a field-of-view or border test within its margin).
 * Returns the number of voxels updated. */
int64_t orc_tsdf_integrate(const orc_tsdf_box* B, const orc_camera* cam, const double R[9], const double t[3],
                           const double* depth, const uint8_t* allocated, double* D, double* Wt, int32_t* obs,
                           uint8_t* fragile) {
    int64_t updated = 0;
    const double vs = B->voxel_size;
    for (int bz = B->b0[2]; bz < B->b0[2] + B->nb[2]; ++bz)
        for (int by = B->b0[1]; by < B->b0[1] + B->nb[1]; ++by)
            for (int bx = B->b0[0]; bx < B->b0[0] + B->nb[0]; ++bx) {
                const size_t s = block_slot(B, bx, by, bz);
                if (!allocated[s]) continue;
                int any = 0;
                for (int k = 0; k < TSDF_BLOCK; ++k)
                    for (int j = 0; j < TSDF_BLOCK; ++j)
                        for (int i = 0; i < TSDF_BLOCK; ++i) {
                            const size_t v = s * 512 + (size_t)(k * 8 + j) * 8 + i;
                            const double X[3] = { ((double)bx * 8 + i + 0.5) * vs, ((double)by * 8 + j + 0.5) * vs,
                                                  ((double)bz * 8 + k + 0.5) * vs };
                            double Xd[3], uv[2];
                            for (int a = 0; a < 3; ++a) Xd[a] = R[3 * a] * X[0] + R[3 * a + 1] * X[1] + R[3 * a + 2] * X[2] + t[a];
                            const double range = sqrt(Xd[0] * Xd[0] + Xd[1] * Xd[1] + Xd[2] * Xd[2]);
                            const double th = atan2(sqrt(Xd[0] * Xd[0] + Xd[1] * Xd[1]), Xd[2]);
                            if (fragile && fabs(th - cam->theta_max) < 1e-5) fragile[v] = 1;
                            if (!orc_project(cam, Xd, uv)) continue; /* unified model */
                            const double pu = floor(uv[0] + 0.5), pv = floor(uv[1] + 0.5); /* nearest pixel */
                            if (fragile && (fabs(uv[0] + 0.5 - floor(uv[0] + 0.5 + 0.5)) < 1e-3 ||
                                            fabs(uv[1] + 0.5 - floor(uv[1] + 0.5 + 0.5)) < 1e-3)) fragile[v] = 1;
                            if (pu < 0.0 || pv < 0.0 || pu > cam->width - 1 || pv > cam->height - 1) continue;
                            const double d = depth[(size_t)pv * cam->width + (size_t)pu];
                            if (!(d > 0.0)) continue;
                            const double eta = d - range;
                            if (fragile && fabs(eta + B->mu) < 1e-5 * (B->mu + range)) fragile[v] = 1;
                            if (eta < -B->mu) continue; /* "not smaller than -mu" */
                            double sample = eta / B->mu;
                            if (sample > 1.0) sample = 1.0;
                            if (fragile && fabs(eta - B->mu) < 1e-5 * (B->mu + range)) fragile[v] = 1; /* clamp on / off: continuous, harmless */
                            D[v] = (Wt[v] * D[v] + sample) / (Wt[v] + 1.0);
                            Wt[v] = Wt[v] + 1.0 < (double)B->w_max ? Wt[v] + 1.0 : (double)B->w_max;
                            any = 1;
                            ++updated;
                        }
                if (any) obs[s] += 1;
            }
    return updated;
}

/* Points of the map ("only consider voxel blocks with at least 3 observations"; SPEC.md extract_points):
 * for every voxel of a block with obs >= min_obs and each of its +x, +y, +z neighbours (inside the box, in a block with
 * obs >= min_obs), a point where D changes sign between two voxels that both carry weight, placed by linear
 * interpolation of D.  points: up to cap * 3 doubles; returns the number found (may exceed cap). */
int64_t orc_tsdf_extract(const orc_tsdf_box* B, const uint8_t* allocated, const double* D, const double* Wt,
                         const int32_t* obs, int min_obs, double* points, int64_t cap) {
    int64_t n = 0;
    const double vs = B->voxel_size;
    const int nx = B->nb[0] * 8, ny = B->nb[1] * 8, nz = B->nb[2] * 8;
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                const size_t s0 = ((size_t)(z / 8) * B->nb[1] + (size_t)(y / 8)) * B->nb[0] + (size_t)(x / 8);
                if (!allocated[s0] || obs[s0] < min_obs) continue;
                const size_t v0 = s0 * 512 + (size_t)((z % 8) * 8 + (y % 8)) * 8 + (x % 8);
                if (!(Wt[v0] > 0.0)) continue;
                for (int a = 0; a < 3; ++a) {
                    const int x1 = x + (a == 0), y1 = y + (a == 1), z1 = z + (a == 2);
                    if (x1 >= nx || y1 >= ny || z1 >= nz) continue;
                    const size_t s1 = ((size_t)(z1 / 8) * B->nb[1] + (size_t)(y1 / 8)) * B->nb[0] + (size_t)(x1 / 8);
                    if (!allocated[s1] || obs[s1] < min_obs) continue;
                    const size_t v1 = s1 * 512 + (size_t)((z1 % 8) * 8 + (y1 % 8)) * 8 + (x1 % 8);
                    if (!(Wt[v1] > 0.0)) continue;
                    const double d0 = D[v0], d1 = D[v1];
                    if (!((d0 > 0.0 && d1 < 0.0) || (d0 < 0.0 && d1 > 0.0))) continue;
                    const double f = d0 / (d0 - d1); /* zero of the linear interpolant between the two centres */
                    if (n < cap) {
                        points[3 * n + 0] = ((double)B->b0[0] * 8 + x + 0.5 + (a == 0 ? f : 0.0)) * vs;
                        points[3 * n + 1] = ((double)B->b0[1] * 8 + y + 0.5 + (a == 1 ? f : 0.0)) * vs;
                        points[3 * n + 2] = ((double)B->b0[2] * 8 + z + 0.5 + (a == 2 ? f : 0.0)) * vs;
                    }
                    ++n;
                }
            }
    return n;
}
