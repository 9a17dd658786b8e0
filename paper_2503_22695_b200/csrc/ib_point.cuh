// ib_point.cuh -- one point against the grid, no shared memory: delta weights in registers,
// sum-factorised contraction, grid read through L1/L2, spread with native fp64 global reductions.
// Used by variant 0 (ib_spread_interp.cu) and for the points of sparsely filled tiles (ib_tiled.cu).
#pragma once
#include "ib_common.cuh"

struct ib_stencil {
    int ix[2][4], iy[2][4], iz[2][4];      // wrapped indices, [0] face-aligned, [1] centre-aligned
    double wx[2][4], wy[2][4], wz[2][4];
};

// periodic == 0: faces outside 0..n-1 do not exist (index -1: skipped by the caller)
__device__ __forceinline__ void ib_axis(double x, double x0, double h, double inv_h, int n, int periodic,
                                        int idx[2][4], double wt[2][4])
{
    double sf = ib_scaled(x, x0, h, inv_h);
#pragma unroll
    for (int o = 0; o < 2; ++o) {
        double s = o ? sf - 0.5 : sf;
        double fl = floor(s);
        ib_phi4(s - fl, wt[o]);
        if (periodic) {
            int i0 = ib_wrap((int)fl - 1, n);
#pragma unroll
            for (int m = 0; m < 4; ++m) {
                int i = i0 + m;
                idx[o][m] = i >= n ? i - n : i;
            }
        } else {
#pragma unroll
            for (int m = 0; m < 4; ++m) {
                int i = (int)fl - 1 + m;
                idx[o][m] = (i < 0 || i >= n) ? -1 : i;
            }
        }
    }
}

// G[c] (already divided by h^3) is spread to frc[c]; U[c] receives the interpolated fld[c].
template <int DO_SPREAD, int DO_INTERP>
__device__ __forceinline__ void ib_point_direct(double x, double y, double z, const double G[3],
                                                const double *const fld[3], double *const frc[3],
                                                const ib_grid_desc &g, double inv_h, double U[3])
{
    ib_stencil s;
    ib_axis(x, g.x0, g.h, inv_h, g.nx, g.periodic, s.ix, s.wx);
    ib_axis(y, g.y0, g.h, inv_h, g.ny, g.periodic, s.iy, s.wy);
    ib_axis(z, g.z0, g.h, inv_h, g.nz, g.periodic, s.iz, s.wz);
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const int ox = (c == 0) ? 0 : 1, oy = (c == 1) ? 0 : 1, oz = (c == 2) ? 0 : 1;
        double acc = 0.0;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            double gk = DO_SPREAD ? G[c] * s.wz[oz][k] : 0.0;
            double ak = 0.0;
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                if (s.iz[oz][k] < 0 || s.iy[oy][j] < 0) continue;           // outside a bounded grid
                int64_t row = ((int64_t)s.iz[oz][k] * g.ny + s.iy[oy][j]) * g.nx;
                if (DO_INTERP) {
                    double r = 0.0;
#pragma unroll
                    for (int i = 0; i < 4; ++i)
                        if (s.ix[ox][i] >= 0) r = fma(__ldg(fld[c] + row + s.ix[ox][i]), s.wx[ox][i], r);
                    ak = fma(r, s.wy[oy][j], ak);
                }
                if (DO_SPREAD) {
                    double gjk = gk * s.wy[oy][j];
#pragma unroll
                    for (int i = 0; i < 4; ++i)
                        if (s.ix[ox][i] >= 0) atomicAdd(frc[c] + row + s.ix[ox][i], gjk * s.wx[ox][i]);
                }
            }
            if (DO_INTERP) acc = fma(ak, s.wz[oz][k], acc);
        }
        U[c] = acc;
    }
}

// The same with 4 lanes per point, lane q = the q-th face of every x-row of the support: the 4 lanes of a
// group hit 4 consecutive faces, so a warp's RED or load touches 8-16 sectors instead of 32 (the direct path of
// the sparse tiles is bound by L2 reduction traffic and by instruction issue).  Written for few instructions:
// the 1-D weight sets are kept as (a, q) pairs (ib_aq), every lane forms only its own x-weight, row and plane
// offsets are 32-bit and formed once per component, the component loop is unrolled so that the alignment of
// each direction is a compile-time choice.  PER: periodic grid (bounded: faces outside 0..n-1 are skipped).
// All 4 lanes must call; qmask = the group's lanes.  U is complete in every lane of the group.
struct ib_axis2 {
    int i0[2];                 // first face of the support, unwrapped: [0] face-aligned, [1] centre-aligned
    double2 aq[2];
};
__device__ __forceinline__ void ib_axis_aq(double x, double x0, double h, double inv_h, ib_axis2 &A)
{
    const double sf = ib_scaled(x, x0, h, inv_h);
#pragma unroll
    for (int o = 0; o < 2; ++o) {
        const double s = o ? sf - 0.5 : sf, fl = floor(s);
        A.i0[o] = (int)fl - 1;
        A.aq[o] = ib_aq(s - fl);
    }
}
// face m of a support starting at i0: index in 0..n-1, or -1 outside a bounded grid
template <int PER>
__device__ __forceinline__ int ib_face_index(int w0, int i0, int m, int n)
{
    if (PER) { const int i = w0 + m; return i >= n ? i - n : i; }       // w0 = i0 wrapped once
    const int i = i0 + m;
    return (i < 0 || i >= n) ? -1 : i;
}

template <int DO_SPREAD, int DO_INTERP, int PER>
__device__ __forceinline__ void ib_point_quad(double x, double y, double z, const double G[3],
                                              const double *const fld[3], double *const frc[3],
                                              const ib_grid_desc &g, double inv_h, int q, unsigned qmask, double U[3])
{
    ib_axis2 ax, ay, az;
    ib_axis_aq(x, g.x0, g.h, inv_h, ax);
    ib_axis_aq(y, g.y0, g.h, inv_h, ay);
    ib_axis_aq(z, g.z0, g.h, inv_h, az);
    // lane q's own x-weight from (a, q):  w = sg q + (sa a + ca)
    const double wsa = q < 2 ? 1.0 : -1.0, wca = q < 2 ? 0.0 : 0.5, wsg = (q == 1 || q == 2) ? 1.0 : -1.0;
    const int nxy = g.nx * g.ny;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const int ox = (c == 0) ? 0 : 1, oy = (c == 1) ? 0 : 1, oz = (c == 2) ? 0 : 1;
        const double wx = fma(wsg, ax.aq[ox].y, fma(wsa, ax.aq[ox].x, wca));
        const int ix = ib_face_index<PER>(PER ? ib_wrap(ax.i0[ox], g.nx) : 0, ax.i0[ox], q, g.nx);
        const int wy0 = PER ? ib_wrap(ay.i0[oy], g.ny) : 0, wz0 = PER ? ib_wrap(az.i0[oz], g.nz) : 0;
        const double ya = ay.aq[oy].x, yq = ay.aq[oy].y, za = az.aq[oz].x, zq = az.aq[oz].y;
        const double wy[4] = {ya - yq, ya + yq, (0.5 - ya) + yq, (0.5 - ya) - yq};
        const double wz[4] = {za - zq, za + zq, (0.5 - za) + zq, (0.5 - za) - zq};
        int offy[4], offz[4];                              // 32-bit face offsets (n_cells < 2^31); < 0: outside
#pragma unroll
        for (int m = 0; m < 4; ++m) {
            const int j = ib_face_index<PER>(wy0, ay.i0[oy], m, g.ny), k = ib_face_index<PER>(wz0, az.i0[oz], m, g.nz);
            offy[m] = (PER || j >= 0) ? j * g.nx + ix : -1;
            offz[m] = (PER || k >= 0) ? k * nxy : -1;
        }
        const bool xin = PER || ix >= 0;
        const double gx = DO_SPREAD ? G[c] * wx : 0.0;
        const double *fc = fld[c];
        double *rc = frc[c];
        double acc = 0.0;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const double gk = gx * wz[k];
            double ak = 0.0;
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                if (!PER && (!xin || offy[j] < 0 || offz[k] < 0)) continue;           // outside a bounded grid
                const unsigned at = (unsigned)(offz[k] + offy[j]);
                if (DO_INTERP) ak = fma(__ldg(fc + at), wy[j], ak);
                if (DO_SPREAD) atomicAdd(rc + at, gk * wy[j]);
            }
            if (DO_INTERP) acc = fma(ak, wz[k], acc);
        }
        if (DO_INTERP) {
            acc *= wx;
            acc += __shfl_xor_sync(qmask, acc, 1);
            acc += __shfl_xor_sync(qmask, acc, 2);
        }
        U[c] = acc;
    }
}
