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
// group hit 4 consecutive faces, so a warp's RED or load touches 8-16 sectors instead of 32 (the direct path
// of the sparse tiles is bound by L2 reduction traffic, not by arithmetic; every lane recomputes the weights).
// All 4 lanes must call; qmask = the group's lanes.  U is complete in every lane of the group.
template <int DO_SPREAD, int DO_INTERP>
__device__ __forceinline__ void ib_point_quad(double x, double y, double z, const double G[3],
                                              const double *const fld[3], double *const frc[3],
                                              const ib_grid_desc &g, double inv_h, int q, unsigned qmask, double U[3])
{
    ib_stencil s;
    ib_axis(x, g.x0, g.h, inv_h, g.nx, g.periodic, s.ix, s.wx);
    ib_axis(y, g.y0, g.h, inv_h, g.ny, g.periodic, s.iy, s.wy);
    ib_axis(z, g.z0, g.h, inv_h, g.nz, g.periodic, s.iz, s.wz);
    int ixq[2];
    double wxq[2];
#pragma unroll
    for (int o = 0; o < 2; ++o) {                       // selects, not indexing: the arrays stay in registers
        ixq[o] = q == 0 ? s.ix[o][0] : q == 1 ? s.ix[o][1] : q == 2 ? s.ix[o][2] : s.ix[o][3];
        wxq[o] = q == 0 ? s.wx[o][0] : q == 1 ? s.wx[o][1] : q == 2 ? s.wx[o][2] : s.wx[o][3];
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const int ox = (c == 0) ? 0 : 1, oy = (c == 1) ? 0 : 1, oz = (c == 2) ? 0 : 1;
        const bool xin = ixq[ox] >= 0;
        const double gx = DO_SPREAD ? G[c] * wxq[ox] : 0.0;
        double acc = 0.0;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const double gk = gx * s.wz[oz][k];
            double ak = 0.0;
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                if (s.iz[oz][k] < 0 || s.iy[oy][j] < 0 || !xin) continue;           // outside a bounded grid
                const int64_t at = ((int64_t)s.iz[oz][k] * g.ny + s.iy[oy][j]) * g.nx + ixq[ox];
                if (DO_INTERP) ak = fma(__ldg(fld[c] + at), s.wy[oy][j], ak);
                if (DO_SPREAD) atomicAdd(frc[c] + at, gk * s.wy[oy][j]);
            }
            if (DO_INTERP) acc = fma(ak, s.wz[oz][k], acc);
        }
        if (DO_INTERP) {
            acc *= wxq[ox];
            acc += __shfl_xor_sync(qmask, acc, 1);
            acc += __shfl_xor_sync(qmask, acc, 2);
        }
        U[c] = acc;
    }
}
