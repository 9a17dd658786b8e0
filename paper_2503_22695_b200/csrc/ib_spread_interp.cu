// ib_spread_interp.cu -- spreading (Eq.(24)-(26) L211-217, L253-257) and interpolation
// (Eq.(27)-(29) L222-229, L243-247) on the MAC grid with the Peskin 4-point delta (L52 -> ref.1).
//   f_c[i0+m] += G_{s,c} phi(s1-i0_1-m1) phi(..) phi(..) / h^3 ,   U_{s,c} = sum_m u_c[i0+m] phi phi phi
// component c on its own staggered lattice, offsets u (0,1/2,1/2), v (1/2,0,1/2), w (1/2,1/2,0).
//
// variant 0 (this file, ibk_point_*): one thread per point, weights in registers, sum-factorised
//   contraction, grid read through L1/L2, spread with native fp64 global reductions (RED.ADD.F64).
// variant 1 (ib_tiled.cu): points sorted by Eulerian cell, shared-memory halo tile per 8^3 tile.
#include "ib_common.cuh"

struct ib_stencil {
    int ix[2][4], iy[2][4], iz[2][4];      // wrapped indices, [0] face-aligned, [1] centre-aligned
    double wx[2][4], wy[2][4], wz[2][4];
};

__device__ __forceinline__ void ib_axis(double x, double x0, double h, double inv_h, int n,
                                        int idx[2][4], double wt[2][4])
{
    double sf = ib_scaled(x, x0, h, inv_h);
#pragma unroll
    for (int o = 0; o < 2; ++o) {
        double s = o ? sf - 0.5 : sf;
        double fl = floor(s);
        ib_phi4(s - fl, wt[o]);
        int i0 = ib_wrap((int)fl - 1, n);
#pragma unroll
        for (int m = 0; m < 4; ++m) {
            int i = i0 + m;
            idx[o][m] = i >= n ? i - n : i;
        }
    }
}

template <int DO_SPREAD, int DO_INTERP>
__global__ void __launch_bounds__(128)
ibk_point_kernel(int64_t P, const double *__restrict__ xp, const double *__restrict__ Gp,
                 const double *__restrict__ u, const double *__restrict__ v, const double *__restrict__ w,
                 double *__restrict__ fu, double *__restrict__ fv, double *__restrict__ fw,
                 double *__restrict__ Up, ib_grid_desc g, double inv_h, long long *status)
{
    int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= P) return;
    double x = __ldg(xp + p), y = __ldg(xp + P + p), z = __ldg(xp + 2 * P + p);
    if (!(isfinite(x) && isfinite(y) && isfinite(z))) {
        ib_latch(status, IB_ERR_NONFINITE, p);
        if (DO_INTERP) { Up[p] = 0.0; Up[P + p] = 0.0; Up[2 * P + p] = 0.0; }
        return;
    }
    ib_stencil s;
    ib_axis(x, g.x0, g.h, inv_h, g.nx, s.ix, s.wx);
    ib_axis(y, g.y0, g.h, inv_h, g.ny, s.iy, s.wy);
    ib_axis(z, g.z0, g.h, inv_h, g.nz, s.iz, s.wz);
    const double ih3 = inv_h * inv_h * inv_h;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const int ox = (c == 0) ? 0 : 1, oy = (c == 1) ? 0 : 1, oz = (c == 2) ? 0 : 1;
        const double *fld = (c == 0) ? u : (c == 1) ? v : w;
        double *frc = (c == 0) ? fu : (c == 1) ? fv : fw;
        double Gc = DO_SPREAD ? __ldg(Gp + c * P + p) * ih3 : 0.0;
        double acc = 0.0;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            double gk = Gc * s.wz[oz][k];
            double ak = 0.0;
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                int64_t row = ((int64_t)s.iz[oz][k] * g.ny + s.iy[oy][j]) * g.nx;
                if (DO_INTERP) {
                    double r = 0.0;
#pragma unroll
                    for (int i = 0; i < 4; ++i) r = fma(__ldg(fld + row + s.ix[ox][i]), s.wx[ox][i], r);
                    ak = fma(r, s.wy[oy][j], ak);
                }
                if (DO_SPREAD) {
                    double gjk = gk * s.wy[oy][j];
#pragma unroll
                    for (int i = 0; i < 4; ++i) atomicAdd(frc + row + s.ix[ox][i], gjk * s.wx[ox][i]);
                }
            }
            if (DO_INTERP) acc = fma(ak, s.wz[oz][k], acc);
        }
        if (DO_INTERP) Up[c * P + p] = acc;
    }
}

ib_status ibk_spread_interp(ib_ctx *c, const double *xp, const double *Gp, int64_t P,
                            const double *u, const double *v, const double *w,
                            double *fu, double *fv, double *fw, double *Up, int accumulate,
                            cudaStream_t st)
{
    const bool sp = Gp != nullptr, in = Up != nullptr;
    if (sp && !accumulate) {
        size_t nb = (size_t)c->n_cells * sizeof(double);
        ib_prof_begin(c, IB_PHASE_ZERO, st);
        IB_CUDA_TRY(cudaMemsetAsync(fu, 0, nb, st));
        IB_CUDA_TRY(cudaMemsetAsync(fv, 0, nb, st));
        IB_CUDA_TRY(cudaMemsetAsync(fw, 0, nb, st));
        ib_prof_end(c, IB_PHASE_ZERO, st);
    }
    if (P == 0) return IB_OK;
    if (c->variant == 1) return ibk_tiled_spread_interp(c, 0, xp, Gp, P, nullptr, nullptr, u, v, w, fu, fv, fw, Up, 0, st);
    unsigned nb = ib_blocks(P, 128);
    ib_prof_begin(c, IB_PHASE_SPREAD_INTERP, st);
    if (sp && in)
        ibk_point_kernel<1, 1><<<nb, 128, 0, st>>>(P, xp, Gp, u, v, w, fu, fv, fw, Up, c->grid, c->inv_h, c->d_status);
    else if (sp)
        ibk_point_kernel<1, 0><<<nb, 128, 0, st>>>(P, xp, Gp, u, v, w, fu, fv, fw, Up, c->grid, c->inv_h, c->d_status);
    else if (in)
        ibk_point_kernel<0, 1><<<nb, 128, 0, st>>>(P, xp, Gp, u, v, w, fu, fv, fw, Up, c->grid, c->inv_h, c->d_status);
    ib_prof_end(c, IB_PHASE_SPREAD_INTERP, st);
    c->launches++;
    IB_CUDA_TRY(cudaGetLastError());
    return IB_OK;
}
