// ib_spread_interp.cu -- spreading (Eq.(24)-(26) L211-217, L253-257) and interpolation
// (Eq.(27)-(29) L222-229, L243-247) on the MAC grid with the Peskin 4-point delta (L52 -> ref.1).
//   f_c[i0+m] += G_{s,c} phi(s1-i0_1-m1) phi(..) phi(..) / h^3 ,   U_{s,c} = sum_m u_c[i0+m] phi phi phi
// component c on its own staggered lattice, offsets u (0,1/2,1/2), v (1/2,0,1/2), w (1/2,1/2,0).
//
// variant 0 (this file, ibk_point_*): one thread per point, weights in registers, sum-factorised
//   contraction, grid read through L1/L2, spread with native fp64 global reductions (RED.ADD.F64).
// variant 1 (ib_tiled.cu): points sorted by Eulerian cell, shared-memory halo tile per 8^3 tile.
#include "ib_point.cuh"

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
    if (!g.periodic && !ib_in_box(x, y, z, g, inv_h)) {
        ib_latch(status, IB_ERR_OUT_OF_DOMAIN, p);
        if (DO_INTERP) { Up[p] = 0.0; Up[P + p] = 0.0; Up[2 * P + p] = 0.0; }
        return;
    }
    const double ih3 = inv_h * inv_h * inv_h;
    double G[3] = {0, 0, 0}, U[3];
    if (DO_SPREAD) { G[0] = __ldg(Gp + p) * ih3; G[1] = __ldg(Gp + P + p) * ih3; G[2] = __ldg(Gp + 2 * P + p) * ih3; }
    const double *const fld[3] = {u, v, w};
    double *const frc[3] = {fu, fv, fw};
    ib_point_direct<DO_SPREAD, DO_INTERP>(x, y, z, G, fld, frc, g, inv_h, U);
    if (DO_INTERP) { Up[p] = U[0]; Up[P + p] = U[1]; Up[2 * P + p] = U[2]; }
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
