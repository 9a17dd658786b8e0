// ib_tiled.cu -- variant 1 of spread/interp: points sorted by Eulerian cell, shared-memory halo tile.
#include "ib_common.cuh"

ib_status ibk_tiled_spread_interp(ib_ctx *c, const double *xp, const double *Gp, int64_t P,
                                  const double *u, const double *v, const double *w,
                                  double *fu, double *fv, double *fw, double *Up, cudaStream_t st)
{
    (void)c; (void)xp; (void)Gp; (void)P; (void)u; (void)v; (void)w; (void)fu; (void)fv; (void)fw; (void)Up; (void)st;
    return IB_ERR_UNSUPPORTED;
}
