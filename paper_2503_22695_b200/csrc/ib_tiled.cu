// ib_tiled.cu -- variant 1 of spread (Eq.(24)-(26)) and interpolation (Eq.(27)-(29)):
// points sorted by Eulerian half-cell, one CTA per 4x4x4-cell tile with an 8x8x8 shared-memory halo
// of u,v,w and of the force accumulators, register-resident 4x4x4 stencil slabs.
//
// Why half-cells: component c lives on its own staggered lattice (MAC grid, L205).  In the
// direction d == c the 4-point support of a point is fixed by its cell; in the other two it is
// fixed by the cell of the lattice shifted by h/2.  Sorting by half-cell ("octant cell", 8^3 per
// tile) makes every cell of every shifted lattice a union of <= 4 contiguous runs of the sorted
// order, so all points of one work item (shifted cell, component) share ONE 4x4x4 window.
//
// Work item = (shifted cell, component).  A group of 4 lanes owns it: lane q keeps the z-plane q of
// the window -- 16 velocity values and 16 force accumulators -- in registers and loops over the
// item's points.  Per point and lane: 21 DFMA for interpolation (+2 shuffle-adds), 21 for
// spreading; the delta weights of 4 points are computed by the 4 lanes (one point each, one sqrt
// per 1-D weight set) and exchanged through a 464-byte shared-memory staging record.  Force is
// reduced in registers over all points of the item, then in shared memory over the items of the
// tile (fp64 CAS adds: Blackwell has no native shared fp64 add), then ONE global RED.ADD.F64 per
// touched face of the halo (coalesced rows of 8).
#include "ib_common.cuh"

#define TT 4                    // tile edge in cells
#define TH 8                    // halo edge
#define TH3 512
#define NOC 512                 // half-cells per tile (8^3)
#define NITEM 300               // 3 components x (4*5*5) shifted cells
#define TB 128                  // threads per CTA
#define NWARP (TB / 32)
#define REC 14                  // staging record: wx[4] wy[4] wz[4] G pad (doubles)
#define GSTRIDE 58              // doubles per group staging block (4 records = 56, +2: bank spread, 16B aligned)
#define NBIN 66

struct ib_tiled_params {
    const double *xp, *Gp;
    int64_t P;
    const double *fld[3];
    double *frc[3];
    double *Up;
    const uint32_t *skey;
    const int32_t *perm;
    const int32_t *tile_start;
    const int32_t *tile_list;
    int32_t *counters;          // [0] number of non-empty tiles, [1] work counter
    ib_grid_desc g;
    double inv_h, ih3;
    long long *status;
};

// internal sort key: tile4-major, half-cell (8^3) within the tile
__global__ void __launch_bounds__(256)
ibk_keys_half(int64_t P, const double *__restrict__ xp, ib_grid_desc g, double inv_h,
              uint32_t *__restrict__ key32, long long *status)
{
    int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= P) return;
    double x[3] = {__ldg(xp + p), __ldg(xp + P + p), __ldg(xp + 2 * P + p)};
    const double org[3] = {g.x0, g.y0, g.z0};
    const int n[3] = {g.nx, g.ny, g.nz};
    if (!(isfinite(x[0]) && isfinite(x[1]) && isfinite(x[2]))) {
        ib_latch(status, IB_ERR_NONFINITE, p);
        x[0] = org[0]; x[1] = org[1]; x[2] = org[2];
    }
    int h2[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        double sc = __dmul_rn(__dsub_rn(x[d], org[d]), inv_h);
        long long c2 = (long long)floor(2.0 * sc);
        c2 %= 2 * n[d];
        if (c2 < 0) c2 += 2 * n[d];
        h2[d] = (int)c2;
    }
    int ntx = g.nx / TT, nty = g.ny / TT;
    uint32_t t = (uint32_t)(((h2[2] >> 3) * nty + (h2[1] >> 3)) * ntx + (h2[0] >> 3));
    uint32_t l = (uint32_t)((((h2[2] & 7) << 3) | (h2[1] & 7)) << 3 | (h2[0] & 7));
    key32[p] = t * NOC + l;
}

__global__ void __launch_bounds__(256)
ibk_tile_compact(const int32_t *__restrict__ tile_start, int n_tiles, int32_t *__restrict__ tile_list,
                 int32_t *__restrict__ counters)
{
    int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n_tiles) return;
    if (tile_start[t + 1] > tile_start[t]) tile_list[atomicAdd(&counters[0], 1)] = t;
}

// decode a work item: component c, shifted-cell coordinates l[3]
__device__ __forceinline__ void ib_item_decode(int it, int &c, int l[3])
{
    c = it / 100;
    int r = it - c * 100;
    int nx = (c == 0) ? 4 : 5, ny = (c == 1) ? 4 : 5;
    l[0] = r % nx;
    l[1] = (r / nx) % ny;
    l[2] = r / (nx * ny);
}

// half-cell range [lo,hi] (clipped to the tile) covered by shifted cell l in direction d of comp c
__device__ __forceinline__ void ib_half_range(int c, int d, int l, int &lo, int &hi)
{
    if (d == c) { lo = 2 * l; hi = 2 * l + 1; }
    else { lo = max(2 * l - 1, 0); hi = min(2 * l, 7); }
}

template <int DO_SPREAD, int DO_INTERP>
__global__ void __launch_bounds__(TB, 4)
ibk_tiled_kernel(ib_tiled_params pr)
{
    extern __shared__ __align__(16) double smem[];
    double *su = smem;                                   // [3][512]
    double *sf = su + 3 * TH3;                           // [3][512]
    double *stg = sf + 3 * TH3;                          // [NWARP*8][GSTRIDE]
    int *oc_start = (int *)(stg + NWARP * 8 * GSTRIDE);  // [513]
    int *item_cnt = oc_start + NOC + 1;                  // [NITEM]
    int *order = item_cnt + NITEM;                       // [NITEM]
    int *bins = order + NITEM;                           // [NBIN]
    __shared__ int s_tile, s_nitems;

    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int grp = lane >> 2, q = lane & 3;
    const unsigned gmask = 0xFu << (lane & ~3);
    const int n[3] = {pr.g.nx, pr.g.ny, pr.g.nz};
    const double org[3] = {pr.g.x0, pr.g.y0, pr.g.z0};
    const int ntx = n[0] / TT, nty = n[1] / TT;
    const int64_t P = pr.P;

    for (;;) {
        if (tid == 0) s_tile = atomicAdd(&pr.counters[1], 1);
        __syncthreads();
        const int ti = s_tile;
        if (ti >= pr.counters[0]) break;
        const int tile = __ldg(pr.tile_list + ti);
        const int beg = __ldg(pr.tile_start + tile), end = __ldg(pr.tile_start + tile + 1);
        const int t3[3] = {tile % ntx, (tile / ntx) % nty, tile / (ntx * nty)};
        // halo origin (global index of halo entry 0), wrapped
        int h0[3];
#pragma unroll
        for (int d = 0; d < 3; ++d) h0[d] = ib_wrap(TT * t3[d] - 2, n[d]);

        // ---- phase 0: halo load, zero accumulators and counters -------------------------------
        for (int i = tid; i <= NOC; i += TB) oc_start[i] = 0;
        for (int i = tid; i < NBIN; i += TB) bins[i] = 0;
        for (int idx = tid; idx < 3 * TH3; idx += TB) {
            if (DO_SPREAD) sf[idx] = 0.0;
            if (DO_INTERP) {
                int c = idx >> 9, r = idx & 511;
                int i = h0[0] + (r & 7), j = h0[1] + ((r >> 3) & 7), k = h0[2] + (r >> 6);
                i -= (i >= n[0]) ? n[0] : 0; j -= (j >= n[1]) ? n[1] : 0; k -= (k >= n[2]) ? n[2] : 0;
                su[idx] = __ldg(pr.fld[c] + ((int64_t)k * n[1] + j) * n[0] + i);
            }
        }
        __syncthreads();
        // ---- phase 1: points per half-cell, exclusive scan -------------------------------------
        for (int r = beg + tid; r < end; r += TB) atomicAdd(&oc_start[__ldg(pr.skey + r) & (NOC - 1)], 1);
        __syncthreads();
        {
            int v0 = oc_start[4 * tid], v1 = oc_start[4 * tid + 1], v2 = oc_start[4 * tid + 2], v3 = oc_start[4 * tid + 3];
            int s = v0 + v1 + v2 + v3, inc = s;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                int t = __shfl_up_sync(0xffffffffu, inc, o);
                if (lane >= o) inc += t;
            }
            __shared__ int wsum[NWARP];
            if (lane == 31) wsum[wid] = inc;
            __syncthreads();
            int off = 0;
            for (int w = 0; w < wid; ++w) off += wsum[w];
            int ex = off + inc - s;
            oc_start[4 * tid] = ex; oc_start[4 * tid + 1] = ex + v0; oc_start[4 * tid + 2] = ex + v0 + v1;
            oc_start[4 * tid + 3] = ex + v0 + v1 + v2;
            if (tid == TB - 1) oc_start[NOC] = ex + s;
        }
        __syncthreads();
        // ---- phase 2: points per work item, order items by count (descending) ------------------
        for (int it = tid; it < NITEM; it += TB) {
            int c, l[3], lo[3], hi[3];
            ib_item_decode(it, c, l);
#pragma unroll
            for (int d = 0; d < 3; ++d) ib_half_range(c, d, l[d], lo[d], hi[d]);
            int cnt = 0;
            for (int z2 = lo[2]; z2 <= hi[2]; ++z2)
                for (int y2 = lo[1]; y2 <= hi[1]; ++y2) {
                    int b = (z2 * 8 + y2) * 8;
                    cnt += oc_start[b + hi[0] + 1] - oc_start[b + lo[0]];
                }
            item_cnt[it] = cnt;
            atomicAdd(&bins[min(cnt, NBIN - 1)], 1);
        }
        __syncthreads();
        if (wid == 0) {                       // descending exclusive scan of the bins (bin 0 dropped)
            int carry = 0;
            for (int b0 = NBIN - 1; b0 >= 1; b0 -= 32) {
                int b = b0 - lane;
                int v = (b >= 1) ? bins[b] : 0, inc = v;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    int t = __shfl_up_sync(0xffffffffu, inc, o);
                    if (lane >= o) inc += t;
                }
                if (b >= 1) bins[b] = carry + inc - v;
                carry += __shfl_sync(0xffffffffu, inc, 31);
            }
            if (lane == 0) s_nitems = carry;
        }
        __syncthreads();
        for (int it = tid; it < NITEM; it += TB) {
            int cnt = item_cnt[it];
            if (cnt > 0) order[atomicAdd(&bins[min(cnt, NBIN - 1)], 1)] = it;
        }
        __syncthreads();
        const int nitems = s_nitems;

        // ---- phase 3: the items ----------------------------------------------------------------
        double *mystg = stg + (wid * 8 + grp) * GSTRIDE;
        for (int base = wid * 8; base < nitems; base += NWARP * 8) {
            const int wi = base + grp;
            const bool have = wi < nitems;
            int c = 0, l[3] = {0, 0, 0};
            if (have) ib_item_decode(order[wi], c, l);
            // runs of the sorted order that make up this item
            int rstart[4], rend[4], npts = 0;
            {
                int lo[3], hi[3];
#pragma unroll
                for (int d = 0; d < 3; ++d) ib_half_range(c, d, l[d], lo[d], hi[d]);
#pragma unroll
                for (int rr = 0; rr < 4; ++rr) {
                    int z2 = lo[2] + (rr >> 1), y2 = lo[1] + (rr & 1);
                    bool ok = have && z2 <= hi[2] && y2 <= hi[1];
                    int b = (z2 * 8 + y2) * 8;
                    int s0 = ok ? oc_start[b + lo[0]] : 0, s1 = ok ? oc_start[b + hi[0] + 1] : 0;
                    rstart[rr] = s0 - npts;          // rank = rstart + virtual index
                    npts += s1 - s0;
                    rend[rr] = npts;                 // virtual indices < rend belong to runs <= rr
                }
            }
            int nmax = npts;
#pragma unroll
            for (int o = 16; o >= 4; o >>= 1) nmax = max(nmax, __shfl_xor_sync(0xffffffffu, nmax, o));
            // window origin inside the halo, expected wrapped global index of window entry 1
            int o3[3], e3[3];
            double off3[3];
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                o3[d] = l[d] + ((d == c) ? 1 : 0);
                off3[d] = (d == c) ? 0.0 : 0.5;
                int e = h0[d] + o3[d] + 1;
                e3[d] = e >= n[d] ? e - n[d] : e;
            }
            const double *suc = su + c * TH3 + ((o3[2] + q) * TH + o3[1]) * TH + o3[0];
            double *sfc = sf + c * TH3 + ((o3[2] + q) * TH + o3[1]) * TH + o3[0];
            double uu[4][4], ff[4][4];
#pragma unroll
            for (int j = 0; j < 4; ++j)
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    uu[j][i] = DO_INTERP ? suc[j * TH + i] : 0.0;
                    ff[j][i] = 0.0;
                }
            const double *Gc = DO_SPREAD ? pr.Gp + (int64_t)c * P : nullptr;
            double *Uc = DO_INTERP ? pr.Up + (int64_t)c * P : nullptr;

            for (int r0 = 0; r0 < nmax; r0 += 4) {
                // -- lane q prepares point r0+q: delta weights of the 3 directions on comp c's lattice
                const int vi = r0 + q;
                const bool valid = vi < npts;
                int rank = vi + ((vi < rend[0]) ? rstart[0] : (vi < rend[1]) ? rstart[1] : (vi < rend[2]) ? rstart[2] : rstart[3]);
                int id = valid ? __ldg(pr.perm + beg + rank) : 0;
                double wgt[3][4];
#pragma unroll
                for (int d = 0; d < 3; ++d) {
                    double xd = __ldg(pr.xp + (int64_t)d * P + id);
                    double s = ib_scaled(xd, org[d], pr.g.h, pr.inv_h) - off3[d];
                    double fl = floor(s);
                    double r = s - fl;
                    // binning and weights round differently at exact cell boundaries: re-express r
                    // relative to the item's window and clamp (phi is continuous, A19)
                    // (grid dims are multiples of 8, so the index difference mod 8 tells -1/0/+1 apart)
                    int dm = ((int)fl - e3[d]) & 7;
                    r += (dm == 1) ? 1.0 : ((dm == 7) ? -1.0 : 0.0);
                    r = fmin(fmax(r, 0.0), 1.0);
                    ib_phi4(r, wgt[d]);
                }
                double Gv = (DO_SPREAD && valid) ? __ldg(Gc + id) * pr.ih3 : 0.0;
                if (!valid) {
#pragma unroll
                    for (int m = 0; m < 4; ++m) wgt[2][m] = 0.0;
                }
                double *rec = mystg + q * REC;
                *reinterpret_cast<double2 *>(rec + 0) = make_double2(wgt[0][0], wgt[0][1]);
                *reinterpret_cast<double2 *>(rec + 2) = make_double2(wgt[0][2], wgt[0][3]);
                *reinterpret_cast<double2 *>(rec + 4) = make_double2(wgt[1][0], wgt[1][1]);
                *reinterpret_cast<double2 *>(rec + 6) = make_double2(wgt[1][2], wgt[1][3]);
                *reinterpret_cast<double2 *>(rec + 8) = make_double2(wgt[2][0], wgt[2][1]);
                *reinterpret_cast<double2 *>(rec + 10) = make_double2(wgt[2][2], wgt[2][3]);
                rec[12] = Gv;
                __syncwarp();
#pragma unroll
                for (int jp = 0; jp < 4; ++jp) {
                    const double *rj = mystg + jp * REC;
                    double2 a0 = *reinterpret_cast<const double2 *>(rj + 0), a1 = *reinterpret_cast<const double2 *>(rj + 2);
                    double2 b0 = *reinterpret_cast<const double2 *>(rj + 4), b1 = *reinterpret_cast<const double2 *>(rj + 6);
                    const double wx[4] = {a0.x, a0.y, a1.x, a1.y}, wy[4] = {b0.x, b0.y, b1.x, b1.y};
                    const double wz = rj[8 + q];
                    if (DO_INTERP) {
                        double acc = 0.0;
#pragma unroll
                        for (int j = 0; j < 4; ++j) {
                            double rr = uu[j][0] * wx[0];
                            rr = fma(uu[j][1], wx[1], rr);
                            rr = fma(uu[j][2], wx[2], rr);
                            rr = fma(uu[j][3], wx[3], rr);
                            acc = fma(rr, wy[j], acc);
                        }
                        double pv = acc * wz;
                        pv += __shfl_xor_sync(0xffffffffu, pv, 1);
                        pv += __shfl_xor_sync(0xffffffffu, pv, 2);
                        int idj = __shfl_sync(0xffffffffu, id, (lane & ~3) + jp);
                        if (q == 0 && r0 + jp < npts) Uc[idj] = pv;
                    }
                    if (DO_SPREAD) {
                        double gz = rj[12] * wz;
#pragma unroll
                        for (int j = 0; j < 4; ++j) {
                            double gj = gz * wy[j];
#pragma unroll
                            for (int i = 0; i < 4; ++i) ff[j][i] = fma(gj, wx[i], ff[j][i]);
                        }
                    }
                }
                __syncwarp();
            }
            if (DO_SPREAD && have) {
#pragma unroll
                for (int j = 0; j < 4; ++j)
#pragma unroll
                    for (int i = 0; i < 4; ++i) atomicAdd(sfc + j * TH + i, ff[j][i]);
            }
        }
        __syncthreads();
        // ---- phase 4: one global reduction per touched face of the halo ------------------------
        if (DO_SPREAD) {
            for (int idx = tid; idx < 3 * TH3; idx += TB) {
                double val = sf[idx];
                if (val != 0.0) {
                    int c = idx >> 9, r = idx & 511;
                    int i = h0[0] + (r & 7), j = h0[1] + ((r >> 3) & 7), k = h0[2] + (r >> 6);
                    i -= (i >= n[0]) ? n[0] : 0; j -= (j >= n[1]) ? n[1] : 0; k -= (k >= n[2]) ? n[2] : 0;
                    atomicAdd(pr.frc[c] + ((int64_t)k * n[1] + j) * n[0] + i, val);
                }
            }
        }
        __syncthreads();
    }
    (void)gmask;
}

// ---- radix sort plumbing shared with ib_binsort.cu ---------------------------------------------
ib_status ibk_sort_keys_inplace(ib_ctx *c, int64_t P, int bits, cudaStream_t st);
__global__ void ibk_tile_starts_shift(const uint32_t *__restrict__ skeys, int64_t P, int n_tiles, int shift,
                                      int32_t *__restrict__ tile_start);

template <int S, int I>
static ib_status launch_tiled(ib_ctx *c, const ib_tiled_params &pr, cudaStream_t st)
{
    static int configured = 0;
    const size_t smem = (size_t)(6 * TH3 + NWARP * 8 * GSTRIDE) * sizeof(double) + (NOC + 1 + 2 * NITEM + NBIN + 3) * sizeof(int);
    if (!configured) {
        IB_CUDA_TRY(cudaFuncSetAttribute(ibk_tiled_kernel<S, I>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        configured = 1;
    }
    cudaDeviceProp prop;
    static int sms = 0;
    if (!sms) {
        IB_CUDA_TRY(cudaGetDeviceProperties(&prop, c->device));
        sms = prop.multiProcessorCount;
    }
    ibk_tiled_kernel<S, I><<<sms * 4, TB, smem, st>>>(pr);
    c->launches++;
    return IB_OK;
}

ib_status ibk_tiled_spread_interp(ib_ctx *c, const double *xp, const double *Gp, int64_t P,
                                  const double *u, const double *v, const double *w,
                                  double *fu, double *fv, double *fw, double *Up, cudaStream_t st)
{
    ib_status rs = ibk_sort_reserve(c, P);
    if (rs != IB_OK) return rs;
    const int n_tiles = (int)(c->n_cells / (TT * TT * TT));
    ib_prof_begin(c, IB_PHASE_SORT, st);
    ibk_keys_half<<<ib_blocks(P, 256), 256, 0, st>>>(P, xp, c->grid, c->inv_h, c->d_key[0], c->d_status);
    c->launches++;
    int bits = 1;
    while ((1ll << bits) < (int64_t)n_tiles * NOC) ++bits;
    rs = ibk_sort_keys_inplace(c, P, bits, st);
    if (rs != IB_OK) return rs;
    IB_CUDA_TRY(cudaMemsetAsync(c->d_tile_count, 0, 2 * sizeof(int32_t), st));
    ibk_tile_starts_shift<<<ib_blocks(P + 1, 256), 256, 0, st>>>(c->d_key[0], P, n_tiles, 9, c->d_cell_start);
    ibk_tile_compact<<<ib_blocks(n_tiles, 256), 256, 0, st>>>(c->d_cell_start, n_tiles, c->d_tile_list, c->d_tile_count);
    c->launches += 2;
    ib_prof_end(c, IB_PHASE_SORT, st);

    ib_tiled_params pr;
    pr.xp = xp; pr.Gp = Gp; pr.P = P;
    pr.fld[0] = u; pr.fld[1] = v; pr.fld[2] = w;
    pr.frc[0] = fu; pr.frc[1] = fv; pr.frc[2] = fw;
    pr.Up = Up;
    pr.skey = c->d_key[0]; pr.perm = c->d_val[0];
    pr.tile_start = c->d_cell_start; pr.tile_list = c->d_tile_list; pr.counters = c->d_tile_count;
    pr.g = c->grid; pr.inv_h = c->inv_h; pr.ih3 = c->inv_h * c->inv_h * c->inv_h;
    pr.status = c->d_status;
    ib_prof_begin(c, IB_PHASE_SPREAD_INTERP, st);
    if (Gp && Up) rs = launch_tiled<1, 1>(c, pr, st);
    else if (Gp) rs = launch_tiled<1, 0>(c, pr, st);
    else rs = launch_tiled<0, 1>(c, pr, st);
    ib_prof_end(c, IB_PHASE_SPREAD_INTERP, st);
    if (rs != IB_OK) return rs;
    IB_CUDA_TRY(cudaGetLastError());
    return IB_OK;
}
