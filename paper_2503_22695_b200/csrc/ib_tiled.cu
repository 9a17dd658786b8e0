// ib_tiled.cu -- variant 1 of spread (Eq.(24)-(26)) and interpolation (Eq.(27)-(29)):
// points grouped by 4x4x4-cell tile (ib_bin.cu); persistent CTAs pull chunks of one tile from a work
// list, keep an 8x8x8 halo of u,v,w in shared memory and hold 4x4x4 stencil windows in registers.
//
// Per chunk the CTA stages the tile-relative scaled coordinates of the points in shared memory and
// sorts them by half-cell ("octant", 8^3 per tile) with a shared-memory counting sort.  Why half-cells:
// component c lives on its own staggered lattice (MAC grid, L205).  In the direction d == c the
// 4-point support of a point is fixed by its cell; in the other two it is fixed by the cell of the
// lattice shifted by h/2.  With the points ordered by half-cell every cell of every shifted lattice is
// a union of <= 4 contiguous runs, so all points of one work item (shifted cell, component) share ONE
// 4x4x4 window.
//
// Work item = (shifted cell, component); items are ordered by point count and pulled by the warps, 8
// at a time.  A group of 4 lanes owns an item: lane q keeps the x-column q of the window -- 16
// velocity values and 16 force accumulators -- in registers and loops over the item's points in quads.
// Per point and lane: 21 DFMA for interpolation, 21 for spreading.  The delta weights of a quad are
// computed by the 4 lanes (one point each, one branch-free sqrt per 1-D weight set) into a
// double-buffered shared-memory record while the group consumes the previous quad; index, force and
// id of the quad after that are already in flight.  Force is reduced in registers over all points of
// the item and flushed with RED.ADD.F64 straight to the grid: the 4 lanes of a group hit 4 consecutive
// faces (Blackwell has no native shared-memory fp64 add; the CAS loop measured 34 wavefronts each).
// Tiles with fewer than IB_SMALL_TILE points skip all of this (ibk_small_tiles, ib_point.cuh).
#include "ib_point.cuh"

#define TT 4                    // tile edge in cells
#define TH 8                    // halo edge
#define TH3 512
#define NOC 512                 // half-cells per tile (8^3)
#define NITEM 300               // 3 components x (4*5*5) shifted cells
#define TB 192                  // threads per CTA (2 CTAs/SM at <= 168 registers)
#define NCTA 2
#define NWARP (TB / 32)
#define CH IB_CHUNK             // points staged per work item (9 per thread)
#define REC 14                  // staging record: wx[4] wy[4] wz[4] G pad (doubles)
#define GBUF 56                 // doubles per staging buffer of a group (4 records)
#define GSTRIDE 120             // doubles per group: two buffers + pad (60 16-byte units = 4 mod 8: conflict-free STS.128)
#define SZ 68                   // z-plane stride of the halo in doubles (64 + 4: the 4 lanes of a group hit distinct banks)
#define SU3 (TH * SZ)           // one component of the halo
#define NBIN 66

struct ib_tiled_params {
    const double *sx, *sG;      // [3][P] records grouped by tile
    const int32_t *sid;         // [P] point id of record
    int64_t P;
    const double *fld[3];
    double *frc[3];
    double *Up;
    const int4 *work;           // {tile, first record, points, 0} per chunk
    int32_t *counters;          // [0] number of work items, [1] work counter, [3] zero, [IB_SLAB0 + k] first item of slab k
    int wb, we, wc;             // this launch covers the work items counters[wb] <= w < counters[we]; counters[wc] counts them
    ib_grid_desc g;
    double inv_h, ih3;
};

// decode a work item: component c, shifted-cell coordinates l[3]  (c*100 + (l2*ny + l1)*nx + l0 with
// nx = 4 if c == 0 else 5, ny = 4 if c == 1 else 5; compile-time constant divisors only)
__device__ __forceinline__ void ib_item_decode(int it, int &c, int l[3])
{
    // written without branches: the compiler merges a three-way branch into selects of the DIVISORS and
    // then divides by a run-time value (three I2F/MUFU.RCP sequences per item in the SASS)
    c = it / 100;
    const int r = it - c * 100;
    const int q20 = r / 20, q25 = r / 25;
    l[2] = (c == 2) ? q25 : q20;
    const int rem = r - ((c == 2) ? 25 * q25 : 20 * q20);      // index in the z-plane: nx*ny = 20 or 25
    const int q5 = rem / 5;
    l[1] = (c == 0) ? (rem >> 2) : q5;
    l[0] = (c == 0) ? (rem & 3) : rem - 5 * q5;
}

// the same, packed into 11 bits for the sorted item list (the item loop unpacks instead of dividing)
__device__ __forceinline__ unsigned short ib_item_code(int it)
{
    int c, l[3];
    ib_item_decode(it, c, l);
    return (unsigned short)(c | (l[0] << 2) | (l[1] << 5) | (l[2] << 8));
}
__device__ __forceinline__ void ib_item_unpack(int code, int &c, int l[3])
{
    c = code & 3; l[0] = (code >> 2) & 7; l[1] = (code >> 5) & 7; l[2] = code >> 8;
}

// half-cell range [lo,hi] (clipped to the tile) covered by shifted cell l in direction d of comp c
__device__ __forceinline__ void ib_half_range(int c, int d, int l, int &lo, int &hi)
{
    if (d == c) { lo = 2 * l; hi = 2 * l + 1; }
    else { lo = max(2 * l - 1, 0); hi = min(2 * l, 7); }
}

// scaled coordinate of a point relative to the origin of its tile, xi in [0,4) up to rounding:
// s = (x-x0)/h to ~1 ulp; the tile is the one the binning formula (A21) assigned, so the integer
// part comes from that formula and only the fraction from s.
__device__ __forceinline__ double ib_tile_coord(double x, double x0, double h, double inv_h)
{
    double sc = __dmul_rn(__dsub_rn(x, x0), inv_h);
    double fl = floor(sc);
    // grid dims are multiples of 8, so the periodically wrapped cell index is congruent to the
    // unwrapped one modulo the tile edge 4
    return (ib_scaled(x, x0, h, inv_h) - fl) + (double)((long long)fl & (TT - 1));
}

__device__ __forceinline__ int ib_octant_key(double a, double b, double c)
{
    int hx = min(max((int)floor(2.0 * a), 0), 7), hy = min(max((int)floor(2.0 * b), 0), 7),
        hz = min(max((int)floor(2.0 * c), 0), 7);
    return (hz * 8 + hy) * 8 + hx;
}

__device__ __forceinline__ void ib_prefetch_l2(const void *p)
{
    asm volatile("prefetch.global.L2 [%0];" ::"l"(p));
}

// PER: periodic grid (compile-time, so that the periodic kernel carries none of the wall predicates)
template <int DO_SPREAD, int DO_INTERP, int PER>
__global__ void __launch_bounds__(TB, NCTA)
ibk_tiled_kernel(ib_tiled_params pr)
{
    extern __shared__ __align__(16) double smem[];
    double *su = smem;                                   // [3][8][SZ] halo of u,v,w
    double *sxi = su + 3 * SU3;                          // [3][CH] tile-relative scaled coordinates
    double *stg = sxi + 3 * CH;                          // [NWARP*8][GSTRIDE]
    int *oc_cur = (int *)(stg + NWARP * 8 * GSTRIDE);    // [512]
    int *bins = oc_cur + NOC;                            // [68]
    unsigned short *oc_start = (unsigned short *)(bins + 68);   // [516]
    unsigned short *item_cnt = oc_start + 516;           // [NITEM]
    unsigned short *order = item_cnt + NITEM;            // [NITEM]
    unsigned short *sidx = order + NITEM;                // [CH]
    __shared__ int s_nitems, s_next;
    __shared__ int4 s_work, s_nwk;
    __shared__ int wsum[NWARP];

    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int grp = lane >> 2, q = lane & 3;
    const int n[3] = {pr.g.nx, pr.g.ny, pr.g.nz};
    const double org[3] = {pr.g.x0, pr.g.y0, pr.g.z0};
    const int ntx = n[0] / TT, nty = n[1] / TT;
    const int64_t P = pr.P;

    if (tid == 0) {
        const int w = pr.counters[pr.wb] + atomicAdd(&pr.counters[pr.wc], 1);
        s_work = (w < pr.counters[pr.we]) ? __ldg(pr.work + w) : make_int4(-1, 0, 0, 0);
        s_next = 0;
    }
    for (int i = tid; i < NOC; i += TB) oc_cur[i] = 0;
    for (int i = tid; i < 68; i += TB) bins[i] = 0;
    __syncthreads();
    for (;;) {
        const int4 wk = s_work;                      // published by the barrier that ended the previous item
        if (wk.x < 0) break;
        // the next work item is claimed and read now; its latency hides behind this item's processing
        int4 nwk = make_int4(-1, 0, 0, 0);
        if (tid == 0) {
            const int w = pr.counters[pr.wb] + atomicAdd(&pr.counters[pr.wc], 1);
            if (w < pr.counters[pr.we]) nwk = __ldg(pr.work + w);
            s_nwk = nwk;                                 // read behind the next barrier (prefetch of its records)
        }
        const int tile = wk.x, cb = wk.y, cn = wk.z;
#ifndef IB_NO_PF
        // this chunk's forces and ids are first needed after the staging and the sort: pull them into L2 now
        // (one 128-byte line per 16 doubles / 32 ids; the item loop then waits on L2, not on DRAM)
        if (16 * tid < cn) {
            if (DO_SPREAD) {
#pragma unroll
                for (int d = 0; d < 3; ++d) ib_prefetch_l2(pr.sG + (int64_t)d * P + cb + 16 * tid);
            }
            if (DO_INTERP && 32 * tid < cn) ib_prefetch_l2(pr.sid + cb + 32 * tid);
        }
#endif
        const int t3[3] = {tile % ntx, (tile / ntx) % nty, tile / (ntx * nty)};
        int h0[3];                                       // halo origin (global index of halo entry 0), wrapped
#pragma unroll
        for (int d = 0; d < 3; ++d) h0[d] = PER ? ib_wrap(TT * t3[d] - 2, n[d]) : TT * t3[d] - 2;

        // ---- halo load, zero the accumulators ---------------------------------------------------
#ifndef IB_NO_HALO
        if (DO_INTERP) {
            for (int idx = tid; idx < 3 * TH3; idx += TB) {
                int c = idx >> 9, r = idx & 511;
                int i = h0[0] + (r & 7), j = h0[1] + ((r >> 3) & 7), k = h0[2] + (r >> 6);
                double val = 0.0;                        // faces outside a bounded grid read as zero (never used: weight dropped)
                if (PER) { i -= (i >= n[0]) ? n[0] : 0; j -= (j >= n[1]) ? n[1] : 0; k -= (k >= n[2]) ? n[2] : 0; }
                if (PER || (i >= 0 && i < n[0] && j >= 0 && j < n[1] && k >= 0 && k < n[2]))
                    val = __ldg(pr.fld[c] + ((int64_t)k * n[1] + j) * n[0] + i);
                su[c * SU3 + (r >> 6) * SZ + (r & 63)] = val;
            }
        }
#endif

        {
            // ---- stage the chunk, count points per half-cell -----------------------------------
            {
                double xr[CH / TB][3];                   // all loads of the chunk in flight at once
#pragma unroll
                for (int k = 0; k < CH / TB; ++k) {
                    const int i = tid + k * TB;
#pragma unroll
                    for (int d = 0; d < 3; ++d)
                        xr[k][d] = (i < cn) ? __ldcs(pr.sx + (int64_t)d * P + cb + i) : 0.0;
                }
#pragma unroll
                for (int k = 0; k < CH / TB; ++k) {
                    const int i = tid + k * TB;
                    if (i < cn) {
                        double xi[3];
#pragma unroll
                        for (int d = 0; d < 3; ++d) {
                            xi[d] = ib_tile_coord(xr[k][d], org[d], pr.g.h, pr.inv_h);
                            sxi[d * CH + i] = xi[d];
                        }
                        atomicAdd(&oc_cur[ib_octant_key(xi[0], xi[1], xi[2])], 1);
                    }
                }
            }
            __syncthreads();
#ifndef IB_NO_PF
            {                                            // the next chunk's coordinates -> L2 while this one is processed
                const int4 nx4 = s_nwk;
                if (nx4.x >= 0) {
                    for (int i = 16 * tid; i < 3 * CH; i += 16 * TB) {
                        const int d = i / CH, o = i - d * CH;          // CH is a multiple of 16
                        if (o < nx4.z) ib_prefetch_l2(pr.sx + (int64_t)d * P + nx4.y + o);
                    }
                }
            }
#endif
            {                                            // exclusive scan of the 512 counts, SCK per thread
                constexpr int SCK = (NOC + TB - 1) / TB;
                int v[SCK], s = 0;
#pragma unroll
                for (int k = 0; k < SCK; ++k) {
                    v[k] = (SCK * tid + k < NOC) ? oc_cur[SCK * tid + k] : 0;
                    s += v[k];
                }
                int inc = s;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    int t = __shfl_up_sync(0xffffffffu, inc, o);
                    if (lane >= o) inc += t;
                }
                if (lane == 31) wsum[wid] = inc;
                __syncthreads();
                int ex = inc - s;
                for (int w = 0; w < wid; ++w) ex += wsum[w];
#pragma unroll
                for (int k = 0; k < SCK; ++k) {
                    if (SCK * tid + k < NOC) { oc_start[SCK * tid + k] = ex; oc_cur[SCK * tid + k] = ex; }
                    ex += v[k];
                }
                if (tid == TB - 1) oc_start[NOC] = ex;
            }
            __syncthreads();
#ifndef IB_NO_PASS2
            for (int i = tid; i < cn; i += TB) {
                int key = ib_octant_key(sxi[i], sxi[CH + i], sxi[2 * CH + i]);
                sidx[atomicAdd(&oc_cur[key], 1)] = (unsigned short)i;
            }
#endif
            // ---- points per work item, order items by count (descending) -----------------------
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
                if (cnt > 0) order[atomicAdd(&bins[min(cnt, NBIN - 1)], 1)] = ib_item_code(it);
            }
            __syncthreads();
            const int nitems = s_nitems;
            // the half-cell cursors and the count bins are dead from here on: reset them for the next
            // work item (their next use lies behind the barriers that end this one)
            for (int i = tid; i < NOC; i += TB) oc_cur[i] = 0;
            for (int i = tid; i < 68; i += TB) bins[i] = 0;

            // ---- the items --------------------------------------------------------------------------
            double *mystg = stg + (wid * 8 + grp) * GSTRIDE;
            for (;;) {
                int base = 0;
                if (lane == 0) base = atomicAdd(&s_next, 8);     // warps pull 8 items at a time (largest first)
                base = __shfl_sync(0xffffffffu, base, 0);
                if (base >= nitems) break;
#ifdef IB_NO_ITEMS
                if (base >= 0) break;
#endif
                const int wi = base + grp;
                const bool have = wi < nitems;
                int c = 0, l[3] = {0, 0, 0};
                if (have) ib_item_unpack(order[wi], c, l);
                // runs of the half-cell order that make up this item
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
                // window origin inside the halo; base3[d] = scaled coordinate of the point minus
                // base3 is r in [0,1): d == c: cell l; d != c: shifted cell covers xi-1/2 in [l-1,l)
                int o3[3];
                double base3[3];
#pragma unroll
                for (int d = 0; d < 3; ++d) {
                    o3[d] = l[d] + ((d == c) ? 1 : 0);
                    base3[d] = (d == c) ? (double)l[d] : (double)l[d] - 0.5;
                }
                const double *suc = su + c * SU3 + o3[2] * SZ + o3[1] * TH + o3[0] + q;   // lane q owns x-column q
                double uu[4][4], ff[4][4];
#pragma unroll
                for (int j = 0; j < 4; ++j)
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        uu[j][i] = DO_INTERP ? suc[i * SZ + j * TH] : 0.0;            // [y j][z i]
                        ff[j][i] = 0.0;
                    }
                const double *Gc = DO_SPREAD ? pr.sG + (int64_t)c * P + cb : nullptr;
                double *Uc = DO_INTERP ? pr.Up + (int64_t)c * P : nullptr;

                // Software pipeline over quads of 4 points: while the group consumes quad k from one staging
                // buffer, lane q computes the delta weights of its point of quad k+1 into the other buffer and
                // the index / force / id of its point of quad k+2 are in flight.  One __syncwarp per quad.
                int si1, id0 = 0, id1 = 0;
                bool valid0, valid1;
                double G1 = 0.0;
#define IB_FETCH(R0, SI, GV, ID, VALID)                                                                      \
    {                                                                                                        \
        const int vi = (R0) + q;                                                                             \
        VALID = vi < npts;                                                                                   \
        int rank = vi + ((vi < rend[0]) ? rstart[0] : (vi < rend[1]) ? rstart[1] : (vi < rend[2]) ? rstart[2] : rstart[3]); \
        SI = VALID ? (int)sidx[rank] : 0;                                                                    \
        GV = (DO_SPREAD && VALID) ? __ldcs(Gc + SI) : 0.0;                                                   \
        if (DO_INTERP && VALID) ID = __ldcs(pr.sid + cb + SI);                                               \
    }
#define IB_WEIGHTS(BUF, SI, GV, VALID)                                                                       \
    {                                                                                                        \
        double wgt[3][4];                                                                                    \
        _Pragma("unroll") for (int d = 0; d < 3; ++d) {                                                      \
            /* r in [0,1] up to rounding at cell boundaries, where the formula continues phi smoothly (A19) */ \
            ib_phi4((VALID) ? sxi[d * CH + SI] - base3[d] : 0.0, wgt[d]); /* padding lanes: any r in range */ \
        }                                                                                                    \
        if (!(VALID)) { _Pragma("unroll") for (int m = 0; m < 4; ++m) wgt[2][m] = 0.0; }                     \
        double *rec = mystg + (BUF) * GBUF + q * REC;                                                        \
        *reinterpret_cast<double2 *>(rec + 0) = make_double2(wgt[0][0], wgt[0][1]);                          \
        *reinterpret_cast<double2 *>(rec + 2) = make_double2(wgt[0][2], wgt[0][3]);                          \
        *reinterpret_cast<double2 *>(rec + 4) = make_double2(wgt[1][0], wgt[1][1]);                          \
        *reinterpret_cast<double2 *>(rec + 6) = make_double2(wgt[1][2], wgt[1][3]);                          \
        *reinterpret_cast<double2 *>(rec + 8) = make_double2(wgt[2][0], wgt[2][1]);                          \
        *reinterpret_cast<double2 *>(rec + 10) = make_double2(wgt[2][2], wgt[2][3]);                         \
        rec[12] = (GV) * pr.ih3;                                                                             \
    }
                {
                    int si0;
                    double G0 = 0.0;
                    IB_FETCH(0, si0, G0, id0, valid0)
                    IB_WEIGHTS(0, si0, G0, valid0)
                }
                IB_FETCH(4, si1, G1, id1, valid1)
                __syncwarp();
                int buf = 0;
#ifdef IB_NO_MAIN
                nmax = 0;
#endif
                for (int r0 = 0; r0 < nmax; r0 += 4, buf ^= 1) {
                    // -- weights of quad r0+4 into the other buffer, fetch quad r0+8
                    int si2 = 0, id2 = 0;
                    bool valid2 = false;
                    double G2 = 0.0;
                    if (r0 + 4 < nmax) {
                        IB_WEIGHTS(buf ^ 1, si1, G1, valid1)
                        IB_FETCH(r0 + 8, si2, G2, id2, valid2)
                    }
                    // -- consume quad r0
                    const double *cur = mystg + buf * GBUF;
                    double mine = 0.0;
#pragma unroll
                    for (int jp = 0; jp < 4; ++jp) {
                        const double *rj = cur + jp * REC;
                        double2 a0 = *reinterpret_cast<const double2 *>(rj + 4), a1 = *reinterpret_cast<const double2 *>(rj + 6);
                        double2 b0 = *reinterpret_cast<const double2 *>(rj + 8), b1 = *reinterpret_cast<const double2 *>(rj + 10);
                        const double wy[4] = {a0.x, a0.y, a1.x, a1.y}, wz[4] = {b0.x, b0.y, b1.x, b1.y};
                        const double wx = rj[q];
                        if (DO_INTERP) {
                            double rr[4];
#pragma unroll
                            for (int j = 0; j < 4; ++j) {
                                rr[j] = uu[j][0] * wz[0];
                                rr[j] = fma(uu[j][1], wz[1], rr[j]);
                                rr[j] = fma(uu[j][2], wz[2], rr[j]);
                                rr[j] = fma(uu[j][3], wz[3], rr[j]);
                            }
                            double pv = fma(rr[0], wy[0], rr[1] * wy[1]) + fma(rr[2], wy[2], rr[3] * wy[3]);
                            pv *= wx;
                            pv += __shfl_xor_sync(0xffffffffu, pv, 1);
                            pv += __shfl_xor_sync(0xffffffffu, pv, 2);
                            if (q == jp) mine = pv;
                        }
                        if (DO_SPREAD) {
                            double gx = rj[12] * wx;
#pragma unroll
                            for (int j = 0; j < 4; ++j) {
                                double gj = gx * wy[j];
#pragma unroll
                                for (int i = 0; i < 4; ++i) ff[j][i] = fma(gj, wz[i], ff[j][i]);
                            }
                        }
                    }
                    if (DO_INTERP && valid0) __stcs(Uc + id0, mine);
                    valid0 = valid1; id0 = id1;
                    si1 = si2; G1 = G2; id1 = id2; valid1 = valid2;
                    __syncwarp();
                }
#undef IB_FETCH
#undef IB_WEIGHTS
#ifdef IB_NO_FLUSH
                if (DO_SPREAD && have && ff[0][0] == 123.456) {
#else
                if (DO_SPREAD && have) {
#endif
                    // lane q flushes x-column q: for every (y,z) the 4 lanes of the group hit 4 consecutive faces
                    // (bounded grid: faces outside 0..n-1 do not exist -- their share of the force is dropped, A26)
                    constexpr bool per = PER != 0;
                    int gi = h0[0] + o3[0] + q;
                    if (per) gi -= (gi >= n[0]) ? n[0] : 0;
                    const bool xin = per || (gi >= 0 && gi < n[0]);
                    int gj[4], gk[4];
                    bool jin[4], kin[4];
#pragma unroll
                    for (int m = 0; m < 4; ++m) {
                        gj[m] = h0[1] + o3[1] + m; gk[m] = h0[2] + o3[2] + m;
                        if (per) { gj[m] -= (gj[m] >= n[1]) ? n[1] : 0; gk[m] -= (gk[m] >= n[2]) ? n[2] : 0; }
                        jin[m] = per || (gj[m] >= 0 && gj[m] < n[1]);
                        kin[m] = per || (gk[m] >= 0 && gk[m] < n[2]);
                    }
                    double *fp = pr.frc[c] + gi;
                    int ok[4], oj[4];                                  // 32-bit face offsets (n_cells < 2^31)
#pragma unroll
                    for (int m = 0; m < 4; ++m) { ok[m] = gk[m] * n[1] * n[0]; oj[m] = gj[m] * n[0]; }
#pragma unroll
                    for (int i = 0; i < 4; ++i)
#pragma unroll
                        for (int j = 0; j < 4; ++j)
                            if (xin && kin[i] && jin[j]) atomicAdd(fp + (ok[i] + oj[j]), ff[j][i]);
                }
            }
        }
        __syncthreads();                              // every warp has left the item loop and read s_work
        if (tid == 0) { s_work = nwk; s_next = 0; }
        __syncthreads();                              // buffers are reused by the next work item
    }
}


// Points of tiles with fewer than IB_SMALL_TILE points are not worth a halo and a sort: one thread per
// point of the compact list written by ibk_tile_scan, every point treated directly against the grid.
// 8 resident CTAs = 64 registers, 32 warps per SM: the kernel waits on dependent loads and REDs, not on issue slots,
// so the few spilled values (<= 170 B) cost less than the warps gain (5/6/8/10/12/16 CTAs measured: DESIGN.md s.9)
#ifndef IB_SMALL_MINB
#define IB_SMALL_MINB 8
#endif
template <int DO_SPREAD, int DO_INTERP>
__global__ void __launch_bounds__(128, IB_SMALL_MINB)
ibk_small_tiles(ib_tiled_params pr, const int32_t *__restrict__ small_rec, const int32_t *__restrict__ counters)
{
    // 4 lanes per point (ib_point_quad); the list length is known on the device only, so the grid is sized for
    // the device and strides over the list
    const int q = threadIdx.x & 3;
    const unsigned qmask = 0xFu << (threadIdx.x & 28);
    const int64_t P = pr.P;
    const int n = counters[2], stride = (gridDim.x * blockDim.x) >> 2;
    for (int i = (blockIdx.x * blockDim.x + threadIdx.x) >> 2; i < n; i += stride) {
        const int r = __ldg(small_rec + i);
        double G[3] = {0, 0, 0}, U[3];
        if (DO_SPREAD) { G[0] = pr.sG[r] * pr.ih3; G[1] = pr.sG[P + r] * pr.ih3; G[2] = pr.sG[2 * P + r] * pr.ih3; }
        ib_point_quad<DO_SPREAD, DO_INTERP>(pr.sx[r], pr.sx[P + r], pr.sx[2 * P + r], G, pr.fld, pr.frc, pr.g, pr.inv_h, q, qmask, U);
        if (DO_INTERP && q == 0) {
            const int id = pr.sid[r];
            pr.Up[id] = U[0]; pr.Up[P + id] = U[1]; pr.Up[2 * P + id] = U[2];
        }
    }
}

// blocks of the sparse-tile kernel: enough for the longest possible list, at most 16 per SM (grid stride)
static int ib_small_blocks(int64_t nsmall_max, int sms)
{
    const int64_t need = (nsmall_max * 4 + 127) / 128;
    const int64_t cap = (int64_t)(sms > 0 ? sms : 148) * 16;
    return (int)(need < 1 ? 1 : (need < cap ? need : cap));
}

template <int S, int I, int PER>
static ib_status launch_tiled_p(ib_ctx *c, const ib_tiled_params &pr, bool with_small, cudaStream_t st)
{
    static unsigned char configured[64] = {0};           // per device: function attributes belong to the device's context
    static int sm_count[64] = {0};
    const int dv = c->device & 63;
    const size_t smem = (size_t)(3 * SU3 + 3 * CH + NWARP * 8 * GSTRIDE) * sizeof(double) +
                        (NOC + 68) * sizeof(int) + (516 + 2 * NITEM + CH) * sizeof(unsigned short);
    static_assert(CH % TB == 0, "chunk must be a whole number of points per thread");
    if (!configured[dv]) {
        IB_CUDA_TRY(cudaFuncSetAttribute(ibk_tiled_kernel<S, I, PER>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        configured[dv] = 1;
    }
    if (!sm_count[dv]) IB_CUDA_TRY(cudaDeviceGetAttribute(&sm_count[dv], cudaDevAttrMultiProcessorCount, c->device));
    const int sms = sm_count[dv];
    // the few points of sparsely filled tiles go one by one on a second stream, beside the tile kernel
    const int64_t nsmall_max = min((int64_t)pr.P, (c->n_cells / (TT * TT * TT)) * (int64_t)(IB_SMALL_TILE - 1));
    const bool beside = !c->profile && with_small;
    cudaStream_t s3 = beside ? c->side2 : st;
    if (beside) {
        IB_CUDA_TRY(cudaEventRecord(c->ev_sfork, st));
        IB_CUDA_TRY(cudaStreamWaitEvent(s3, c->ev_sfork, 0));
    }
    if (with_small) ibk_small_tiles<S, I><<<ib_small_blocks(nsmall_max, sms), 128, 0, s3>>>(pr, c->d_small_rec, c->d_tile_count);
    if (beside) IB_CUDA_TRY(cudaEventRecord(c->ev_sjoin, s3));
    ibk_tiled_kernel<S, I, PER><<<sms * NCTA, TB, smem, st>>>(pr);
    if (beside) IB_CUDA_TRY(cudaStreamWaitEvent(st, c->ev_sjoin, 0));
    c->launches += with_small ? 2 : 1;
    return IB_OK;
}

template <int S, int I>
static ib_status launch_tiled(ib_ctx *c, const ib_tiled_params &pr, bool with_small, cudaStream_t st)
{
    return c->grid.periodic ? launch_tiled_p<S, I, 1>(c, pr, with_small, st) : launch_tiled_p<S, I, 0>(c, pr, with_small, st);
}

// mesh != 0: points are the sub-points of the mesh at node positions x with force coefficients Fhat
// (xp/Gp ignored); mesh == 0: the cloud xp/Gp.  Gp/Fhat NULL = interpolate only; Up NULL = spread only.
ib_status ibk_tiled_spread_interp(ib_ctx *c, int mesh, const double *xp, const double *Gp, int64_t P,
                                  const double *x, const double *Fhat,
                                  const double *u, const double *v, const double *w,
                                  double *fu, double *fv, double *fw, double *Up, int counted, cudaStream_t st)
{
    ib_status rs = ibk_bin_reserve(c, P);
    if (rs != IB_OK) return rs;
    const bool spread = mesh ? (Fhat != nullptr) : (Gp != nullptr);
    ib_prof_begin(c, IB_PHASE_SORT, st);
    rs = ibk_bin_points(c, mesh, xp, Gp, P, x, Fhat, Up, counted ? 2 : 3, st);   // counted: phase 1 already enqueued
    ib_prof_end(c, IB_PHASE_SORT, st);
    if (rs != IB_OK) return rs;

    return ibk_tiled_launch(c, P, spread, Up != nullptr, u, v, w, fu, fv, fw, Up, -1, st);
}

static void fill_params(ib_ctx *c, ib_tiled_params &pr, int64_t P, const double *u, const double *v, const double *w,
                        double *fu, double *fv, double *fw, double *Up, int slab)
{
    pr.sx = c->d_sx; pr.sG = c->d_sG; pr.sid = c->d_sid; pr.P = P;
    pr.fld[0] = u; pr.fld[1] = v; pr.fld[2] = w;
    pr.frc[0] = fu; pr.frc[1] = fv; pr.frc[2] = fw;
    pr.Up = Up;
    pr.work = c->d_work; pr.counters = c->d_tile_count;
    pr.wb = slab < 0 ? 3 : IB_SLAB0 + slab;
    pr.we = slab < 0 ? 0 : IB_SLAB0 + slab + 1;
    pr.wc = slab < 0 ? 1 : IB_SLABC0 + slab;
    pr.g = c->grid; pr.inv_h = c->inv_h; pr.ih3 = c->inv_h * c->inv_h * c->inv_h;
}

// The tile kernel (and the direct path of the sparse tiles) over records that are already binned.
// Spreading and interpolation may be launched separately over the same records (ib_coupling_step_host
// overlaps them with the host copies): the work counter is reset on the stream before every launch.
// slab < 0: all work items, and the sparse tiles beside them; slab k >= 0: the work items of z-slab k only
// (the tile layers [k L, (k+1) L), L = ib_slab_layers) with a work counter of its own, so that slabs may run
// on different streams at once; the sparse tiles are then the caller's to launch (ibk_small_launch).
ib_status ibk_tiled_launch(ib_ctx *c, int64_t P, int do_spread, int do_interp,
                           const double *u, const double *v, const double *w,
                           double *fu, double *fv, double *fw, double *Up, int slab, cudaStream_t st)
{
    ib_status rs = IB_OK;
    ib_tiled_params pr;
    fill_params(c, pr, P, u, v, w, fu, fv, fw, Up, slab);
    const bool with_small = slab < 0;
    IB_CUDA_TRY(cudaMemsetAsync(c->d_tile_count + pr.wc, 0, sizeof(int32_t), st));
    ib_prof_begin(c, IB_PHASE_SPREAD_INTERP, st);
    if (do_spread && do_interp) rs = launch_tiled<1, 1>(c, pr, with_small, st);
    else if (do_spread) rs = launch_tiled<1, 0>(c, pr, with_small, st);
    else rs = launch_tiled<0, 1>(c, pr, with_small, st);
    ib_prof_end(c, IB_PHASE_SPREAD_INTERP, st);
    if (rs != IB_OK) return rs;
    IB_CUDA_TRY(cudaGetLastError());
    return IB_OK;
}

// the direct path of the sparse tiles alone, on the given stream
ib_status ibk_small_launch(ib_ctx *c, int64_t P, int do_spread, int do_interp,
                           const double *u, const double *v, const double *w,
                           double *fu, double *fv, double *fw, double *Up, cudaStream_t st)
{
    ib_tiled_params pr;
    fill_params(c, pr, P, u, v, w, fu, fv, fw, Up, -1);
    const int64_t nsmall_max = min((int64_t)P, (c->n_cells / (TT * TT * TT)) * (int64_t)(IB_SMALL_TILE - 1));
    const int nb = ib_small_blocks(nsmall_max, 0);
    if (do_spread && do_interp) ibk_small_tiles<1, 1><<<nb, 128, 0, st>>>(pr, c->d_small_rec, c->d_tile_count);
    else if (do_spread) ibk_small_tiles<1, 0><<<nb, 128, 0, st>>>(pr, c->d_small_rec, c->d_tile_count);
    else ibk_small_tiles<0, 1><<<nb, 128, 0, st>>>(pr, c->d_small_rec, c->d_tile_count);
    c->launches += 1;
    IB_CUDA_TRY(cudaGetLastError());
    return IB_OK;
}
