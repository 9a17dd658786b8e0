// ib_tiled.cu -- variant 1 of spread (Eq.(24)-(26)) and interpolation (Eq.(27)-(29)):
// points grouped by 4x4x4-cell tile (ib_bin.cu); one persistent, warp-specialised CTA per SM pulls work items
// (runs of z-layers of one tile, <= IB_CHUNK points) from a work list, keeps an 8x8x8 halo of u,v,w in shared
// memory and holds the stencil windows in registers (the producer / consumer split is described at the kernel).
//
// Per work item the producer warps compute, one thread per point, the tile-relative scaled coordinates and from them
// the six 1-D delta-weight sets of the point (3 directions x {face-aligned, centre-aligned}: component c
// lives on its own staggered lattice, MAC grid L205), once, and stores them in shared memory in half-cell
// order ("octant", 8^3 per tile; shared-memory counting sort).  Why half-cells: in the direction d == c the
// 4-point support of a point is fixed by its cell; in the other two it is fixed by the cell of the lattice
// shifted by h/2.  With the points ordered by half-cell every cell of every shifted lattice is a union of
// <= 4 contiguous runs, so all points of one item (shifted cell, component) share ONE 4x4x4 window.
//
// A weight set is stored as the pair (a, q) it is made of: the Peskin 4-point weights of a point at
// fraction r are  w0 = a - q, w1 = a + q, w2 = (1/2 - a) + q, w3 = (1/2 - a) - q  with a = 3/8 - r/4 and
// q = sqrt(1 + 4r - 4r^2)/8 (ib_phi4).  They are affine in (a, q), so a 4-term contraction with them is a
// 3-term one in the basis {1, a, q}:
//     sum_i w_i u_i = S0 + a Sa + q Sq,   S0 = (u2+u3)/2,  Sa = u0+u1-u2-u3,  Sq = -u0+u1+u2-u3,
// and the transpose for spreading: accumulate the moments M0 = sum g, Ma = sum g a, Mq = sum g q over the
// points, then  f0 = Ma-Mq, f1 = Ma+Mq, f2 = M0/2-Ma+Mq, f3 = M0/2-Ma-Mq.  The y and z directions of a window
// are kept in that basis (3x3 = 9 values instead of 4x4 = 16), x stays in weight form across 4 lanes.
//
// Items are cut into units of <= PCAP points, ordered by point count and pulled by the consumer warps in
// batches of 8 units of one component.  A group of 4 lanes owns a unit: lane q keeps the x-column q of the window -- 9 transformed velocity values and 9 force moments -- in
// registers and loops over the unit's points: per point and lane 9 DFMA for interpolation, 12 for
// spreading, 2 for its own x-weight, against 21 + 21 in weight form.  The moments are transformed back once
// per unit and flushed with RED.ADD.F64 straight to the grid: the 4 lanes of a group hit 4 consecutive
// faces (Blackwell has no native shared-memory fp64 add; the CAS loop measured 34 wavefronts each).
// Tiles with fewer than IB_SMALL_TILE points skip all of this (ibk_small_tiles, ib_point.cuh).
#include <cassert>
#include <cuda.h>               // CUtensorMap and its enums only: the encoder is fetched through the runtime, libcuda is not linked
#include "ib_point.cuh"

#define TT 4                    // tile edge in cells
#define TH 8                    // halo edge
#define TH3 512
#define NOC 512                 // half-cells per tile (8^3)
#define NITEM 300               // 3 components x (4*5*5) shifted cells
#define TB 512                  // threads per CTA: one CTA per SM, 16 warps
#define NWARP (TB / 32)
#ifndef IB_TILED_PRODUCER_WARPS
#define IB_TILED_PRODUCER_WARPS 6   // of the 16 warps (the others run the items); 5 / 7 / 8 measured
#endif
#define CH IB_CHUNK             // records staged per work item
#define SZ 64                   // z-plane stride of the halo in doubles: dense 8 x 8 x 8, the layout a TMA box load writes
#define SU3 (TH * SZ)           // one component of the halo
#ifndef PCAP
#define PCAP 24                 // an item with more points is cut into units of PCAP points (each with a window of its own); 16 / 20 / 24 / 28 / 32 measured on the final kernel
#endif
#define NBIN (PCAP + 1)         // units are ordered by point count 0..PCAP
#define NORD ((100 + IB_CHUNK / PCAP + 7) & ~7)   // units per component: one per item + IB_CHUNK / PCAP whole ones, in whole batches

struct ib_tiled_params {
    const double *rec;          // [P][8] records grouped by bin: {x, y, z, id | G0, G1, G2, -} (ib_bin.cu)
    int64_t P;
    const double *fld[3];
    double *frc[3];
    double *Up;
    const int4 *work;           // {tile, first record, points, tile coordinates tx | ty << 10 | tz << 20} per work item
    int32_t *counters;          // [0] number of work items, [1] work counter, [3] zero, [IB_SLAB0 + k] first item of slab k
    int wb, we, wc;             // this launch covers the work items counters[wb] <= w < counters[we]; counters[wc] counts them
    ib_grid_desc g;
    double inv_h, ih3;
    int use_tma;                // tm[] are valid: the halo of a tile that does not wrap comes by one TMA box load per component
    alignas(64) CUtensorMap tm[3];   // u, v, w as 3-D fp64 tensors (nx, ny, nz), box 8 x 8 x 8, out-of-range elements read as zero
};

// decode an item: component c, shifted-cell coordinates l[3]  (c*100 + (l2*ny + l1)*nx + l0 with
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
    const int ci = __double2int_rd(__dmul_rn(__dsub_rn(x, x0), inv_h));       // floor: the cell of A21 before the wrap
    // grid dims are multiples of 8, so the periodically wrapped cell index is congruent to the
    // unwrapped one modulo the tile edge 4.  s - fl is exact, so (s - fl) + (ci & 3) = s - (fl - (ci & 3)) in one rounding
    return ib_scaled(x, x0, h, inv_h) - ib_i2d(ci & ~(TT - 1));
}

__device__ __forceinline__ void ib_prefetch_l2(const void *p)
{
    asm volatile("prefetch.global.L2 [%0];" ::"l"(p));
}

// one 32-byte half of a record, streaming
__device__ __forceinline__ void ib_load_rec(const double *p, double v[4])
{
    asm volatile("ld.global.cs.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(v[0]), "=d"(v[1]), "=d"(v[2]), "=d"(v[3]) : "l"(p));
}

// 4 values along one direction of a window -> their 3 coefficients in the basis {1, a, q}
__device__ __forceinline__ void ib_to_basis(double u0, double u1, double u2, double u3, double &s0, double &sa, double &sq)
{
    const double p = u2 + u3;
    s0 = 0.5 * p;
    sa = (u0 + u1) - p;
    sq = (u1 - u0) + (u2 - u3);
}

// 3 moments along one direction -> the 4 face values (transpose of ib_to_basis)
__device__ __forceinline__ void ib_from_basis(double m0, double ma, double mq, double f[4])
{
    const double t = fma(0.5, m0, -ma);
    f[0] = ma - mq;
    f[1] = ma + mq;
    f[2] = t + mq;
    f[3] = t - mq;
}

// shared-memory addresses (32-bit, shared window) of one work item's arrays, and per-lane constants.  They are
// made opaque to the compiler once (ib_opaque): it otherwise re-derives them inside the point loop to save
// registers (10 of 70 instructions per point in the SASS of the first version).
struct ib_tile_smem {
    unsigned su, sets, sGs, sids;    // [3][8][SZ] halo, [6][CH] (a,q) pairs, [3][CH] force, [CH] ids
    const uint4 *item_runs;          // [NITEM + 1]
    const unsigned *item_win;        // [NITEM + 1]
};

__device__ __forceinline__ void ib_opaque(unsigned &v) { asm volatile("" : "+r"(v)); }
__device__ __forceinline__ void ib_opaque(double &v) { asm volatile("" : "+d"(v)); }
__device__ __forceinline__ double2 ib_lds128(unsigned a)
{
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(a));
    return v;
}
__device__ __forceinline__ double ib_lds64(unsigned a)
{
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ unsigned ib_lds32(unsigned a)
{
    unsigned v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a));
    return v;
}

// record of virtual point index vi of an item made of <= 4 runs (rstart/rend: see the caller)
__device__ __forceinline__ int ib_item_rec(int vi, const int rstart[4], const int rend[3])
{
    int off = rstart[0];
    off = (vi >= rend[0]) ? rstart[1] : off;
    off = (vi >= rend[1]) ? rstart[2] : off;
    off = (vi >= rend[2]) ? rstart[3] : off;
    return vi + off;
}

// One batch of 8 units of component C (the same for the whole warp): the group of 4 lanes owns the unit `part`
// of item `it` (an empty slot of the batch gets the item NITEM, which has no points).  One instantiation serves
// the three components: three copies of this loop do not fit the instruction cache of a scheduler (measured:
// 1.9 "no instruction" stalls per issue).
template <int DO_SPREAD, int DO_INTERP, int PER>
__device__ __forceinline__ void ib_run_batch(int C, const ib_tiled_params &pr, const ib_tile_smem &sm, int it, int part, int q,
                                             const int h0[3], const int n[3], double wsa, double wca, double wsg)
{
    const unsigned full = 0xffffffffu;
    // runs of the half-cell order that make up this item
    int rstart[4], rend[3], npts = 0;
    {
        const uint4 rn4 = sm.item_runs[it];
        const unsigned rn[4] = {rn4.x, rn4.y, rn4.z, rn4.w};
#pragma unroll
        for (int rr = 0; rr < 4; ++rr) {
            const int s0 = (int)(rn[rr] & 0xffffu), s1 = (int)(rn[rr] >> 16);
            rstart[rr] = s0 - npts;          // record = rstart + virtual index
            npts += s1 - s0;
            if (rr < 3) rend[rr] = npts;     // virtual indices < rend belong to runs <= rr
        }
    }
    // this group's unit: the virtual points [vlo, vlo + nun) of the item
    const int vlo = part * PCAP, nun = min(PCAP, npts - vlo);       // <= 0 for the empty slot
    assert(it <= NITEM && npts <= CH && (it == NITEM || nun > 0));
    int nmax = nun;
#pragma unroll
    for (int o = 16; o >= 4; o >>= 1) nmax = max(nmax, __shfl_xor_sync(full, nmax, o));
    // window: offset of its origin in the halo (with the component), origin o3 = l + (d == C)
    const unsigned win = sm.item_win[it];
    // lane q owns x-column q of the window; y and z in the basis {1, a, q}: S[by][bz]
    double S[3][3], M[3][3];
    if (DO_INTERP) {
        const unsigned suc = sm.su + ((win & 0xffffu) + q) * 8u;
        double t[4][3];
#pragma unroll
        for (int j = 0; j < 4; ++j)
            ib_to_basis(ib_lds64(suc + j * TH * 8), ib_lds64(suc + (j * TH + SZ) * 8), ib_lds64(suc + (j * TH + 2 * SZ) * 8),
                        ib_lds64(suc + (j * TH + 3 * SZ) * 8), t[j][0], t[j][1], t[j][2]);
#pragma unroll
        for (int bz = 0; bz < 3; ++bz) ib_to_basis(t[0][bz], t[1][bz], t[2][bz], t[3][bz], S[0][bz], S[1][bz], S[2][bz]);
    }
#pragma unroll
    for (int by = 0; by < 3; ++by)
#pragma unroll
        for (int bz = 0; bz < 3; ++bz) M[by][bz] = 0.0;
    unsigned ax = sm.sets + (C != 0 ? CH * 16 : 0), ay = sm.sets + (C != 1 ? 3 * CH * 16 : 2 * CH * 16),
             az = sm.sets + (C != 2 ? 5 * CH * 16 : 4 * CH * 16), ag = sm.sGs + C * (CH * 8);
    double *Uc = DO_INTERP ? pr.Up + (int64_t)C * pr.P : nullptr;
    unsigned qq = (unsigned)q;
    ib_opaque(ax); ib_opaque(ay); ib_opaque(az); ib_opaque(ag); ib_opaque(qq);      // kept in registers, not re-derived per point
    asm volatile("" : "+l"(Uc));

    // 4 points per step: the x-sums of the 4 interpolated values are reduced across the 4 lanes in a
    // transposing butterfly (3 shuffles instead of 8), which leaves point k's value in lane k -- one store
    // instruction per 4 points
    double ra0 = 0.0, ra1 = 0.0, rs0 = 0.0, rs1 = 0.0;                      // the reduction of a step is finished in the next one (its second shuffle and the
                                                       // store run beside the loads of the next four points)
    for (int v0 = 0; v0 < nmax; v0 += 4) {
        if (DO_INTERP && v0 > 0) {
            const bool hi1 = (qq & 1u) != 0;
            ra0 += __shfl_xor_sync(full, rs0, 2);
            ra1 += __shfl_xor_sync(full, rs1, 2);
            double tot = hi1 ? ra1 : ra0;
            tot += __shfl_xor_sync(full, hi1 ? ra0 : ra1, 1);
            if (v0 - 4 + (int)qq < nun) __stcs(Uc + ib_lds32(sm.sids + 4u * (unsigned)ib_item_rec(vlo + v0 - 4 + (int)qq, rstart, rend)), tot);
        }
        double pv[4];
        // two points in one straight line of code (their loads and dependent chains overlap); the second pair
        // of a step only when the longest unit of the batch reaches it
#pragma unroll
        for (int kp = 0; kp < 4; kp += 2) {
            pv[kp] = 0.0; pv[kp + 1] = 0.0;
            if (kp == 0 || v0 + kp < nmax) {                  // warp-uniform
                // all the loads of the pair first (the asm loads keep their order), then the arithmetic
                bool valid[2];
                double2 X[2], Y[2], Z[2];
                double gl[2];
#pragma unroll
                for (int k = 0; k < 2; ++k) {
                    valid[k] = v0 + kp + k < nun;
                    const int rec = valid[k] ? ib_item_rec(vlo + v0 + kp + k, rstart, rend) : 0;   // padding: record 0 exists, its force is replaced by zero
                    assert(rec >= 0 && rec < CH);
                    const unsigned r16 = (unsigned)rec << 4;
                    X[k] = ib_lds128(ax + r16); Y[k] = ib_lds128(ay + r16); Z[k] = ib_lds128(az + r16);
                    gl[k] = DO_SPREAD ? ib_lds64(ag + ((unsigned)rec << 3)) : 0.0;
                }
#pragma unroll
                for (int k = 0; k < 2; ++k) {
                    const double wx = fma(wsg, X[k].y, fma(wsa, X[k].x, wca));
                    if (DO_INTERP) {
                        const double c0 = fma(Z[k].y, S[0][2], fma(Z[k].x, S[0][1], S[0][0]));
                        const double c1 = fma(Z[k].y, S[1][2], fma(Z[k].x, S[1][1], S[1][0]));
                        const double c2 = fma(Z[k].y, S[2][2], fma(Z[k].x, S[2][1], S[2][0]));
                        pv[kp + k] = fma(Y[k].y, c2, fma(Y[k].x, c1, c0)) * wx;
                    }
                    if (DO_SPREAD) {
                        const double g0 = (valid[k] ? gl[k] : 0.0) * wx, g1 = g0 * Y[k].x, g2 = g0 * Y[k].y;
                        M[0][0] += g0; M[0][1] = fma(g0, Z[k].x, M[0][1]); M[0][2] = fma(g0, Z[k].y, M[0][2]);
                        M[1][0] += g1; M[1][1] = fma(g1, Z[k].x, M[1][1]); M[1][2] = fma(g1, Z[k].y, M[1][2]);
                        M[2][0] += g2; M[2][1] = fma(g2, Z[k].x, M[2][1]); M[2][2] = fma(g2, Z[k].y, M[2][2]);
                    }
                }
            }
        }
        if (DO_INTERP) {
            const bool hi2 = (qq & 2u) != 0;
            rs0 = hi2 ? pv[0] : pv[2]; rs1 = hi2 ? pv[1] : pv[3];
            ra0 = hi2 ? pv[2] : pv[0];
            ra1 = hi2 ? pv[3] : pv[1];
        }
    }
    if (DO_INTERP && nmax > 0) {
        // the last step of the batch; lane q holds the value of point v0 + q
        const int v0 = (nmax - 1) & ~3;
        const bool hi1 = (qq & 1u) != 0;
        ra0 += __shfl_xor_sync(full, rs0, 2);
        ra1 += __shfl_xor_sync(full, rs1, 2);
        double tot = hi1 ? ra1 : ra0;
        tot += __shfl_xor_sync(full, hi1 ? ra0 : ra1, 1);
        if (v0 + (int)qq < nun) __stcs(Uc + ib_lds32(sm.sids + 4u * (unsigned)ib_item_rec(vlo + v0 + (int)qq, rstart, rend)), tot);
    }
    if (DO_SPREAD && nun > 0) {
        // moments -> face values ff[y j][z i] of x-column q
        double t[4][3], ff[4][4];
#pragma unroll
        for (int bz = 0; bz < 3; ++bz) {
            double f4[4];
            ib_from_basis(M[0][bz], M[1][bz], M[2][bz], f4);
#pragma unroll
            for (int j = 0; j < 4; ++j) t[j][bz] = f4[j];
        }
#pragma unroll
        for (int j = 0; j < 4; ++j) ib_from_basis(t[j][0], t[j][1], t[j][2], ff[j]);
        // lane q flushes x-column q: for every (y,z) the 4 lanes of the group hit 4 consecutive faces
        // (bounded grid: faces outside 0..n-1 do not exist -- their share of the force is dropped, A26)
        constexpr bool per = PER != 0;
        int gi = h0[0] + (int)((win >> 16) & 15u) + q;
        if (per) gi -= (gi >= n[0]) ? n[0] : 0;
        const bool xin = per || (gi >= 0 && gi < n[0]);
        const int j0 = h0[1] + (int)((win >> 20) & 15u), k0 = h0[2] + (int)((win >> 24) & 15u), nxy = n[0] * n[1];
        unsigned ok[4], oj[4];                             // 32-bit face offsets (n_cells < 2^31)
        bool jin[4], kin[4];
#pragma unroll
        for (int m = 0; m < 4; ++m) {
            int gj = j0 + m, gk = k0 + m;
            if (per) { gj -= (gj >= n[1]) ? n[1] : 0; gk -= (gk >= n[2]) ? n[2] : 0; }
            jin[m] = per || (gj >= 0 && gj < n[1]);
            kin[m] = per || (gk >= 0 && gk < n[2]);
            oj[m] = (unsigned)(gj * n[0] + gi);
            ok[m] = (unsigned)(gk * nxy);
        }
        double *fp = pr.frc[C];
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j)
                if (xin && kin[i] && jin[j]) atomicAdd(fp + (ok[i] + oj[j]), ff[j][i]);
    }
}

// ---- warp-specialised persistent kernel ----------------------------------------------------------------
// One CTA per SM, 16 warps: NPW "producer" warps turn work items into shared-memory records (coordinates ->
// half-cell sort -> (a,q) sets, runs and ordered units of the items; one thread starts the TMA box loads of the
// halo, whose bytes the consumers await on a barrier of their own), NCW "consumer" warps run the
// batches of units.  Two record buffers: the producers fill buffer k+1 while the consumers work through
// buffer k.  full[b] / empty[b] are mbarriers (producers -> consumers: one arrival; consumers -> producers:
// one per consumer warp).  No barrier ever joins the two groups: a consumer warp that finds no more batches
// in a buffer moves on to the next, the producers wait only for the buffer they are about to overwrite.
// (The first version had all warps walk through the phases of a work item together: a quarter of the warp
// time went to the barriers between the phases and to the tail of the item loop.)
#define NPW IB_TILED_PRODUCER_WARPS
#define NCW (NWARP - NPW)
#define TBP (NPW * 32)                                  // producer threads
#define KPT ((CH + TBP - 1) / TBP)                      // points per producer thread
#define NIT ((NITEM + TBP - 1) / TBP)                   // items per producer thread in the counting pass
#define SCK ((NOC + TBP - 1) / TBP)                     // half-cell counters per producer thread in the scan

// byte offsets inside one record buffer
#define OFF_SU 0
#define OFF_SETS (OFF_SU + 3 * SU3 * 8)
#define OFF_SG (OFF_SETS + 6 * CH * 16)
#define OFF_RUNS (OFF_SG + 3 * CH * 8)
#define OFF_SIDS (OFF_RUNS + (NITEM + 1) * 16)
#define OFF_ORDER (OFF_SIDS + CH * 4)
#define OFF_CTL (OFF_ORDER + ((3 * NORD * 2 + 15) & ~15))
#define BUF_BYTES ((OFF_CTL + 48 + 127) & ~127)          // ctl: {nbatch, ncomp[3], next, h0[3], halo barrier phase + 1 or 0}; the halo of the next buffer stays 128-byte aligned
// after the two buffers: producer-private scratch and the static window table
#define OFF_OCCNT (2 * BUF_BYTES)
#define OFF_BINS (OFF_OCCNT + NOC * 4)
#define OFF_OCSTART (OFF_BINS + ((3 * NBIN * 4 + 15) & ~15))
#define OFF_WIN (OFF_OCSTART + ((516 * 2 + 15) & ~15))
#define OFF_MISC (OFF_WIN + ((NITEM + 1) * 4 + 15) / 16 * 16)      // wsum[NPW], work slots int4[2], mbarriers
#define TILED_SMEM_BYTES (OFF_MISC + 16 * 4 + 2 * 16 + 6 * 8)

__device__ __forceinline__ void ib_mbar_init(unsigned a, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(a), "r"(count) : "memory");
}
__device__ __forceinline__ void ib_mbar_arrive(unsigned a)
{
    asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.shared::cta.b64 st, [%0];\n\t}" ::"r"(a) : "memory");
}
__device__ __forceinline__ void ib_mbar_wait(unsigned a, unsigned parity)
{
    asm volatile("{\n\t.reg .pred p;\n"
                 "IB_MBAR_WAIT:\n\t"
                 "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1, 0x989680;\n\t"
                 "@p bra IB_MBAR_DONE;\n\t"
                 "bra IB_MBAR_WAIT;\n"
                 "IB_MBAR_DONE:\n\t}" ::"r"(a), "r"(parity) : "memory");
}
__device__ __forceinline__ void ib_mbar_expect_tx(unsigned a, unsigned bytes)
{
    asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.expect_tx.shared::cta.b64 st, [%0], %1;\n\t}" ::"r"(a), "r"(bytes) : "memory");
}
// one 8 x 8 x 8 box of a 3-D tensor -> shared memory; elements outside the tensor arrive as zeros
__device__ __forceinline__ void ib_tma_box(unsigned dst, const CUtensorMap *tm, int x, int y, int z, unsigned bar)
{
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
                 ::"r"(dst), "l"(tm), "r"(x), "r"(y), "r"(z), "r"(bar) : "memory");
}
__device__ __forceinline__ void ib_producer_sync()
{
    asm volatile("bar.sync 1, %0;" ::"n"(TBP) : "memory");
}

// PER: periodic grid (compile-time, so that the periodic kernel carries none of the wall predicates)
template <int DO_SPREAD, int DO_INTERP, int PER>
__global__ void __launch_bounds__(TB, 1)
ibk_tiled_kernel(const __grid_constant__ ib_tiled_params pr)
{
    extern __shared__ __align__(1024) unsigned char smraw[];
    int *oc_cnt = reinterpret_cast<int *>(smraw + OFF_OCCNT);                       // [NOC] points per half-cell
    int *bins = reinterpret_cast<int *>(smraw + OFF_BINS);                          // [3][NBIN] units per component and point count
    unsigned short *oc_start = reinterpret_cast<unsigned short *>(smraw + OFF_OCSTART);   // [516] first record of a half-cell
    unsigned *item_win = reinterpret_cast<unsigned *>(smraw + OFF_WIN);             // [NITEM + 1] window of an item: halo offset | o3x << 16 | o3y << 20 | o3z << 24
    int *wsum = reinterpret_cast<int *>(smraw + OFF_MISC);                          // [16]
    int4 *s_wk = reinterpret_cast<int4 *>(smraw + OFF_MISC + 64);                   // work item of the even / odd iteration
    const unsigned mbar = (unsigned)__cvta_generic_to_shared(smraw + OFF_MISC + 96);   // full[0], full[1], empty[0], empty[1], halo[0], halo[1]

    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int n[3] = {pr.g.nx, pr.g.ny, pr.g.nz};

    if (tid == 0) {
        ib_mbar_init(mbar + 0, 1); ib_mbar_init(mbar + 8, 1);
        ib_mbar_init(mbar + 16, NCW); ib_mbar_init(mbar + 24, NCW);
        ib_mbar_init(mbar + 32, 1); ib_mbar_init(mbar + 40, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");      // the TMA unit sees the initialised barriers
        const int w = pr.counters[pr.wb] + atomicAdd(&pr.counters[pr.wc], 1);
        s_wk[0] = (w < pr.counters[pr.we]) ? __ldg(pr.work + w) : make_int4(-1, 0, 0, 0);
    }
    for (int i = tid; i < NOC; i += TB) oc_cnt[i] = 0;
    for (int i = tid; i < 3 * NBIN; i += TB) bins[i] = 0;
    // the windows of the items do not depend on the work item; item NITEM (in both buffers) has no points
    for (int it = tid; it <= NITEM; it += TB) {
        int c = 0, l[3] = {0, 0, 0};
        if (it < NITEM) ib_item_decode(it, c, l);
        const int o3[3] = {l[0] + (c == 0 ? 1 : 0), l[1] + (c == 1 ? 1 : 0), l[2] + (c == 2 ? 1 : 0)};
        item_win[it] = (unsigned)(c * SU3 + o3[2] * SZ + o3[1] * TH + o3[0]) | (o3[0] << 16) | (o3[1] << 20) | (o3[2] << 24);
    }
    if (tid < 2) reinterpret_cast<uint4 *>(smraw + tid * BUF_BYTES + OFF_RUNS)[NITEM] = make_uint4(0, 0, 0, 0);
    __syncthreads();                                 // the only CTA-wide barrier of the kernel

    if (wid < NPW) {
        // =================================== producers ==========================================================
        const double org[3] = {pr.g.x0, pr.g.y0, pr.g.z0};
        int wfirst = 0, wlast = 0, wnext = 0;            // thread 0: the launch's range of work items, the index claimed for the next one
        if (tid == 0) { wfirst = pr.counters[pr.wb]; wlast = pr.counters[pr.we]; wnext = wfirst + atomicAdd(&pr.counters[pr.wc], 1); }
        unsigned halo_phase = 0;                         // bit b: phase of halo[b] that the next TMA load into buffer b completes
        for (int iter = 0;; ++iter) {
            const int b = iter & 1;
            unsigned char *buf = smraw + b * BUF_BYTES;
            const int4 wk = s_wk[b];
            if (wk.x < 0) {
                // no more work: an empty buffer with nbatch < 0 tells the consumers to stop
                if (tid == 0) {
                    if (iter >= 2) ib_mbar_wait(mbar + 16 + 8 * b, ((iter >> 1) - 1) & 1);
                    reinterpret_cast<int *>(buf + OFF_CTL)[0] = -1;
                    ib_mbar_arrive(mbar + 8 * b);
                }
                break;
            }
            const int cb = wk.y, cn = wk.z;
            // Work items are claimed two ahead, so that thread 0 never waits for a round trip to the L2 (the atomic on
            // the one counter of all CTAs takes about 2000 cycles, the load of the work item 700 more): the atomic
            // issued now names the item after the next one and is not looked at before the next iteration; the
            // index it returned last time is used now, and the work item loaded with it is stored into the other slot
            // (every producer has read that one at the top of the previous iteration) inside the scan
            int wnn = 0;
            if (tid == 0) wnn = wfirst + atomicAdd(&pr.counters[pr.wc], 1);
            // ---- coordinates of the records, one thread per point: tile coordinates, half-cell, rank inside it.
            // Nothing here touches the record buffers: it overlaps the consumers' work on both of them.
            double xi[KPT][3];
            int ks[KPT], idr[KPT];
            {
                double xr[KPT][4];
#pragma unroll
                for (int k = 0; k < KPT; ++k) {
                    const int i = tid + k * TBP;
                    xr[k][0] = xr[k][1] = xr[k][2] = xr[k][3] = 0.0;
                    if (i < cn) ib_load_rec(pr.rec + (size_t)(cb + i) * 8, xr[k]);
                    idr[k] = (int)__double_as_longlong(xr[k][3]);
                }
#pragma unroll
                for (int k = 0; k < KPT; ++k) {
                    const int i = tid + k * TBP;
                    ks[k] = -1;
                    if (i < cn) {
                        int key = 0;
#pragma unroll
                        for (int d = 2; d >= 0; --d) {
                            xi[k][d] = ib_tile_coord(xr[k][d], org[d], pr.g.h, pr.inv_h);
                            key = key * 8 + min(max(__double2int_rd(2.0 * xi[k][d]), 0), 7);
                        }
                        ks[k] = key | (atomicAdd(&oc_cnt[key], 1) << 9);
                    }
                }
            }
            int4 wk_next = make_int4(-1, 0, 0, 0);
            if (tid == 0 && wnext < wlast) wk_next = __ldg(pr.work + wnext);
            ib_producer_sync();
            for (int i = tid; i < 3 * NBIN; i += TBP) bins[i] = 0;      // read last before the closing barrier of the previous iteration
            {                                            // exclusive scan of the 512 counts
                int v[SCK], s = 0;
#pragma unroll
                for (int k = 0; k < SCK; ++k) {
                    v[k] = (SCK * tid + k < NOC) ? oc_cnt[SCK * tid + k] : 0;
                    s += v[k];
                }
                int inc = s;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    int t = __shfl_up_sync(0xffffffffu, inc, o);
                    if (lane >= o) inc += t;
                }
                if (lane == 31) wsum[wid] = inc;
                if (tid == 0) { s_wk[b ^ 1] = wk_next; wnext = wnn; }
                ib_producer_sync();
                int ex = inc - s;
                for (int w = 0; w < wid; ++w) ex += wsum[w];
#pragma unroll
                for (int k = 0; k < SCK; ++k) {
                    if (SCK * tid + k < NOC) { oc_start[SCK * tid + k] = ex; oc_cnt[SCK * tid + k] = 0; }   // counts: ready for the next work item
                    ex += v[k];
                }
                if (tid == TBP - 1) oc_start[NOC] = ex;
            }
            {                                            // the next work item's records -> L2 while this one is processed
                const int4 nx4 = s_wk[b ^ 1];
                if (nx4.x >= 0)
                    for (int i = 2 * tid; i < nx4.z; i += 2 * TBP) ib_prefetch_l2(pr.rec + (size_t)(nx4.y + i) * 8);   // two records per 128-byte line
            }
            ib_producer_sync();
            // ---- from here on the record buffer is written: the consumers must have left its previous contents
            if (iter >= 2) ib_mbar_wait(mbar + 16 + 8 * b, ((iter >> 1) - 1) & 1);
            double *su = reinterpret_cast<double *>(buf + OFF_SU);
            double2 *sets = reinterpret_cast<double2 *>(buf + OFF_SETS);
            double *sGs = reinterpret_cast<double *>(buf + OFF_SG);
            uint4 *item_runs = reinterpret_cast<uint4 *>(buf + OFF_RUNS);
            int *sids = reinterpret_cast<int *>(buf + OFF_SIDS);
            unsigned short *order = reinterpret_cast<unsigned short *>(buf + OFF_ORDER);
            int *ctl = reinterpret_cast<int *>(buf + OFF_CTL);
            const int t3[3] = {wk.w & 1023, (wk.w >> 10) & 1023, wk.w >> 20};     // tile coordinates, packed by ibk_tile_scan
            int h0[3];                                       // halo origin (global index of halo entry 0), wrapped
#pragma unroll
            for (int d = 0; d < 3; ++d) h0[d] = PER ? ib_wrap(TT * t3[d] - 2, n[d]) : TT * t3[d] - 2;
            // ---- halo: one TMA box load per component (8 x 8 x 8 doubles; what lies outside a bounded grid arrives as
            // zeros, which is what A26 asks for); the halo of a tile at the edge of a periodic grid wraps around, which a
            // box cannot: it is put together from asynchronous 8-byte copies, as is every halo when there are no tensor maps
            bool tma = false;
            if (DO_INTERP) {
                tma = pr.use_tma != 0;
                if (PER) {
#pragma unroll
                    for (int d = 0; d < 3; ++d) tma = tma && t3[d] > 0 && TT * t3[d] + 6 <= n[d];
                }
            }
            int halo_tag = 0;                                // phase of halo[b] + 1 for the consumers to wait on; 0: none
            if (DO_INTERP && tma) {
                halo_tag = 1 + (int)((halo_phase >> b) & 1u);
                halo_phase ^= 1u << b;
                if (tid == 0) {
                    const unsigned hb = mbar + 32 + 8 * b, dst = (unsigned)__cvta_generic_to_shared(su);
                    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");      // earlier generic-proxy accesses to the buffer come first
                    ib_mbar_expect_tx(hb, 3 * TH3 * 8);
#pragma unroll
                    for (int c = 0; c < 3; ++c) ib_tma_box(dst + c * (SU3 * 8), &pr.tm[c], TT * t3[0] - 2, TT * t3[1] - 2, TT * t3[2] - 2, hb);
                }
            } else if (DO_INTERP) {
                for (int idx = tid; idx < 3 * TH3; idx += TBP) {
                    int c = idx >> 9, r = idx & 511;
                    int i = h0[0] + (r & 7), j = h0[1] + ((r >> 3) & 7), k = h0[2] + (r >> 6);
                    if (PER) { i -= (i >= n[0]) ? n[0] : 0; j -= (j >= n[1]) ? n[1] : 0; k -= (k >= n[2]) ? n[2] : 0; }
                    // faces outside a bounded grid read as zero (source size 0: their weight meets no force and no velocity)
                    const bool in = PER || (i >= 0 && i < n[0] && j >= 0 && j < n[1] && k >= 0 && k < n[2]);
                    const double *src = in ? pr.fld[c] + ((int64_t)k * n[1] + j) * n[0] + i : pr.fld[c];
                    const unsigned dst = (unsigned)__cvta_generic_to_shared(su + c * SU3 + (r >> 6) * SZ + (r & 63));
                    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(dst), "l"(src), "r"(in ? 8 : 0) : "memory");
                }
                asm volatile("cp.async.commit_group;" ::: "memory");
            }
            // ---- items: runs of records and point count; rank among the units of equal component and count ----
            int my_nf[NIT], my_rf[NIT], my_rem[NIT], my_rr[NIT];     // whole units of the item and their first rank, points and rank of the last unit
#pragma unroll
            for (int j = 0; j < NIT; ++j) {
                const int it = tid + j * TBP;
                my_nf[j] = 0; my_rf[j] = 0; my_rem[j] = 0; my_rr[j] = 0;
                if (it < NITEM) {
                    int c, l[3], lo[3], hi[3];
                    ib_item_decode(it, c, l);
#pragma unroll
                    for (int d = 0; d < 3; ++d) ib_half_range(c, d, l[d], lo[d], hi[d]);
                    unsigned rn[4];
                    int cnt = 0;
#pragma unroll
                    for (int rr = 0; rr < 4; ++rr) {
                        const int z2 = lo[2] + (rr >> 1), y2 = lo[1] + (rr & 1);
                        const bool ok = z2 <= hi[2] && y2 <= hi[1];
                        const int bb = (z2 * 8 + y2) * 8;
                        const unsigned s0 = ok ? oc_start[bb + lo[0]] : 0, s1 = ok ? oc_start[bb + hi[0] + 1] : 0;
                        rn[rr] = s0 | (s1 << 16);
                        cnt += (int)(s1 - s0);
                    }
                    item_runs[it] = make_uint4(rn[0], rn[1], rn[2], rn[3]);
                    my_nf[j] = cnt / PCAP;
                    my_rem[j] = cnt - PCAP * my_nf[j];
                    if (my_nf[j] > 0) my_rf[j] = atomicAdd(&bins[c * NBIN + PCAP], my_nf[j]);
                    if (my_rem[j] > 0) my_rr[j] = atomicAdd(&bins[c * NBIN + my_rem[j]], 1);
                }
            }
            // ---- the records, in half-cell order: six (a,q) sets, force / h^3, id ------------------------
#pragma unroll
            for (int k = 0; k < KPT; ++k) {
                if (ks[k] >= 0) {
                    const int i = tid + k * TBP;
                    double Gr[4] = {0.0, 0.0, 0.0, 0.0};
                    if (DO_SPREAD) ib_load_rec(pr.rec + (size_t)(cb + i) * 8 + 4, Gr);
                    const int key = ks[k] & 511;
                    const int pos = oc_start[key] + (ks[k] >> 9);
                    assert(pos >= 0 && pos < cn && cn <= CH);
#pragma unroll
                    for (int d = 0; d < 3; ++d) {
                        // face-aligned: cell hd >> 1; centre-aligned: shifted cell (hd + 1) >> 1 covers xi - 1/2 in [l-1, l).
                        // r in [0,1] up to rounding at cell boundaries, where the formula continues phi smoothly (A19)
                        const int hd = (key >> (3 * d)) & 7;
                        sets[(2 * d) * CH + pos] = ib_aq(xi[k][d] - ib_i2d(hd >> 1));
                        sets[(2 * d + 1) * CH + pos] = ib_aq(xi[k][d] + 0.5 - ib_i2d((hd + 1) >> 1));
                    }
                    if (DO_SPREAD) {
#pragma unroll
                        for (int d = 0; d < 3; ++d) sGs[d * CH + pos] = Gr[d] * pr.ih3;
                    }
                    if (DO_INTERP) sids[pos] = idr[k];
                }
            }
            if (DO_INTERP) asm volatile("cp.async.wait_group 0;" ::: "memory");      // this thread's part of the halo has landed
            ib_producer_sync();
            // ---- order the units by component, then by point count (descending): every warp scans the 3 x PCAP
            // bins for itself (lane l: the units of PCAP - l points).  Unit k of component c goes to order[c][k] as
            // item | part << 9; batch b of the item loop is the 8 units 8 (b / 3) ... of component b % 3, so that the
            // batches come in roughly descending size whatever their component (longest first keeps the warps level
            // at the end of the work item).
            {
                int pre[3], ncomp[3];
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    const int v = lane < PCAP ? bins[c * NBIN + PCAP - lane] : 0;
                    int inc = v;
#pragma unroll
                    for (int o = 1; o < 32; o <<= 1) {
                        int t = __shfl_up_sync(0xffffffffu, inc, o);
                        if (lane >= o) inc += t;
                    }
                    pre[c] = inc - v;
                    ncomp[c] = __shfl_sync(0xffffffffu, inc, 31);
                }
                static_assert(PCAP <= 32 && PCAP % 4 == 0, "one lane per unit size; the item loop steps by 4 points");
#pragma unroll
                for (int j = 0; j < NIT; ++j) {
                    if (wid * 32 + j * TBP < NITEM) {                // warp-uniform: some lane of this warp has an item
                        const int it = tid + j * TBP;
                        const int c = it >= 200 ? 2 : (it >= 100 ? 1 : 0);
                        // the owner lane of the size cannot know the asker's component, so all three prefixes travel
                        const int owner = PCAP - max(my_rem[j], 1);
                        const int a0 = __shfl_sync(0xffffffffu, pre[0], owner), a1 = __shfl_sync(0xffffffffu, pre[1], owner),
                                  a2 = __shfl_sync(0xffffffffu, pre[2], owner);
                        unsigned short *oc = order + c * NORD;
                        assert(ncomp[c] <= NORD && my_rf[j] + my_nf[j] <= ncomp[c]);
                        for (int pp = 0; pp < my_nf[j]; ++pp) oc[my_rf[j] + pp] = (unsigned short)(it | (pp << 9));   // units of PCAP points come first
                        if (my_rem[j] > 0) oc[(c == 0 ? a0 : (c == 1 ? a1 : a2)) + my_rr[j]] = (unsigned short)(it | (my_nf[j] << 9));
                    }
                }
                if (tid == 0) {
                    ctl[1] = ncomp[0]; ctl[2] = ncomp[1]; ctl[3] = ncomp[2];
                    ctl[4] = 0;                                  // batch counter
                    ctl[5] = h0[0]; ctl[6] = h0[1]; ctl[7] = h0[2];
                    ctl[8] = halo_tag;
                    ctl[0] = 3 * ((max(ncomp[0], max(ncomp[1], ncomp[2])) + 7) >> 3);
                }
            }
            ib_producer_sync();                              // every producer's records and units are written ...
            if (tid == 0) ib_mbar_arrive(mbar + 8 * b);      // ... and, through this arrival, visible to the consumers
        }
    } else {
        // =================================== consumers ==========================================================
        const int grp = lane >> 2, q = lane & 3;
        // lane q's own x-weight from (a, q):  w = sg q + (sa a + ca)
        double wsa = q < 2 ? 1.0 : -1.0, wca = q < 2 ? 0.0 : 0.5, wsg = (q == 1 || q == 2) ? 1.0 : -1.0;
        ib_opaque(wsa); ib_opaque(wca); ib_opaque(wsg);
        for (int iter = 0;; ++iter) {
            const int b = iter & 1;
            unsigned char *buf = smraw + b * BUF_BYTES;
            ib_mbar_wait(mbar + 8 * b, (iter >> 1) & 1);
            int *ctl = reinterpret_cast<int *>(buf + OFF_CTL);
            const int nbatch = ctl[0];
            if (nbatch < 0) break;
            const int ncomp[3] = {ctl[1], ctl[2], ctl[3]};
            const int h0[3] = {ctl[5], ctl[6], ctl[7]};
            if (DO_INTERP && ctl[8] != 0) ib_mbar_wait(mbar + 32 + 8 * b, (unsigned)(ctl[8] - 1));      // the halo came by TMA: wait for its bytes
            const unsigned short *order = reinterpret_cast<const unsigned short *>(buf + OFF_ORDER);
            ib_tile_smem sm;
            sm.su = (unsigned)__cvta_generic_to_shared(buf + OFF_SU); sm.sets = (unsigned)__cvta_generic_to_shared(buf + OFF_SETS);
            sm.sGs = (unsigned)__cvta_generic_to_shared(buf + OFF_SG); sm.sids = (unsigned)__cvta_generic_to_shared(buf + OFF_SIDS);
            ib_opaque(sm.su); ib_opaque(sm.sets); ib_opaque(sm.sGs); ib_opaque(sm.sids);
            sm.item_runs = reinterpret_cast<const uint4 *>(buf + OFF_RUNS); sm.item_win = item_win;
            // batches of 8 units of one component; the next batch is claimed one batch ahead: the shared-memory
            // atomic and its broadcast are out of the way
            int bnext = 0;
            if (lane == 0) bnext = atomicAdd(&ctl[4], 1);
            for (;;) {
                const int bt = __shfl_sync(0xffffffffu, bnext, 0);
                if (bt >= nbatch) break;
                if (lane == 0) bnext = atomicAdd(&ctl[4], 1);
                const int c = bt % 3, k8 = (bt / 3) * 8;                                 // warp-uniform
                const int nc = c == 0 ? ncomp[0] : (c == 1 ? ncomp[1] : ncomp[2]);
                if (k8 >= nc) continue;                                                // this component has fewer batches
                const int un = k8 + grp < nc ? (int)order[c * NORD + k8 + grp] : NITEM;      // empty slot: the item without points
                ib_run_batch<DO_SPREAD, DO_INTERP, PER>(c, pr, sm, un & 511, un >> 9, q, h0, n, wsa, wca, wsg);
            }
            __syncwarp();
            if (lane == 0) ib_mbar_arrive(mbar + 16 + 8 * b);    // this warp has left the buffer
        }
    }
}


// Points of tiles with fewer than IB_SMALL_TILE points are not worth a halo and a sort: 4 lanes per point of
// the compact list written by ibk_tile_scan, every point treated directly against the grid (ib_point_quad).
// The spreading half is bound by the L2 reduction units (48 sectors per point), the rest by dependent loads.
// 3 resident CTAs of 128 threads per SM measured best on the sparse workloads (2 / 4 / 5 / 6 / 8: DESIGN.md): the
// compiler keeps all offsets and weights of a component in registers, and the kernel leaves the L2 more room
#ifndef IB_SMALL_MINB
#define IB_SMALL_MINB 3
#endif
#define IB_SMALL_TB 128
template <int DO_SPREAD, int DO_INTERP, int PER>
__global__ void __launch_bounds__(IB_SMALL_TB, IB_SMALL_MINB)
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
        const double *rc = pr.rec + (size_t)r * 8;
        if (DO_SPREAD) { G[0] = rc[4] * pr.ih3; G[1] = rc[5] * pr.ih3; G[2] = rc[6] * pr.ih3; }
        ib_point_quad<DO_SPREAD, DO_INTERP, PER>(rc[0], rc[1], rc[2], G, pr.fld, pr.frc, pr.g, pr.inv_h, q, qmask, U);
        if (DO_INTERP && q == 0) {
            const int id = (int)__double_as_longlong(rc[3]);
            pr.Up[id] = U[0]; pr.Up[P + id] = U[1]; pr.Up[2 * P + id] = U[2];
        }
    }
}

// blocks of the sparse-tile kernel: enough for the longest possible list, at most 64 per SM (grid stride; 3 are
// resident -- many short CTAs level the end of the kernel: 3 / 6 / 16 / 256 / 2048 per SM measured)
static int ib_small_blocks(int64_t nsmall_max, int sms)
{
    const int64_t need = (nsmall_max * 4 + IB_SMALL_TB - 1) / IB_SMALL_TB;
    const int64_t cap = (int64_t)(sms > 0 ? sms : 148) * 64;
    return (int)(need < 1 ? 1 : (need < cap ? need : cap));
}

template <int S, int I, int PER>
static ib_status launch_tiled_p(ib_ctx *c, const ib_tiled_params &pr, bool with_small, cudaStream_t st)
{
    const size_t smem = TILED_SMEM_BYTES;
    static_assert(CH % 16 == 0 && TILED_SMEM_BYTES <= 227 * 1024, "staging layout");
    // per context (a context belongs to one device and, by the header's contract, to one thread at a time)
    unsigned char &configured = c->tiled_cfg[S * 4 + I * 2 + PER];
    if (!configured) {
        IB_CUDA_TRY(cudaFuncSetAttribute(ibk_tiled_kernel<S, I, PER>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        configured = 1;
    }
    if (!c->sm_count) IB_CUDA_TRY(cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, c->device));
    const int sms = c->sm_count;
    // the few points of sparsely filled tiles go one by one on a second stream, beside the tile kernel
    const int64_t nsmall_max = min((int64_t)pr.P, (c->n_cells / (TT * TT * TT)) * (int64_t)(IB_SMALL_TILE - 1));
    const bool beside = !c->profile && with_small;
    cudaStream_t s3 = beside ? c->side2 : st;
    if (beside) {
        IB_CUDA_TRY(cudaEventRecord(c->ev_sfork, st));
        IB_CUDA_TRY(cudaStreamWaitEvent(s3, c->ev_sfork, 0));
    }
    if (with_small) ibk_small_tiles<S, I, PER><<<ib_small_blocks(nsmall_max, sms), IB_SMALL_TB, 0, s3>>>(pr, c->d_small_rec, c->d_tile_count);
    if (beside) IB_CUDA_TRY(cudaEventRecord(c->ev_sjoin, s3));
    ibk_tiled_kernel<S, I, PER><<<sms, TB, smem, st>>>(pr);
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

// cuTensorMapEncodeTiled of the driver, through the runtime's entry-point query (the library does not link libcuda)
typedef CUresult (*ib_tma_encode_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                     const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                     CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static ib_tma_encode_fn ib_tma_encoder()
{
    static ib_tma_encode_fn fn = []() -> ib_tma_encode_fn {
        void *f = nullptr;
        cudaDriverEntryPointQueryResult q = cudaDriverEntryPointSymbolNotFound;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess) {
            (void)cudaGetLastError();
            return nullptr;
        }
        return reinterpret_cast<ib_tma_encode_fn>(f);
    }();
    return fn;
}

// u, v, w as 3-D tensors for the halo loads of the tile kernel.  Returns false (the kernel then copies every halo
// element by element) when the driver has no encoder or refuses the arrays: a pointer that is not 16-byte aligned.
static bool ib_halo_maps(const ib_grid_desc &g, const double *const fld[3], CUtensorMap tm[3])
{
    ib_tma_encode_fn enc = ib_tma_encoder();
    if (!enc) return false;
    const cuuint64_t dims[3] = {(cuuint64_t)g.nx, (cuuint64_t)g.ny, (cuuint64_t)g.nz};
    const cuuint64_t strides[2] = {(cuuint64_t)g.nx * 8, (cuuint64_t)g.nx * g.ny * 8};
    const cuuint32_t box[3] = {TH, TH, TH}, estr[3] = {1, 1, 1};
    for (int c = 0; c < 3; ++c) {
        if (!fld[c] || (reinterpret_cast<uintptr_t>(fld[c]) & 15u)) return false;
        if (enc(&tm[c], CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, const_cast<double *>(fld[c]), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
            return false;
    }
    return true;
}

static void fill_params(ib_ctx *c, ib_tiled_params &pr, int64_t P, const double *u, const double *v, const double *w,
                        double *fu, double *fv, double *fw, double *Up, int slab)
{
    memset(&pr, 0, sizeof(pr));
    pr.rec = c->d_rec; pr.P = P;
    pr.fld[0] = u; pr.fld[1] = v; pr.fld[2] = w;
    pr.frc[0] = fu; pr.frc[1] = fv; pr.frc[2] = fw;
    pr.Up = Up;
    pr.work = c->d_work; pr.counters = c->d_tile_count;
    pr.wb = slab < 0 ? 3 : IB_SLAB0 + slab;
    pr.we = slab < 0 ? 0 : IB_SLAB0 + slab + 1;
    pr.wc = slab < 0 ? 1 : IB_SLABC0 + slab;
    pr.g = c->grid; pr.inv_h = c->inv_h; pr.ih3 = c->inv_h * c->inv_h * c->inv_h;
    pr.use_tma = (u && v && w && Up) ? (ib_halo_maps(c->grid, pr.fld, pr.tm) ? 1 : 0) : 0;
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
    if (slab >= 0) IB_CUDA_TRY(cudaMemsetAsync(c->d_tile_count + pr.wc, 0, sizeof(int32_t), st));   // slab < 0: ibk_tile_scan has just reset counters[1]
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
    const bool per = c->grid.periodic != 0;
    if (do_spread && do_interp) {
        if (per) ibk_small_tiles<1, 1, 1><<<nb, IB_SMALL_TB, 0, st>>>(pr, c->d_small_rec, c->d_tile_count);
        else ibk_small_tiles<1, 1, 0><<<nb, IB_SMALL_TB, 0, st>>>(pr, c->d_small_rec, c->d_tile_count);
    } else if (do_spread) {
        if (per) ibk_small_tiles<1, 0, 1><<<nb, IB_SMALL_TB, 0, st>>>(pr, c->d_small_rec, c->d_tile_count);
        else ibk_small_tiles<1, 0, 0><<<nb, IB_SMALL_TB, 0, st>>>(pr, c->d_small_rec, c->d_tile_count);
    } else {
        if (per) ibk_small_tiles<0, 1, 1><<<nb, IB_SMALL_TB, 0, st>>>(pr, c->d_small_rec, c->d_tile_count);
        else ibk_small_tiles<0, 1, 0><<<nb, IB_SMALL_TB, 0, st>>>(pr, c->d_small_rec, c->d_tile_count);
    }
    c->launches += 1;
    IB_CUDA_TRY(cudaGetLastError());
    return IB_OK;
}
