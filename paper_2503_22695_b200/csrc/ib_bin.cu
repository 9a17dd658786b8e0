// ib_bin.cu -- tile-level counting sort of the Lagrangian force points (SURVEY.md §8(a) a4+a5 fused).
// Not in the paper (north_star: "points binned and sorted by Eulerian cell").
//
// Points are grouped by 4x4x4-cell tile, and inside a tile by z-layer of cells, with a counting sort over
// the bins (tile, layer): count pass -> two-kernel scan (which also emits the tile kernel's work list and
// the list of points of sparsely filled tiles) -> scatter pass that writes the point records (x_s, G_s,
// id) contiguously per bin.  A work item of the tile kernel is a run of whole layers of one tile with at
// most IB_CHUNK points (a layer with more is cut into equal pieces), so the points of a work item are
// neighbours in space and share their stencil windows however densely a tile is filled.  The order of
// points inside a bin is whatever the atomics give; the tile kernel (ib_tiled.cu) sorts them by
// half-cell in shared memory.  Two point sources:
//   cloud : xp/Gp arrays given by the caller (ib_spread / ib_interp, nodal rule of L241)
//   mesh  : sub-points generated on the fly from the element nodes -- x_s = sum_a N_a(xi_s) x_a,
//           G_s = W_s sum_a N_a(xi_s) Fhat_a (reading A13) -- one thread per row of n1 sub-points,
//           so the element-ordered xp/Gp arrays never touch HBM in ib_coupling_step.
// The cell of a point is the binning formula of A21 (IEEE double, no contraction); positions are
// computed with explicit __fma_rn/__dmul_rn so that the count and scatter passes agree bit for bit.
#include <cassert>
#include "ib_common.cuh"

#define BT 4                       // tile edge in cells

struct ib_bin_params {
    // cloud source
    int64_t P;
    const double *xp, *Gp;
    // mesh source
    int64_t n_rows, n_elems, n_nodes;
    int un1, un2, un3;             // uniform nsub (un1 == 0: per-element nsub / row_off / pt_off)
    // uniform nsub: what every row would otherwise divide for (host: ib_bin_uniform)
    int rpe, epc;                  // rows per element n2 n3; elements per CTA of 256 rows when rpe divides 256
    unsigned rpe_m16, n2_m16;      // ceil(2^16 / rpe), ceil(2^16 / n2): a / d = (a * m16) >> 16 for a < 512
    double rn2, rn3;               // 1.0 / n2, 1.0 / n3 (IEEE division, the value the device would form)
    int prefetch_w;                // scatter pass of a large mesh: the quadrature weights of a row are asked for (L1) before the binning
    const int32_t *nsub;
    const int64_t *pt_off, *row_off;
    const int32_t *conn;
    const double *x, *Fhat, *Wp;
    // grid
    ib_grid_desc g;
    double inv_h;
    // bins
    int32_t *tile_cur;             // count pass: counts; scatter pass: running cursors
    double *rec;                   // [P][8] records: {x, y, z, id | G0, G1, G2, -} (two 32-byte halves)
    double *Up;                    // non-finite points get Up = 0 (scatter pass), may be NULL
    long long *status;
};

// bin of a point: 4 x (tile index) + (z-layer of the cell inside its tile)
__device__ __forceinline__ int ib_tile_of(double x, double y, double z, const ib_grid_desc &g, double inv_h)
{
    int cx = ib_cell(x, g.x0, inv_h, g.nx), cy = ib_cell(y, g.y0, inv_h, g.ny), cz = ib_cell(z, g.z0, inv_h, g.nz);
    return ((((cz >> 2) * (g.ny / BT) + (cy >> 2)) * (g.nx / BT) + (cx >> 2)) << 2) | (cz & 3);
}

// The points of a CTA are neighbours in space (rows of the same few elements) and fall into a handful of bins:
// they are counted per CTA in a small shared-memory hash table (native 32-bit shared atomics), and the CTA then
// makes ONE global atomic per distinct bin -- instead of a warp match and a global atomic per point and warp,
// whose returned slot every store of the scatter pass had to wait for.
#define HT 128
struct ib_bin_hash { int key[HT], cnt[HT], base[HT]; };
#define IB_CODE_NONE (-1)          // no record (invalid point)

__device__ __forceinline__ void ib_hash_clear(ib_bin_hash &h)
{
    for (int i = threadIdx.x; i < HT; i += blockDim.x) { h.key[i] = -1; h.cnt[i] = 0; }
}
// count the point in; returns slot | rank << 8, or (table full after 32 probes: clouds scattered all over the
// grid) INT_MIN | the global slot taken at once
template <int SCATTER>
__device__ __forceinline__ int ib_hash_insert(ib_bin_hash &h, int bin, int32_t *tile_cur)
{
    unsigned s = ((unsigned)bin * 2654435761u) >> 25;
    for (int t = 0; t < 32; ++t) {
        const int k = atomicCAS(&h.key[s], -1, bin);
        if (k == -1 || k == bin) return (int)s | (atomicAdd(&h.cnt[s], 1) << 8);
        s = (s + 1) & (HT - 1);
    }
    const int pos = atomicAdd(&tile_cur[bin], 1);
    return SCATTER ? (int)(0x80000000u | (unsigned)pos) : IB_CODE_NONE;
}
// one global atomic per distinct bin of the CTA; barriers inside: every thread of the CTA must call
template <int SCATTER>
__device__ __forceinline__ void ib_hash_flush(ib_bin_hash &h, int32_t *tile_cur)
{
    __syncthreads();
    for (int i = threadIdx.x; i < HT; i += blockDim.x)
        if (h.key[i] >= 0) {
            const int b = atomicAdd(&tile_cur[h.key[i]], h.cnt[i]);
            if (SCATTER) h.base[i] = b;
        }
    if (SCATTER) __syncthreads();
}
__device__ __forceinline__ int ib_hash_pos(const ib_bin_hash &h, int code)
{
    return code < 0 ? (int)((unsigned)code & 0x7fffffffu) : h.base[code & 255] + (code >> 8);
}

// one record: two 32-byte stores, streaming (the records exceed L2 and are read once, oldest first, so keeping
// them out of L2 leaves room for the grid halos)
__device__ __forceinline__ void ib_store_rec(double *rec, int pos, double x, double y, double z, int id,
                                             bool with_g, double g0, double g1, double g2)
{
    double *r = rec + (size_t)pos * 8;
    asm volatile("st.global.cs.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(r), "d"(x), "d"(y), "d"(z), "d"(__longlong_as_double((long long)id)) : "memory");
    if (with_g) asm volatile("st.global.cs.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(r + 4), "d"(g0), "d"(g1), "d"(g2), "d"(0.0) : "memory");
}

// ---- cloud source ------------------------------------------------------------------------------
template <int SCATTER>
__global__ void __launch_bounds__(256)
ibk_bin_cloud(ib_bin_params pr)
{
    __shared__ ib_bin_hash h;
    ib_hash_clear(h);
    __syncthreads();
    const int64_t P = pr.P;
    int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    bool valid = p < P;
    double x = 0, y = 0, z = 0;
    if (valid) {
        x = __ldg(pr.xp + p); y = __ldg(pr.xp + P + p); z = __ldg(pr.xp + 2 * P + p);
        if (!(isfinite(x) && isfinite(y) && isfinite(z))) {
            if (SCATTER) {
                ib_latch(pr.status, IB_ERR_NONFINITE, p);
                if (pr.Up) { pr.Up[p] = 0.0; pr.Up[P + p] = 0.0; pr.Up[2 * P + p] = 0.0; }
            }
            valid = false;
        } else if (!pr.g.periodic && !ib_in_box(x, y, z, pr.g, pr.inv_h)) {
            if (SCATTER) {
                ib_latch(pr.status, IB_ERR_OUT_OF_DOMAIN, p);
                if (pr.Up) { pr.Up[p] = 0.0; pr.Up[P + p] = 0.0; pr.Up[2 * P + p] = 0.0; }
            }
            valid = false;
        }
    }
    const int code = valid ? ib_hash_insert<SCATTER>(h, ib_tile_of(x, y, z, pr.g, pr.inv_h), pr.tile_cur) : IB_CODE_NONE;
    ib_hash_flush<SCATTER>(h, pr.tile_cur);
    if (SCATTER && valid) {
        const int pos = ib_hash_pos(h, code);
        assert(pos >= 0 && pos < P);
        const bool wg = pr.Gp != nullptr;
        ib_store_rec(pr.rec, pos, x, y, z, (int)p, wg, wg ? __ldg(pr.Gp + p) : 0.0, wg ? __ldg(pr.Gp + P + p) : 0.0,
                     wg ? __ldg(pr.Gp + 2 * P + p) : 0.0);
    }
}

// ---- mesh source: one thread per row (e, m2, m3) of n1 sub-points ----------------------------------
__device__ __forceinline__ int64_t ib_find_row_elem(const int64_t *__restrict__ off, int64_t n_elems, int64_t r)
{
    int64_t lo = 0, hi = n_elems;                 // off[lo] <= r < off[hi]
    while (hi - lo > 1) {
        int64_t mid = (lo + hi) >> 1;
        if (__ldg(off + mid) <= r) lo = mid; else hi = mid;
    }
    return lo;
}

// bilinear combination of the 4 nodes (ja,ka) of one x-face of the element, no contraction freedom
__device__ __forceinline__ double ib_face_lerp(double w00, double w10, double w01, double w11,
                                               double v0, double v2, double v4, double v6)
{
    return __fma_rn(w11, v6, __fma_rn(w01, v4, __fma_rn(w10, v2, __dmul_rn(w00, v0))));
}

// STAGE: uniform nsub with 4 <= n2*n3 dividing 256 -- the CTA's 256 rows are 256/(n2 n3) whole elements,
// whose node positions (and force coefficients) are staged once in shared memory instead of being
// gathered by every row.
// N1: the number of sub-points of a row when the rule is uniform with 2 or 4 of them (the loops over the points of a
// row are unrolled for registers: 8 copies of which a 4-point rule skips half -- the code of the generic kernel is
// 5,900 instructions long and a row executes 1,100 of them, which the instruction cache does not like); 0: any rule
template <int SCATTER, int STAGE, int N1>
__global__ void __launch_bounds__(256, 4)
ibk_bin_mesh(ib_bin_params pr)
{
    constexpr int NJ = N1 > 0 ? N1 : 8;
    __shared__ double s_nd[STAGE ? 16 * 8 * 6 : 1];       // [element of the CTA][local node][x0 x1 x2 F0 F1 F2]
    __shared__ ib_bin_hash h;
    __shared__ long long s_e0;                            // uniform rule, rows not staged: element and row inside it of the CTA's first row
    __shared__ int s_r0;
    ib_hash_clear(h);
    if (!STAGE && threadIdx.x == 0 && pr.un1 > 0) {       // one 64-bit division per CTA instead of one per row
        const long long base = (long long)blockIdx.x * blockDim.x;
        s_e0 = base / pr.rpe;
        s_r0 = (int)(base - s_e0 * pr.rpe);
    }
    if (!STAGE) __syncthreads();
    if (STAGE) {
        const int epc = pr.epc;
        const int64_t e_first = (int64_t)blockIdx.x * epc;
        for (int i = threadIdx.x; i < epc * 8; i += 256) {
            const int64_t ee = e_first + (i >> 3);
            if (ee < pr.n_elems) {
                const int nd = __ldg(pr.conn + ee * 8 + (i & 7));
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    s_nd[i * 6 + c] = __ldg(pr.x + (int64_t)c * pr.n_nodes + nd);
                    if (SCATTER && pr.Fhat) s_nd[i * 6 + 3 + c] = __ldg(pr.Fhat + (int64_t)c * pr.n_nodes + nd);
                }
            }
        }
        __syncthreads();
    }
    int64_t row = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    bool live = row < pr.n_rows;
    int64_t e = 0, p0 = 0;
    int n1 = 0, n2 = 1, n3 = 1, m2 = 0, m3 = 0;
    if (live) {
        int r;
        if (pr.un1 > 0) {
            n1 = N1 > 0 ? N1 : pr.un1; n2 = pr.un2; n3 = pr.un3;
            const int rpe = pr.rpe;
            // row = 256 blockIdx + thread: the element comes from the CTA's first row and a division of a number
            // below 512 by rpe <= 64, which is a multiplication (exact: a (m16 d - 2^16) < 2^16 for a < 512, d <= 64)
            const int rr = (STAGE ? 0 : s_r0) + (int)threadIdx.x;
            const int el = (int)(((unsigned)rr * pr.rpe_m16) >> 16);
            e = (STAGE ? (int64_t)blockIdx.x * pr.epc : (int64_t)s_e0) + el;
            r = rr - el * rpe;
            assert(e == row / rpe && r == (int)(row - e * rpe));
            p0 = e * (int64_t)(n1 * rpe) + (int64_t)r * n1;
        } else {
            e = ib_find_row_elem(pr.row_off, pr.n_elems, row);
            n1 = __ldg(pr.nsub + 3 * e); n2 = __ldg(pr.nsub + 3 * e + 1); n3 = __ldg(pr.nsub + 3 * e + 2);
            r = (int)(row - __ldg(pr.row_off + e));
            p0 = __ldg(pr.pt_off + e) + (int64_t)r * n1;
        }
        if (pr.un1 > 0) { m3 = (int)(((unsigned)r * pr.n2_m16) >> 16); m2 = r - m3 * n2; }
        else { m2 = r % n2; m3 = r / n2; }
        assert(m3 == r / n2 && m2 == r % n2);
    }
    double L[3] = {0, 0, 0}, D[3] = {0, 0, 0}, LF[3] = {0, 0, 0}, DF[3] = {0, 0, 0};
    bool finite = true;
    if (live) {
        int nd[8] = {0, 0, 0, 0, 0, 0, 0, 0};
        const double *sn = s_nd;
        if (STAGE) {
            sn = s_nd + (int)(e - (int64_t)blockIdx.x * pr.epc) * 48;
        } else {
            const int4 *cp = reinterpret_cast<const int4 *>(pr.conn + e * 8);
            int4 c0 = __ldg(cp), c1 = __ldg(cp + 1);
            nd[0] = c0.x; nd[1] = c0.y; nd[2] = c0.z; nd[3] = c0.w;
            nd[4] = c1.x; nd[5] = c1.y; nd[6] = c1.z; nd[7] = c1.w;
        }
        // N-weights of the row: 1/2 (1 +- xi) with xi = -1 + (2m+1)/n  ->  (m + 1/2)/n and its complement
        const double rn2 = pr.un1 > 0 ? pr.rn2 : 1.0 / (double)n2, rn3 = pr.un1 > 0 ? pr.rn3 : 1.0 / (double)n3;
        double b1 = ((double)m2 + 0.5) * rn2, g1 = ((double)m3 + 0.5) * rn3;
        double b0 = 1.0 - b1, g0 = 1.0 - g1;
        double w00 = __dmul_rn(b0, g0), w10 = __dmul_rn(b1, g0), w01 = __dmul_rn(b0, g1), w11 = __dmul_rn(b1, g1);
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const double *xc = pr.x + (int64_t)c * pr.n_nodes;
            double v[8];
#pragma unroll
            for (int a = 0; a < 8; ++a) {
                v[a] = STAGE ? sn[a * 6 + c] : __ldg(xc + nd[a]);
                finite = finite && isfinite(v[a]);
            }
            L[c] = ib_face_lerp(w00, w10, w01, w11, v[0], v[2], v[4], v[6]);
            double R = ib_face_lerp(w00, w10, w01, w11, v[1], v[3], v[5], v[7]);
            D[c] = __dsub_rn(R, L[c]);
            if (SCATTER && pr.Fhat) {
                const double *fc = pr.Fhat + (int64_t)c * pr.n_nodes;
#pragma unroll
                for (int a = 0; a < 8; ++a) v[a] = STAGE ? sn[a * 6 + 3 + c] : __ldg(fc + nd[a]);
                LF[c] = ib_face_lerp(w00, w10, w01, w11, v[0], v[2], v[4], v[6]);
                DF[c] = ib_face_lerp(w00, w10, w01, w11, v[1], v[3], v[5], v[7]) - LF[c];
            }
        }
        if (!finite) {
            if (SCATTER) {
                ib_latch(pr.status, IB_ERR_NONFINITE, e);
                if (pr.Up)
                    for (int j = 0; j < n1; ++j) { pr.Up[p0 + j] = 0.0; pr.Up[pr.P + p0 + j] = 0.0; pr.Up[2 * pr.P + p0 + j] = 0.0; }
            }
            live = false;
        }
    }
    // the weights W_s of the row are read after two barriers: their line is on its way meanwhile (large meshes only:
    // at C1 the extra instruction costs 2 us of a 13 us kernel, at C3 it takes 3 % off the scatter pass)
    if (SCATTER && pr.prefetch_w && live && pr.Fhat) asm volatile("prefetch.global.L1 [%0];" ::"l"(pr.Wp + p0));
    // ---- the n1 points of the row: position, bin, count in the CTA's table ------------------------------
    const double rn1 = 1.0 / (double)(n1 > 0 ? n1 : 1);
    int code[NJ];                                  // nsub <= 8 (ib_create)
#pragma unroll
    for (int j = 0; j < NJ; ++j) {
        code[j] = IB_CODE_NONE;
        if (live && j < n1) {
            const double t = ((double)j + 0.5) * rn1;
            const double x = __fma_rn(t, D[0], L[0]), y = __fma_rn(t, D[1], L[1]), z = __fma_rn(t, D[2], L[2]);
            if (!pr.g.periodic && !ib_in_box(x, y, z, pr.g, pr.inv_h)) {      // outside a bounded grid
                if (SCATTER) {
                    ib_latch(pr.status, IB_ERR_OUT_OF_DOMAIN, e);
                    if (pr.Up) { pr.Up[p0 + j] = 0.0; pr.Up[pr.P + p0 + j] = 0.0; pr.Up[2 * pr.P + p0 + j] = 0.0; }
                }
            } else {
                const int c = ib_hash_insert<SCATTER>(h, ib_tile_of(x, y, z, pr.g, pr.inv_h), pr.tile_cur);
                code[j] = SCATTER ? c : 0;
            }
        }
    }
    ib_hash_flush<SCATTER>(h, pr.tile_cur);
    if (SCATTER) {
#pragma unroll
        for (int j = 0; j < NJ; ++j) {
            if (live && j < n1 && code[j] != IB_CODE_NONE) {
                const double t = ((double)j + 0.5) * rn1;
                const double x = __fma_rn(t, D[0], L[0]), y = __fma_rn(t, D[1], L[1]), z = __fma_rn(t, D[2], L[2]);
                const int pos = ib_hash_pos(h, code[j]);
                assert(pos >= 0 && pos < pr.P);
                double g0 = 0.0, g1 = 0.0, g2 = 0.0;
                if (pr.Fhat) {
                    const double W = __ldg(pr.Wp + p0 + j);
                    g0 = W * fma(t, DF[0], LF[0]); g1 = W * fma(t, DF[1], LF[1]); g2 = W * fma(t, DF[2], LF[2]);
                }
                ib_store_rec(pr.rec, pos, x, y, z, (int)(p0 + j), pr.Fhat != nullptr, g0, g1, g2);
            }
        }
    }
}

// ---- scan over the tiles (two small kernels, one thread per tile = 4 bins): start offsets, cursors, work
// list, compact list of the records of sparsely filled tiles ------------------------------------------
#define SCT 1024
#define IB_MIN_CHUNK 128           // smallest work item of the tile kernel (points) that the work list is cut into

__device__ __forceinline__ void ib_block_scan2(int &a, int &b, int *ws, int *wl, int &ta, int &tb)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    int ia = a, ib = b;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int x = __shfl_up_sync(0xffffffffu, ia, o), y = __shfl_up_sync(0xffffffffu, ib, o);
        if (lane >= o) { ia += x; ib += y; }
    }
    if (lane == 31) { ws[wid] = ia; wl[wid] = ib; }
    __syncthreads();
    if (wid == 0) {
        int x = ws[lane], y = wl[lane], ix = x, iy = y;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int p = __shfl_up_sync(0xffffffffu, ix, o), r = __shfl_up_sync(0xffffffffu, iy, o);
            if (lane >= o) { ix += p; iy += r; }
        }
        ws[lane] = ix - x; wl[lane] = iy - y;
        if (lane == 31) { ws[32] = ix; wl[32] = iy; }
    }
    __syncthreads();
    ta = ws[32]; tb = wl[32];
    a = ws[wid] + ia - a;                          // exclusive prefixes
    b = wl[wid] + ib - b;
}

// Work items of one tile whose 4 z-layers hold c.x .. c.w points (records start at `first`): runs of whole
// layers with at most `chunk` points; a layer with more is cut into equal pieces.  chunk = IB_CHUNK (the
// tile kernel's staging capacity) for large clouds, smaller for small ones so that a few densely filled
// tiles still spread over many CTAs.  EMIT: write {tile, first record, points, tile coordinates} to work[l ...].
// Returns the number of work items (0 for a sparsely filled tile: its points go one by one).
template <int EMIT>
__device__ __forceinline__ int ib_tile_chunks(const int4 c, int chunk, int tile, int first, int4 *__restrict__ work, int l, int ntx, int nty)
{
    const int tw = EMIT ? ((tile % ntx) | (((tile / ntx) % nty) << 10) | ((tile / (ntx * nty)) << 20)) : 0;   // tile coordinates (grids up to 4096 cells an edge)
    const int cnt[4] = {c.x, c.y, c.z, c.w};
    if (c.x + c.y + c.z + c.w < IB_SMALL_TILE) return 0;
    int n = 0, acc = 0, beg = first;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        if (cnt[k] > chunk) {
            if (acc > 0) {
                if (EMIT) work[l + n] = make_int4(tile, beg, acc, tw);
                ++n; beg += acc; acc = 0;
            }
            const int pieces = (cnt[k] + chunk - 1) / chunk, per = (cnt[k] + pieces - 1) / pieces;
            for (int o = 0; o < cnt[k]; o += per) {
                if (EMIT) work[l + n] = make_int4(tile, beg + o, min(per, cnt[k] - o), tw);
                ++n;
            }
            beg += cnt[k];
        } else if (acc + cnt[k] > chunk) {
            if (EMIT) work[l + n] = make_int4(tile, beg, acc, tw);
            ++n; beg += acc; acc = cnt[k];
        } else acc += cnt[k];
    }
    if (acc > 0) {
        if (EMIT) work[l + n] = make_int4(tile, beg, acc, tw);
        ++n;
    }
    return n;
}

__global__ void __launch_bounds__(SCT)
ibk_tile_partials(const int32_t *__restrict__ tile_cur, int n_tiles, int chunk, int2 *__restrict__ partial)
{
    __shared__ int ws[33], wl[33];
    const int t = blockIdx.x * SCT + threadIdx.x;
    int s = 0, l = 0;
    if (t < n_tiles) {
        const int4 c = *reinterpret_cast<const int4 *>(tile_cur + 4 * t);
        s = c.x + c.y + c.z + c.w;
        l = ib_tile_chunks<0>(c, chunk, t, 0, nullptr, 0, 1, 1);
    }
    int ts, tl;
    ib_block_scan2(s, l, ws, wl, ts, tl);
    if (threadIdx.x == 0) partial[blockIdx.x] = make_int2(ts, tl);
}

// start offsets and cursors of the bins, and the work list
__global__ void __launch_bounds__(SCT)
ibk_tile_scan(int32_t *__restrict__ tile_cur, int n_tiles, int chunk, const int2 *__restrict__ partial,
              int32_t *__restrict__ tile_start, int4 *__restrict__ work, int32_t *__restrict__ small_rec,
              int32_t *__restrict__ counters, int slab_tiles, int ntx, int nty, int work_cap)
{
    __shared__ int ws[33], wl[33];
    __shared__ int base_s, base_l, base_m;
    if (threadIdx.x < 32) {
        int s = 0, l = 0;
        for (int b = threadIdx.x; b < (int)blockIdx.x; b += 32) { int2 p = partial[b]; s += p.x; l += p.y; }
#pragma unroll
        for (int o = 16; o >= 1; o >>= 1) { s += __shfl_xor_sync(0xffffffffu, s, o); l += __shfl_xor_sync(0xffffffffu, l, o); }
        if (threadIdx.x == 0) { base_s = s; base_l = l; }
    }
    const int t = blockIdx.x * SCT + threadIdx.x;
    int4 c = make_int4(0, 0, 0, 0);
    if (t < n_tiles) c = *reinterpret_cast<const int4 *>(tile_cur + 4 * t);
    const int tot = c.x + c.y + c.z + c.w;
    int s = tot, l = ib_tile_chunks<0>(c, chunk, t, 0, nullptr, 0, 1, 1);
    int ts, tl;
    ib_block_scan2(s, l, ws, wl, ts, tl);          // includes the barrier that publishes base_s/base_l
    s += base_s; l += base_l;
    // first work item of every slab of slab_tiles tiles: ib_coupling_step_host launches the tile kernel slab
    // by slab so that the copies of f overlap the spreading of the next slab
    if (t < n_tiles && t % slab_tiles == 0) counters[IB_SLAB0 + t / slab_tiles] = l;
    if (t < n_tiles) {
        const int4 st = make_int4(s, s + c.x, s + c.x + c.y, s + c.x + c.y + c.z);
        *reinterpret_cast<int4 *>(tile_start + 4 * t) = st;
        *reinterpret_cast<int4 *>(tile_cur + 4 * t) = st;
        assert(l + ib_tile_chunks<0>(c, chunk, t, 0, nullptr, 0, 1, 1) <= work_cap);
        ib_tile_chunks<1>(c, chunk, t, s, work, l, ntx, nty);
    }
    {   // records of sparsely filled tiles: a compact list (order across CTAs is whatever the atomic gives)
        int m = (t < n_tiles && tot < IB_SMALL_TILE) ? tot : 0, zero = 0, tm, tz;
        const int mine = m;
        __syncthreads();                           // the first scan's totals have been read by every thread
        ib_block_scan2(m, zero, ws, wl, tm, tz);
        if (threadIdx.x == 0) base_m = tm ? atomicAdd(&counters[2], tm) : 0;
        __syncthreads();
        m += base_m;
        for (int o = 0; o < mine; ++o) small_rec[m + o] = s + o;
    }
    if (blockIdx.x == gridDim.x - 1 && threadIdx.x == 0) {
        tile_start[4 * n_tiles] = base_s + ts;
        counters[0] = base_l + tl;
        counters[1] = 0;
        for (int k = (n_tiles + slab_tiles - 1) / slab_tiles; k <= IB_MAX_SLABS; ++k) counters[IB_SLAB0 + k] = base_l + tl;
    }
}

// phases: 1 = count pass + scan (needs only the positions), 2 = scatter pass (needs the forces too)
ib_status ibk_bin_points(ib_ctx *c, int mesh, const double *xp, const double *Gp, int64_t P,
                         const double *x, const double *Fhat, double *Up, int phases, cudaStream_t st)
{
    const int n_tiles = (int)(c->n_cells / (BT * BT * BT));
    ib_bin_params pr;
    memset(&pr, 0, sizeof(pr));
    pr.P = P; pr.xp = xp; pr.Gp = Gp;
    pr.n_rows = c->n_rows; pr.n_elems = c->n_elems; pr.n_nodes = c->n_nodes;
    pr.un1 = c->un[0]; pr.un2 = c->un[1]; pr.un3 = c->un[2];
    if (pr.un1 > 0) {
        pr.rpe = pr.un2 * pr.un3;
        pr.epc = 256 / pr.rpe;
        pr.rpe_m16 = (65536u + (unsigned)pr.rpe - 1u) / (unsigned)pr.rpe;
        pr.n2_m16 = (65536u + (unsigned)pr.un2 - 1u) / (unsigned)pr.un2;
        pr.rn2 = 1.0 / (double)pr.un2;
        pr.rn3 = 1.0 / (double)pr.un3;
    }
    pr.nsub = c->d_nsub; pr.pt_off = c->d_pt_off; pr.row_off = c->d_row_off; pr.conn = c->d_conn;
    pr.x = x; pr.Fhat = Fhat; pr.Wp = c->d_Wp;
    pr.g = c->grid; pr.inv_h = c->inv_h;
    pr.tile_cur = c->d_tile_cur; pr.rec = c->d_rec;
    pr.Up = Up; pr.status = c->d_status;
    pr.prefetch_w = P >= 262144;
    const int64_t nthr = mesh ? c->n_rows : P;
    const int rpe = c->un[1] * c->un[2];
    const bool stage = c->un[0] > 0 && rpe >= 16 && 256 % rpe == 0;     // <= 16 elements per CTA fit the staging array
    if (phases & 1) {
        IB_CUDA_TRY(cudaMemsetAsync(c->d_tile_count, 0, ((size_t)c->tile_hdr + (size_t)n_tiles * 4) * sizeof(int32_t), st));   // counters and bins
        if (mesh && stage && c->un[0] == 4) ibk_bin_mesh<0, 1, 4><<<ib_blocks(nthr, 256), 256, 0, st>>>(pr);
        else if (mesh && stage && c->un[0] == 2) ibk_bin_mesh<0, 1, 2><<<ib_blocks(nthr, 256), 256, 0, st>>>(pr);
        else if (mesh && stage) ibk_bin_mesh<0, 1, 0><<<ib_blocks(nthr, 256), 256, 0, st>>>(pr);
        else if (mesh) ibk_bin_mesh<0, 0, 0><<<ib_blocks(nthr, 256), 256, 0, st>>>(pr);
        else ibk_bin_cloud<0><<<ib_blocks(nthr, 256), 256, 0, st>>>(pr);
        const int nsb = (n_tiles + SCT - 1) / SCT;
        int2 *partial = reinterpret_cast<int2 *>(c->d_tile_count + IB_TILE_HDR);
        // a small cloud is cut into about one work item per SM (measured at C2, 65 k points: 66 us per step against
        // 76 with four items per SM -- every work item has a fixed cost, and a CTA with one item has nothing to
        // overlap anyway); from IB_CHUNK points per SM on the items have the tile kernel's full staging capacity
        if (!c->sm_count) IB_CUDA_TRY(cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, c->device));
        int chunk = (int)((P / (c->sm_count > 0 ? c->sm_count : 148) + 31) / 32 * 32);
        chunk = chunk < IB_MIN_CHUNK ? IB_MIN_CHUNK : (chunk > IB_CHUNK ? IB_CHUNK : chunk);
        if (nsb > 1) ibk_tile_partials<<<nsb, SCT, 0, st>>>(c->d_tile_cur, n_tiles, chunk, partial);   // one CTA needs no partial sums
        ibk_tile_scan<<<nsb, SCT, 0, st>>>(c->d_tile_cur, n_tiles, chunk, partial, c->d_tile_start, c->d_work, c->d_small_rec, c->d_tile_count,
                                           ib_slab_tiles(c), c->grid.nx / BT, c->grid.ny / BT, (int)c->work_cap);
        c->launches += 3;
    }
    if (phases & 2) {
        if (mesh && stage && c->un[0] == 4) ibk_bin_mesh<1, 1, 4><<<ib_blocks(nthr, 256), 256, 0, st>>>(pr);
        else if (mesh && stage && c->un[0] == 2) ibk_bin_mesh<1, 1, 2><<<ib_blocks(nthr, 256), 256, 0, st>>>(pr);
        else if (mesh && stage) ibk_bin_mesh<1, 1, 0><<<ib_blocks(nthr, 256), 256, 0, st>>>(pr);
        else if (mesh) ibk_bin_mesh<1, 0, 0><<<ib_blocks(nthr, 256), 256, 0, st>>>(pr);
        else ibk_bin_cloud<1><<<ib_blocks(nthr, 256), 256, 0, st>>>(pr);
        c->launches += 1;
    }
    IB_CUDA_TRY(cudaGetLastError());
    return IB_OK;
}

ib_status ibk_bin_reserve(ib_ctx *c, int64_t P)
{
    if (P <= c->bin_cap) return IB_OK;
    c->gstate = 0;                                  // a captured step holds the old buffers
    if (c->d_rec) cudaFree(c->d_rec);
    if (c->d_work) cudaFree(c->d_work);
    if (c->d_small_rec) cudaFree(c->d_small_rec);
    c->d_small_rec = nullptr;
    c->d_rec = nullptr; c->d_work = nullptr;
    c->bin_cap = 0;
    int64_t cap = P + P / 8 + 1024;
    if (cudaMalloc(&c->d_rec, (size_t)cap * 8 * sizeof(double)) != cudaSuccess) return IB_ERR_ALLOC;
    {   // a tile with >= IB_SMALL_TILE points gives at most 4 runs of layers plus one piece per IB_MIN_CHUNK points
        const int64_t n_tiles = c->n_cells / (BT * BT * BT), dense = cap / IB_SMALL_TILE + 1;
        c->work_cap = 4 * (dense < n_tiles ? dense : n_tiles) + cap / IB_MIN_CHUNK + 8;
    }
    if (cudaMalloc(&c->d_work, (size_t)c->work_cap * sizeof(int4)) != cudaSuccess) return IB_ERR_ALLOC;
    if (cudaMalloc(&c->d_small_rec, (size_t)cap * sizeof(int32_t)) != cudaSuccess) return IB_ERR_ALLOC;
    c->bin_cap = cap;
    return IB_OK;
}
