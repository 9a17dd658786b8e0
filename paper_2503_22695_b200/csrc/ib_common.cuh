// ib_common.cuh -- device helpers and the host-side context of libibcouple (CUDA path only).
// Shares nothing with oracle/.  Citations are to /root/reference/PAPER.md lines (see include/ibcouple.h).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/ibcouple.h"

#define IB_TILE 8              // tile edge of the binning key (A21)
#define IB_TILE_CELLS 512
#ifndef IB_SMALL_TILE
#define IB_SMALL_TILE 64         // tiles with fewer points skip the tile kernel: their points go one by one (ib_point.cuh); 32/48/80/96/128/192 measured
#endif
#ifndef IB_CHUNK
#define IB_CHUNK 768             // points per work item of the tile kernel = records it stages in shared memory (ib_bin.cu emits the work list); the largest that two record buffers leave room for (576 ... 768 measured: the larger the better)
#endif
#define IB_SLAB0 4                // d_tile_count[IB_SLAB0 + k] = first work item of z-slab k (ib_tile_scan)
#define IB_MAX_SLABS 32
#define IB_SLABC0 40              // d_tile_count[IB_SLABC0 + k] = work counter of slab k
#define IB_TILE_HDR 80            // ints of d_tile_count before the partial sums of the scan
#ifndef IB_HOST_SLABS
#define IB_HOST_SLABS 8           // z-slabs ib_coupling_step_host cuts the step into
#endif
static_assert(IB_HOST_SLABS >= 1 && IB_HOST_SLABS <= IB_MAX_SLABS, "IB_HOST_SLABS out of range");
static_assert(IB_SLAB0 + IB_MAX_SLABS < IB_SLABC0 && IB_SLABC0 + IB_MAX_SLABS <= IB_TILE_HDR, "d_tile_count header layout");

// ---------------------------------------------------------------------------------------------
// host-side context
// ---------------------------------------------------------------------------------------------
struct ib_ctx {
    int device;
    ib_grid_desc grid;
    double inv_h;
    int64_t n_nodes, n_elems, n_points, n_cells;
    int nodal;                 // nsub == NULL
    int uniform_S;             // all elements share one nsub triple (0 if not)
    int n_mats;
    int variant;
    // static mesh (device copies)
    int32_t *d_conn;           // [n_elems][8]
    double *d_X;               // [3][n_nodes]
    double *d_fib;             // [6][n_elems]
    int32_t *d_mat_id;         // [n_elems]
    int32_t *d_nsub;           // [n_elems][3]
    int64_t *d_pt_off;         // [n_elems+1]
    ib_material *d_mats;
    int elem_type, npe;        // IB_ELEM_HEX8 / IB_ELEM_TET4, nodes per element
    int32_t *d_adj;            // hex: [8][n_nodes] slot = e*8+a or -1 (ELL, ascending element id)
    int32_t *d_node_off, *d_node_slot;   // tets: CSR node -> slots e*4+a (ascending), valence is unbounded
    double *d_Wp;              // [P] sub-point weights W_s
    double *d_wa;              // [n_nodes] lumped weights
    double *d_geo;             // [10][8 n_elems] reference J0^-1 and det J0 per Gauss point
    // per-step scratch
    double *d_Ce;              // [3][n_elems*8] per-element nodal contributions
    double *d_Fhat;            // [3][n_nodes]
    double *d_B;               // [3][n_nodes] (when caller passes B == NULL)
    double *d_xp, *d_Gp, *d_Up;   // [3][P]
    // sort scratch (grown on demand)
    int64_t sort_cap;
    uint32_t *d_key[2];
    int32_t *d_val[2];
    uint32_t *d_hist;
    int64_t hist_cap;
    // tile-level counting sort of the points (ib_bin.cu), tiles of 4x4x4 cells
    int64_t n_rows;            // rows (e,m2,m3) of sub-points of the mesh source
    int un[3];                 // uniform nsub triple, un[0] == 0 if elements differ
    int64_t *d_row_off;        // [n_elems+1]
    int32_t *d_tile_cur;       // [n_tiles] counts, then running cursors
    int32_t *d_tile_start;     // [n_tiles+1]
    int4 *d_work;              // work list of the tile kernel: {tile, first record, points, packed tile coordinates} per work item
    int64_t work_cap;
    int32_t *d_small_rec;      // records of tiles with < IB_SMALL_TILE points (count in d_tile_count[2])
    int32_t *d_tile_count;     // [0] number of non-empty tiles, [1] work counter; d_tile_cur follows it in the same block
    int tile_hdr;              // ints of d_tile_count before d_tile_cur
    int64_t bin_cap;
    double *d_rec;             // [P][8] point records grouped by bin: {x, y, z, id | G0, G1, G2, -}
    // host staging for the *_host entry point
    double *d_hx, *d_hu, *d_hv, *d_hw, *d_hfu, *d_hfv, *d_hfw, *d_hUn, *d_hB;
    // status latch: one packed word (ib_latch)
    long long *d_status;
    cudaStream_t last_stream;
    cudaStream_t side;         // internal stream: work that needs only the positions overlaps the FE force
    cudaEvent_t ev_fork, ev_join, ev_aux;
    cudaStream_t side2;        // the direct path of the sparse tiles runs beside the tile kernel
    cudaEvent_t ev_sfork, ev_sjoin;
    cudaStream_t side3;        // ib_coupling_step_host: f goes back to the host slab by slab on this stream
    cudaStream_t side4;        // ... and the odd slabs of the tile kernel run on this one
    cudaEvent_t ev_slab[IB_MAX_SLABS], ev_h2d[IB_MAX_SLABS];
    cudaEvent_t ev_zero;       // ... f has been zero-filled
    int64_t launches;
    unsigned char tiled_cfg[8];  // ibk_tiled_kernel<S,I,PER>: dynamic shared memory size has been set
    int sm_count;
    // NEXT-4 boundary loads (ib_set_tethers / ib_set_surface / ib_set_loads)
    int32_t *d_teth_ids, *d_faces;
    int64_t n_teth, n_faces;
    int npf;
    double kappa_t, qt0[3], p_load;
    // CUDA graph of ib_coupling_step (replayed when the same pointers come in again on a capturable stream)
    int graph_on, gstate;      // gstate: 0 none, 1 key seen once (ran eagerly), 2 captured
    cudaGraphExec_t gexec;
    const void *gkey[11];
    int64_t g_launches;
    // optional per-phase event timing
    int profile;
    void *prof;                // std::vector<ib_prof_rec>* (ib_context.cu)
};

// z-slabs of the tile list (tiles are numbered z-major): tile layers per slab and tiles per slab.  The
// scan handles 4 tiles per thread, so a tile layer must be a multiple of 4 tiles; otherwise one slab.
static inline int ib_slab_layers(const ib_ctx *c)
{
    const int ntz = c->grid.nz / 4, per = (c->grid.nx / 4) * (c->grid.ny / 4);
    const int K = ntz / 2 < IB_HOST_SLABS ? ntz / 2 : IB_HOST_SLABS;     // at least two tile layers per slab
    if (per % 4 != 0 || K < 2) return ntz;
    return (ntz + K - 1) / K;
}
static inline int ib_slab_tiles(const ib_ctx *c)
{
    const int per = (c->grid.nx / 4) * (c->grid.ny / 4);
    const int t = ib_slab_layers(c) * per;
    return (t + 3) / 4 * 4;
}
static inline int ib_slab_count(const ib_ctx *c)
{
    const int ntz = c->grid.nz / 4, L = ib_slab_layers(c);
    return (ntz + L - 1) / L;
}

void ib_prof_begin(ib_ctx *c, int phase, cudaStream_t st);
void ib_prof_end(ib_ctx *c, int phase, cudaStream_t st);

#ifdef NDEBUG
#define IB_CUDA_WHERE(e) ((void)0)
#else            /* checked test builds say which call failed */
#include <cstdio>
#define IB_CUDA_WHERE(e) fprintf(stderr, "[ibcouple] %s at %s:%d\n", cudaGetErrorString(e), __FILE__, __LINE__)
#endif
#define IB_CUDA_TRY(expr)                                   \
    do {                                                    \
        cudaError_t _e = (expr);                            \
        if (_e != cudaSuccess) { IB_CUDA_WHERE(_e); return IB_ERR_CUDA; } \
    } while (0)

static inline unsigned ib_blocks(int64_t n, int per) { return (unsigned)((n + per - 1) / per); }

// ---------------------------------------------------------------------------------------------
// device helpers
// ---------------------------------------------------------------------------------------------
// One word holds (code, id): code in the top 8 bits, 2^48-1 - id below, kept with atomicMax -- so the
// reported pair is always one error: the highest code seen (OUT_OF_DOMAIN > NONFINITE > INVERTED) with the
// smallest id that raised THAT code.  0 = no error.  ib_check unpacks it (ib_status_unpack).
#define IB_STATUS_IDMASK 0xFFFFFFFFFFFFull
__device__ __forceinline__ void ib_latch(long long *status, int code, long long id)
{
    atomicMax((unsigned long long *)status, ((unsigned long long)code << 56) | (IB_STATUS_IDMASK - ((unsigned long long)id & IB_STATUS_IDMASK)));
}
static inline void ib_status_unpack(unsigned long long w, int *code, long long *id)
{
    *code = (int)(w >> 56);
    *id = w ? (long long)(IB_STATUS_IDMASK - (w & IB_STATUS_IDMASK)) : -1;
}

// sqrt(a) for a in [1/64, 1/32] (the argument (1+4r-4r^2)/64 of the kernel): reciprocal-square-root seed
// from the upper word (MUFU.RSQ64H, ~2^-20; the float route costs two conversions more on the same unit),
// one Goldschmidt step (~2^-39) and one residual correction (~2^-77, i.e. rounding level) -- no special
// cases, no branches, 7 fp64 operations.
__device__ __forceinline__ double ib_sqrt_seeded(double a)
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(a));               // one MUFU.RSQ64H
    double g = a * y, h = 0.5 * y;
    double r = fma(-g, h, 0.5);
    g = fma(g, r, g);
    h = fma(h, r, h);
    return fma(fma(-g, g, a), h, g);
}

// (double)v for |v| < 2^31 without the conversion unit: the integer goes into the low word of 2^52 + 2^31 + v
// (exact), one fp64 subtraction takes the offset out again
__device__ __forceinline__ double ib_i2d(int v)
{
    return __hiloint2double(0x43300000, v ^ (int)0x80000000) - 4503601774854144.0;
}

// Peskin 4-point kernel (PAPER.md L52 -> ref.1): the four weights of the support that starts at
// i0 = floor(s) - 1, with r = s - floor(s) in [0,1):
//   phi(1+r) = (3-2r-q)/8, phi(r) = (3-2r+q)/8, phi(1-r) = (1+2r+q)/8, phi(2-r) = (1+2r-q)/8,
//   q = sqrt(1+4r-4r^2)  (one square root serves all four; q/8 = sqrt((1+4r-4r^2)/64) directly).
__device__ __forceinline__ void ib_phi4(double r, double w[4])
{
    double q = ib_sqrt_seeded(fma(0.0625 * r, 1.0 - r, 0.015625));
    double a = fma(-0.25, r, 0.375);
    double b = fma(0.25, r, 0.125);
    w[0] = a - q;
    w[1] = a + q;
    w[2] = b + q;
    w[3] = b - q;
}

// The same as the pair (a, q) the four weights are made of:  w0 = a - q, w1 = a + q, w2 = (1/2 - a) + q,
// w3 = (1/2 - a) - q  with a = 3/8 - r/4, q = sqrt(1 + 4r - 4r^2)/8.
__device__ __forceinline__ double2 ib_aq(double r)
{
    return make_double2(fma(-0.25, r, 0.375), ib_sqrt_seeded(fma(0.0625 * r, 1.0 - r, 0.015625)));
}

// scaled coordinate s = (x - x0)/h, computed as a product with 1/h plus one residual correction
// so that it agrees with true division to ~1 ulp.
__device__ __forceinline__ double ib_scaled(double x, double x0, double h, double inv_h)
{
    double d = x - x0;
    double s = d * inv_h;
    double res = fma(-s, h, d);
    return fma(res, inv_h, s);
}

__device__ __forceinline__ int ib_wrap(int i, int n)
{
    i %= n;
    return i < 0 ? i + n : i;
}

// Binning cell index of A21: floor((x - x0) * inv_h) mod n, in IEEE double with NO contraction.
__device__ __forceinline__ int ib_cell(double x, double x0, double inv_h, int n)
{
    const double sc = __dmul_rn(__dsub_rn(x, x0), inv_h);
    const int ci = __double2int_rd(sc);                   // floor in one conversion (saturates far outside)
    if ((unsigned)ci < (unsigned)n) return ci;            // inside the box: no wrap, no 64-bit modulo
    long long c = (long long)floor(sc);
    c %= n;
    if (c < 0) c += n;
    return (int)c;
}

// bounded grid (periodic == 0, reading A26): is the point inside the box [x0, x0 + n h)^3 ?
__device__ __forceinline__ bool ib_in_box(double x, double y, double z, const ib_grid_desc &g, double inv_h)
{
    const double fx = floor(__dmul_rn(__dsub_rn(x, g.x0), inv_h)), fy = floor(__dmul_rn(__dsub_rn(y, g.y0), inv_h)),
                 fz = floor(__dmul_rn(__dsub_rn(z, g.z0), inv_h));
    return fx >= 0.0 && fx < (double)g.nx && fy >= 0.0 && fy < (double)g.ny && fz >= 0.0 && fz < (double)g.nz;
}

// Q1 shape functions at xi (local node a = ia + 2 ja + 4 ka)
__device__ __forceinline__ void ib_shape(double x0, double x1, double x2, double N[8])
{
    double a0 = 0.5 * (1.0 - x0), a1 = 0.5 * (1.0 + x0);
    double b0 = 0.5 * (1.0 - x1), b1 = 0.5 * (1.0 + x1);
    double c0 = 0.5 * (1.0 - x2), c1 = 0.5 * (1.0 + x2);
    double ab00 = a0 * b0, ab10 = a1 * b0, ab01 = a0 * b1, ab11 = a1 * b1;
    N[0] = ab00 * c0; N[1] = ab10 * c0; N[2] = ab01 * c0; N[3] = ab11 * c0;
    N[4] = ab00 * c1; N[5] = ab10 * c1; N[6] = ab01 * c1; N[7] = ab11 * c1;
}

// shape-function gradients wrt xi
__device__ __forceinline__ void ib_dshape(double x0, double x1, double x2, double dN[8][3])
{
#pragma unroll
    for (int a = 0; a < 8; ++a) {
        double s0 = (a & 1) ? 1.0 : -1.0, s1 = (a & 2) ? 1.0 : -1.0, s2 = (a & 4) ? 1.0 : -1.0;
        double f0 = fma(s0, x0, 1.0), f1 = fma(s1, x1, 1.0), f2 = fma(s2, x2, 1.0);
        dN[a][0] = 0.125 * s0 * f1 * f2;
        dN[a][1] = 0.125 * f0 * s1 * f2;
        dN[a][2] = 0.125 * f0 * f1 * s2;
    }
}

// sub-point reference coordinate: xi = -1 + (2m+1)/n
__device__ __forceinline__ double ib_subxi(int m, int n) { return -1.0 + (double)(2 * m + 1) / (double)n; }

__device__ __forceinline__ double ib_det3(const double A[3][3])
{
    return A[0][0] * (A[1][1] * A[2][2] - A[1][2] * A[2][1])
         - A[0][1] * (A[1][0] * A[2][2] - A[1][2] * A[2][0])
         + A[0][2] * (A[1][0] * A[2][1] - A[1][1] * A[2][0]);
}

// internal launchers (defined across the .cu files)
ib_status ibk_fe_force(ib_ctx *c, const double *x, double *B, double *Fhat, cudaStream_t st);
ib_status ibk_points(ib_ctx *c, const double *x, const double *Fhat, double *xp, double *Gp, cudaStream_t st);
ib_status ibk_restrict(ib_ctx *c, const double *Up, double *Un, cudaStream_t st);
ib_status ibk_precompute_weights(ib_ctx *c, cudaStream_t st);
ib_status ibk_fe_precompute(ib_ctx *c, cudaStream_t st);
ib_status ibk_bin_sort(ib_ctx *c, const double *xp, int64_t P, int64_t *key_out, int32_t *perm_out,
                       int build_cells, cudaStream_t st);
ib_status ibk_spread_interp(ib_ctx *c, const double *xp, const double *Gp, int64_t P,
                            const double *u, const double *v, const double *w,
                            double *fu, double *fv, double *fw, double *Up, int accumulate,
                            cudaStream_t st);
ib_status ibk_sort_reserve(ib_ctx *c, int64_t P);
ib_status ibk_bin_reserve(ib_ctx *c, int64_t P);
ib_status ibk_tiled_spread_interp(ib_ctx *c, int mesh, const double *xp, const double *Gp, int64_t P,
                                  const double *x, const double *Fhat,
                                  const double *u, const double *v, const double *w,
                                  double *fu, double *fv, double *fw, double *Up, int counted, cudaStream_t st);
ib_status ibk_tiled_launch(ib_ctx *c, int64_t P, int do_spread, int do_interp,
                           const double *u, const double *v, const double *w,
                           double *fu, double *fv, double *fw, double *Up, int slab, cudaStream_t st);
ib_status ibk_small_launch(ib_ctx *c, int64_t P, int do_spread, int do_interp,
                           const double *u, const double *v, const double *w,
                           double *fu, double *fv, double *fw, double *Up, cudaStream_t st);
ib_status ibk_bin_points(ib_ctx *c, int mesh, const double *xp, const double *Gp, int64_t P,
                         const double *x, const double *Fhat, double *Up, int phases, cudaStream_t st);
