// ib_binsort.cu -- bin Lagrangian points by Eulerian cell and stable-sort them.
// Not in the paper; north_star requirement; definition = reading A21:
//   c_d = floor((x_d - x0_d) * inv_h) mod n_d  (IEEE double, no contraction), tile edge T = 8,
//   key = ((tz*nty+ty)*ntx+tx)*512 + ((lz*8+ly)*8+lx),  perm = stable sort of point ids by key.
// Hand-written LSD radix sort, 8-bit digits, only the ceil(log2(n_cells)) significant bits:
// per pass  histogram -> exclusive scan -> stable scatter (warp match_any ranking).
#include "ib_common.cuh"

#define RS_THREADS 256
#define RS_ITEMS 16
#define RS_TILE (RS_THREADS * RS_ITEMS)          // 4096 keys per block
#define RS_WARPS (RS_THREADS / 32)
#define RS_WITEMS (RS_TILE / RS_WARPS)           // 512 consecutive keys per warp

__global__ void __launch_bounds__(256)
ibk_keys(int64_t P, const double *__restrict__ xp, ib_grid_desc g, double inv_h,
         uint32_t *__restrict__ key32, int64_t *__restrict__ key64, long long *status)
{
    int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= P) return;
    double x = __ldg(xp + p), y = __ldg(xp + P + p), z = __ldg(xp + 2 * P + p);
    if (!(isfinite(x) && isfinite(y) && isfinite(z))) {
        ib_latch(status, IB_ERR_NONFINITE, p);
        x = g.x0; y = g.y0; z = g.z0;
    }
    int cx = ib_cell(x, g.x0, inv_h, g.nx), cy = ib_cell(y, g.y0, inv_h, g.ny), cz = ib_cell(z, g.z0, inv_h, g.nz);
    int ntx = g.nx / IB_TILE, nty = g.ny / IB_TILE;
    uint32_t t = (uint32_t)(((cz >> 3) * nty + (cy >> 3)) * ntx + (cx >> 3));
    uint32_t l = (uint32_t)((((cz & 7) << 3) | (cy & 7)) << 3 | (cx & 7));
    uint32_t k = t * IB_TILE_CELLS + l;
    key32[p] = k;
    if (key64) key64[p] = (int64_t)k;
}

__global__ void __launch_bounds__(RS_THREADS)
ibk_radix_hist(const uint32_t *__restrict__ keys, int64_t P, int shift, uint32_t *__restrict__ hist,
               int nblocks)
{
    __shared__ uint32_t h[256];
    h[threadIdx.x] = 0;
    __syncthreads();
    int64_t base = (int64_t)blockIdx.x * RS_TILE;
#pragma unroll
    for (int i = 0; i < RS_ITEMS; ++i) {
        int64_t idx = base + i * RS_THREADS + threadIdx.x;
        if (idx < P) atomicAdd(&h[(keys[idx] >> shift) & 255u], 1u);
    }
    __syncthreads();
    hist[(int64_t)threadIdx.x * nblocks + blockIdx.x] = h[threadIdx.x];
}

// ---- generic exclusive scan of uint32 (three kernels, 2048 elements per block) ----------------
#define SC_THREADS 256
#define SC_ITEMS 8
#define SC_TILE (SC_THREADS * SC_ITEMS)

__device__ __forceinline__ uint32_t ib_block_exclusive_scan(uint32_t v, uint32_t *total)
{
    __shared__ uint32_t ws[32];
    __shared__ uint32_t tot;
    int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    uint32_t inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        uint32_t n = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += n;
    }
    if (lane == 31) ws[wid] = inc;
    __syncthreads();
    if (wid == 0) {
        uint32_t s = (lane < (int)(blockDim.x >> 5)) ? ws[lane] : 0;
        uint32_t si = s;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t n = __shfl_up_sync(0xffffffffu, si, o);
            if (lane >= o) si += n;
        }
        ws[lane] = si - s;
        if (lane == 31) tot = si;
    }
    __syncthreads();
    uint32_t r = inc - v + ws[wid];
    if (total) *total = tot;
    __syncthreads();
    return r;
}

__global__ void __launch_bounds__(SC_THREADS)
ibk_scan_reduce(const uint32_t *__restrict__ in, int64_t n, uint32_t *__restrict__ sums)
{
    int64_t base = (int64_t)blockIdx.x * SC_TILE + (int64_t)threadIdx.x * SC_ITEMS;
    uint32_t s = 0;
#pragma unroll
    for (int i = 0; i < SC_ITEMS; ++i)
        if (base + i < n) s += in[base + i];
    uint32_t tot;
    ib_block_exclusive_scan(s, &tot);
    if (threadIdx.x == 0) sums[blockIdx.x] = tot;
}

__global__ void __launch_bounds__(1024)
ibk_scan_sums(uint32_t *__restrict__ sums, int n)
{
    __shared__ uint32_t carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (int base = 0; base < n; base += 1024) {
        int i = base + threadIdx.x;
        uint32_t v = i < n ? sums[i] : 0, tot;
        uint32_t ex = ib_block_exclusive_scan(v, &tot);
        uint32_t c = carry;
        if (i < n) sums[i] = ex + c;
        __syncthreads();
        if (threadIdx.x == 0) carry = c + tot;
        __syncthreads();
    }
}

__global__ void __launch_bounds__(SC_THREADS)
ibk_scan_apply(uint32_t *__restrict__ data, int64_t n, const uint32_t *__restrict__ sums)
{
    int64_t base = (int64_t)blockIdx.x * SC_TILE + (int64_t)threadIdx.x * SC_ITEMS;
    uint32_t v[SC_ITEMS], s = 0;
#pragma unroll
    for (int i = 0; i < SC_ITEMS; ++i) {
        v[i] = (base + i < n) ? data[base + i] : 0;
        s += v[i];
    }
    uint32_t ex = ib_block_exclusive_scan(s, nullptr) + sums[blockIdx.x];
#pragma unroll
    for (int i = 0; i < SC_ITEMS; ++i) {
        if (base + i < n) data[base + i] = ex;
        ex += v[i];
    }
}

// ---- stable scatter ---------------------------------------------------------------------------
__global__ void __launch_bounds__(RS_THREADS)
ibk_radix_scatter(const uint32_t *__restrict__ keys_in, const int32_t *__restrict__ vals_in,
                  uint32_t *__restrict__ keys_out, int32_t *__restrict__ vals_out, int64_t P, int shift,
                  const uint32_t *__restrict__ hist, int nblocks)
{
    __shared__ uint32_t wh[RS_WARPS][256];
    int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    for (int i = threadIdx.x; i < RS_WARPS * 256; i += RS_THREADS) (&wh[0][0])[i] = 0;
    __syncthreads();
    int64_t wbase = (int64_t)blockIdx.x * RS_TILE + (int64_t)wid * RS_WITEMS;
    uint32_t k[RS_ITEMS];
    const unsigned lt = (1u << lane) - 1u;
#pragma unroll
    for (int i = 0; i < RS_ITEMS; ++i) {
        int64_t idx = wbase + i * 32 + lane;
        bool ok = idx < P;
        k[i] = ok ? keys_in[idx] : 0xffffffffu;
        unsigned d = (k[i] >> shift) & 255u;
        unsigned act = __ballot_sync(0xffffffffu, ok);
        if (ok) {
            unsigned peers = __match_any_sync(act, d);
            if ((peers & lt) == 0) wh[wid][d] += __popc(peers);
        }
        __syncwarp();
    }
    __syncthreads();
    {
        unsigned d = threadIdx.x;
        uint32_t run = hist[(int64_t)d * nblocks + blockIdx.x];
#pragma unroll
        for (int w = 0; w < RS_WARPS; ++w) {
            uint32_t t = wh[w][d];
            wh[w][d] = run;
            run += t;
        }
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < RS_ITEMS; ++i) {
        int64_t idx = wbase + i * 32 + lane;
        bool ok = idx < P;
        unsigned d = (k[i] >> shift) & 255u;
        unsigned act = __ballot_sync(0xffffffffu, ok);
        if (ok) {
            unsigned peers = __match_any_sync(act, d);
            uint32_t pos = wh[wid][d] + __popc(peers & lt);
            __syncwarp(act);
            if ((peers & lt) == 0) wh[wid][d] += __popc(peers);
            keys_out[pos] = k[i];
            vals_out[pos] = vals_in ? vals_in[idx] : (int32_t)idx;
        }
        __syncwarp();
    }
}

// start rank of every tile (n_tiles+1 entries) from the sorted keys; tile = key >> shift
__global__ void __launch_bounds__(256)
ibk_tile_starts_shift(const uint32_t *__restrict__ skeys, int64_t P, int n_tiles, int shift,
                      int32_t *__restrict__ tile_start)
{
    int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (r > P) return;
    int t = (r < P) ? (int)(skeys[r] >> shift) : n_tiles;
    int tp = (r > 0) ? (int)(skeys[r - 1] >> shift) : -1;
    for (int tt = tp + 1; tt <= t; ++tt) tile_start[tt] = (int32_t)r;
}

__global__ void ibk_copy_perm(const int32_t *__restrict__ in, int32_t *__restrict__ out, int64_t P)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < P) out[i] = in[i];
}

ib_status ibk_sort_reserve(ib_ctx *c, int64_t P)
{
    if (P <= c->sort_cap) return IB_OK;
    for (int i = 0; i < 2; ++i) {
        if (c->d_key[i]) cudaFree(c->d_key[i]);
        if (c->d_val[i]) cudaFree(c->d_val[i]);
        c->d_key[i] = nullptr; c->d_val[i] = nullptr;
    }
    if (c->d_hist) cudaFree(c->d_hist);
    c->d_hist = nullptr;
    c->sort_cap = 0;
    int64_t cap = P + P / 8 + 1024;
    for (int i = 0; i < 2; ++i) {
        if (cudaMalloc(&c->d_key[i], cap * sizeof(uint32_t)) != cudaSuccess) return IB_ERR_ALLOC;
        if (cudaMalloc(&c->d_val[i], cap * sizeof(int32_t)) != cudaSuccess) return IB_ERR_ALLOC;
    }
    int64_t nb = (cap + RS_TILE - 1) / RS_TILE;
    int64_t hl = 256 * nb;
    int64_t nsum = (hl + SC_TILE - 1) / SC_TILE;
    c->hist_cap = hl + nsum + 16;
    if (cudaMalloc(&c->d_hist, c->hist_cap * sizeof(uint32_t)) != cudaSuccess) return IB_ERR_ALLOC;
    c->sort_cap = cap;
    return IB_OK;
}

// LSD radix sort of the `bits` low bits of the keys in d_key[0] (values = point ids, implicit
// iota on the first pass). On return the sorted keys / permutation are in d_key[0] / d_val[0]
// (copied back when the pass count is odd).
ib_status ibk_sort_keys_inplace(ib_ctx *c, int64_t P, int bits, cudaStream_t st)
{
    if (P <= 0) return IB_OK;
    int passes = (bits + 7) / 8;
    int nb = (int)((P + RS_TILE - 1) / RS_TILE);
    int64_t hl = 256ll * nb;
    int nsum = (int)((hl + SC_TILE - 1) / SC_TILE);
    uint32_t *sums = c->d_hist + hl;
    int cur = 0;
    for (int ps = 0; ps < passes; ++ps) {
        int shift = 8 * ps;
        ibk_radix_hist<<<nb, RS_THREADS, 0, st>>>(c->d_key[cur], P, shift, c->d_hist, nb);
        ibk_scan_reduce<<<nsum, SC_THREADS, 0, st>>>(c->d_hist, hl, sums);
        ibk_scan_sums<<<1, 1024, 0, st>>>(sums, nsum);
        ibk_scan_apply<<<nsum, SC_THREADS, 0, st>>>(c->d_hist, hl, sums);
        ibk_radix_scatter<<<nb, RS_THREADS, 0, st>>>(c->d_key[cur], ps == 0 ? nullptr : c->d_val[cur],
                                                     c->d_key[cur ^ 1], c->d_val[cur ^ 1], P, shift,
                                                     c->d_hist, nb);
        c->launches += 5;
        cur ^= 1;
    }
    if (cur != 0) {
        IB_CUDA_TRY(cudaMemcpyAsync(c->d_key[0], c->d_key[1], P * sizeof(uint32_t), cudaMemcpyDeviceToDevice, st));
        IB_CUDA_TRY(cudaMemcpyAsync(c->d_val[0], c->d_val[1], P * sizeof(int32_t), cudaMemcpyDeviceToDevice, st));
    }
    IB_CUDA_TRY(cudaGetLastError());
    return IB_OK;
}

ib_status ibk_bin_sort(ib_ctx *c, const double *xp, int64_t P, int64_t *key_out, int32_t *perm_out,
                       int build_cells, cudaStream_t st)
{
    ib_status rs = ibk_sort_reserve(c, P);
    if (rs != IB_OK) return rs;
    (void)build_cells;
    if (P > 0) {
        ibk_keys<<<ib_blocks(P, 256), 256, 0, st>>>(P, xp, c->grid, c->inv_h, c->d_key[0], key_out, c->d_status);
        c->launches++;
        int bits = 1;
        while ((1ll << bits) < c->n_cells) ++bits;
        rs = ibk_sort_keys_inplace(c, P, bits, st);
        if (rs != IB_OK) return rs;
        if (perm_out) {
            ibk_copy_perm<<<ib_blocks(P, 256), 256, 0, st>>>(c->d_val[0], perm_out, P);
            c->launches++;
        }
    }
    IB_CUDA_TRY(cudaGetLastError());
    return IB_OK;
}

// ---- ib_bin_sort_static: the same sort without a context and without any allocation ------------------------
// (include/ibcouple.h).  The kernels are the ones above; the scratch that ibk_sort_reserve takes from cudaMalloc
// is ONE file-scope device array here, sized for IB_BIN_SORT_STATIC_MAX_POINTS points.  Every GPU that loads
// the library holds it until the process exits; all calls on a device share it.
#include <cmath>
#include <mutex>

#define IBS_MAXP IB_BIN_SORT_STATIC_MAX_POINTS
#define IBS_NB ((IBS_MAXP + RS_TILE - 1) / RS_TILE)            // blocks of the histogram / scatter kernels at the limit
#define IBS_HL (256 * IBS_NB)                                  // histogram entries
#define IBS_NSUM ((IBS_HL + SC_TILE - 1) / SC_TILE)            // block sums of the scan
// layout, in 32-bit words; every part starts on a 256-byte boundary
#define IBS_OFF_STATUS 0                                       // 2 x 64 bit: the status latch (ib_latch)
#define IBS_OFF_KEY 64                                         // [2][IBS_MAXP] keys, ping and pong
#define IBS_OFF_VAL (IBS_OFF_KEY + 2 * IBS_MAXP)               // [2][IBS_MAXP] point ids
#define IBS_OFF_HIST (IBS_OFF_VAL + 2 * IBS_MAXP)              // [256][blocks] digit counts
#define IBS_OFF_SUMS (IBS_OFF_HIST + IBS_HL)                   // [IBS_NSUM]
#define IBS_WORDS (IBS_OFF_SUMS + ((IBS_NSUM + 63) & ~63))
static_assert(IBS_MAXP % 64 == 0 && IBS_HL % 64 == 0, "parts of the scratch array stay 256-byte aligned");
static_assert(IBS_WORDS * 4ll == 4260352ll, "include/ibcouple.h and README.md state this size");

static __device__ __align__(256) uint32_t ib_static_scratch[IBS_WORDS];

// In host code `ib_static_scratch` is a stand-in for the symbol, not a device address: the address comes from
// cudaGetSymbolAddress, once per device, with that device current.
#define IBS_MAX_DEVICES 64
static std::mutex ibs_mutex;
static uint32_t *ibs_dev_ptr[IBS_MAX_DEVICES];

static ib_status ibs_scratch(uint32_t **out)
{
    int dev = -1;
    IB_CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= IBS_MAX_DEVICES) return IB_ERR_UNSUPPORTED;
    std::lock_guard<std::mutex> lock(ibs_mutex);
    if (!ibs_dev_ptr[dev]) {
        void *p = nullptr;
        IB_CUDA_TRY(cudaGetSymbolAddress(&p, ib_static_scratch));
        if (!p) return IB_ERR_CUDA;
        ibs_dev_ptr[dev] = static_cast<uint32_t *>(p);
    }
    *out = ibs_dev_ptr[dev];
    return IB_OK;
}

extern "C" ib_status ib_bin_sort_static(const ib_grid_desc *g, const double *xp, int64_t P, int64_t *key_out,
                                        int32_t *perm_out, int32_t check, void *stream)
{
    if (!g || P < 0 || (P > 0 && !xp)) return IB_ERR_INVALID_ARG;
    if (g->nx <= 0 || g->ny <= 0 || g->nz <= 0 || (g->nx % IB_TILE) || (g->ny % IB_TILE) || (g->nz % IB_TILE))
        return IB_ERR_INVALID_ARG;
    if (!(g->h > 0.0) || !std::isfinite(g->h) || !std::isfinite(g->x0) || !std::isfinite(g->y0) || !std::isfinite(g->z0))
        return IB_ERR_INVALID_ARG;
    const int64_t n_cells = (int64_t)g->nx * g->ny * g->nz;
    if (n_cells > (int64_t)INT32_MAX) return IB_ERR_INVALID_ARG;
    if (P > (int64_t)IBS_MAXP) return IB_ERR_TOO_LARGE;        // the scratch array holds no more
    uint32_t *scr = nullptr;
    ib_status rs = ibs_scratch(&scr);
    if (rs != IB_OK) return rs;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    long long *status = reinterpret_cast<long long *>(scr + IBS_OFF_STATUS);
    uint32_t *key[2] = {scr + IBS_OFF_KEY, scr + IBS_OFF_KEY + IBS_MAXP};
    int32_t *val[2] = {reinterpret_cast<int32_t *>(scr + IBS_OFF_VAL), reinterpret_cast<int32_t *>(scr + IBS_OFF_VAL + IBS_MAXP)};
    uint32_t *hist = scr + IBS_OFF_HIST, *sums = scr + IBS_OFF_SUMS;
    // the array keeps the last call's contents.  The status word must start at zero; everything else that is
    // read below is written first (keys and ids [0, P), all 256 x nb histogram entries, all nsum block sums)
    IB_CUDA_TRY(cudaMemsetAsync(status, 0, 2 * sizeof(long long), st));
    if (P > 0) {
        ibk_keys<<<ib_blocks(P, 256), 256, 0, st>>>(P, xp, *g, 1.0 / g->h, key[0], key_out, status);
        int bits = 1;
        while ((1ll << bits) < n_cells) ++bits;
        const int passes = (bits + 7) / 8;
        const int nb = (int)((P + RS_TILE - 1) / RS_TILE);
        const int64_t hl = 256ll * nb;
        const int nsum = (int)((hl + SC_TILE - 1) / SC_TILE);
        int cur = 0;
        for (int ps = 0; ps < passes; ++ps) {
            const int shift = 8 * ps;
            ibk_radix_hist<<<nb, RS_THREADS, 0, st>>>(key[cur], P, shift, hist, nb);
            ibk_scan_reduce<<<nsum, SC_THREADS, 0, st>>>(hist, hl, sums);
            ibk_scan_sums<<<1, 1024, 0, st>>>(sums, nsum);
            ibk_scan_apply<<<nsum, SC_THREADS, 0, st>>>(hist, hl, sums);
            ibk_radix_scatter<<<nb, RS_THREADS, 0, st>>>(key[cur], ps == 0 ? nullptr : val[cur], key[cur ^ 1], val[cur ^ 1],
                                                         P, shift, hist, nb);
            cur ^= 1;
        }
        if (perm_out) ibk_copy_perm<<<ib_blocks(P, 256), 256, 0, st>>>(val[cur], perm_out, P);
        IB_CUDA_TRY(cudaGetLastError());
    }
    if (check) {
        unsigned long long w[2] = {0, 0};
        IB_CUDA_TRY(cudaMemcpyAsync(w, status, sizeof(w), cudaMemcpyDeviceToHost, st));
        IB_CUDA_TRY(cudaStreamSynchronize(st));
        int code = 0;
        long long id = -1;
        ib_status_unpack(w[0], &code, &id);
        if (code != 0) return static_cast<ib_status>(code);
    }
    return IB_OK;
}
