// ib_context.cu -- C-ABI entry points of libibcouple (include/ibcouple.h): context lifetime,
// argument validation, and the per-step calls that enqueue the kernels of the other files.
#include <climits>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>
#include <nvtx3/nvToolsExt.h>
#include "ib_common.cuh"

#define ST(s) ((cudaStream_t)(s))

static ib_status dev_alloc(void **p, size_t bytes)
{
    *p = nullptr;
    if (bytes == 0) bytes = 16;
    return cudaMalloc(p, bytes) == cudaSuccess ? IB_OK : IB_ERR_ALLOC;
}

template <class T>
static ib_status dev_upload(T **dst, const T *src, size_t n)
{
    ib_status s = dev_alloc((void **)dst, n * sizeof(T));
    if (s != IB_OK) return s;
    if (n && cudaMemcpy(*dst, src, n * sizeof(T), cudaMemcpyHostToDevice) != cudaSuccess) return IB_ERR_CUDA;
    return IB_OK;
}

struct ib_prof_rec { int phase; cudaEvent_t e0, e1; };
typedef std::vector<ib_prof_rec> ib_prof_vec;

// Every phase of a step is an NVTX range on the calling thread (names a timeline of the three streams; costs a
// function-pointer check when no tool is attached) and, with ib_profile_enable, a pair of CUDA events.
static const char *const ib_phase_name[IB_PHASE_COUNT] = {"ib:fe_force", "ib:points(count+scan)", "ib:sort(scatter)",
                                                          "ib:spread+interp", "ib:restrict", "ib:zero f"};

void ib_prof_begin(ib_ctx *c, int phase, cudaStream_t st)
{
    nvtxRangePushA(ib_phase_name[phase]);
    if (!c->profile) return;
    ib_prof_vec *v = (ib_prof_vec *)c->prof;
    ib_prof_rec r;
    r.phase = phase;
    cudaEventCreate(&r.e0);
    cudaEventCreate(&r.e1);
    cudaEventRecord(r.e0, st);
    v->push_back(r);
}

void ib_prof_end(ib_ctx *c, int phase, cudaStream_t st)
{
    nvtxRangePop();
    if (!c->profile) return;
    ib_prof_vec *v = (ib_prof_vec *)c->prof;
    for (size_t i = v->size(); i-- > 0;)
        if ((*v)[i].phase == phase) { cudaEventRecord((*v)[i].e1, st); return; }
}

extern "C" ib_status ib_profile_enable(ib_ctx *c, int32_t on)
{
    if (!c) return IB_ERR_INVALID_ARG;
    if (!c->prof) c->prof = new ib_prof_vec();
    c->profile = on ? 1 : 0;
    c->gstate = 0;
    return IB_OK;
}

extern "C" ib_status ib_profile_read(ib_ctx *c, double *ms_sum, int64_t *calls)
{
    if (!c || !ms_sum || !calls) return IB_ERR_INVALID_ARG;
    for (int i = 0; i < IB_PHASE_COUNT; ++i) { ms_sum[i] = 0.0; calls[i] = 0; }
    if (!c->prof) return IB_OK;
    ib_prof_vec *v = (ib_prof_vec *)c->prof;
    for (auto &r : *v) {
        float ms = 0.f;
        if (cudaEventSynchronize(r.e1) == cudaSuccess && cudaEventElapsedTime(&ms, r.e0, r.e1) == cudaSuccess) {
            ms_sum[r.phase] += ms;
            calls[r.phase]++;
        }
        cudaEventDestroy(r.e0);
        cudaEventDestroy(r.e1);
    }
    v->clear();
    return IB_OK;
}

extern "C" const char *ib_status_string(ib_status s)
{
    switch (s) {
    case IB_OK: return "IB_OK";
    case IB_ERR_INVALID_ARG: return "IB_ERR_INVALID_ARG";
    case IB_ERR_UNSUPPORTED: return "IB_ERR_UNSUPPORTED";
    case IB_ERR_ALLOC: return "IB_ERR_ALLOC";
    case IB_ERR_CUDA: return "IB_ERR_CUDA";
    case IB_ERR_INVERTED_ELEMENT: return "IB_ERR_INVERTED_ELEMENT";
    case IB_ERR_NONFINITE: return "IB_ERR_NONFINITE";
    case IB_ERR_OUT_OF_DOMAIN: return "IB_ERR_OUT_OF_DOMAIN";
    case IB_ERR_TOO_LARGE: return "IB_ERR_TOO_LARGE";
    }
    return "IB_ERR_UNKNOWN";
}

static ib_status reset_status(ib_ctx *c, cudaStream_t st)
{
    IB_CUDA_TRY(cudaMemsetAsync(c->d_status, 0, 2 * sizeof(long long), st));
    return IB_OK;
}

extern "C" ib_status ib_destroy(ib_ctx *c)
{
    if (!c) return IB_ERR_INVALID_ARG;
    cudaSetDevice(c->device);
    void *ptrs[] = {c->d_conn, c->d_X, c->d_fib, c->d_mat_id, c->d_nsub, c->d_pt_off, c->d_mats, c->d_adj,
                    c->d_Wp, c->d_wa, c->d_geo, c->d_node_off, c->d_node_slot, c->d_teth_ids, c->d_faces, c->d_Ce, c->d_Fhat, c->d_B, c->d_xp, c->d_Gp, c->d_Up, c->d_key[0],
                    c->d_key[1], c->d_val[0], c->d_val[1], c->d_hist, c->d_tile_start, c->d_work, c->d_small_rec,
                    c->d_row_off, c->d_rec,
                    c->d_tile_count, c->d_hx, c->d_hu, c->d_hfu,
                    c->d_hUn, c->d_hB, c->d_status};
    for (void *p : ptrs)
        if (p) cudaFree(p);
    if (c->gexec) cudaGraphExecDestroy(c->gexec);
    if (c->side) cudaStreamDestroy(c->side);
    if (c->ev_fork) cudaEventDestroy(c->ev_fork);
    if (c->ev_join) cudaEventDestroy(c->ev_join);
    if (c->ev_aux) cudaEventDestroy(c->ev_aux);
    if (c->side2) cudaStreamDestroy(c->side2);
    if (c->ev_sfork) cudaEventDestroy(c->ev_sfork);
    if (c->ev_sjoin) cudaEventDestroy(c->ev_sjoin);
    if (c->side3) cudaStreamDestroy(c->side3);
    if (c->side4) cudaStreamDestroy(c->side4);
    for (cudaEvent_t e : c->ev_h2d)
        if (e) cudaEventDestroy(e);
    if (c->ev_zero) cudaEventDestroy(c->ev_zero);
    for (cudaEvent_t e : c->ev_slab)
        if (e) cudaEventDestroy(e);
    if (c->prof) {
        double ms[IB_PHASE_COUNT];
        int64_t n[IB_PHASE_COUNT];
        ib_profile_read(c, ms, n);
        delete (ib_prof_vec *)c->prof;
    }
    delete c;
    return IB_OK;
}

extern "C" ib_status ib_create(ib_ctx **out, const ib_grid_desc *g, const ib_mesh_desc *m, int32_t device)
{
    if (!out) return IB_ERR_INVALID_ARG;
    *out = nullptr;
    if (!g || !m) return IB_ERR_INVALID_ARG;
    if (g->nx <= 0 || g->ny <= 0 || g->nz <= 0 || (g->nx % IB_TILE) || (g->ny % IB_TILE) || (g->nz % IB_TILE))
        return IB_ERR_INVALID_ARG;
    if (!(g->h > 0.0) || !std::isfinite(g->h) || !std::isfinite(g->x0) || !std::isfinite(g->y0) || !std::isfinite(g->z0))
        return IB_ERR_INVALID_ARG;
    if ((int64_t)g->nx * g->ny * g->nz > (int64_t)INT32_MAX) return IB_ERR_INVALID_ARG;
    if (g->nx > 4096 || g->ny > 4096 || g->nz > 8192) return IB_ERR_UNSUPPORTED;      // tile coordinates are packed 10 + 10 + 11 bits in the work list
    if (m->n_nodes < 0 || m->n_elems < 0 || m->n_nodes > INT32_MAX || m->n_elems > INT32_MAX / 8) return IB_ERR_INVALID_ARG;
    if (m->n_elems > 0 && (!m->conn || !m->X_ref || !m->mats || m->n_mats <= 0)) return IB_ERR_INVALID_ARG;
    if (m->elem_type < IB_ELEM_HEX8 || m->elem_type > IB_ELEM_TET10) return IB_ERR_INVALID_ARG;
    if (m->elem_type != IB_ELEM_HEX8 && m->nsub) return IB_ERR_UNSUPPORTED;       // tets: nodal coupling only
    const int npe = m->elem_type == IB_ELEM_TET4 ? 4 : (m->elem_type == IB_ELEM_TET10 ? 10 : 8);
    if (m->n_nodes > 0 && !m->X_ref) return IB_ERR_INVALID_ARG;
    for (int i = 0; i < m->n_mats; ++i)
        if (m->mats[i].law < IB_LAW_NEOHOOKEAN || m->mats[i].law > IB_LAW_FR2) return IB_ERR_INVALID_ARG;

    // host-side validation and topology
    const int64_t nn = m->n_nodes, ne = m->n_elems;
    std::vector<int64_t> off((size_t)ne + 1, 0), roff((size_t)ne + 1, 0);
    int uniform = 0;
    if (m->nsub) {
        for (int64_t e = 0; e < ne; ++e) {
            const int32_t *s = m->nsub + 3 * e;
            if (s[0] < 1 || s[1] < 1 || s[2] < 1 || s[0] > 8 || s[1] > 8 || s[2] > 8) return IB_ERR_INVALID_ARG;
            off[e + 1] = off[e] + (int64_t)s[0] * s[1] * s[2];
            roff[e + 1] = roff[e] + (int64_t)s[1] * s[2];
        }
        if (off[ne] > (int64_t)INT32_MAX) return IB_ERR_INVALID_ARG;
        uniform = ne > 0 ? m->nsub[0] * m->nsub[1] * m->nsub[2] : 0;
        for (int64_t e = 1; e < ne && uniform; ++e)
            if (m->nsub[3 * e] != m->nsub[0] || m->nsub[3 * e + 1] != m->nsub[1] || m->nsub[3 * e + 2] != m->nsub[2])
                uniform = 0;
    }
    std::vector<int32_t> adj((size_t)8 * (nn > 0 ? nn : 1), -1), node_off((size_t)nn + 1, 0), node_slot;
    {
        std::vector<int32_t> cnt((size_t)(nn > 0 ? nn : 1), 0);
        for (int64_t e = 0; e < ne; ++e) {
            if (m->mat_id && (m->mat_id[e] < 0 || m->mat_id[e] >= m->n_mats)) return IB_ERR_INVALID_ARG;
            for (int a = 0; a < npe; ++a) {
                int32_t n = m->conn[e * npe + a];
                if (n < 0 || n >= nn) return IB_ERR_INVALID_ARG;
                if (npe == 8) {
                    if (cnt[n] >= 8) return IB_ERR_UNSUPPORTED;
                    adj[(size_t)cnt[n] * nn + n] = (int32_t)(e * 8 + a);      // ascending element id
                }
                cnt[n]++;
            }
        }
        if (m->nsub)                                      // a node of no element has lumped weight 0: 1/w_a would put NaN into Fhat and Un
            for (int64_t n = 0; n < nn; ++n)
                if (cnt[n] == 0) return IB_ERR_INVALID_ARG;
        if (npe != 8) {                                   // CSR: tets share nodes with any number of neighbours
            for (int64_t n = 0; n < nn; ++n) node_off[n + 1] = node_off[n] + cnt[n];
            node_slot.resize((size_t)ne * npe + 1);
            std::vector<int32_t> cur(node_off.begin(), node_off.end() - 1);
            for (int64_t e = 0; e < ne; ++e)
                for (int a = 0; a < npe; ++a) node_slot[cur[m->conn[e * npe + a]]++] = (int32_t)(e * npe + a);
        }
    }

    if (cudaSetDevice(device) != cudaSuccess) return IB_ERR_CUDA;
    ib_ctx *c = new (std::nothrow) ib_ctx();
    if (!c) return IB_ERR_ALLOC;
    memset(c, 0, sizeof(*c));
    c->device = device;
    c->grid = *g;
    c->inv_h = 1.0 / g->h;
    c->n_nodes = nn;
    c->n_elems = ne;
    c->n_cells = (int64_t)g->nx * g->ny * g->nz;
    c->nodal = m->nsub == nullptr;
    c->n_points = c->nodal ? nn : off[ne];
    c->uniform_S = uniform;
    c->n_rows = roff[ne];
    if (uniform) { c->un[0] = m->nsub[0]; c->un[1] = m->nsub[1]; c->un[2] = m->nsub[2]; }
    c->n_mats = m->n_mats;
    c->elem_type = m->elem_type;
    c->npe = npe;
    c->variant = 1;
    c->graph_on = 1;

    ib_status s = IB_OK;
#define TRY(x) do { if (s == IB_OK) s = (x); } while (0)
    TRY(dev_upload(&c->d_conn, m->conn, (size_t)ne * npe));
    TRY(dev_upload(&c->d_X, m->X_ref, (size_t)nn * 3));
    if (m->fibers) TRY(dev_upload(&c->d_fib, m->fibers, (size_t)ne * 6));
    if (m->mat_id) TRY(dev_upload(&c->d_mat_id, m->mat_id, (size_t)ne));
    if (m->nsub) TRY(dev_upload(&c->d_nsub, m->nsub, (size_t)ne * 3));
    TRY(dev_upload(&c->d_pt_off, off.data(), (size_t)ne + 1));
    TRY(dev_upload(&c->d_mats, m->mats, (size_t)(m->n_mats > 0 ? m->n_mats : 0)));
    TRY(dev_upload(&c->d_adj, adj.data(), (size_t)8 * (nn > 0 ? nn : 1)));
    if (npe != 8) {
        TRY(dev_upload(&c->d_node_off, node_off.data(), (size_t)nn + 1));
        TRY(dev_upload(&c->d_node_slot, node_slot.data(), node_slot.size()));
    }
    const size_t P = (size_t)c->n_points;
    TRY(dev_alloc((void **)&c->d_wa, (size_t)nn * sizeof(double)));
    TRY(dev_alloc((void **)&c->d_Ce, (size_t)ne * 3 * (npe > 8 ? npe : 8) * sizeof(double)));
    TRY(dev_alloc((void **)&c->d_geo, (size_t)ne * 80 * sizeof(double)));
    TRY(dev_alloc((void **)&c->d_Fhat, (size_t)nn * 3 * sizeof(double)));
    TRY(dev_alloc((void **)&c->d_B, (size_t)nn * 3 * sizeof(double)));
    if (!c->nodal) {
        TRY(dev_alloc((void **)&c->d_Wp, P * sizeof(double)));
        TRY(dev_alloc((void **)&c->d_xp, P * 3 * sizeof(double)));
        TRY(dev_alloc((void **)&c->d_Gp, P * 3 * sizeof(double)));
        TRY(dev_alloc((void **)&c->d_Up, P * 3 * sizeof(double)));
    }
    const int n_tiles = (int)(c->n_cells / 64);          // 4x4x4-cell tiles of the tiled path
    // counters + scan partials, then the bins (4 z-layer bins per tile): one block, zeroed by one memset per step
    c->tile_hdr = (IB_TILE_HDR + 2 * (n_tiles / 1024 + 2) + 3) & ~3;
    TRY(dev_alloc((void **)&c->d_tile_count, (size_t)(c->tile_hdr + 4 * n_tiles + 4) * sizeof(int32_t)));
    if (s == IB_OK) c->d_tile_cur = c->d_tile_count + c->tile_hdr;
    TRY(dev_alloc((void **)&c->d_tile_start, (size_t)(4 * n_tiles + 4) * sizeof(int32_t)));
    TRY(dev_upload(&c->d_row_off, roff.data(), (size_t)ne + 1));
    TRY(dev_alloc((void **)&c->d_status, 2 * sizeof(long long)));
    if (s == IB_OK && (cudaStreamCreateWithFlags(&c->side, cudaStreamNonBlocking) != cudaSuccess ||
                       cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
                       cudaEventCreateWithFlags(&c->ev_join, cudaEventDisableTiming) != cudaSuccess ||
                       cudaEventCreateWithFlags(&c->ev_aux, cudaEventDisableTiming) != cudaSuccess ||
                       cudaStreamCreateWithFlags(&c->side2, cudaStreamNonBlocking) != cudaSuccess ||
                       cudaEventCreateWithFlags(&c->ev_sfork, cudaEventDisableTiming) != cudaSuccess ||
                       cudaEventCreateWithFlags(&c->ev_sjoin, cudaEventDisableTiming) != cudaSuccess))
        s = IB_ERR_CUDA;
    if (s == IB_OK && cudaEventCreateWithFlags(&c->ev_zero, cudaEventDisableTiming) != cudaSuccess) s = IB_ERR_CUDA;
    if (s == IB_OK && (cudaStreamCreateWithFlags(&c->side3, cudaStreamNonBlocking) != cudaSuccess ||
                       cudaStreamCreateWithFlags(&c->side4, cudaStreamNonBlocking) != cudaSuccess))
        s = IB_ERR_CUDA;
    for (int k = 0; k < IB_MAX_SLABS && s == IB_OK; ++k)
        if (cudaEventCreateWithFlags(&c->ev_slab[k], cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&c->ev_h2d[k], cudaEventDisableTiming) != cudaSuccess)
            s = IB_ERR_CUDA;
    if (s == IB_OK) s = reset_status(c, 0);
    if (s == IB_OK) s = ibk_sort_reserve(c, c->n_points);
    if (s == IB_OK) s = ibk_bin_reserve(c, c->n_points);
    if (s == IB_OK) s = ibk_precompute_weights(c, 0);
    if (s == IB_OK && npe == 8) s = ibk_fe_precompute(c, 0);
    if (s == IB_OK && cudaDeviceSynchronize() != cudaSuccess) s = IB_ERR_CUDA;
#undef TRY
    if (s == IB_OK) {
        unsigned long long hs = 0;
        int code = 0;
        long long id = -1;
        if (cudaMemcpy(&hs, c->d_status, sizeof(hs), cudaMemcpyDeviceToHost) != cudaSuccess) s = IB_ERR_CUDA;
        else {
            ib_status_unpack(hs, &code, &id);
            if (code != 0) s = (ib_status)code;                     // inverted reference element
        }
    }
    if (s != IB_OK) { ib_destroy(c); return s; }
    *out = c;
    return IB_OK;
}

extern "C" int64_t ib_num_points(const ib_ctx *c) { return c ? c->n_points : -1; }
extern "C" int64_t ib_num_nodes(const ib_ctx *c) { return c ? c->n_nodes : -1; }
extern "C" int64_t ib_num_elems(const ib_ctx *c) { return c ? c->n_elems : -1; }
extern "C" int64_t ib_launch_count(const ib_ctx *c) { return c ? c->launches : -1; }

extern "C" ib_status ib_set_variant(ib_ctx *c, int32_t variant)
{
    if (!c || (variant != 0 && variant != 1)) return IB_ERR_INVALID_ARG;
    c->variant = variant;
    c->gstate = 0;
    return IB_OK;
}

static ib_status replace_ids(int32_t **dst, const int32_t *src, size_t n)
{
    if (*dst) { cudaFree(*dst); *dst = nullptr; }
    return n ? dev_upload(dst, src, n) : IB_OK;
}

extern "C" ib_status ib_set_tethers(ib_ctx *c, int64_t n, const int32_t *ids, double kappa)
{
    if (!c || n < 0 || (n > 0 && !ids) || !std::isfinite(kappa)) return IB_ERR_INVALID_ARG;
    {
        std::vector<unsigned char> seen((size_t)(c->n_nodes > 0 ? c->n_nodes : 1), 0);      // the kernel adds without atomics: ids must be distinct
        for (int64_t k = 0; k < n; ++k) {
            if (ids[k] < 0 || ids[k] >= c->n_nodes || seen[ids[k]]) return IB_ERR_INVALID_ARG;
            seen[ids[k]] = 1;
        }
    }
    if (cudaSetDevice(c->device) != cudaSuccess) return IB_ERR_CUDA;
    cudaDeviceSynchronize();
    c->gstate = 0;
    c->n_teth = 0;
    ib_status s = replace_ids(&c->d_teth_ids, ids, (size_t)n);
    if (s != IB_OK) return s;
    c->n_teth = n;
    c->kappa_t = kappa;
    return IB_OK;
}

extern "C" ib_status ib_set_surface(ib_ctx *c, int64_t n_faces, int32_t npf, const int32_t *faces)
{
    if (!c || n_faces < 0 || (n_faces > 0 && (!faces || (npf != 3 && npf != 4 && npf != 6)))) return IB_ERR_INVALID_ARG;
    for (int64_t k = 0; k < n_faces * npf; ++k)
        if (faces[k] < 0 || faces[k] >= c->n_nodes) return IB_ERR_INVALID_ARG;
    if (cudaSetDevice(c->device) != cudaSuccess) return IB_ERR_CUDA;
    cudaDeviceSynchronize();
    c->gstate = 0;
    c->n_faces = 0;
    ib_status s = replace_ids(&c->d_faces, faces, (size_t)(n_faces * npf));
    if (s != IB_OK) return s;
    c->n_faces = n_faces;
    c->npf = npf;
    return IB_OK;
}

extern "C" ib_status ib_set_loads(ib_ctx *c, const double *qt0, double p)
{
    if (!c || !std::isfinite(p)) return IB_ERR_INVALID_ARG;
    for (int k = 0; k < 3; ++k) {
        if (qt0 && !std::isfinite(qt0[k])) return IB_ERR_INVALID_ARG;
        c->qt0[k] = qt0 ? qt0[k] : 0.0;
    }
    c->p_load = p;
    c->gstate = 0;                                   // the load values are kernel arguments of a captured step
    return IB_OK;
}

extern "C" ib_status ib_set_graph(ib_ctx *c, int32_t on)
{
    if (!c) return IB_ERR_INVALID_ARG;
    c->graph_on = on ? 1 : 0;
    c->gstate = 0;
    return IB_OK;
}

static inline ib_status enter(ib_ctx *c, void *stream)
{
    if (!c) return IB_ERR_INVALID_ARG;
    if (cudaSetDevice(c->device) != cudaSuccess) return IB_ERR_CUDA;
    c->last_stream = ST(stream);
    return IB_OK;
}

extern "C" ib_status ib_fe_force(ib_ctx *c, const double *x, double *B, void *stream)
{
    ib_status s = enter(c, stream);
    if (s != IB_OK) return s;
    if (!x || !B) return IB_ERR_INVALID_ARG;
    return ibk_fe_force(c, x, B, nullptr, ST(stream));
}

__global__ void ibk_scale_by_inv(int64_t n_nodes, const double *__restrict__ B, const double *__restrict__ wa,
                                 double *__restrict__ Fhat)
{
    int64_t n = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= n_nodes) return;
    double r = 1.0 / wa[n];
    Fhat[n] = B[n] * r; Fhat[n_nodes + n] = B[n_nodes + n] * r; Fhat[2 * n_nodes + n] = B[2 * n_nodes + n] * r;
}

extern "C" ib_status ib_points(ib_ctx *c, const double *x, const double *B, double *xp, double *Gp, void *stream)
{
    ib_status s = enter(c, stream);
    if (s != IB_OK) return s;
    if ((xp && !x) || (Gp && !B)) return IB_ERR_INVALID_ARG;
    cudaStream_t st = ST(stream);
    const size_t nb = (size_t)c->n_nodes * 3 * sizeof(double);
    if (c->nodal) {
        if (xp && nb) IB_CUDA_TRY(cudaMemcpyAsync(xp, x, nb, cudaMemcpyDeviceToDevice, st));
        if (Gp && nb) IB_CUDA_TRY(cudaMemcpyAsync(Gp, B, nb, cudaMemcpyDeviceToDevice, st));
        return IB_OK;
    }
    if (Gp && c->n_nodes > 0) {
        ibk_scale_by_inv<<<ib_blocks(c->n_nodes, 256), 256, 0, st>>>(c->n_nodes, B, c->d_wa, c->d_Fhat);
        c->launches++;
    }
    return ibk_points(c, x, c->d_Fhat, xp, Gp, st);
}

extern "C" ib_status ib_restrict(ib_ctx *c, const double *Up, double *Un, void *stream)
{
    ib_status s = enter(c, stream);
    if (s != IB_OK) return s;
    if (!Up || !Un) return IB_ERR_INVALID_ARG;
    if (c->nodal) {
        const size_t nb = (size_t)c->n_nodes * 3 * sizeof(double);
        if (nb) IB_CUDA_TRY(cudaMemcpyAsync(Un, Up, nb, cudaMemcpyDeviceToDevice, ST(stream)));
        return IB_OK;
    }
    return ibk_restrict(c, Up, Un, ST(stream));
}

extern "C" ib_status ib_bin_sort(ib_ctx *c, const double *xp, int64_t P, int64_t *key_out, int32_t *perm_out,
                                 void *stream)
{
    ib_status s = enter(c, stream);
    if (s != IB_OK) return s;
    if (P < 0 || P > (int64_t)INT32_MAX || (P > 0 && !xp)) return IB_ERR_INVALID_ARG;
    return ibk_bin_sort(c, xp, P, key_out, perm_out, 0, ST(stream));
}

extern "C" ib_status ib_spread(ib_ctx *c, const double *xp, const double *Gp, int64_t P, double *fu, double *fv,
                               double *fw, int32_t accumulate, void *stream)
{
    ib_status s = enter(c, stream);
    if (s != IB_OK) return s;
    if (P < 0 || P > (int64_t)INT32_MAX || !fu || !fv || !fw || (P > 0 && (!xp || !Gp))) return IB_ERR_INVALID_ARG;
    if (P == 0) {
        if (!accumulate) {
            size_t nb = (size_t)c->n_cells * sizeof(double);
            IB_CUDA_TRY(cudaMemsetAsync(fu, 0, nb, ST(stream)));
            IB_CUDA_TRY(cudaMemsetAsync(fv, 0, nb, ST(stream)));
            IB_CUDA_TRY(cudaMemsetAsync(fw, 0, nb, ST(stream)));
        }
        return IB_OK;
    }
    return ibk_spread_interp(c, xp, Gp, P, nullptr, nullptr, nullptr, fu, fv, fw, nullptr, accumulate, ST(stream));
}

extern "C" ib_status ib_interp(ib_ctx *c, const double *xp, int64_t P, const double *u, const double *v,
                               const double *w, double *Up, void *stream)
{
    ib_status s = enter(c, stream);
    if (s != IB_OK) return s;
    if (P < 0 || P > (int64_t)INT32_MAX || !u || !v || !w || (P > 0 && (!xp || !Up))) return IB_ERR_INVALID_ARG;
    if (P == 0) return IB_OK;
    return ibk_spread_interp(c, xp, nullptr, P, u, v, w, nullptr, nullptr, nullptr, Up, 0, ST(stream));
}

static ib_status coupling_step_body(ib_ctx *c, const double *x, const double *u, const double *v,
                                    const double *w, double *fu, double *fv, double *fw, double *Un,
                                    double *B, cudaStream_t st)
{
    ib_status s = IB_OK;
    double *Bd = B ? B : c->d_B;
    if (c->nodal) {
        // the paper's nodal rule verbatim (L241-257): points = nodes, spread B itself, Un = U^IB
        ib_prof_begin(c, IB_PHASE_FE_FORCE, st);
        s = ibk_fe_force(c, x, Bd, nullptr, st);
        ib_prof_end(c, IB_PHASE_FE_FORCE, st);
        if (s != IB_OK) return s;
        return ibk_spread_interp(c, x, Bd, c->n_nodes, u, v, w, fu, fv, fw, Un, 0, st);
    }
    if (c->variant == 1) {
        // Fork: zero-fill of f and the count pass + scan of the point binning need only the positions,
        // so they run on the context's side stream while the FE force runs on the caller's stream.
        const size_t gb = (size_t)c->n_cells * sizeof(double);
        const bool overlap = !c->profile && c->n_points > 0;      // per-phase timing wants the phases in sequence
        cudaStream_t s2 = overlap ? c->side : st;
        if (overlap) {
            IB_CUDA_TRY(cudaEventRecord(c->ev_fork, st));
            IB_CUDA_TRY(cudaStreamWaitEvent(s2, c->ev_fork, 0));
        }
        // the zero-fill of f is a branch of its own (third stream): neither the force nor the binning waits for it
        cudaStream_t sz = overlap ? c->side2 : st;
        if (overlap) IB_CUDA_TRY(cudaStreamWaitEvent(sz, c->ev_fork, 0));
        ib_prof_begin(c, IB_PHASE_ZERO, st);
        IB_CUDA_TRY(cudaMemsetAsync(fu, 0, gb, sz));
        IB_CUDA_TRY(cudaMemsetAsync(fv, 0, gb, sz));
        IB_CUDA_TRY(cudaMemsetAsync(fw, 0, gb, sz));
        ib_prof_end(c, IB_PHASE_ZERO, st);
        if (overlap) IB_CUDA_TRY(cudaEventRecord(c->ev_zero, sz));
        if (c->n_points > 0) {
            s = ibk_bin_reserve(c, c->n_points);
            if (s != IB_OK) return s;
            ib_prof_begin(c, IB_PHASE_POINTS, st);
            s = ibk_bin_points(c, 1, nullptr, nullptr, c->n_points, x, nullptr, nullptr, 1, s2);
            ib_prof_end(c, IB_PHASE_POINTS, st);
            if (s != IB_OK) return s;
        }
        if (overlap) IB_CUDA_TRY(cudaEventRecord(c->ev_join, s2));
        ib_prof_begin(c, IB_PHASE_FE_FORCE, st);
        s = ibk_fe_force(c, x, Bd, c->d_Fhat, st);
        ib_prof_end(c, IB_PHASE_FE_FORCE, st);
        if (s != IB_OK) return s;
        if (overlap) {
            IB_CUDA_TRY(cudaStreamWaitEvent(st, c->ev_join, 0));
            IB_CUDA_TRY(cudaStreamWaitEvent(st, c->ev_zero, 0));
        }
        if (c->n_points > 0)
            s = ibk_tiled_spread_interp(c, 1, nullptr, nullptr, c->n_points, x, c->d_Fhat, u, v, w, fu, fv, fw,
                                        c->d_Up, 1, st);
    } else {
        ib_prof_begin(c, IB_PHASE_FE_FORCE, st);
        s = ibk_fe_force(c, x, Bd, c->d_Fhat, st);
        ib_prof_end(c, IB_PHASE_FE_FORCE, st);
        if (s != IB_OK) return s;
        ib_prof_begin(c, IB_PHASE_POINTS, st);
        s = ibk_points(c, x, c->d_Fhat, c->d_xp, c->d_Gp, st);
        ib_prof_end(c, IB_PHASE_POINTS, st);
        if (s != IB_OK) return s;
        s = ibk_spread_interp(c, c->d_xp, c->d_Gp, c->n_points, u, v, w, fu, fv, fw, c->d_Up, 0, st);
    }
    if (s != IB_OK) return s;
    ib_prof_begin(c, IB_PHASE_RESTRICT, st);
    s = ibk_restrict(c, c->d_Up, Un, st);
    ib_prof_end(c, IB_PHASE_RESTRICT, st);
    return s;
}

__global__ void ibk_axpy(int64_t n, const double *__restrict__ x, double a, const double *__restrict__ y,
                         double *__restrict__ out)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = fma(a, y[i], x[i]);
}

extern "C" ib_status ib_step_eq16(ib_ctx *c, const double *x, const double *u, const double *v, const double *w,
                                  double dt, double *x_new, double *fu, double *fv, double *fw, double *Un,
                                  double *B, void *stream)
{
    ib_status s = enter(c, stream);
    if (s != IB_OK) return s;
    if (!x || !u || !v || !w || !x_new || x_new == x || !fu || !fv || !fw || !Un || !std::isfinite(dt))
        return IB_ERR_INVALID_ARG;
    cudaStream_t st = ST(stream);
    double *Bd = B ? B : c->d_B;
    const int64_t n3 = 3 * c->n_nodes;
    // 1. U^IB = I(X^n, u^n), projected to the nodes
    if (c->nodal) {
        if (c->n_nodes > 0) s = ibk_spread_interp(c, x, nullptr, c->n_nodes, u, v, w, nullptr, nullptr, nullptr, Un, 0, st);
    } else {
        if (c->n_points > 0) {
            if (c->variant == 1)
                s = ibk_tiled_spread_interp(c, 1, nullptr, nullptr, c->n_points, x, nullptr, u, v, w, nullptr, nullptr,
                                            nullptr, c->d_Up, 0, st);
            else {
                s = ibk_points(c, x, nullptr, c->d_xp, nullptr, st);
                if (s == IB_OK) s = ibk_spread_interp(c, c->d_xp, nullptr, c->n_points, u, v, w, nullptr, nullptr, nullptr,
                                                      c->d_Up, 0, st);
            }
        }
        if (s == IB_OK) s = ibk_restrict(c, c->d_Up, Un, st);
    }
    if (s != IB_OK) return s;
    // 2. x_new = x + dt Un
    if (n3 > 0) {
        ibk_axpy<<<ib_blocks(n3, 256), 256, 0, st>>>(n3, x, dt, Un, x_new);
        c->launches++;
    }
    // 3. F^{n+1} at the new positions
    s = ibk_fe_force(c, x_new, Bd, c->nodal ? nullptr : c->d_Fhat, st);
    if (s != IB_OK) return s;
    // 4. f = E(X^n, F^{n+1}): spread at the OLD positions
    const size_t gb = (size_t)c->n_cells * sizeof(double);
    if (c->nodal) return ibk_spread_interp(c, x, Bd, c->n_nodes, nullptr, nullptr, nullptr, fu, fv, fw, nullptr, 0, st);
    if (c->variant == 1) {
        IB_CUDA_TRY(cudaMemsetAsync(fu, 0, gb, st));
        IB_CUDA_TRY(cudaMemsetAsync(fv, 0, gb, st));
        IB_CUDA_TRY(cudaMemsetAsync(fw, 0, gb, st));
        if (c->n_points == 0) return IB_OK;
        return ibk_tiled_spread_interp(c, 1, nullptr, nullptr, c->n_points, x, c->d_Fhat, nullptr, nullptr, nullptr, fu, fv,
                                       fw, nullptr, 0, st);
    }
    s = ibk_points(c, x, c->d_Fhat, c->d_xp, c->d_Gp, st);
    if (s != IB_OK) return s;
    return ibk_spread_interp(c, c->d_xp, c->d_Gp, c->n_points, nullptr, nullptr, nullptr, fu, fv, fw, nullptr, 0, st);
}

extern "C" ib_status ib_coupling_step(ib_ctx *c, const double *x, const double *u, const double *v,
                                      const double *w, double *fu, double *fv, double *fw, double *Un,
                                      double *B, void *stream)
{
    ib_status s = enter(c, stream);
    if (s != IB_OK) return s;
    if (!x || !u || !v || !w || !fu || !fv || !fw || !Un) return IB_ERR_INVALID_ARG;
    cudaStream_t st = ST(stream);
    const bool capturable = c->graph_on && !c->profile && st != 0 && st != cudaStreamLegacy && st != cudaStreamPerThread;
    if (!capturable) return coupling_step_body(c, x, u, v, w, fu, fv, fw, Un, B, st);
    const void *key[11] = {x, u, v, w, fu, fv, fw, Un, B, (const void *)st, (const void *)(intptr_t)c->variant};
    const bool same = c->gstate != 0 && memcmp(key, c->gkey, sizeof(key)) == 0;
    if (same && c->gstate == 2) {
        IB_CUDA_TRY(cudaGraphLaunch(c->gexec, st));
        c->launches += c->g_launches;
        return IB_OK;
    }
    if (same && c->gstate == 1) {
        // second call with these pointers: everything lazy (attributes, buffers) exists -> capture
        if (c->gexec) { cudaGraphExecDestroy(c->gexec); c->gexec = nullptr; }
        const int64_t l0 = c->launches;
        if (cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
            s = coupling_step_body(c, x, u, v, w, fu, fv, fw, Un, B, st);
            cudaGraph_t g = nullptr;
            cudaError_t e = cudaStreamEndCapture(st, &g);
            if (s == IB_OK && e == cudaSuccess && g && cudaGraphInstantiate(&c->gexec, g, 0) == cudaSuccess) {
                cudaGraphDestroy(g);
                c->g_launches = c->launches - l0;
                c->launches = l0;
                c->gstate = 2;
                IB_CUDA_TRY(cudaGraphLaunch(c->gexec, st));
                c->launches += c->g_launches;
                return IB_OK;
            }
            if (g) cudaGraphDestroy(g);
            cudaGetLastError();
            c->launches = l0;
        }
        c->gstate = 0;
        c->graph_on = 0;                                   // capture is not possible here: stay eager
        return coupling_step_body(c, x, u, v, w, fu, fv, fw, Un, B, st);
    }
    memcpy(c->gkey, key, sizeof(key));
    c->gstate = 1;
    return coupling_step_body(c, x, u, v, w, fu, fv, fw, Un, B, st);
}

static ib_status host_step_pipelined(ib_ctx *c, const double *x_h, const double *u_h, const double *v_h, const double *w_h,
                                     double *fu_h, double *fv_h, double *fw_h, double *Un_h, double *B_h, int packed, cudaStream_t st);
static ib_status host_step(ib_ctx *c, const double *x_h, const double *u_h, const double *v_h, const double *w_h, double *fu_h,
                           double *fv_h, double *fw_h, double *Un_h, double *B_h, int packed, void *stream);

extern "C" ib_status ib_coupling_step_host(ib_ctx *c, const double *x_h, const double *u_h, const double *v_h,
                                           const double *w_h, double *fu_h, double *fv_h, double *fw_h,
                                           double *Un_h, double *B_h, void *stream)
{
    return host_step(c, x_h, u_h, v_h, w_h, fu_h, fv_h, fw_h, Un_h, B_h, 0, stream);
}

static ib_status host_step(ib_ctx *c, const double *x_h, const double *u_h, const double *v_h, const double *w_h, double *fu_h,
                           double *fv_h, double *fw_h, double *Un_h, double *B_h, int packed, void *stream)
{
    ib_status s = enter(c, stream);
    if (s != IB_OK) return s;
    if (!x_h || !u_h || !v_h || !w_h || !fu_h || !fv_h || !fw_h || !Un_h) return IB_ERR_INVALID_ARG;
    cudaStream_t st = ST(stream);
    const size_t nb = (size_t)c->n_nodes * 3 * sizeof(double), gb = (size_t)c->n_cells * sizeof(double);
    if (!c->d_hx) {
        ib_status a = IB_OK;
        double **bufs[] = {&c->d_hx, &c->d_hUn, &c->d_hB};
        for (auto b : bufs) if (a == IB_OK) a = dev_alloc((void **)b, nb);
        // u,v,w and fu,fv,fw are one [3][n_cells] block each: a caller whose host arrays are laid out the same way
        // (ib_coupling_step_host3) gets one copy per slab and direction instead of three
        if (a == IB_OK) a = dev_alloc((void **)&c->d_hu, 3 * gb);
        if (a == IB_OK) a = dev_alloc((void **)&c->d_hfu, 3 * gb);
        if (a != IB_OK) return a;
        c->d_hv = c->d_hu + c->n_cells; c->d_hw = c->d_hu + 2 * c->n_cells;
        c->d_hfv = c->d_hfu + c->n_cells; c->d_hfw = c->d_hfu + 2 * c->n_cells;
    }
    const bool pipelined = c->variant == 1 && !c->nodal && !c->profile && c->n_points > 0;
    if (!pipelined) {
        IB_CUDA_TRY(cudaMemcpyAsync(c->d_hx, x_h, nb, cudaMemcpyHostToDevice, st));
        IB_CUDA_TRY(cudaMemcpyAsync(c->d_hu, u_h, gb, cudaMemcpyHostToDevice, st));
        IB_CUDA_TRY(cudaMemcpyAsync(c->d_hv, v_h, gb, cudaMemcpyHostToDevice, st));
        IB_CUDA_TRY(cudaMemcpyAsync(c->d_hw, w_h, gb, cudaMemcpyHostToDevice, st));
        s = ib_coupling_step(c, c->d_hx, c->d_hu, c->d_hv, c->d_hw, c->d_hfu, c->d_hfv, c->d_hfw, c->d_hUn,
                             B_h ? c->d_hB : nullptr, stream);
        if (s != IB_OK) return s;
        IB_CUDA_TRY(cudaMemcpyAsync(fu_h, c->d_hfu, gb, cudaMemcpyDeviceToHost, st));
        IB_CUDA_TRY(cudaMemcpyAsync(fv_h, c->d_hfv, gb, cudaMemcpyDeviceToHost, st));
        IB_CUDA_TRY(cudaMemcpyAsync(fw_h, c->d_hfw, gb, cudaMemcpyDeviceToHost, st));
        IB_CUDA_TRY(cudaMemcpyAsync(Un_h, c->d_hUn, nb, cudaMemcpyDeviceToHost, st));
        if (B_h) IB_CUDA_TRY(cudaMemcpyAsync(B_h, c->d_hB, nb, cudaMemcpyDeviceToHost, st));
        IB_CUDA_TRY(cudaStreamSynchronize(st));
        return IB_OK;
    }
    s = host_step_pipelined(c, x_h, u_h, v_h, w_h, fu_h, fv_h, fw_h, Un_h, B_h, packed, st);
    if (s != IB_OK) {
        // copies to and from the caller's host buffers may still be in flight on the internal streams: no
        // return before they have drained
        cudaStream_t all[5] = {st, c->side, c->side2, c->side3, c->side4};
        for (cudaStream_t q : all) cudaStreamSynchronize(q);
        cudaGetLastError();
    }
    return s;
}

extern "C" ib_status ib_coupling_step_host3(ib_ctx *c, const double *x_h, const double *uvw_h, double *f_h, double *Un_h,
                                            double *B_h, void *stream)
{
    if (!c || !uvw_h || !f_h) return IB_ERR_INVALID_ARG;
    return host_step(c, x_h, uvw_h, uvw_h + c->n_cells, uvw_h + 2 * c->n_cells, f_h, f_h + c->n_cells, f_h + 2 * c->n_cells, Un_h,
                     B_h, 1, stream);
}

static ib_status host_step_pipelined(ib_ctx *c, const double *x_h, const double *u_h, const double *v_h, const double *w_h,
                                     double *fu_h, double *fv_h, double *fw_h, double *Un_h, double *B_h, int packed, cudaStream_t st)
{
    ib_status s = IB_OK;
    const size_t nb = (size_t)c->n_nodes * 3 * sizeof(double), gb = (size_t)c->n_cells * sizeof(double);
    // Pipelined in z-slabs of the tile list (tiles are numbered z-major).  The force side of the step needs
    // only x, so it runs while u,v,w cross the bus, slab by slab, on a side stream.  The fused
    // spread + interpolate kernel of slab k needs the velocity layers of slab k and 2 more on either side
    // and a point reaches at most 2 cells beyond its own 4-cell tile layer, so after slab k every z-layer
    // below the last tile layer of that slab is final and goes back to the host on a third stream while the
    // next slabs run; the first tile layer (periodic wrap of the last slab) goes last.  Consecutive slabs
    // alternate between two streams so that the tail of one kernel is filled by the next.
    //   st / side4 : H2D x | FE force | scatter, sparse tiles: spread | SPREAD+INTERP slab 0 | 1 | ... | restrict | D2H Un, B
    //   side       :       H2D u,v,w wrap layers + slab 0 | slab 1 | ...
    //   side2      :       zero f, count pass, scan                      ...      sparse tiles: interpolate
    //   side3      :                                                        D2H f layers of slab 0 | slab 1 | ...
    cudaStream_t s2 = c->side, s3 = c->side3, s4 = c->side4, ss = c->side2;
    double *Bd = B_h ? c->d_hB : c->d_B;
    const int K = ib_slab_count(c), nz = c->grid.nz, zs = 4 * ib_slab_layers(c);
    const size_t plane = (size_t)c->grid.nx * c->grid.ny, pb = plane * sizeof(double);
    const int z_first = nz < 4 ? nz : 4;          // wrap margin: the last z_first layers come first, the first go back last
    // z-layers [z0, z0 + nl) of the three components: one 2-D copy (3 rows, pitch n_cells) when the host arrays
    // are one [3][n_cells] block like the device's, else three copies
    // (only on the caller's word -- ib_coupling_step_host3: three arrays that merely happen to be adjacent may be
    // separate allocations, which one copy cannot span)
    const bool upack = packed != 0, fpack = packed != 0;
    auto h2d3 = [&](int z0, int nl, cudaStream_t q) -> cudaError_t {
        if (nl <= 0) return cudaSuccess;
        if (upack) return cudaMemcpy2DAsync(c->d_hu + z0 * plane, gb, u_h + z0 * plane, gb, (size_t)nl * pb, 3, cudaMemcpyHostToDevice, q);
        const double *uh[3] = {u_h, v_h, w_h};
        double *ud[3] = {c->d_hu, c->d_hv, c->d_hw};
        for (int d = 0; d < 3; ++d) {
            cudaError_t e = cudaMemcpyAsync(ud[d] + z0 * plane, uh[d] + z0 * plane, (size_t)nl * pb, cudaMemcpyHostToDevice, q);
            if (e != cudaSuccess) return e;
        }
        return cudaSuccess;
    };
    auto d2h3 = [&](int z0, int nl, cudaStream_t q) -> cudaError_t {
        if (nl <= 0) return cudaSuccess;
        if (fpack) return cudaMemcpy2DAsync(fu_h + z0 * plane, gb, c->d_hfu + z0 * plane, gb, (size_t)nl * pb, 3, cudaMemcpyDeviceToHost, q);
        double *fh[3] = {fu_h, fv_h, fw_h}, *fd[3] = {c->d_hfu, c->d_hfv, c->d_hfw};
        for (int d = 0; d < 3; ++d) {
            cudaError_t e = cudaMemcpyAsync(fh[d] + z0 * plane, fd[d] + z0 * plane, (size_t)nl * pb, cudaMemcpyDeviceToHost, q);
            if (e != cudaSuccess) return e;
        }
        return cudaSuccess;
    };
    // x first: the force side waits for it, and the copy engine serves the H2D copies of all streams in turn
    IB_CUDA_TRY(cudaMemcpyAsync(c->d_hx, x_h, nb, cudaMemcpyHostToDevice, st));
    IB_CUDA_TRY(cudaEventRecord(c->ev_fork, st));             // orders the side streams after x and earlier work on st
    IB_CUDA_TRY(cudaStreamWaitEvent(s2, c->ev_fork, 0));
    // zero-fill of f and the count pass of the binning beside the FE force, as in ib_coupling_step
    IB_CUDA_TRY(cudaStreamWaitEvent(ss, c->ev_fork, 0));
    IB_CUDA_TRY(cudaMemsetAsync(c->d_hfu, 0, 3 * gb, ss));
    IB_CUDA_TRY(cudaEventRecord(c->ev_zero, ss));             // f is zero
    s = ibk_bin_reserve(c, c->n_points);
    if (s == IB_OK) s = ibk_bin_points(c, 1, nullptr, nullptr, c->n_points, c->d_hx, nullptr, nullptr, 1, ss);
    IB_CUDA_TRY(cudaEventRecord(c->ev_join, ss));
    if (s == IB_OK) s = ibk_fe_force(c, c->d_hx, Bd, c->d_Fhat, st);
    if (s != IB_OK) return s;
    {
        if (K > 1) IB_CUDA_TRY(h2d3(nz - z_first, z_first, s2));
        // copy k ends 4 layers into slab k+1: with the wrap layers it is all that the kernel of slab k reads
        const int z_last = K > 1 ? nz - z_first : nz;
        for (int k = 0; k < K; ++k) {
            const int z0 = k == 0 ? 0 : (zs * k + 4 < z_last ? zs * k + 4 : z_last);
            const int z1 = (k == K - 1 || zs * (k + 1) + 4 > z_last) ? z_last : zs * (k + 1) + 4;
            IB_CUDA_TRY(h2d3(z0, z1 - z0, s2));
            IB_CUDA_TRY(cudaEventRecord(c->ev_h2d[k], s2));
        }
    }
    // While the device is busy with all that, the host finds the z-layers the structure can reach: the
    // sub-points are convex combinations of the nodes, a support reaches less than 3 cells, so outside
    // [f_lo, f_hi) the force stays the zero it was filled with and goes back right away (the D2H engine has
    // nothing else to do yet).  Not used when the structure comes within 4 layers of the z-walls (periodic wrap).
    int f_lo = 0, f_hi = nz;
    bool band = false;
    {
        const double *zh = x_h + 2 * c->n_nodes;
        double zmin = zh[0], zmax = zh[0];
        for (int64_t n = 1; n < c->n_nodes; ++n) {
            zmin = zh[n] < zmin ? zh[n] : zmin;
            zmax = zh[n] > zmax ? zh[n] : zmax;
        }
        const double lo = floor((zmin - c->grid.z0) * c->inv_h) - 4.0, hi = floor((zmax - c->grid.z0) * c->inv_h) + 6.0;
        if (lo >= (double)z_first && hi <= (double)(nz - z_first) && hi > lo) {      // false for NaN as well
            f_lo = (int)lo; f_hi = (int)hi; band = true;
        }
    }
    if (band) {
        IB_CUDA_TRY(cudaStreamWaitEvent(s3, c->ev_zero, 0));
        IB_CUDA_TRY(d2h3(0, f_lo, s3));
        IB_CUDA_TRY(d2h3(f_hi, nz - f_hi, s3));
    }
    IB_CUDA_TRY(cudaStreamWaitEvent(st, c->ev_join, 0));
    if (s == IB_OK) s = ibk_bin_points(c, 1, nullptr, nullptr, c->n_points, c->d_hx, c->d_Fhat, c->d_Up, 2, st);
    // the sparse tiles are spread before the first slab: beside it they would find no free SM until it ends
    if (s == IB_OK) s = ibk_small_launch(c, c->n_points, 1, 0, nullptr, nullptr, nullptr, c->d_hfu, c->d_hfv, c->d_hfw, nullptr, st);
    if (s != IB_OK) return s;
    IB_CUDA_TRY(cudaEventRecord(c->ev_aux, st));              // the records are binned
    IB_CUDA_TRY(cudaStreamWaitEvent(s4, c->ev_aux, 0));
    {
        int z_done = band ? f_lo : z_first;
        for (int k = 0; k < K; ++k) {
            cudaStream_t sk = (k & 1) ? s4 : st;
            IB_CUDA_TRY(cudaStreamWaitEvent(sk, c->ev_h2d[k], 0));
            s = ibk_tiled_launch(c, c->n_points, 1, 1, c->d_hu, c->d_hv, c->d_hw, c->d_hfu, c->d_hfv, c->d_hfw,
                                 c->d_Up, k, sk);
            if (s != IB_OK) return s;
            IB_CUDA_TRY(cudaEventRecord(c->ev_slab[k], sk));
            int z_end = (k == K - 1) ? nz : zs * (k + 1) - 4;
            if (z_end > f_hi) z_end = f_hi;                   // f_hi = nz without a band
            if (z_end < z_done) z_end = z_done;
            IB_CUDA_TRY(cudaStreamWaitEvent(s3, c->ev_slab[k], 0));
            IB_CUDA_TRY(d2h3(z_done, z_end - z_done, s3));
            z_done = z_end;
        }
        if (!band) IB_CUDA_TRY(d2h3(0, z_first, s3));
    }
    IB_CUDA_TRY(cudaStreamWaitEvent(ss, c->ev_aux, 0));
    IB_CUDA_TRY(cudaStreamWaitEvent(ss, c->ev_h2d[K - 1], 0));
    s = ibk_small_launch(c, c->n_points, 0, 1, c->d_hu, c->d_hv, c->d_hw, nullptr, nullptr, nullptr, c->d_Up, ss);
    if (s != IB_OK) return s;
    IB_CUDA_TRY(cudaEventRecord(c->ev_sfork, ss));            // the sparse tiles are interpolated
    IB_CUDA_TRY(cudaStreamWaitEvent(st, c->ev_sfork, 0));
    for (int k = 1; k < K; k += 2) IB_CUDA_TRY(cudaStreamWaitEvent(st, c->ev_slab[k], 0));
    s = ibk_restrict(c, c->d_Up, c->d_hUn, st);
    if (s != IB_OK) return s;
    IB_CUDA_TRY(cudaMemcpyAsync(Un_h, c->d_hUn, nb, cudaMemcpyDeviceToHost, st));
    if (B_h) IB_CUDA_TRY(cudaMemcpyAsync(B_h, c->d_hB, nb, cudaMemcpyDeviceToHost, st));
    IB_CUDA_TRY(cudaStreamSynchronize(st));
    IB_CUDA_TRY(cudaStreamSynchronize(s2));
    IB_CUDA_TRY(cudaStreamSynchronize(s3));
    return IB_OK;
}

extern "C" ib_status ib_check(ib_ctx *c, int64_t *first_bad)
{
    if (!c) return IB_ERR_INVALID_ARG;
    if (cudaSetDevice(c->device) != cudaSuccess) return IB_ERR_CUDA;
    if (first_bad) *first_bad = -1;
    if (cudaStreamSynchronize(c->last_stream) != cudaSuccess) return IB_ERR_CUDA;
    unsigned long long hs = 0;
    IB_CUDA_TRY(cudaMemcpy(&hs, c->d_status, sizeof(hs), cudaMemcpyDeviceToHost));
    if (cudaGetLastError() != cudaSuccess) return IB_ERR_CUDA;
    int code = 0;
    long long id = -1;
    ib_status_unpack(hs, &code, &id);
    if (code == 0) return IB_OK;
    if (first_bad) *first_bad = id;
    ib_status r = reset_status(c, c->last_stream);
    if (r != IB_OK) return r;
    cudaStreamSynchronize(c->last_stream);
    return (ib_status)code;
}

// ---------------------------------------------------------------------------------------------
// FP64 FMA peak probe (denominator of the "alu" roofline; MEASURED_PEAKS.json has no fp64 figure)
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
ibk_dfma_probe(double *out, int iters, double a, double b)
{
    double r0 = threadIdx.x, r1 = r0 + 1, r2 = r0 + 2, r3 = r0 + 3, r4 = r0 + 4, r5 = r0 + 5, r6 = r0 + 6, r7 = r0 + 7;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            r0 = fma(r0, a, b); r1 = fma(r1, a, b); r2 = fma(r2, a, b); r3 = fma(r3, a, b);
            r4 = fma(r4, a, b); r5 = fma(r5, a, b); r6 = fma(r6, a, b); r7 = fma(r7, a, b);
        }
    }
    double s = r0 + r1 + r2 + r3 + r4 + r5 + r6 + r7;
    if (s == 123.456) out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

extern "C" ib_status ib_probe_dfma(int32_t device, double *dfma_per_s, double *ms_out)
{
    if (!dfma_per_s) return IB_ERR_INVALID_ARG;
    if (cudaSetDevice(device) != cudaSuccess) return IB_ERR_CUDA;
    cudaDeviceProp prop;
    IB_CUDA_TRY(cudaGetDeviceProperties(&prop, device));
    double *d = nullptr;
    int blocks = prop.multiProcessorCount * 8, iters = 4096;
    IB_CUDA_TRY(cudaMalloc(&d, (size_t)blocks * 256 * sizeof(double)));
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    float best = 1e30f;
    for (int rep = 0; rep < 5; ++rep) {
        cudaEventRecord(e0);
        ibk_dfma_probe<<<blocks, 256>>>(d, iters, 0.999999, 1e-9);
        cudaEventRecord(e1);
        if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(d); return IB_ERR_CUDA; }
        float ms;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(d);
    double n = (double)blocks * 256.0 * iters * 64.0;
    *dfma_per_s = n / (best * 1e-3);
    if (ms_out) *ms_out = best;
    return IB_OK;
}
