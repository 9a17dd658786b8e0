/*
 * ibcouple.h -- C ABI of libibcouple: the Lagrangian-Eulerian coupling step of the matrix-free
 * immersed boundary (IB) method of arXiv 2503.22695, hand-written CUDA for NVIDIA B200 (sm_100a).
 *
 * One time step's coupling (Eq.(16), Eq.(20)-(22) L191-196) has three parts:
 *   (1) the hyperelastic finite-element nodal force, Eq.(20) L191 / L249-251, with F, J (L28-32)
 *       and P = dW/dF (L42-44) per element at 2x2x2 Gauss points, for the neo-Hookean (L441-445)
 *       and Holzapfel-Ogden (Eq.(12)-(15) L147-155) laws, accumulated to nodes with no assembled
 *       sparse matrix (abstract, L13);
 *   (2) spreading of that force to the staggered (MAC, L205) grid with the regularised delta
 *       delta_h, Eq.(24)-(26) L211-217 / L253-257 (Peskin 4-point kernel, ref. 1 L474);
 *   (3) interpolation of the MAC velocity to the Lagrangian points, Eq.(27)-(29) L222-229 /
 *       L243-247, followed by the lumped L2 projection onto the nodes (L233-237, L241).
 *
 * Data layout:
 *   grid arrays u,v,w,fu,fv,fw : nx*ny*nz doubles each, x fastest: idx = (k*ny + j)*nx + i,
 *       periodic in all three directions; u[i,j,k] lives at (x0+i h, y0+(j+1/2)h, z0+(k+1/2)h),
 *       v at ((i+1/2)h, j h, (k+1/2)h), w at ((i+1/2)h, (j+1/2)h, k h) (+origin).
 *       nx, ny, nz must be multiples of 8 (tile edge of the binning key).
 *   node arrays X_ref, x, B, Un : component-major [3][n_nodes] doubles.
 *   point arrays xp, Gp, Up     : component-major [3][P] doubles.
 *   conn [n_elems][8] int32, local node a = ia + 2 ja + 4 ka (Q1 hexahedron; [n_elems][4] for P1 tets);
 *   fibers [6][n_elems] doubles = (e_f, e_s) per element, unit and orthogonal;
 *   nsub [n_elems][3] int32 sub-point counts (n1,n2,n3) per element, each in 1..8.
 *
 * Ownership: every pointer is owned by the caller. ib_create COPIES the static mesh description
 * (host pointers) to the device; the context owns those copies and all scratch. Pointers passed
 * to the per-step calls are DEVICE pointers unless the name ends in _host.
 * Streams: `stream` is a cudaStream_t passed as void* (NULL = default stream). Per-step calls
 * only enqueue work and return; they never synchronise. Device-detected errors (inverted
 * element, non-finite input) are latched in a device status word and reported by ib_check().
 * Thread safety: one context may be used from one host thread / one stream at a time.
 */
#ifndef IBCOUPLE_H
#define IBCOUPLE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ib_ctx ib_ctx;

typedef enum {
    IB_OK = 0,
    IB_ERR_INVALID_ARG = 1,      /* NULL pointer, negative size, h <= 0, bad mat_id / nsub / dims      */
    IB_ERR_UNSUPPORTED = 2,      /* hex node shared by more than 8 elements; sub-points on tetrahedra   */
    IB_ERR_ALLOC = 3,            /* cudaMalloc / malloc failed                                          */
    IB_ERR_CUDA = 4,             /* a CUDA runtime call failed (no device, launch error)                */
    IB_ERR_INVERTED_ELEMENT = 5, /* det J0 <= 0 or J <= 0 at a Gauss point (reported by ib_check)       */
    IB_ERR_NONFINITE = 6,        /* NaN/Inf position (reported by ib_check)                             */
    IB_ERR_OUT_OF_DOMAIN = 7,    /* point outside a bounded (periodic == 0) grid (reported by ib_check) */
    IB_ERR_TOO_LARGE = 8         /* ib_bin_sort_static: more points than its fixed scratch area holds  */
} ib_status;

/* Uniform MAC grid. periodic = 1: indices wrap in all three directions (the configs).
 * periodic = 0 (NEXT-4; the paper's box has Dirichlet walls, L200; reading A26): the arrays hold the faces
 * 0..n-1 of every component, a delta support that reaches outside is truncated, and a point outside
 * [x0, x0 + n h) is skipped (U = 0) and latched as IB_ERR_OUT_OF_DOMAIN. */
typedef struct {
    int32_t nx, ny, nz;
    double h, x0, y0, z0;
    int32_t periodic;
} ib_grid_desc;

typedef enum { IB_LAW_NEOHOOKEAN = 0, IB_LAW_HO = 1, IB_LAW_MSR = 2, IB_LAW_FR2 = 3 } ib_law;

/* Material row. HO (Eq.(12)-(15)): a,b isotropic; af,bf / as_,bs fibre and sheet; afs,bfs
 * coupling; kappa = kappa_stab of U(J) = kappa/2 (ln J)^2 (L94). neo-Hookean (L441-445):
 * a = mu (= 2 alpha), b = 0, fibre constants ignored.
 * NEXT-2 laws: IB_LAW_MSR, modified standard reinforcing model Eq.(7): a = G_T (b = 0),
 * af = G_L, bf = E_L.  IB_LAW_FR2, fibre-reinforced model 2 Eq.(10)-(11) L136-141: a = 2 C10 C01,
 * b = C01, af, bf, fibre term on I4f without the tension switch.  Fibre-reinforced model 1,
 * Eq.(8)-(9) L128-134, is IB_LAW_HO with a = 2 C1, b = 0, as_ = afs = 0.
 * Ta: active tension T_a(t) of L317-331, P += Ta (1 + 4.9 (sqrt(I4f) - 1)) F e_f (x) e_f; 0 = passive. */
typedef struct {
    int32_t law;
    double a, b, af, bf, as_, bs, afs, bfs, kappa;
    double Ta;
} ib_material;

/* Static mesh description; all pointers are HOST pointers, copied by ib_create. */
typedef struct {
    int64_t n_nodes, n_elems;
    const int32_t *conn;      /* [n_elems][8]                                            */
    const double *X_ref;      /* [3][n_nodes] reference coordinates                      */
    const double *fibers;     /* [6][n_elems] or NULL (then e_f = e_x, e_s = e_y)        */
    const int32_t *mat_id;    /* [n_elems] or NULL (all 0)                               */
    const int32_t *nsub;      /* [n_elems][3] or NULL = nodal rule of L241 (points=nodes)*/
    const ib_material *mats;  /* [n_mats]                                                */
    int32_t n_mats;
    int32_t elem_type;        /* IB_ELEM_HEX8 (0): conn [n_elems][8]; IB_ELEM_TET4 (1), NEXT-3: P1
                                 tetrahedra, conn [n_elems][4] with det [X1-X0,X2-X0,X3-X0] > 0, one
                                 quadrature point, nodal coupling only (nsub must be NULL, L241);
                                 IB_ELEM_TET10 (2): P2 tetrahedra (L265), conn [n_elems][10] = 4 vertices then the
                                 mid-edge nodes of edges 01,12,02,03,13,23; 4-point degree-2 rule (reading A25);
                                 nodal coupling only */
} ib_mesh_desc;
enum { IB_ELEM_HEX8 = 0, IB_ELEM_TET4 = 1, IB_ELEM_TET10 = 2 };

/* Create a context: validates, copies the mesh, builds the node->element adjacency (hexahedra: at most 8
 * incident elements per node, else IB_ERR_UNSUPPORTED; tetrahedra: any valence), and precomputes on the
 * device the reference geometry of the Gauss points, the sub-point weights W_s = det J0(xi_s) 8/(n1 n2 n3)
 * and the lumped nodal weights w_a = sum W_s N_a(xi_s) (L235, L241). An inverted reference element
 * (det J0 <= 0) makes ib_create return IB_ERR_INVERTED_ELEMENT.
 * `device` is the CUDA device ordinal. Synchronous. */
ib_status ib_create(ib_ctx **ctx, const ib_grid_desc *grid, const ib_mesh_desc *mesh, int32_t device);
ib_status ib_destroy(ib_ctx *ctx);

/* Number of Lagrangian force points P (= n_nodes in nodal mode), nodes, elements. */
int64_t ib_num_points(const ib_ctx *ctx);
int64_t ib_num_nodes(const ib_ctx *ctx);
int64_t ib_num_elems(const ib_ctx *ctx);

/* (1) FE nodal force  B_a = - sum_q P(F(X_q)) grad_X phi_a(X_q) w_q   (Eq.(20)).
 * x [3][n_nodes] current positions (in); B [3][n_nodes] (out, overwritten). Deterministic:
 * element contributions are gathered per node in fixed order, no atomics. */
ib_status ib_fe_force(ib_ctx *ctx, const double *x, double *B, void *stream);

/* Lagrangian force points of the sub-point rule at the current configuration:
 * xp [3][P] = sum_a N_a(xi_s) x_a ; Gp [3][P] = W_s sum_a N_a(xi_s) B_a / w_a (either may be NULL;
 * B may be NULL iff Gp is NULL). In nodal mode xp = x, Gp = B. */
ib_status ib_points(ib_ctx *ctx, const double *x, const double *B, double *xp, double *Gp, void *stream);

/* Lumped L2 projection (L233-237) of point values to nodes: Un_a = (1/w_a) sum_s W_s N_a(xi_s) Up_s.
 * Deterministic (per-node gather). In nodal mode Un = Up. */
ib_status ib_restrict(ib_ctx *ctx, const double *Up, double *Un, void *stream);

/* Bin points by Eulerian cell and sort (stable): c_d = floor((xp_d - x0_d) * (1.0/h)) mod n_d,
 * key = ((tz*nty+ty)*ntx+tx)*512 + ((lz*8+ly)*8+lx) with t = c div 8, l = c mod 8;
 * perm_out[r] = id of the point of rank r (ties keep ascending id); key_out[p] = key of point p.
 * Bit-exact against the definition. key_out or perm_out may be NULL. P <= 2^31-1. */
ib_status ib_bin_sort(ib_ctx *ctx, const double *xp, int64_t P, int64_t *key_out, int32_t *perm_out,
                      void *stream);

/* The same bin sort (same definition, same kernels, bit-identical key_out / perm_out) for callers that must
 * not allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  It takes
 * no context and calls no cudaMalloc / cudaFree or allocating library routine: its scratch (two key and two
 * id buffers, the digit histograms of the radix sort, the status word) lives in ONE file-scope
 * `static __device__` array of the library, 4,260,352 bytes, which every GPU that loads the library holds
 * until the process exits.  Hence the limit: P <= IB_BIN_SORT_STATIC_MAX_POINTS, beyond it the call returns
 * IB_ERR_TOO_LARGE and does nothing.
 *   grid   HOST pointer; validated like ib_create's (dimensions multiples of 8, h > 0, ...): IB_ERR_INVALID_ARG.
 *   xp     DEVICE [3][P] (may be NULL iff P == 0); key_out DEVICE [P] or NULL; perm_out DEVICE [P] or NULL.
 *   stream the cudaStream_t to enqueue on (NULL: the default stream); it must belong to the CURRENT device,
 *          whose copy of the scratch array is used.
 *   check  0: asynchronous, like ib_bin_sort.  A non-finite coordinate is binned at the grid origin (as by
 *          ib_bin_sort) and only latched in the scratch array.  != 0: the call also synchronises the stream and
 *          returns IB_ERR_NONFINITE if a coordinate was NaN/Inf (key_out / perm_out are still written).
 * All calls on one device share the array, which keeps the last call's contents (the call clears the status
 * word; every other word it reads it has written first).  Two calls that overlap on the GPU -- different
 * streams, or two host threads -- RACE on it: serialise them (one stream, or events).  Calls on different
 * devices are independent. */
#define IB_BIN_SORT_STATIC_MAX_POINTS 262144
ib_status ib_bin_sort_static(const ib_grid_desc *grid, const double *xp, int64_t P, int64_t *key_out,
                             int32_t *perm_out, int32_t check, void *stream);

/* (2) Spread, Eq.(24)-(26): f_c[face] (+)= sum_s Gp_{s,c} delta_h(x_face - xp_s), delta_h =
 * h^-3 phi phi phi on component c's own staggered lattice. accumulate == 0 zero-fills fu,fv,fw
 * first. Generic over arbitrary point clouds. Sums are reordered (atomics): not bit-reproducible. */
ib_status ib_spread(ib_ctx *ctx, const double *xp, const double *Gp, int64_t P,
                    double *fu, double *fv, double *fw, int32_t accumulate, void *stream);

/* (3) Interpolate, Eq.(27)-(29): Up_{s,c} = sum_faces u_c[face] delta_h(x_face - xp_s) h^3. */
ib_status ib_interp(ib_ctx *ctx, const double *xp, int64_t P, const double *u, const double *v,
                    const double *w, double *Up, void *stream);

/* The whole coupling step at one position array x (BASELINE.json "one coupling step"):
 *   B = fe_force(x); points; f = spread(xp, Gp) (overwrites fu,fv,fw); Up = interp(xp,u,v,w);
 *   Un = restrict(Up).   B may be NULL (not returned).  In nodal mode (nsub == NULL, the paper's rule
 *   L241-257) the points are the nodes: f = spread(x, B), Un = interp(x, u,v,w).  Work that needs only x
 *   runs on context-owned side streams beside the FE force; everything is ordered after earlier work on
 *   `stream` and complete, in stream order, when the call's last kernel on `stream` is. */
ib_status ib_coupling_step(ib_ctx *ctx, const double *x, const double *u, const double *v,
                           const double *w, double *fu, double *fv, double *fw, double *Un,
                           double *B, void *stream);

/* NEXT-1: one time step of the paper's explicit coupling, Eq.(16), with a
 * frozen velocity field -- the same operators in the paper's order:
 *   U^IB = I(X^n, u^n)                      interpolate at the CURRENT positions (L173), project to the
 *                                           nodes (L233-237)                       -> Un [3][n_nodes]
 *   x_new = x + dt * Un                     move the structure (L173)             -> x_new [3][n_nodes]
 *   B = fe_force(x_new)                     F^{n+1} from P^{n+1} (L169, L191)     -> B (may be NULL)
 *   f = E(X^n, F^{n+1})                     spread with deltas centred at the OLD positions x (L171, L193)
 * fu,fv,fw are overwritten. x_new must not alias x. */
ib_status ib_step_eq16(ib_ctx *ctx, const double *x, const double *u, const double *v, const double *w,
                       double dt, double *x_new, double *fu, double *fv, double *fw, double *Un, double *B,
                       void *stream);

/* Same step with HOST buffers: copies x,u,v,w host->device, runs the step, copies fu,fv,fw,Un
 * (and B if non-NULL) device->host, then synchronises. Buffers should be pinned for full PCIe rate.
 * In the default variant the step is pipelined in z-slabs of the grid (up to 8): the force side, which
 * needs only x, runs while u,v,w cross the bus slab by slab; the fused spread + interpolate kernel of a
 * slab starts when the velocity layers of that slab and its neighbours have arrived; the layers of
 * fu,fv,fw that a finished slab can no longer touch travel back while the next slabs run (layers out of
 * the structure's reach -- found from the z-range of x_host -- go back as soon as they are zero-filled). The host
 * arrays are therefore written in pieces: none of them is valid before the call returns. */
ib_status ib_coupling_step_host(ib_ctx *ctx, const double *x_host, const double *u_host,
                                const double *v_host, const double *w_host, double *fu_host,
                                double *fv_host, double *fw_host, double *Un_host, double *B_host,
                                void *stream);

/* The same with the three velocity components, and the three force components, each in ONE host array
 * [3][n_cells] (u then v then w; fu then fv then fw): every slab then crosses the bus as one copy per direction
 * instead of three (three small copies in flight in both directions measured 40 GB/s where one gets 55).
 * (Three separate arrays that happen to be adjacent do not qualify: one copy cannot span allocations.) */
ib_status ib_coupling_step_host3(ib_ctx *ctx, const double *x_host, const double *uvw_host, double *f_host,
                                 double *Un_host, double *B_host, void *stream);

/* Synchronise the last used stream and report the latched device status. first_bad_index (may be
 * NULL) receives the smallest offending element or node id, or -1. Clears the latch. */
ib_status ib_check(ib_ctx *ctx, int64_t *first_bad_index);

/* Number of kernel launches enqueued by this context since creation (for bench accounting). */
int64_t ib_launch_count(const ib_ctx *ctx);

/* Select the kernel variant used by spread/interp/coupling_step: 0 = reference path (one thread
 * per point, global atomics), 1 = tiled path (points sorted by cell, shared-memory halo tile).
 * Default 1. Returns IB_ERR_INVALID_ARG for other values. */
ib_status ib_set_variant(ib_ctx *ctx, int32_t variant);

/* NEXT-4: solid boundary loads (Table 3 row "Solid boundary" L398). Once set they are ADDED to
 * the nodal force by ib_fe_force and by every step (before the force is spread); B is then no longer
 * bit-reproducible (the surface loads are accumulated with atomics).
 *  tethers  (L263 "fixed left face ... penalty parameter kappa = 10^6", L425): reading A24, a penalty spring
 *           to the reference position, B_a += kappa (X_a - x_a) for the listed nodes (host ids, distinct).
 *  surface  boundary faces, host array [n_faces][nodes_per_face], 4 = bilinear quads in cyclic order,
 *           3 = linear triangles, 6 = quadratic triangles (3 vertices, then the middles of the edges
 *           v0v1, v1v2, v2v0; reading A27: symmetric 6-point rule of degree 4, exact for the pressure term),
 *           normal pointing out of the solid.
 *  loads    qt0 = q(t) t0 (host, 3 doubles or NULL): dead traction per unit REFERENCE area (L263),
 *           B_a += q t0 int N_a dA;   p: follower pressure on the CURRENT faces (L303, L315),
 *           B_a -= p int N_a n da.  Call again every step with the current q(t), p_endo(t).
 * n = 0 / n_faces = 0 removes the load. */
ib_status ib_set_tethers(ib_ctx *ctx, int64_t n, const int32_t *node_ids, double kappa);
ib_status ib_set_surface(ib_ctx *ctx, int64_t n_faces, int32_t nodes_per_face, const int32_t *faces);
ib_status ib_set_loads(ib_ctx *ctx, const double *qt0, double p);

/* CUDA graph replay of ib_coupling_step (default on): when the call comes in a second time with the same
 * pointers on the same non-default stream, the step's ~16 launches on three streams are captured once
 * and replayed with one cudaGraphLaunch afterwards (the small configs are launch-latency bound). The
 * legacy default stream cannot be captured: there the step is always enqueued kernel by kernel. */
ib_status ib_set_graph(ib_ctx *ctx, int32_t on);

/* Per-phase device timing with CUDA events recorded on the launching stream (used by bench.py for
 * the roofline of the dominant kernel). Phases of ib_coupling_step / ib_spread / ib_interp: */
enum { IB_PHASE_FE_FORCE = 0, IB_PHASE_POINTS = 1, IB_PHASE_SORT = 2, IB_PHASE_SPREAD_INTERP = 3,
       IB_PHASE_RESTRICT = 4, IB_PHASE_ZERO = 5, IB_PHASE_COUNT = 6 };
ib_status ib_profile_enable(ib_ctx *ctx, int32_t on);
/* Synchronises the recorded events, adds up milliseconds and call counts per phase since the last
 * read into ms_sum[IB_PHASE_COUNT] / calls[IB_PHASE_COUNT], and resets the accumulators. */
ib_status ib_profile_read(ib_ctx *ctx, double *ms_sum, int64_t *calls);

/* FP64 FMA peak probe: runs a register-only DFMA loop on `device`; returns achieved DFMA/s in
 * *dfma_per_s and the kernel time in *ms. Used by bench.py for the "alu" roofline denominator. */
ib_status ib_probe_dfma(int32_t device, double *dfma_per_s, double *ms);

const char *ib_status_string(ib_status s);

#ifdef __cplusplus
}
#endif
#endif /* IBCOUPLE_H */
