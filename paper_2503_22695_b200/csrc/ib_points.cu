// ib_points.cu -- Lagrangian force points of the sub-point rule, prolongation and restriction
// (reading A13 of PAPER.md L233-237, L241):
//   W_s  = det J0(xi_s) 8/(n1 n2 n3)                       (precomputed, reference is static)
//   w_a  = sum_{e contains a} sum_s W_s N_a(xi_s)          (precomputed, lumped mass)
//   x_s  = sum_a N_a(xi_s) x_a ;  G_s = W_s sum_a N_a(xi_s) Fhat_a,  Fhat_a = B_a / w_a
//   Un_a = (1/w_a) sum_{e,s} W_s N_a(xi_s) Up_s            (lumped L2 projection)
// Node sums use the same deterministic ELL gather as the FE force (no atomics).
#include "ib_common.cuh"

__device__ __forceinline__ int64_t ib_find_elem(const int64_t *__restrict__ off, int64_t n_elems, int64_t p)
{
    int64_t lo = 0, hi = n_elems;                 // off[lo] <= p < off[hi]
    while (hi - lo > 1) {
        int64_t mid = (lo + hi) >> 1;
        if (__ldg(off + mid) <= p) lo = mid; else hi = mid;
    }
    return lo;
}

struct ib_sub {
    int64_t e;
    int s, n1, n2, n3;
};

__device__ __forceinline__ ib_sub ib_locate(int64_t p, int64_t n_elems, int uniform_S,
                                            const int32_t *__restrict__ nsub,
                                            const int64_t *__restrict__ off)
{
    ib_sub r;
    if (uniform_S > 0) {
        r.e = p / uniform_S;
        r.s = (int)(p - r.e * uniform_S);
        r.n1 = __ldg(nsub); r.n2 = __ldg(nsub + 1); r.n3 = __ldg(nsub + 2);
    } else {
        r.e = ib_find_elem(off, n_elems, p);
        r.s = (int)(p - __ldg(off + r.e));
        r.n1 = __ldg(nsub + 3 * r.e); r.n2 = __ldg(nsub + 3 * r.e + 1); r.n3 = __ldg(nsub + 3 * r.e + 2);
    }
    return r;
}

__device__ __forceinline__ void ib_sub_shape(const ib_sub &r, double N[8])
{
    int m1 = r.s % r.n1, m2 = (r.s / r.n1) % r.n2, m3 = r.s / (r.n1 * r.n2);
    ib_shape(ib_subxi(m1, r.n1), ib_subxi(m2, r.n2), ib_subxi(m3, r.n3), N);
}

// W_s for every sub-point (create time)
__global__ void __launch_bounds__(256)
ibk_subpoint_weights(int64_t P, int64_t n_elems, int64_t n_nodes, int uniform_S,
                     const int32_t *__restrict__ nsub, const int64_t *__restrict__ off,
                     const int32_t *__restrict__ conn, const double *__restrict__ X,
                     double *__restrict__ Wp, long long *status)
{
    int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= P) return;
    ib_sub r = ib_locate(p, n_elems, uniform_S, nsub, off);
    int m1 = r.s % r.n1, m2 = (r.s / r.n1) % r.n2, m3 = r.s / (r.n1 * r.n2);
    double dN[8][3];
    ib_dshape(ib_subxi(m1, r.n1), ib_subxi(m2, r.n2), ib_subxi(m3, r.n3), dN);
    double J0[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
#pragma unroll
    for (int a = 0; a < 8; ++a) {
        int n = __ldg(conn + r.e * 8 + a);
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            double Xa = __ldg(X + c * n_nodes + n);
#pragma unroll
            for (int d = 0; d < 3; ++d) J0[c][d] = fma(Xa, dN[a][d], J0[c][d]);
        }
    }
    double dj = ib_det3(J0);
    if (!(dj > 0.0)) ib_latch(status, IB_ERR_INVERTED_ELEMENT, r.e);
    Wp[p] = dj * 8.0 / (double)(r.n1 * r.n2 * r.n3);
}

// per element, per local node a: sum_s W_s N_a(xi_s) [* Up_s,c]   (8 lanes per element, lane = node)
template <int WITH_U>
__global__ void __launch_bounds__(256)
ibk_elem_node_sums(int64_t n_elems, int64_t P, const int32_t *__restrict__ nsub,
                   const int64_t *__restrict__ off, const double *__restrict__ Wp,
                   const double *__restrict__ Up, double *__restrict__ Ce)
{
    int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    int64_t e = t >> 3;
    int a = (int)(t & 7);
    if (e >= n_elems) return;
    int n1 = __ldg(nsub + 3 * e), n2 = __ldg(nsub + 3 * e + 1), n3 = __ldg(nsub + 3 * e + 2);
    int64_t p0 = __ldg(off + e);
    double s1 = (a & 1) ? 1.0 : -1.0, s2 = (a & 2) ? 1.0 : -1.0, s3 = (a & 4) ? 1.0 : -1.0;
    double acc0 = 0.0, acc1 = 0.0, acc2 = 0.0;
    int s = 0;
    // N_a along one direction at xi = -1 + (2m+1)/n:  1/2 (1 + s xi) = 1/2 (1 - s) + s (2m+1)/(2n) = base + m step
    // (no division inside the loops)
    const double r1 = 1.0 / (double)n1, r2 = 1.0 / (double)n2, r3 = 1.0 / (double)n3;
    const double b1 = fma(0.5 * s1, r1, 0.5 - 0.5 * s1), b2 = fma(0.5 * s2, r2, 0.5 - 0.5 * s2), b3 = fma(0.5 * s3, r3, 0.5 - 0.5 * s3);
    const double t1 = s1 * r1, t2 = s2 * r2, t3 = s3 * r3;
    for (int m3 = 0; m3 < n3; ++m3) {
        const double f3 = fma((double)m3, t3, b3);
        for (int m2 = 0; m2 < n2; ++m2) {
            const double f23 = f3 * fma((double)m2, t2, b2);
#pragma unroll 4
            for (int m1 = 0; m1 < n1; ++m1, ++s) {
                const double Na = f23 * fma((double)m1, t1, b1);
                const double wn = __ldg(Wp + p0 + s) * Na;
                if (WITH_U) {
                    acc0 = fma(wn, __ldg(Up + p0 + s), acc0);
                    acc1 = fma(wn, __ldg(Up + P + p0 + s), acc1);
                    acc2 = fma(wn, __ldg(Up + 2 * P + p0 + s), acc2);
                } else {
                    acc0 += wn;
                }
            }
        }
    }
    int64_t ne8 = n_elems * 8;
    Ce[e * 8 + a] = acc0;
    if (WITH_U) { Ce[ne8 + e * 8 + a] = acc1; Ce[2 * ne8 + e * 8 + a] = acc2; }
}


// Fast path of the restriction for a uniform nsub whose rows-per-element n2*n3 is a power of two <= 32:
// one thread per row (e, m2, m3) of n1 sub-points (coalesced reads of W_s and Up), sum-factorised
// over m1 in the thread, then a butterfly over the rows of the element.
template <int N1>
__global__ void __launch_bounds__(256)
ibk_restrict_rows(int64_t n_rows, int64_t P, int n1r, int n2, int n3, const double *__restrict__ Wp,
                  const double *__restrict__ Up, double *__restrict__ Ce, int64_t ne8)
{
    const int rpe = n2 * n3;
    int64_t row = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const bool live = row < n_rows;
    if (!live) row = n_rows - 1;
    const int64_t e = row / rpe;
    const int r = (int)(row - e * rpe);
    const int m2 = r % n2, m3 = r / n2;
    const int n1 = N1 > 0 ? N1 : n1r;
    const int64_t p0 = row * n1;
    double A0[3] = {0, 0, 0}, A1[3] = {0, 0, 0};
#pragma unroll
    for (int j = 0; j < (N1 > 0 ? N1 : 8); ++j) {
        if (N1 == 0 && j >= n1) break;
        double t = 0.5 * (1.0 + ib_subxi(j, n1));
        double W = __ldcs(Wp + p0 + j);
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            double wu = W * __ldcs(Up + (int64_t)c * P + p0 + j);
            A1[c] = fma(wu, t, A1[c]);
            A0[c] = fma(wu, 1.0 - t, A0[c]);
        }
    }
    const double x2 = ib_subxi(m2, n2), x3 = ib_subxi(m3, n3);
    const double b[2] = {0.5 * (1.0 - x2), 0.5 * (1.0 + x2)}, g[2] = {0.5 * (1.0 - x3), 0.5 * (1.0 + x3)};
    if (N1 == 4 && n2 == 4 && n3 == 4) {
        // 4 x 4 rows per element = 16 adjacent lanes, r = m2 + 4 m3.  Transposing reduction: at each
        // step a lane keeps the half of its values whose target index bit equals its own lane bit and
        // sends the other half (15 double shuffles instead of 96).
        const bool r0 = r & 1, r1 = r & 2, r2 = r & 4;
        const unsigned full = 0xffffffffu;
        const double lv = live ? 1.0 : 0.0;
        double s1[2][3];                               // [ia][c], target ja = r0
#pragma unroll
        for (int ia = 0; ia < 2; ++ia)
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const double Ai = lv * (ia ? A1[c] : A0[c]);
                const double keep = (r0 ? b[1] : b[0]) * Ai, send = (r0 ? b[0] : b[1]) * Ai;
                s1[ia][c] = keep + __shfl_xor_sync(full, send, 1);
            }
        double s2[3];                                  // [c], target ia = r1
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const double keep = r1 ? s1[1][c] : s1[0][c], send = r1 ? s1[0][c] : s1[1][c];
            s2[c] = keep + __shfl_xor_sync(full, send, 2);
        }
        double s3[3];                                  // [c], target ka = r2
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const double keep = (r2 ? g[1] : g[0]) * s2[c], send = (r2 ? g[0] : g[1]) * s2[c];
            s3[c] = keep + __shfl_xor_sync(full, send, 4);
        }
#pragma unroll
        for (int c = 0; c < 3; ++c) s3[c] += __shfl_xor_sync(full, s3[c], 8);
        if (live && !(r & 8)) {
            const int a = (r1 ? 1 : 0) + (r0 ? 2 : 0) + (r2 ? 4 : 0);
#pragma unroll
            for (int c = 0; c < 3; ++c) Ce[c * ne8 + e * 8 + a] = s3[c];
        }
        return;
    }
    double v[8][3];
#pragma unroll
    for (int a = 0; a < 8; ++a) {
        double w = b[(a >> 1) & 1] * g[a >> 2];
        if (!live) w = 0.0;
#pragma unroll
        for (int c = 0; c < 3; ++c) v[a][c] = w * ((a & 1) ? A1[c] : A0[c]);
    }
    for (int o = 1; o < rpe; o <<= 1) {
#pragma unroll
        for (int a = 0; a < 8; ++a)
#pragma unroll
            for (int c = 0; c < 3; ++c) v[a][c] += __shfl_xor_sync(0xffffffffu, v[a][c], o);
    }
    if (live) {
#pragma unroll
        for (int a = 0; a < 8; ++a)
#pragma unroll
            for (int c = 0; c < 3; ++c)
                if ((a * 3 + c) % rpe == r) Ce[c * ne8 + e * 8 + a] = v[a][c];
    }
}

// The restriction for a uniform nsub whose rows-per-element n2*n3 is NOT a power of two (3^3, 5^3, 6^3 ...): a
// butterfly over the rows of an element does not close, so the rows meet in shared memory.  A CTA takes
// 256 / (n2 n3) whole elements; phase 1: one thread per row (e, m2, m3), coalesced reads of W_s and Up, the sum over
// m1 against the two x-shape functions (6 values per row); phase 2: 6 threads per element -- (x-side of the node, component)
// -- add the rows up in fixed order with the y and z shape functions, four nodes each.  Same sums as ibk_elem_node_sums in another
// order, one pass over the points instead of eight.
__global__ void __launch_bounds__(256)
ibk_restrict_rows_smem(int64_t n_elems, int64_t P, int n1, int n2, int n3, const double *__restrict__ Wp,
                       const double *__restrict__ Up, double *__restrict__ Ce, int64_t ne8)
{
    __shared__ double sA[256 * 7];                     // [row of the CTA][A0[3], A1[3], pad]
    const int rpe = n2 * n3, epc = 256 / rpe;
    const int tid = threadIdx.x;
    const int64_t e0 = (int64_t)blockIdx.x * epc;
    if (tid < epc * rpe) {
        const int64_t e = e0 + tid / rpe;
        double A0[3] = {0, 0, 0}, A1[3] = {0, 0, 0};
        if (e < n_elems) {
            const int64_t p0 = (e0 * rpe + tid) * (int64_t)n1;
            const double rn = 1.0 / (double)n1;
            for (int j = 0; j < n1; ++j) {
                const double t = ((double)j + 0.5) * rn;           // 1/2 (1 + xi_j)
                const double W = __ldg(Wp + p0 + j);
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    const double wu = W * __ldg(Up + (int64_t)c * P + p0 + j);
                    A1[c] = fma(wu, t, A1[c]);
                    A0[c] = fma(wu, 1.0 - t, A0[c]);
                }
            }
        }
#pragma unroll
        for (int c = 0; c < 3; ++c) { sA[tid * 7 + c] = A0[c]; sA[tid * 7 + 3 + c] = A1[c]; }
    }
    __syncthreads();
    // phase 2: thread = (element, x-side ia, component); it walks the element's rows once and forms the four
    // (ja, ka) sums of its column of nodes together
    if (tid < epc * 6) {
        const int el = tid / 6, k = tid - el * 6, ia = k / 3, c = k - ia * 3;
        const int64_t e = e0 + el;
        if (e >= n_elems) return;
        const double r2 = 1.0 / (double)n2, r3 = 1.0 / (double)n3;
        const double *row = sA + (el * rpe) * 7 + ia * 3 + c;
        double acc[2][2] = {{0.0, 0.0}, {0.0, 0.0}};      // [ka][ja]
        double t3 = 0.5 * r3;
        for (int m3 = 0; m3 < n3; ++m3, t3 += r3) {
            double p0 = 0.0, p1 = 0.0, t2 = 0.5 * r2;
            for (int m2 = 0; m2 < n2; ++m2, t2 += r2) {
                const double v = row[(m3 * n2 + m2) * 7];
                p1 = fma(t2, v, p1);
                p0 = fma(1.0 - t2, v, p0);
            }
            acc[0][0] = fma(1.0 - t3, p0, acc[0][0]); acc[0][1] = fma(1.0 - t3, p1, acc[0][1]);
            acc[1][0] = fma(t3, p0, acc[1][0]); acc[1][1] = fma(t3, p1, acc[1][1]);
        }
        double *out = Ce + c * ne8 + e * 8 + ia;
#pragma unroll
        for (int ka = 0; ka < 2; ++ka)
#pragma unroll
            for (int ja = 0; ja < 2; ++ja) out[2 * ja + 4 * ka] = acc[ka][ja];
    }
}

// per node gather of Ce; mode 0: w_a = sum ; mode 1: Un_c = sum_c / w_a
template <int WITH_U>
__global__ void __launch_bounds__(256)
ibk_node_gather_w(int64_t n_nodes, int64_t ne8, const int32_t *__restrict__ adj,
                  const double *__restrict__ Ce, double *__restrict__ wa, double *__restrict__ Un)
{
    int64_t n = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= n_nodes) return;
    double s0 = 0.0, s1 = 0.0, s2 = 0.0;
#pragma unroll
    for (int j = 0; j < 8; ++j) {
        int slot = __ldg(adj + j * n_nodes + n);
        if (slot >= 0) {
            s0 += __ldg(Ce + slot);
            if (WITH_U) { s1 += __ldg(Ce + ne8 + slot); s2 += __ldg(Ce + 2 * ne8 + slot); }
        }
    }
    if (WITH_U) {
        double r = 1.0 / __ldg(wa + n);
        Un[n] = s0 * r; Un[n_nodes + n] = s1 * r; Un[2 * n_nodes + n] = s2 * r;
    } else {
        wa[n] = s0;
    }
}

// x_s and G_s for every sub-point
__global__ void __launch_bounds__(256)
ibk_points_kernel(int64_t P, int64_t n_elems, int64_t n_nodes, int uniform_S,
                  const int32_t *__restrict__ nsub, const int64_t *__restrict__ off,
                  const int32_t *__restrict__ conn, const double *__restrict__ x,
                  const double *__restrict__ Fhat, const double *__restrict__ Wp,
                  double *__restrict__ xp, double *__restrict__ Gp)
{
    int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= P) return;
    ib_sub r = ib_locate(p, n_elems, uniform_S, nsub, off);
    double N[8];
    ib_sub_shape(r, N);
    int nd[8];
    {
        const int4 *cp = reinterpret_cast<const int4 *>(conn + r.e * 8);
        int4 c0 = __ldg(cp), c1 = __ldg(cp + 1);
        nd[0] = c0.x; nd[1] = c0.y; nd[2] = c0.z; nd[3] = c0.w;
        nd[4] = c1.x; nd[5] = c1.y; nd[6] = c1.z; nd[7] = c1.w;
    }
    if (xp) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            double v = 0.0;
#pragma unroll
            for (int a = 0; a < 8; ++a) v = fma(N[a], __ldg(x + c * n_nodes + nd[a]), v);
            xp[c * P + p] = v;
        }
    }
    if (Gp) {
        double W = __ldg(Wp + p);
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            double v = 0.0;
#pragma unroll
            for (int a = 0; a < 8; ++a) v = fma(N[a], __ldg(Fhat + c * n_nodes + nd[a]), v);
            Gp[c * P + p] = W * v;
        }
    }
}

ib_status ibk_precompute_weights(ib_ctx *c, cudaStream_t st)
{
    if (c->nodal || c->n_points == 0) return IB_OK;
    ibk_subpoint_weights<<<ib_blocks(c->n_points, 256), 256, 0, st>>>(
        c->n_points, c->n_elems, c->n_nodes, c->uniform_S, c->d_nsub, c->d_pt_off, c->d_conn, c->d_X,
        c->d_Wp, c->d_status);
    ibk_elem_node_sums<0><<<ib_blocks(c->n_elems * 8, 256), 256, 0, st>>>(
        c->n_elems, c->n_points, c->d_nsub, c->d_pt_off, c->d_Wp, nullptr, c->d_Ce);
    ibk_node_gather_w<0><<<ib_blocks(c->n_nodes, 256), 256, 0, st>>>(c->n_nodes, c->n_elems * 8, c->d_adj,
                                                                      c->d_Ce, c->d_wa, nullptr);
    c->launches += 3;
    IB_CUDA_TRY(cudaGetLastError());
    return IB_OK;
}

ib_status ibk_points(ib_ctx *c, const double *x, const double *Fhat, double *xp, double *Gp, cudaStream_t st)
{
    if (c->n_points == 0) return IB_OK;
    ibk_points_kernel<<<ib_blocks(c->n_points, 256), 256, 0, st>>>(
        c->n_points, c->n_elems, c->n_nodes, c->uniform_S, c->d_nsub, c->d_pt_off, c->d_conn, x, Fhat,
        c->d_Wp, xp, Gp);
    c->launches++;
    IB_CUDA_TRY(cudaGetLastError());
    return IB_OK;
}

ib_status ibk_restrict(ib_ctx *c, const double *Up, double *Un, cudaStream_t st)
{
    if (c->n_elems == 0 || c->n_nodes == 0) return IB_OK;
    const int rpe = c->un[1] * c->un[2];
    if (c->un[0] > 0 && rpe <= 32 && (rpe & (rpe - 1)) == 0)
    {
        if (c->un[0] == 4)
            ibk_restrict_rows<4><<<ib_blocks(c->n_rows, 256), 256, 0, st>>>(c->n_rows, c->n_points, 4, c->un[1], c->un[2],
                                                                          c->d_Wp, Up, c->d_Ce, c->n_elems * 8);
        else
            ibk_restrict_rows<0><<<ib_blocks(c->n_rows, 256), 256, 0, st>>>(c->n_rows, c->n_points, c->un[0], c->un[1],
                                                                          c->un[2], c->d_Wp, Up, c->d_Ce, c->n_elems * 8);
    }
    else if (c->un[0] > 0 && rpe <= 256)
    {
        const int epc = 256 / rpe;
        ibk_restrict_rows_smem<<<ib_blocks(c->n_elems, epc), 256, 0, st>>>(c->n_elems, c->n_points, c->un[0], c->un[1], c->un[2],
                                                                          c->d_Wp, Up, c->d_Ce, c->n_elems * 8);
    }
    else
        ibk_elem_node_sums<1><<<ib_blocks(c->n_elems * 8, 256), 256, 0, st>>>(
            c->n_elems, c->n_points, c->d_nsub, c->d_pt_off, c->d_Wp, Up, c->d_Ce);
    ibk_node_gather_w<1><<<ib_blocks(c->n_nodes, 256), 256, 0, st>>>(c->n_nodes, c->n_elems * 8, c->d_adj,
                                                                      c->d_Ce, c->d_wa, Un);
    c->launches += 2;
    IB_CUDA_TRY(cudaGetLastError());
    return IB_OK;
}
