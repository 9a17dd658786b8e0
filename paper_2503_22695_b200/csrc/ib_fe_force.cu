// ib_fe_force.cu -- matrix-free hyperelastic FE nodal force.
//   B_a = - sum_q P(F(X_q)) grad_X phi_a(X_q) w_q          PAPER.md Eq.(20)
//   F = d chi / d X, J = det F                              L28-32
//   P = d Psi / d F for neo-Hookean (L441-445) and Holzapfel-Ogden (Eq.(12)-(15) L147-155)
// "eliminating sparse matrix storage and operations entirely" (L13): one thread per Gauss point,
// the 8 Gauss points of an element sit in 8 adjacent lanes and exchange their 8x3 nodal
// contributions with a transposing shuffle reduction; a second kernel gathers, per node, the
// <= 8 element contributions through an ELL adjacency in fixed order (deterministic, no atomics,
// no CSR, no assembled operator).
#include "ib_common.cuh"

// first Piola-Kirchhoff stress (HO, NH; NEXT-2: Eq.(7), Eq.(10)-(11), active stress). Readings A2 (F^-T in the isotropic term), A3 (symmetric I8 term),
// A6 (NH: a = mu, b = 0), A9 (I4* = max(I4,1)). Returns J.
__device__ __forceinline__ double ib_pk1(const ib_material &m, const double F[3][3], const double ef[3],
                                         const double es[3], double P[3][3])
{
    // cofactor matrix: cof[c][K] = J * F^-T[c][K]
    double cof[3][3];
    cof[0][0] = F[1][1] * F[2][2] - F[1][2] * F[2][1];
    cof[0][1] = F[1][2] * F[2][0] - F[1][0] * F[2][2];
    cof[0][2] = F[1][0] * F[2][1] - F[1][1] * F[2][0];
    cof[1][0] = F[0][2] * F[2][1] - F[0][1] * F[2][2];
    cof[1][1] = F[0][0] * F[2][2] - F[0][2] * F[2][0];
    cof[1][2] = F[0][1] * F[2][0] - F[0][0] * F[2][1];
    cof[2][0] = F[0][1] * F[1][2] - F[0][2] * F[1][1];
    cof[2][1] = F[0][2] * F[1][0] - F[0][0] * F[1][2];
    cof[2][2] = F[0][0] * F[1][1] - F[0][1] * F[1][0];
    double J = F[0][0] * cof[0][0] + F[0][1] * cof[0][1] + F[0][2] * cof[0][2];
    if (!(J > 0.0)) return J;
    double rJ = 1.0 / J;
    double I1 = 0.0;
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int K = 0; K < 3; ++K) I1 = fma(F[c][K], F[c][K], I1);
    double cb = cbrt(J);
    double Jm23 = 1.0 / (cb * cb);
    double lnJ = log(J);
    double e_iso = (m.b != 0.0) ? exp(m.b * (Jm23 * I1 - 3.0)) : 1.0;
    double ciso = m.a * e_iso * Jm23;
    // P = ciso (F - I1/3 F^-T) + kappa lnJ F^-T = ciso F + (kappa lnJ - ciso I1/3)/J cof
    double cvol = (m.kappa * lnJ - ciso * I1 * (1.0 / 3.0)) * rJ;
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int K = 0; K < 3; ++K) P[c][K] = fma(ciso, F[c][K], cvol * cof[c][K]);
    if (m.law != IB_LAW_NEOHOOKEAN || m.Ta != 0.0) {
        double Ff[3], Fs[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            Ff[c] = F[c][0] * ef[0] + F[c][1] * ef[1] + F[c][2] * ef[2];
            Fs[c] = F[c][0] * es[0] + F[c][1] * es[1] + F[c][2] * es[2];
        }
        const double I4f = Ff[0] * Ff[0] + Ff[1] * Ff[1] + Ff[2] * Ff[2];
        double cf = 0.0, cs = 0.0, cfs = 0.0;              // coefficients of Ff(x)ef, Fs(x)es, Ff(x)es + Fs(x)ef
        if (m.law == IB_LAW_HO) {
            double I4s = Fs[0] * Fs[0] + Fs[1] * Fs[1] + Fs[2] * Fs[2];
            double I8 = Ff[0] * Fs[0] + Ff[1] * Fs[1] + Ff[2] * Fs[2];
            double df = fmax(I4f, 1.0) - 1.0, ds = fmax(I4s, 1.0) - 1.0;
            cf = (m.af != 0.0 && df > 0.0) ? 2.0 * m.af * df * exp(m.bf * df * df) : 0.0;
            cs = (m.as_ != 0.0 && ds > 0.0) ? 2.0 * m.as_ * ds * exp(m.bs * ds * ds) : 0.0;
            cfs = (m.afs != 0.0) ? m.afs * I8 * exp(m.bfs * I8 * I8) : 0.0;
        } else if (m.law == IB_LAW_FR2) {
            // Eq.(11): fibre term on I4f itself, no tension switch
            double df = I4f - 1.0;
            cf = (m.af != 0.0) ? 2.0 * m.af * df * exp(m.bf * df * df) : 0.0;
        } else if (m.law == IB_LAW_MSR) {
            // Eq.(7): a = G_T, af = G_L, bf = E_L;  (G_T-G_L)(2 Ff(x)ef - Ff(x)C ef - F C ef(x)ef) + k2/2 (I4f-1) Ff(x)ef
            const double gd = m.a - m.af, k2 = m.bf + m.a - 4.0 * m.af;
            double Cf[3], FCf[3];
#pragma unroll
            for (int K = 0; K < 3; ++K) Cf[K] = F[0][K] * Ff[0] + F[1][K] * Ff[1] + F[2][K] * Ff[2];
#pragma unroll
            for (int c = 0; c < 3; ++c) FCf[c] = F[c][0] * Cf[0] + F[c][1] * Cf[1] + F[c][2] * Cf[2];
            cf = 2.0 * gd + 0.5 * k2 * (I4f - 1.0);
#pragma unroll
            for (int c = 0; c < 3; ++c)
#pragma unroll
                for (int K = 0; K < 3; ++K) P[c][K] -= gd * (Ff[c] * Cf[K] + FCf[c] * ef[K]);
        }
        if (m.Ta != 0.0) cf += m.Ta * (1.0 + 4.9 * (sqrt(I4f) - 1.0));          // active stress, L317-331
#pragma unroll
        for (int c = 0; c < 3; ++c)
#pragma unroll
            for (int K = 0; K < 3; ++K)
                P[c][K] += cf * Ff[c] * ef[K] + cs * Fs[c] * es[K] + cfs * (Ff[c] * es[K] + Fs[c] * ef[K]);
    }
    return J;
}

// Reference geometry of every Gauss point (the reference configuration is static):
// geo[0..8][t] = J0^-1 (rows d, cols I), geo[9][t] = det J0 = quadrature weight w (Gauss weight 1, L251).
__global__ void __launch_bounds__(256)
ibk_fe_geometry(int64_t n_elems, int64_t n_nodes, const int32_t *__restrict__ conn,
                const double *__restrict__ X, double *__restrict__ geo, long long *status)
{
    int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    int64_t e = t >> 3;
    int q = (int)(t & 7);
    if (e >= n_elems) return;
    const double g = 0.57735026918962576451;
    double dN[8][3];
    ib_dshape((q & 1) ? g : -g, (q & 2) ? g : -g, (q & 4) ? g : -g, dN);
    double J0[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
#pragma unroll
    for (int a = 0; a < 8; ++a) {
        int nd = __ldg(conn + e * 8 + a);
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            double Xa = __ldg(X + c * n_nodes + nd);
#pragma unroll
            for (int d = 0; d < 3; ++d) J0[c][d] = fma(Xa, dN[a][d], J0[c][d]);
        }
    }
    double w = ib_det3(J0);
    if (!(w > 0.0)) ib_latch(status, IB_ERR_INVERTED_ELEMENT, e);
    double rw = 1.0 / w;
    const int64_t ng = n_elems * 8;
    geo[0 * ng + t] = (J0[1][1] * J0[2][2] - J0[1][2] * J0[2][1]) * rw;
    geo[1 * ng + t] = (J0[0][2] * J0[2][1] - J0[0][1] * J0[2][2]) * rw;
    geo[2 * ng + t] = (J0[0][1] * J0[1][2] - J0[0][2] * J0[1][1]) * rw;
    geo[3 * ng + t] = (J0[1][2] * J0[2][0] - J0[1][0] * J0[2][2]) * rw;
    geo[4 * ng + t] = (J0[0][0] * J0[2][2] - J0[0][2] * J0[2][0]) * rw;
    geo[5 * ng + t] = (J0[0][2] * J0[1][0] - J0[0][0] * J0[1][2]) * rw;
    geo[6 * ng + t] = (J0[1][0] * J0[2][1] - J0[1][1] * J0[2][0]) * rw;
    geo[7 * ng + t] = (J0[0][1] * J0[2][0] - J0[0][0] * J0[2][1]) * rw;
    geo[8 * ng + t] = (J0[0][0] * J0[1][1] - J0[0][1] * J0[1][0]) * rw;
    geo[9 * ng + t] = w;
}

// One thread per Gauss point; lanes 8g..8g+7 of a warp hold the 8 Gauss points of one element.
#define IB_FE_TB 128             // 3 CTAs of 128 threads per SM (168 registers, no spills) measured best: 256 x 2 (128 registers, spilling) +5 %,
                                 // 128 x 4 / 64 x 8 +3 %, 128 x 5 +15 %
__global__ void __launch_bounds__(IB_FE_TB, 3)
ibk_fe_gauss(int64_t n_elems, int64_t n_nodes, const int32_t *__restrict__ conn,
             const double *__restrict__ geo, const double *__restrict__ x,
             const double *__restrict__ fib, const int32_t *__restrict__ mat_id,
             const ib_material *__restrict__ mats, double *__restrict__ Ce, long long *status)
{
    int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    int64_t e = t >> 3;
    int q = (int)(t & 7);
    bool live = e < n_elems;
    int64_t ee = live ? e : n_elems - 1;          // dead lanes recompute the last element (keeps shuffles uniform)
    const int64_t tt = ee * 8 + q, ng = n_elems * 8;
    int nd[8];
    {
        const int4 *cp = reinterpret_cast<const int4 *>(conn + ee * 8);
        int4 c0 = __ldg(cp), c1 = __ldg(cp + 1);
        nd[0] = c0.x; nd[1] = c0.y; nd[2] = c0.z; nd[3] = c0.w;
        nd[4] = c1.x; nd[5] = c1.y; nd[6] = c1.z; nd[7] = c1.w;
    }
    const double g = 0.57735026918962576451;      // 1/sqrt(3): 2x2x2 Gauss rule, weight 1 (L251)
    double dN[8][3];
    ib_dshape((q & 1) ? g : -g, (q & 2) ? g : -g, (q & 4) ? g : -g, dN);

    // F0_{c d} = sum_a x_{a,c} dN_a/dxi_d ;  F = F0 * J0^-1 with the precomputed reference inverse
    double Fx[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
    bool finite = true;
#pragma unroll
    for (int a = 0; a < 8; ++a) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            double xa = __ldg(x + c * n_nodes + nd[a]);
            finite = finite && isfinite(xa);
#pragma unroll
            for (int d = 0; d < 3; ++d) Fx[c][d] = fma(xa, dN[a][d], Fx[c][d]);
        }
    }
    double Ji[3][3];
#pragma unroll
    for (int d = 0; d < 3; ++d)
#pragma unroll
        for (int I = 0; I < 3; ++I) Ji[d][I] = __ldg(geo + (int64_t)(3 * d + I) * ng + tt);
    const double w = __ldg(geo + 9 * ng + tt);
    double F[3][3];
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int I = 0; I < 3; ++I)
            F[c][I] = Fx[c][0] * Ji[0][I] + Fx[c][1] * Ji[1][I] + Fx[c][2] * Ji[2][I];

    double ef[3] = {1.0, 0.0, 0.0}, es[3] = {0.0, 1.0, 0.0};
    if (fib) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            ef[c] = __ldg(fib + c * n_elems + ee);
            es[c] = __ldg(fib + (3 + c) * n_elems + ee);
        }
    }
    ib_material m = mats[mat_id ? __ldg(mat_id + ee) : 0];
    double P[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
    double J = ib_pk1(m, F, ef, es, P);
    if (live && !finite) ib_latch(status, IB_ERR_NONFINITE, e);
    else if (live && (!(w > 0.0) || !(J > 0.0))) ib_latch(status, IB_ERR_INVERTED_ELEMENT, e);

    // contribution of this Gauss point to node a:  -(P G_a) w,  G_a = J0^-T dN_a  =>  -(P J0^-T) dN_a w
    double Q[3][3];                                // Q_{c d} = -w sum_I P_{cI} Ji[d][I]
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int d = 0; d < 3; ++d)
            Q[c][d] = -w * (P[c][0] * Ji[d][0] + P[c][1] * Ji[d][1] + P[c][2] * Ji[d][2]);
    double v[8][3];
#pragma unroll
    for (int a = 0; a < 8; ++a)
#pragma unroll
        for (int c = 0; c < 3; ++c)
            v[a][c] = Q[c][0] * dN[a][0] + Q[c][1] * dN[a][1] + Q[c][2] * dN[a][2];

    // transposing reduction over the 8 Gauss-point lanes: lane q ends with node q's total
    const unsigned full = 0xffffffffu;
    double s4[4][3];
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            double keep = (q & 4) ? v[a + 4][c] : v[a][c];
            double send = (q & 4) ? v[a][c] : v[a + 4][c];
            s4[a][c] = keep + __shfl_xor_sync(full, send, 4);
        }
    double s2[2][3];
#pragma unroll
    for (int a = 0; a < 2; ++a)
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            double keep = (q & 2) ? s4[a + 2][c] : s4[a][c];
            double send = (q & 2) ? s4[a][c] : s4[a + 2][c];
            s2[a][c] = keep + __shfl_xor_sync(full, send, 2);
        }
    double s1[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        double keep = (q & 1) ? s2[1][c] : s2[0][c];
        double send = (q & 1) ? s2[0][c] : s2[1][c];
        s1[c] = keep + __shfl_xor_sync(full, send, 1);
    }
    if (live) {
        int64_t ne8 = n_elems * 8;
#pragma unroll
        for (int c = 0; c < 3; ++c) Ce[c * ne8 + e * 8 + q] = s1[c];
    }
}

// Per node: sum the <= 8 incident element contributions in ascending element order.
// Optionally also writes Fhat = B / w_a (force density coefficients for the prolongation, A13).
__global__ void __launch_bounds__(256)
ibk_node_gather(int64_t n_nodes, int64_t ne8, const int32_t *__restrict__ adj,
                const double *__restrict__ Ce, const double *__restrict__ wa,
                double *__restrict__ B, double *__restrict__ Fhat)
{
    int64_t n = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= n_nodes) return;
    double s0 = 0.0, s1 = 0.0, s2 = 0.0;
#pragma unroll
    for (int j = 0; j < 8; ++j) {
        int slot = __ldg(adj + j * n_nodes + n);
        if (slot >= 0) {
            s0 += __ldg(Ce + slot);
            s1 += __ldg(Ce + ne8 + slot);
            s2 += __ldg(Ce + 2 * ne8 + slot);
        }
    }
    if (B) { B[n] = s0; B[n_nodes + n] = s1; B[2 * n_nodes + n] = s2; }
    if (Fhat) {
        double r = 1.0 / __ldg(wa + n);
        Fhat[n] = s0 * r; Fhat[n_nodes + n] = s1 * r; Fhat[2 * n_nodes + n] = s2 * r;
    }
}

// ---- NEXT-3: P1 tetrahedra ---------------------------------------------------------------------------
// One thread per element: F is constant, one quadrature point with weight det J0 / 6 (the volume).
// J0 = [X1-X0, X2-X0, X3-X0]; G_a = J0^-T grad_xi N_a (grad_xi N = (-1,-1,-1), e1, e2, e3);
// F = sum_a x_a (x) G_a = [x1-x0, x2-x0, x3-x0] J0^-1;  node a >= 1 gets -w P G_a, node 0 the negative sum.
__global__ void __launch_bounds__(128)
ibk_fe_tet(int64_t n_elems, int64_t n_nodes, const int32_t *__restrict__ conn, const double *__restrict__ X,
           const double *__restrict__ x, const double *__restrict__ fib, const int32_t *__restrict__ mat_id,
           const ib_material *__restrict__ mats, double *__restrict__ Ce, long long *status)
{
    int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n_elems) return;
    const int4 nd = __ldg(reinterpret_cast<const int4 *>(conn) + e);
    const int n4[4] = {nd.x, nd.y, nd.z, nd.w};
    double Xe[4][3], xe[4][3];
    bool finite = true;
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            Xe[a][c] = __ldg(X + c * n_nodes + n4[a]);
            xe[a][c] = __ldg(x + c * n_nodes + n4[a]);
            finite = finite && isfinite(xe[a][c]);
        }
    double J0[3][3], Ds[3][3];                      // [I][d] = X_{d+1,I} - X_{0,I}
#pragma unroll
    for (int I = 0; I < 3; ++I)
#pragma unroll
        for (int d = 0; d < 3; ++d) { J0[I][d] = Xe[d + 1][I] - Xe[0][I]; Ds[I][d] = xe[d + 1][I] - xe[0][I]; }
    const double dj = ib_det3(J0), rd = 1.0 / dj;
    double Ji[3][3];                                 // J0^-1 (rows d, cols I)
    Ji[0][0] = (J0[1][1] * J0[2][2] - J0[1][2] * J0[2][1]) * rd;
    Ji[0][1] = (J0[0][2] * J0[2][1] - J0[0][1] * J0[2][2]) * rd;
    Ji[0][2] = (J0[0][1] * J0[1][2] - J0[0][2] * J0[1][1]) * rd;
    Ji[1][0] = (J0[1][2] * J0[2][0] - J0[1][0] * J0[2][2]) * rd;
    Ji[1][1] = (J0[0][0] * J0[2][2] - J0[0][2] * J0[2][0]) * rd;
    Ji[1][2] = (J0[0][2] * J0[1][0] - J0[0][0] * J0[1][2]) * rd;
    Ji[2][0] = (J0[1][0] * J0[2][1] - J0[1][1] * J0[2][0]) * rd;
    Ji[2][1] = (J0[0][1] * J0[2][0] - J0[0][0] * J0[2][1]) * rd;
    Ji[2][2] = (J0[0][0] * J0[1][1] - J0[0][1] * J0[1][0]) * rd;
    double F[3][3];
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int I = 0; I < 3; ++I) F[c][I] = Ds[c][0] * Ji[0][I] + Ds[c][1] * Ji[1][I] + Ds[c][2] * Ji[2][I];
    double ef[3] = {1.0, 0.0, 0.0}, es[3] = {0.0, 1.0, 0.0};
    if (fib) {
#pragma unroll
        for (int c = 0; c < 3; ++c) { ef[c] = __ldg(fib + c * n_elems + e); es[c] = __ldg(fib + (3 + c) * n_elems + e); }
    }
    ib_material m = mats[mat_id ? __ldg(mat_id + e) : 0];
    double P[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
    double J = ib_pk1(m, F, ef, es, P);
    if (!finite) ib_latch(status, IB_ERR_NONFINITE, e);
    else if (!(dj > 0.0) || !(J > 0.0)) ib_latch(status, IB_ERR_INVERTED_ELEMENT, e);
    const double w = dj * (1.0 / 6.0);
    const int64_t ne4 = n_elems * 4;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        double s0 = 0.0;
#pragma unroll
        for (int d = 0; d < 3; ++d) {               // node d+1: G = row d of J0^-1
            double v = -w * (P[c][0] * Ji[d][0] + P[c][1] * Ji[d][1] + P[c][2] * Ji[d][2]);
            Ce[c * ne4 + e * 4 + d + 1] = v;
            s0 -= v;
        }
        Ce[c * ne4 + e * 4] = s0;
    }
}

// P2 (10-node) tetrahedra, L265: one thread per (element, quadrature point), the 4 points of the
// degree-2 rule (reading A25) in 4 adjacent lanes; N_v = l_v (2 l_v - 1), N_(ab) = 4 l_a l_b with the
// mid-edge nodes in the order 01, 12, 02, 03, 13, 23; the 10 x 3 nodal contributions of the 4 points
// are summed with a butterfly over the 4 lanes.
__global__ void __launch_bounds__(128)
ibk_fe_tet10(int64_t n_elems, int64_t n_nodes, const int32_t *__restrict__ conn, const double *__restrict__ X,
             const double *__restrict__ x, const double *__restrict__ fib, const int32_t *__restrict__ mat_id,
             const ib_material *__restrict__ mats, double *__restrict__ Ce, long long *status)
{
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t e = t >> 2;
    const int q = (int)(t & 3);
    const bool live = e < n_elems;
    const int64_t ee = live ? e : n_elems - 1;
    const double qa = 0.58541019662496845446, qb = 0.13819660112501051518;      // (5 +- 3 sqrt5)/20, (5 - sqrt5)/20
    const double l[4] = {q == 0 ? qa : qb, q == 1 ? qa : qb, q == 2 ? qa : qb, q == 3 ? qa : qb};
    const double dl[4][3] = {{-1, -1, -1}, {1, 0, 0}, {0, 1, 0}, {0, 0, 1}};
    const int ea[6] = {0, 1, 0, 0, 1, 2}, eb[6] = {1, 2, 2, 3, 3, 3};
    double dN[10][3];
#pragma unroll
    for (int v = 0; v < 4; ++v)
#pragma unroll
        for (int d = 0; d < 3; ++d) dN[v][d] = (4.0 * l[v] - 1.0) * dl[v][d];
#pragma unroll
    for (int k = 0; k < 6; ++k)
#pragma unroll
        for (int d = 0; d < 3; ++d) dN[4 + k][d] = 4.0 * (l[ea[k]] * dl[eb[k]][d] + l[eb[k]] * dl[ea[k]][d]);
    double J0[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}}, Fx[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
    bool finite = true;
#pragma unroll
    for (int a = 0; a < 10; ++a) {
        const int nd = __ldg(conn + ee * 10 + a);
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const double Xa = __ldg(X + c * n_nodes + nd), xa = __ldg(x + c * n_nodes + nd);
            finite = finite && isfinite(xa);
#pragma unroll
            for (int d = 0; d < 3; ++d) { J0[c][d] = fma(Xa, dN[a][d], J0[c][d]); Fx[c][d] = fma(xa, dN[a][d], Fx[c][d]); }
        }
    }
    const double dj = ib_det3(J0), rd = 1.0 / dj;
    double Ji[3][3];
    Ji[0][0] = (J0[1][1] * J0[2][2] - J0[1][2] * J0[2][1]) * rd;
    Ji[0][1] = (J0[0][2] * J0[2][1] - J0[0][1] * J0[2][2]) * rd;
    Ji[0][2] = (J0[0][1] * J0[1][2] - J0[0][2] * J0[1][1]) * rd;
    Ji[1][0] = (J0[1][2] * J0[2][0] - J0[1][0] * J0[2][2]) * rd;
    Ji[1][1] = (J0[0][0] * J0[2][2] - J0[0][2] * J0[2][0]) * rd;
    Ji[1][2] = (J0[0][2] * J0[1][0] - J0[0][0] * J0[1][2]) * rd;
    Ji[2][0] = (J0[1][0] * J0[2][1] - J0[1][1] * J0[2][0]) * rd;
    Ji[2][1] = (J0[0][1] * J0[2][0] - J0[0][0] * J0[2][1]) * rd;
    Ji[2][2] = (J0[0][0] * J0[1][1] - J0[0][1] * J0[1][0]) * rd;
    double F[3][3];
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int I = 0; I < 3; ++I) F[c][I] = Fx[c][0] * Ji[0][I] + Fx[c][1] * Ji[1][I] + Fx[c][2] * Ji[2][I];
    double ef[3] = {1.0, 0.0, 0.0}, es[3] = {0.0, 1.0, 0.0};
    if (fib) {
#pragma unroll
        for (int c = 0; c < 3; ++c) { ef[c] = __ldg(fib + c * n_elems + ee); es[c] = __ldg(fib + (3 + c) * n_elems + ee); }
    }
    ib_material m = mats[mat_id ? __ldg(mat_id + ee) : 0];
    double P[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
    const double J = ib_pk1(m, F, ef, es, P);
    if (live && !finite) ib_latch(status, IB_ERR_NONFINITE, e);
    else if (live && (!(dj > 0.0) || !(J > 0.0))) ib_latch(status, IB_ERR_INVERTED_ELEMENT, e);
    const double w = dj * (1.0 / 24.0);
    double Q[3][3];                                  // Q_{c d} = -w sum_I P_{cI} Ji[d][I]
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int d = 0; d < 3; ++d) Q[c][d] = -w * (P[c][0] * Ji[d][0] + P[c][1] * Ji[d][1] + P[c][2] * Ji[d][2]);
    const int64_t ne10 = n_elems * 10;
#pragma unroll
    for (int a = 0; a < 10; ++a)
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            double v = Q[c][0] * dN[a][0] + Q[c][1] * dN[a][1] + Q[c][2] * dN[a][2];
            v += __shfl_xor_sync(0xffffffffu, v, 1);
            v += __shfl_xor_sync(0xffffffffu, v, 2);
            if (live && ((a * 3 + c) & 3) == q) Ce[c * ne10 + e * 10 + a] = v;
        }
}

// Per node: sum its element contributions through the CSR adjacency in ascending slot order.
__global__ void __launch_bounds__(256)
ibk_node_gather_csr(int64_t n_nodes, int64_t ne4, const int32_t *__restrict__ off, const int32_t *__restrict__ slot,
                    const double *__restrict__ Ce, double *__restrict__ B)
{
    int64_t n = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= n_nodes) return;
    double s0 = 0.0, s1 = 0.0, s2 = 0.0;
    for (int k = __ldg(off + n); k < __ldg(off + n + 1); ++k) {
        int sl = __ldg(slot + k);
        s0 += __ldg(Ce + sl); s1 += __ldg(Ce + ne4 + sl); s2 += __ldg(Ce + 2 * ne4 + sl);
    }
    B[n] = s0; B[n_nodes + n] = s1; B[2 * n_nodes + n] = s2;
}

// ---- NEXT-4: solid boundary loads, added to B ----------------------------------------------------------
__global__ void __launch_bounds__(256)
ibk_tethers(int64_t n, int64_t n_nodes, const int32_t *__restrict__ ids, const double *__restrict__ X,
            const double *__restrict__ x, double kappa, double *__restrict__ B)
{
    int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    const int64_t a = ids[k];
#pragma unroll
    for (int c = 0; c < 3; ++c) B[c * n_nodes + a] += kappa * (X[c * n_nodes + a] - x[c * n_nodes + a]);
}

// one thread per face: dead traction q t0 dA on the reference face, follower pressure -p n da on the
// current face; bilinear quads with 2x2 Gauss points, linear triangles with the centroid rule
__global__ void __launch_bounds__(128)
ibk_surface_loads(int64_t n_faces, int npf, int64_t n_nodes, const int32_t *__restrict__ faces,
                  const double *__restrict__ X, const double *__restrict__ x, double q0, double q1, double q2,
                  double p, double *__restrict__ B)
{
    int64_t f = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (f >= n_faces) return;
    int nd[4] = {0, 0, 0, 0};
    double Xf[4][3], xf[4][3];
    for (int a = 0; a < npf; ++a) {
        nd[a] = faces[f * npf + a];
#pragma unroll
        for (int c = 0; c < 3; ++c) { Xf[a][c] = X[c * n_nodes + nd[a]]; xf[a][c] = x[c * n_nodes + nd[a]]; }
    }
    const double qv[3] = {q0, q1, q2};
    double add[4][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
    const double g = 0.57735026918962576451;
    const int nq = npf == 4 ? 4 : 1;
    for (int q = 0; q < nq; ++q) {
        double N[4], d1[4], d2[4], wq;
        if (npf == 4) {
            const double xi = (q & 1) ? g : -g, et = (q & 2) ? g : -g;
#pragma unroll
            for (int a = 0; a < 4; ++a) {
                const double sx = (a == 1 || a == 2) ? 1.0 : -1.0, se = (a >= 2) ? 1.0 : -1.0;
                N[a] = 0.25 * (1.0 + sx * xi) * (1.0 + se * et);
                d1[a] = 0.25 * sx * (1.0 + se * et);
                d2[a] = 0.25 * (1.0 + sx * xi) * se;
            }
            wq = 1.0;
        } else {
            N[0] = N[1] = N[2] = 1.0 / 3.0; N[3] = 0.0;
            d1[0] = -1.0; d1[1] = 1.0; d1[2] = 0.0; d1[3] = 0.0;
            d2[0] = -1.0; d2[1] = 0.0; d2[2] = 1.0; d2[3] = 0.0;
            wq = 0.5;
        }
        double T1[3] = {0, 0, 0}, T2[3] = {0, 0, 0}, t1[3] = {0, 0, 0}, t2[3] = {0, 0, 0};
        for (int a = 0; a < npf; ++a)
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                T1[c] = fma(d1[a], Xf[a][c], T1[c]); T2[c] = fma(d2[a], Xf[a][c], T2[c]);
                t1[c] = fma(d1[a], xf[a][c], t1[c]); t2[c] = fma(d2[a], xf[a][c], t2[c]);
            }
        const double NX[3] = {T1[1] * T2[2] - T1[2] * T2[1], T1[2] * T2[0] - T1[0] * T2[2], T1[0] * T2[1] - T1[1] * T2[0]};
        const double nx[3] = {t1[1] * t2[2] - t1[2] * t2[1], t1[2] * t2[0] - t1[0] * t2[2], t1[0] * t2[1] - t1[1] * t2[0]};
        const double dA = sqrt(NX[0] * NX[0] + NX[1] * NX[1] + NX[2] * NX[2]);
        for (int a = 0; a < npf; ++a)
#pragma unroll
            for (int c = 0; c < 3; ++c) add[a][c] += wq * N[a] * (qv[c] * dA - p * nx[c]);
    }
    for (int a = 0; a < npf; ++a)
#pragma unroll
        for (int c = 0; c < 3; ++c) atomicAdd(B + c * n_nodes + nd[a], add[a][c]);
}

// the same for 6-node (quadratic) triangles, the faces of the P2 tetrahedra: nodes = 3 vertices, then the
// middles of v0v1, v1v2, v2v0; symmetric 6-point rule of degree 4 (reading A27), one thread per face
__global__ void __launch_bounds__(128)
ibk_surface_loads_t6(int64_t n_faces, int64_t n_nodes, const int32_t *__restrict__ faces,
                     const double *__restrict__ X, const double *__restrict__ x, double q0, double q1, double q2,
                     double p, double *__restrict__ B)
{
    int64_t f = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (f >= n_faces) return;
    int nd[6];
    double Xf[6][3], xf[6][3], add[6][3];
#pragma unroll
    for (int a = 0; a < 6; ++a) {
        nd[a] = faces[f * 6 + a];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            Xf[a][c] = X[c * n_nodes + nd[a]]; xf[a][c] = x[c * n_nodes + nd[a]];
            add[a][c] = 0.0;
        }
    }
    const double qv[3] = {q0, q1, q2};
    // a,b = (8 - sqrt10 +- sqrt(38 - 44 sqrt(2/5)))/18; weights (620 +- sqrt(213125 - 53320 sqrt10))/3720, halved (area 1/2)
    const double ta = 0.44594849091596488632, tb = 0.091576213509770743460;
    const double wa = 0.5 * 0.22338158967801146570, wb = 0.5 * 0.10995174365532186764;
#pragma unroll 1
    for (int q = 0; q < 6; ++q) {
        const double t = q < 3 ? ta : tb, wq = q < 3 ? wa : wb;
        const int k = q < 3 ? q : q - 3;
        const double xi = (k == 2) ? 1.0 - 2.0 * t : t, et = (k == 1) ? 1.0 - 2.0 * t : t;
        const double l0 = 1.0 - xi - et, l1 = xi, l2 = et;
        const double N[6] = {l0 * (2.0 * l0 - 1.0), l1 * (2.0 * l1 - 1.0), l2 * (2.0 * l2 - 1.0), 4.0 * l0 * l1, 4.0 * l1 * l2, 4.0 * l2 * l0};
        const double d1[6] = {-(4.0 * l0 - 1.0), 4.0 * l1 - 1.0, 0.0, 4.0 * (l0 - l1), 4.0 * l2, -4.0 * l2};
        const double d2[6] = {-(4.0 * l0 - 1.0), 0.0, 4.0 * l2 - 1.0, -4.0 * l1, 4.0 * l1, 4.0 * (l0 - l2)};
        double T1[3] = {0, 0, 0}, T2[3] = {0, 0, 0}, t1[3] = {0, 0, 0}, t2[3] = {0, 0, 0};
#pragma unroll
        for (int a = 0; a < 6; ++a)
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                T1[c] = fma(d1[a], Xf[a][c], T1[c]); T2[c] = fma(d2[a], Xf[a][c], T2[c]);
                t1[c] = fma(d1[a], xf[a][c], t1[c]); t2[c] = fma(d2[a], xf[a][c], t2[c]);
            }
        const double NX[3] = {T1[1] * T2[2] - T1[2] * T2[1], T1[2] * T2[0] - T1[0] * T2[2], T1[0] * T2[1] - T1[1] * T2[0]};
        const double nx[3] = {t1[1] * t2[2] - t1[2] * t2[1], t1[2] * t2[0] - t1[0] * t2[2], t1[0] * t2[1] - t1[1] * t2[0]};
        const double dA = sqrt(NX[0] * NX[0] + NX[1] * NX[1] + NX[2] * NX[2]);
#pragma unroll
        for (int a = 0; a < 6; ++a)
#pragma unroll
            for (int c = 0; c < 3; ++c) add[a][c] += wq * N[a] * (qv[c] * dA - p * nx[c]);
    }
#pragma unroll
    for (int a = 0; a < 6; ++a)
#pragma unroll
        for (int c = 0; c < 3; ++c) atomicAdd(B + c * n_nodes + nd[a], add[a][c]);
}

__global__ void __launch_bounds__(256)
ibk_fhat(int64_t n_nodes, const double *__restrict__ B, const double *__restrict__ wa, double *__restrict__ Fhat)
{
    int64_t n = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= n_nodes) return;
    const double r = 1.0 / wa[n];
    Fhat[n] = B[n] * r; Fhat[n_nodes + n] = B[n_nodes + n] * r; Fhat[2 * n_nodes + n] = B[2 * n_nodes + n] * r;
}

static bool ib_has_loads(const ib_ctx *c)
{
    return (c->n_teth > 0 && c->kappa_t != 0.0) ||
           (c->n_faces > 0 && (c->p_load != 0.0 || c->qt0[0] != 0.0 || c->qt0[1] != 0.0 || c->qt0[2] != 0.0));
}

static ib_status ib_add_loads(ib_ctx *c, const double *x, double *B, cudaStream_t st)
{
    if (c->n_teth > 0 && c->kappa_t != 0.0) {
        ibk_tethers<<<ib_blocks(c->n_teth, 256), 256, 0, st>>>(c->n_teth, c->n_nodes, c->d_teth_ids, c->d_X, x, c->kappa_t, B);
        c->launches++;
    }
    if (c->n_faces > 0 && (c->p_load != 0.0 || c->qt0[0] != 0.0 || c->qt0[1] != 0.0 || c->qt0[2] != 0.0)) {
        if (c->npf == 6)
            ibk_surface_loads_t6<<<ib_blocks(c->n_faces, 128), 128, 0, st>>>(c->n_faces, c->n_nodes, c->d_faces, c->d_X, x,
                                                                            c->qt0[0], c->qt0[1], c->qt0[2], c->p_load, B);
        else
            ibk_surface_loads<<<ib_blocks(c->n_faces, 128), 128, 0, st>>>(c->n_faces, c->npf, c->n_nodes, c->d_faces, c->d_X, x,
                                                                         c->qt0[0], c->qt0[1], c->qt0[2], c->p_load, B);
        c->launches++;
    }
    IB_CUDA_TRY(cudaGetLastError());
    return IB_OK;
}

ib_status ibk_fe_precompute(ib_ctx *c, cudaStream_t st)
{
    if (c->n_elems == 0) return IB_OK;
    ibk_fe_geometry<<<ib_blocks(c->n_elems * 8, 256), 256, 0, st>>>(c->n_elems, c->n_nodes, c->d_conn, c->d_X, c->d_geo,
                                                                   c->d_status);
    c->launches++;
    IB_CUDA_TRY(cudaGetLastError());
    return IB_OK;
}

ib_status ibk_fe_force(ib_ctx *c, const double *x, double *B, double *Fhat, cudaStream_t st)
{
    if (c->elem_type != IB_ELEM_HEX8) {                   // nodal coupling only: Fhat is never needed
        if (c->n_elems > 0) {
            if (c->elem_type == IB_ELEM_TET4)
                ibk_fe_tet<<<ib_blocks(c->n_elems, 128), 128, 0, st>>>(c->n_elems, c->n_nodes, c->d_conn, c->d_X, x, c->d_fib,
                                                                      c->d_mat_id, c->d_mats, c->d_Ce, c->d_status);
            else
                ibk_fe_tet10<<<ib_blocks(c->n_elems * 4, 128), 128, 0, st>>>(c->n_elems, c->n_nodes, c->d_conn, c->d_X, x,
                                                                            c->d_fib, c->d_mat_id, c->d_mats, c->d_Ce,
                                                                            c->d_status);
            c->launches++;
        }
        if (c->n_nodes > 0) {
            ibk_node_gather_csr<<<ib_blocks(c->n_nodes, 256), 256, 0, st>>>(c->n_nodes, c->n_elems * c->npe, c->d_node_off,
                                                                            c->d_node_slot, c->d_Ce, B);
            c->launches++;
        }
        IB_CUDA_TRY(cudaGetLastError());
        return ib_has_loads(c) ? ib_add_loads(c, x, B, st) : IB_OK;
    }
    if (c->n_elems > 0) {
        int64_t nt = c->n_elems * 8;
        ibk_fe_gauss<<<ib_blocks(nt, IB_FE_TB), IB_FE_TB, 0, st>>>(c->n_elems, c->n_nodes, c->d_conn, c->d_geo, x,
                                                         c->d_fib, c->d_mat_id, c->d_mats, c->d_Ce,
                                                         c->d_status);
        c->launches++;
    }
    if (c->n_nodes > 0) {
        const bool loads = ib_has_loads(c);
        ibk_node_gather<<<ib_blocks(c->n_nodes, 256), 256, 0, st>>>(c->n_nodes, c->n_elems * 8, c->d_adj,
                                                                    c->d_Ce, c->d_wa, B, loads ? nullptr : Fhat);
        c->launches++;
        if (loads) {                                          // Fhat = B / w_a must see the boundary loads too
            ib_status s = ib_add_loads(c, x, B, st);
            if (s != IB_OK) return s;
            if (Fhat) {
                ibk_fhat<<<ib_blocks(c->n_nodes, 256), 256, 0, st>>>(c->n_nodes, B, c->d_wa, Fhat);
                c->launches++;
            }
        }
    }
    IB_CUDA_TRY(cudaGetLastError());
    return IB_OK;
}
