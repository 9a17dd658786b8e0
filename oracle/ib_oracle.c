/*
 * ib_oracle.c -- plain, slow, CPU reference ("oracle") for the Lagrangian-Eulerian coupling step
 * of the immersed boundary method of arXiv 2503.22695 (text in /root/reference/PAPER.md).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code, header, table
 * or helper with paper_2503_22695_b200/csrc (the CUDA path) and neither includes the other.
 *
 * Every function is the paper's definition written out as loops, in the paper's order and
 * notation, with 80-bit long double arithmetic/accumulators so that the oracle is the more
 * accurate side of every comparison.  No blocking, fusion, sorting or reordering.
 * Exception (by specification): oracle_bin_sort evaluates the binning
 * formula in plain IEEE double, because its integer result must be bit-exact.
 *
 * Parity pins (tests/test_oracle_*.py): every function here is pinned by something other than
 * itself -- closed forms, finite differences of the energy, invariants, brute force on tiny
 * grids, the worked example tests/golden/w1_single_point.txt.  Nothing is "parity unpinned".
 *
 * Conventions (SURVEY.md §8 "Conventions"; the paper is silent on all of them):
 *   grid arrays u,v,w,fu,fv,fw: nx*ny*nz doubles, idx=(k*ny+j)*nx+i, periodic wrap;
 *     u[i,j,k] at (x0+i h, y0+(j+1/2)h, z0+(k+1/2)h), v at ((i+1/2)h, j h, (k+1/2)h),
 *     w at ((i+1/2)h,(j+1/2)h, k h) (+origin)            -- MAC grid
 *   mesh: Q1 hexahedra, local node a=ia+2ja+4ka, xi_a=(2ia-1,2ja-1,2ka-1),
 *     N_a(xi)=1/8 prod_d(1+xi_a,d xi_d); conn[e][a]; node arrays component-major [3][n_nodes];
 *     fibres [6][n_elems] = (e_f, e_s); 2x2x2 Gauss points xi=+-1/sqrt(3), weight 1.
 *   force points: per element nsub=(n1,n2,n3); xi_s=(-1+(2m1+1)/n1, ...), s=m1+n1(m2+n2 m3),
 *     W_s=det J0(xi_s) 8/(n1 n2 n3); nsub==NULL selects the paper's nodal rule (L241).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef long double ld;

typedef struct {
    int32_t law;            /* 0 neo-Hookean, 1 Holzapfel-Ogden, 2 modified standard reinforcing (Eq.7),
                               3 fibre-reinforced model 2 (Eq.10-11) */
    double a, b, af, bf, as_, bs, afs, bfs, kappa;
    double Ta;              /* active tension T_a(t) of L317-331 (0 = passive) */
} oracle_material;

typedef struct {
    int32_t nx, ny, nz;
    double h, x0, y0, z0;
    int32_t periodic;       /* 1: indices wrap (configs); 0: bounded box (PAPER.md L200 Dirichlet walls), NEXT-4:
                               reading A26 -- the arrays hold faces 0..n-1 of every component, a support that
                               reaches outside is truncated (those faces belong to the wall / do not exist) */
} oracle_grid;

/* ------------------------------------------------------------------------------------------
 * O1  delta kernel.  PAPER.md L52 and L211 use delta_h without defining it and cite Peskin 2002
 * (ref. 1, L474); reading A1: Peskin's 4-point function
 *   phi(r) = (3 - 2|r| + sqrt(1 + 4|r| - 4 r^2))/8          |r| <= 1
 *          = (5 - 2|r| - sqrt(-7 + 12|r| - 4 r^2))/8        1 <= |r| <= 2
 *          = 0                                              otherwise,
 *   delta_h(x) = h^-3 phi(x1/h) phi(x2/h) phi(x3/h).
 * ---------------------------------------------------------------------------------------- */
static ld phi_l(ld r)
{
    ld a = fabsl(r);
    if (a <= 1.0L) return (3.0L - 2.0L * a + sqrtl(1.0L + 4.0L * a - 4.0L * a * a)) / 8.0L;
    if (a <= 2.0L) {
        ld d = -7.0L + 12.0L * a - 4.0L * a * a;
        if (d < 0.0L) d = 0.0L;                 /* rounding guard at |r| = 2 */
        return (5.0L - 2.0L * a - sqrtl(d)) / 8.0L;
    }
    return 0.0L;
}

double oracle_phi(double r) { return (double)phi_l((ld)r); }

/* ------------------------------------------------------------------------------------------
 * Q1 shape functions (conventions above)
 * ---------------------------------------------------------------------------------------- */
static void shape(const ld xi[3], ld N[8], ld dN[8][3])
{
    for (int a = 0; a < 8; ++a) {
        ld s0 = (a & 1) ? 1.0L : -1.0L, s1 = (a & 2) ? 1.0L : -1.0L, s2 = (a & 4) ? 1.0L : -1.0L;
        ld f0 = 1.0L + s0 * xi[0], f1 = 1.0L + s1 * xi[1], f2 = 1.0L + s2 * xi[2];
        N[a] = 0.125L * f0 * f1 * f2;
        dN[a][0] = 0.125L * s0 * f1 * f2;
        dN[a][1] = 0.125L * f0 * s1 * f2;
        dN[a][2] = 0.125L * f0 * f1 * s2;
    }
}

static ld det3(const ld A[3][3])
{
    return A[0][0] * (A[1][1] * A[2][2] - A[1][2] * A[2][1])
         - A[0][1] * (A[1][0] * A[2][2] - A[1][2] * A[2][0])
         + A[0][2] * (A[1][0] * A[2][1] - A[1][1] * A[2][0]);
}

/* inverse of A (A^-1), returns det */
static ld inv3(const ld A[3][3], ld Ai[3][3])
{
    ld d = det3(A);
    Ai[0][0] = (A[1][1] * A[2][2] - A[1][2] * A[2][1]) / d;
    Ai[0][1] = (A[0][2] * A[2][1] - A[0][1] * A[2][2]) / d;
    Ai[0][2] = (A[0][1] * A[1][2] - A[0][2] * A[1][1]) / d;
    Ai[1][0] = (A[1][2] * A[2][0] - A[1][0] * A[2][2]) / d;
    Ai[1][1] = (A[0][0] * A[2][2] - A[0][2] * A[2][0]) / d;
    Ai[1][2] = (A[0][2] * A[1][0] - A[0][0] * A[1][2]) / d;
    Ai[2][0] = (A[1][0] * A[2][1] - A[1][1] * A[2][0]) / d;
    Ai[2][1] = (A[0][1] * A[2][0] - A[0][0] * A[2][1]) / d;
    Ai[2][2] = (A[0][0] * A[1][1] - A[0][1] * A[1][0]) / d;
    return d;
}

/* reference Jacobian J0_{I d} = sum_a X_{a,I} dN_a/dxi_d at xi */
static void ref_jacobian(const ld Xe[8][3], ld dN[8][3], ld J0[3][3])
{
    for (int I = 0; I < 3; ++I)
        for (int d = 0; d < 3; ++d) {
            ld s = 0.0L;
            for (int a = 0; a < 8; ++a) s += Xe[a][I] * dN[a][d];
            J0[I][d] = s;
        }
}

/* ------------------------------------------------------------------------------------------
 * O3  constitutive laws: first Piola-Kirchhoff stress P = dPsi/dF.
 * Holzapfel-Ogden Psi_4 / P_4: Eq.(12)-(15), L147-155, with
 *   Ibar_1 = J^(-2/3) I_1 (L108), I_4i = e_i.(C e_i), I_8fs = e_f.(C e_s) (L104),
 *   I_4i^* = max(I_4i,1) (L157), U(J) = kappa/2 (ln J)^2 (L94);
 * readings: A2 (F^-T, not F^T, in the isotropic term of Eq.(14)), A3 (symmetric cross term
 *   a_fs I8 exp[b_fs I8^2](F e_f (x) e_s + F e_s (x) e_f) so that P = dPsi/dF), A5, A7.
 * neo-Hookean (L441-445) = HO with a=mu, b=0 and no fibre terms (reading A6: mu = 2 alpha).
 * F is row-major F[c*3+J] = dx_c/dX_J.  Returns 1 if J <= 0 (A10), else 0.
 * ---------------------------------------------------------------------------------------- */
static int pk1_l(const oracle_material *m, const ld F[3][3], const ld ef[3], const ld es[3],
                 ld P[3][3], ld *psi)
{
    ld J = det3(F);
    if (!(J > 0.0L)) return 1;
    ld Fi[3][3];
    inv3(F, Fi);                                   /* F^-1; F^-T_{cJ} = Fi[J][c] */
    ld I1 = 0.0L;
    for (int c = 0; c < 3; ++c)
        for (int K = 0; K < 3; ++K) I1 += F[c][K] * F[c][K];        /* tr(F^T F) */
    ld cb = cbrtl(J);
    ld Jm23 = 1.0L / (cb * cb);                    /* J^(-2/3), A22 */
    ld Ib1 = Jm23 * I1;
    ld lnJ = logl(J);
    ld a = m->a, b = m->b, kap = m->kappa;
    ld e_iso = expl(b * (Ib1 - 3.0L));
    ld W = (b != 0.0L) ? a / (2.0L * b) * e_iso : 0.5L * a * (Ib1 - 3.0L);
    W += 0.5L * kap * lnJ * lnJ;
    for (int c = 0; c < 3; ++c)
        for (int K = 0; K < 3; ++K)
            P[c][K] = a * e_iso * Jm23 * (F[c][K] - (I1 / 3.0L) * Fi[K][c]) + kap * lnJ * Fi[K][c];
    if (m->law == 1) {
        ld Ff[3], Fs[3];
        for (int c = 0; c < 3; ++c) {
            Ff[c] = F[c][0] * ef[0] + F[c][1] * ef[1] + F[c][2] * ef[2];
            Fs[c] = F[c][0] * es[0] + F[c][1] * es[1] + F[c][2] * es[2];
        }
        ld I4f = Ff[0] * Ff[0] + Ff[1] * Ff[1] + Ff[2] * Ff[2];
        ld I4s = Fs[0] * Fs[0] + Fs[1] * Fs[1] + Fs[2] * Fs[2];
        ld I8 = Ff[0] * Fs[0] + Ff[1] * Fs[1] + Ff[2] * Fs[2];
        ld I4fs = I4f > 1.0L ? I4f : 1.0L, I4ss = I4s > 1.0L ? I4s : 1.0L;
        if (m->af != 0.0) {
            ld d = I4fs - 1.0L, ex = expl((ld)m->bf * d * d);
            ld c2 = 2.0L * (ld)m->af * d * ex;
            W += (m->bf != 0.0) ? (ld)m->af / (2.0L * (ld)m->bf) * (ex - 1.0L) : 0.5L * (ld)m->af * d * d;
            for (int c = 0; c < 3; ++c)
                for (int K = 0; K < 3; ++K) P[c][K] += c2 * Ff[c] * ef[K];
        }
        if (m->as_ != 0.0) {
            ld d = I4ss - 1.0L, ex = expl((ld)m->bs * d * d);
            ld c2 = 2.0L * (ld)m->as_ * d * ex;
            W += (m->bs != 0.0) ? (ld)m->as_ / (2.0L * (ld)m->bs) * (ex - 1.0L) : 0.5L * (ld)m->as_ * d * d;
            for (int c = 0; c < 3; ++c)
                for (int K = 0; K < 3; ++K) P[c][K] += c2 * Fs[c] * es[K];
        }
        if (m->afs != 0.0) {
            ld ex = expl((ld)m->bfs * I8 * I8);
            ld c2 = (ld)m->afs * I8 * ex;
            W += (m->bfs != 0.0) ? (ld)m->afs / (2.0L * (ld)m->bfs) * (ex - 1.0L) : 0.5L * (ld)m->afs * I8 * I8;
            for (int c = 0; c < 3; ++c)
                for (int K = 0; K < 3; ++K) P[c][K] += c2 * (Ff[c] * es[K] + Fs[c] * ef[K]);
        }
    }
    /* Modified standard reinforcing model Psi_1 / P_1, Eq.(7) L119-124 (NEXT-2): a = G_T (b = 0),
     * af = G_L, bf = E_L:
     *   Psi += (G_T-G_L)/2 (2 I4f - I5f - 1) + (E_L+G_T-4G_L)/8 (I4f-1)^2,  I5f = e_f.(C^2 e_f) (L104)
     *   P   += (G_T-G_L)(2 F ef(x)ef - F ef (x) C ef - F C ef (x) ef) + (E_L+G_T-4G_L)/2 (I4f-1) F ef(x)ef */
    if (m->law == 2) {
        ld GT = m->a, GL = m->af, EL = m->bf;
        ld Ff[3], Cf[3], FCf[3];
        for (int c = 0; c < 3; ++c) Ff[c] = F[c][0] * ef[0] + F[c][1] * ef[1] + F[c][2] * ef[2];
        for (int K = 0; K < 3; ++K) Cf[K] = F[0][K] * Ff[0] + F[1][K] * Ff[1] + F[2][K] * Ff[2];   /* C ef = F^T F ef */
        for (int c = 0; c < 3; ++c) FCf[c] = F[c][0] * Cf[0] + F[c][1] * Cf[1] + F[c][2] * Cf[2];
        ld I4f = Ff[0] * Ff[0] + Ff[1] * Ff[1] + Ff[2] * Ff[2];
        ld I5f = Cf[0] * Cf[0] + Cf[1] * Cf[1] + Cf[2] * Cf[2];
        ld k2 = EL + GT - 4.0L * GL;
        W += 0.5L * (GT - GL) * (2.0L * I4f - I5f - 1.0L) + 0.125L * k2 * (I4f - 1.0L) * (I4f - 1.0L);
        for (int c = 0; c < 3; ++c)
            for (int K = 0; K < 3; ++K)
                P[c][K] += (GT - GL) * (2.0L * Ff[c] * ef[K] - Ff[c] * Cf[K] - FCf[c] * ef[K])
                         + 0.5L * k2 * (I4f - 1.0L) * Ff[c] * ef[K];
    }
    /* Fibre-reinforced model 2, Psi_3 / P_3, Eq.(10)-(11) L136-141 (NEXT-2; reading A4: C_01 in the
     * exponent of P_3): isotropic part = the exponential term above with a = 2 C10 C01, b = C01
     * and the "-1" of Eq.(10), i.e. an offset C10 = a/(2b), restored; fibre term on I4f itself, NO switch:
     *   Psi += af/(2bf)(exp[bf (I4f-1)^2] - 1),  P += 2 af (I4f-1) exp[bf (I4f-1)^2] F ef(x)ef */
    if (m->law == 3 && b != 0.0L) W -= a / (2.0L * b);
    if (m->law == 3 && m->af != 0.0) {
        ld Ff[3];
        for (int c = 0; c < 3; ++c) Ff[c] = F[c][0] * ef[0] + F[c][1] * ef[1] + F[c][2] * ef[2];
        ld d = Ff[0] * Ff[0] + Ff[1] * Ff[1] + Ff[2] * Ff[2] - 1.0L, ex = expl((ld)m->bf * d * d);
        W += (m->bf != 0.0) ? (ld)m->af / (2.0L * (ld)m->bf) * (ex - 1.0L) : 0.5L * (ld)m->af * d * d;
        for (int c = 0; c < 3; ++c)
            for (int K = 0; K < 3; ++K) P[c][K] += 2.0L * (ld)m->af * d * ex * Ff[c] * ef[K];
    }
    /* Active stress (L317-331, NEXT-2): P^a = F S_a, S_a = T e_f (x) e_f, T = T_a (1 + 4.9 (sqrt(I4f) - 1)).
     * Not hyperelastic: it has no energy, psi is the passive energy only. */
    if (m->Ta != 0.0) {
        ld Ff[3];
        for (int c = 0; c < 3; ++c) Ff[c] = F[c][0] * ef[0] + F[c][1] * ef[1] + F[c][2] * ef[2];
        ld I4f = Ff[0] * Ff[0] + Ff[1] * Ff[1] + Ff[2] * Ff[2];
        ld T = (ld)m->Ta * (1.0L + 4.9L * (sqrtl(I4f) - 1.0L));
        for (int c = 0; c < 3; ++c)
            for (int K = 0; K < 3; ++K) P[c][K] += T * Ff[c] * ef[K];
    }
    if (psi) *psi = W;
    return 0;
}

int oracle_pk1(const oracle_material *m, const double *F, const double *ef, const double *es,
               double *P, double *psi)
{
    ld Fl[3][3], Pl[3][3], f[3] = {1, 0, 0}, s[3] = {0, 1, 0}, W = 0.0L;
    for (int c = 0; c < 3; ++c)
        for (int K = 0; K < 3; ++K) Fl[c][K] = F[c * 3 + K];
    if (ef) for (int i = 0; i < 3; ++i) f[i] = ef[i];
    if (es) for (int i = 0; i < 3; ++i) s[i] = es[i];
    int rc = pk1_l(m, Fl, f, s, Pl, &W);
    if (rc) return rc;
    for (int c = 0; c < 3; ++c)
        for (int K = 0; K < 3; ++K) P[c * 3 + K] = (double)Pl[c][K];
    if (psi) *psi = (double)W;
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * O2  FE nodal force, matrix-free (Eq.(20); L249-251):
 *   F_i = - sum_{(X_q,w_q) in H_q} P^e(X_q) : grad_X phi_i(X_q) w_q
 * per element e, Gauss point q: J0, G_a = J0^-T grad_xi N_a, w = det J0 (weight 1),
 *   F = sum_a x_a (x) G_a (L28-32), P = P(F), B_{a,c} -= sum_J P_{cJ} G_{a,J} w.
 * energy = sum_e sum_q Psi(F_q) w_q (for the -dE/dx pin).  Returns 0, or 1 with *first_bad =
 * element id if det J0 <= 0 or J <= 0 (A10).
 * ---------------------------------------------------------------------------------------- */
int oracle_fe_force(int64_t n_nodes, int64_t n_elems, const int32_t *conn, const double *X,
                    const double *x, const double *fibers, const int32_t *mat_id,
                    const oracle_material *mats, double *B, double *energy, double *minJ,
                    int64_t *first_bad)
{
    ld *Bl = (ld *)calloc((size_t)(3 * n_nodes), sizeof(ld));
    ld E = 0.0L, mj = INFINITY;
    int rc = 0;
    const ld g = 1.0L / sqrtl(3.0L);
    if (first_bad) *first_bad = -1;
    for (int64_t e = 0; e < n_elems && !rc; ++e) {
        ld Xe[8][3], xe[8][3], ef[3] = {1, 0, 0}, es[3] = {0, 1, 0};
        for (int a = 0; a < 8; ++a) {
            int64_t n = conn[e * 8 + a];
            for (int c = 0; c < 3; ++c) { Xe[a][c] = X[c * n_nodes + n]; xe[a][c] = x[c * n_nodes + n]; }
        }
        if (fibers)
            for (int c = 0; c < 3; ++c) { ef[c] = fibers[c * n_elems + e]; es[c] = fibers[(3 + c) * n_elems + e]; }
        const oracle_material *m = &mats[mat_id ? mat_id[e] : 0];
        for (int q = 0; q < 8; ++q) {
            ld xi[3] = {(q & 1) ? g : -g, (q & 2) ? g : -g, (q & 4) ? g : -g};
            ld N[8], dN[8][3], J0[3][3], J0i[3][3];
            shape(xi, N, dN);
            ref_jacobian(Xe, dN, J0);
            ld w = inv3(J0, J0i);
            if (!(w > 0.0L)) { rc = 1; if (first_bad) *first_bad = e; break; }
            ld G[8][3];
            for (int a = 0; a < 8; ++a)
                for (int I = 0; I < 3; ++I) {
                    ld s = 0.0L;
                    for (int d = 0; d < 3; ++d) s += J0i[d][I] * dN[a][d];
                    G[a][I] = s;
                }
            ld F[3][3], P[3][3], W;
            for (int c = 0; c < 3; ++c)
                for (int I = 0; I < 3; ++I) {
                    ld s = 0.0L;
                    for (int a = 0; a < 8; ++a) s += xe[a][c] * G[a][I];
                    F[c][I] = s;
                }
            if (pk1_l(m, F, ef, es, P, &W)) { rc = 1; if (first_bad) *first_bad = e; break; }
            ld J = det3(F);
            if (J < mj) mj = J;
            E += W * w;
            for (int a = 0; a < 8; ++a) {
                int64_t n = conn[e * 8 + a];
                for (int c = 0; c < 3; ++c) {
                    ld s = 0.0L;
                    for (int I = 0; I < 3; ++I) s += P[c][I] * G[a][I];
                    Bl[c * n_nodes + n] -= s * w;
                }
            }
        }
    }
    for (int64_t i = 0; i < 3 * n_nodes; ++i) B[i] = (double)Bl[i];
    if (energy) *energy = (double)E;
    if (minJ) *minJ = (double)mj;
    free(Bl);
    return rc;
}

/* ------------------------------------------------------------------------------------------
 * O2t FE nodal force on P1 (4-node, linear) tetrahedra -- NEXT-3: the paper's cardiac meshes are
 * tetrahedral (L372, L447) and coupled by the nodal rule (L241, L466).  Same weak form (Eq.(20)
 * L191; L249-251) with N_0 = 1-xi-eta-zeta, N_1 = xi, N_2 = eta, N_3 = zeta:
 *   J0_{I d} = sum_a X_{a,I} dN_a/dxi_d = [X_1-X_0, X_2-X_0, X_3-X_0],  G_a = J0^-T grad_xi N_a,
 *   one quadrature point (F is constant per element), weight w = det J0 / 6 (the element volume),
 *   F = sum_a x_a (x) G_a,  B_{a,c} -= sum_J P_{cJ} G_{a,J} w,  energy = sum_e Psi(F_e) w_e.
 * conn is [n_elems][4].  Returns 0, or 1 with *first_bad = element id if det J0 <= 0 or J <= 0.
 * ---------------------------------------------------------------------------------------- */
int oracle_fe_force_tet(int64_t n_nodes, int64_t n_elems, const int32_t *conn, const double *X,
                        const double *x, const double *fibers, const int32_t *mat_id,
                        const oracle_material *mats, double *B, double *energy, double *minJ,
                        int64_t *first_bad)
{
    static const ld dNt[4][3] = {{-1, -1, -1}, {1, 0, 0}, {0, 1, 0}, {0, 0, 1}};
    ld *Bl = (ld *)calloc((size_t)(3 * n_nodes), sizeof(ld));
    ld E = 0.0L, mj = INFINITY;
    int rc = 0;
    for (int64_t e = 0; e < n_elems && !rc; ++e) {
        ld Xe[4][3], xe[4][3], ef[3] = {1, 0, 0}, es[3] = {0, 1, 0};
        for (int a = 0; a < 4; ++a)
            for (int c = 0; c < 3; ++c) {
                Xe[a][c] = X[c * n_nodes + conn[e * 4 + a]];
                xe[a][c] = x[c * n_nodes + conn[e * 4 + a]];
            }
        if (fibers)
            for (int c = 0; c < 3; ++c) { ef[c] = fibers[c * n_elems + e]; es[c] = fibers[(3 + c) * n_elems + e]; }
        const oracle_material *m = &mats[mat_id ? mat_id[e] : 0];
        ld J0[3][3], J0i[3][3];
        for (int I = 0; I < 3; ++I)
            for (int d = 0; d < 3; ++d) {
                ld s = 0.0L;
                for (int a = 0; a < 4; ++a) s += Xe[a][I] * dNt[a][d];
                J0[I][d] = s;
            }
        ld dj = inv3(J0, J0i);
        if (!(dj > 0.0L)) { rc = 1; if (first_bad) *first_bad = e; break; }
        ld w = dj / 6.0L;
        ld G[4][3];
        for (int a = 0; a < 4; ++a)
            for (int I = 0; I < 3; ++I) {
                ld s = 0.0L;
                for (int d = 0; d < 3; ++d) s += J0i[d][I] * dNt[a][d];
                G[a][I] = s;
            }
        ld F[3][3], P[3][3], W;
        for (int c = 0; c < 3; ++c)
            for (int I = 0; I < 3; ++I) {
                ld s = 0.0L;
                for (int a = 0; a < 4; ++a) s += xe[a][c] * G[a][I];
                F[c][I] = s;
            }
        if (pk1_l(m, F, ef, es, P, &W)) { rc = 1; if (first_bad) *first_bad = e; break; }
        ld J = det3(F);
        if (J < mj) mj = J;
        E += W * w;
        for (int a = 0; a < 4; ++a) {
            int64_t n = conn[e * 4 + a];
            for (int c = 0; c < 3; ++c) {
                ld s = 0.0L;
                for (int I = 0; I < 3; ++I) s += P[c][I] * G[a][I];
                Bl[c * n_nodes + n] -= s * w;
            }
        }
    }
    for (int64_t i = 0; i < 3 * n_nodes; ++i) B[i] = (double)Bl[i];
    if (energy) *energy = (double)E;
    if (minJ) *minJ = (double)mj;
    free(Bl);
    return rc;
}

/* ------------------------------------------------------------------------------------------
 * O2q FE nodal force on P2 (10-node, quadratic) tetrahedra -- NEXT-3, second half: "the forces and
 * displacements are discretized using P2 finite elements" (Cook's membrane, L265).  Barycentric
 * coordinates l0 = 1-xi-eta-zeta, l1 = xi, l2 = eta, l3 = zeta; nodes 0-3 vertices, 4-9 the edge
 * mid-points (01, 12, 02, 03, 13, 23):
 *   N_v = l_v (2 l_v - 1),   N_(ab) = 4 l_a l_b,   grad_xi by the product rule,
 *   J0 = sum_a X_a (x) grad_xi N_a (per quadrature point: edges may be curved), G_a = J0^-T grad_xi N_a,
 *   F = sum_a x_a (x) G_a,  B_{a,c} -= sum_J P_{cJ} G_{a,J} w,  w = det J0 * w_q  (Eq.(20)).
 * The paper does not name the quadrature rule; reading A25: the 4-point degree-2 rule, points
 * (a,b,b,b) and permutations in barycentric coordinates, a = (5+3 sqrt5)/20, b = (5-sqrt5)/20, w_q = 1/24.
 * conn is [n_elems][10].
 * ---------------------------------------------------------------------------------------- */
static void p2_shape(const ld l[4], ld dN[10][3])
{
    static const ld dl[4][3] = {{-1, -1, -1}, {1, 0, 0}, {0, 1, 0}, {0, 0, 1}};
    static const int ea[6] = {0, 1, 0, 0, 1, 2}, eb[6] = {1, 2, 2, 3, 3, 3};
    for (int v = 0; v < 4; ++v)
        for (int d = 0; d < 3; ++d) dN[v][d] = (4.0L * l[v] - 1.0L) * dl[v][d];
    for (int e = 0; e < 6; ++e)
        for (int d = 0; d < 3; ++d) dN[4 + e][d] = 4.0L * (l[ea[e]] * dl[eb[e]][d] + l[eb[e]] * dl[ea[e]][d]);
}

int oracle_fe_force_tet10(int64_t n_nodes, int64_t n_elems, const int32_t *conn, const double *X,
                          const double *x, const double *fibers, const int32_t *mat_id,
                          const oracle_material *mats, double *B, double *energy, double *minJ,
                          int64_t *first_bad)
{
    const ld qa = (5.0L + 3.0L * sqrtl(5.0L)) / 20.0L, qb = (5.0L - sqrtl(5.0L)) / 20.0L;
    ld *Bl = (ld *)calloc((size_t)(3 * n_nodes), sizeof(ld));
    ld E = 0.0L, mj = INFINITY;
    int rc = 0;
    for (int64_t e = 0; e < n_elems && !rc; ++e) {
        ld Xe[10][3], xe[10][3], ef[3] = {1, 0, 0}, es[3] = {0, 1, 0};
        for (int a = 0; a < 10; ++a)
            for (int c = 0; c < 3; ++c) {
                Xe[a][c] = X[c * n_nodes + conn[e * 10 + a]];
                xe[a][c] = x[c * n_nodes + conn[e * 10 + a]];
            }
        if (fibers)
            for (int c = 0; c < 3; ++c) { ef[c] = fibers[c * n_elems + e]; es[c] = fibers[(3 + c) * n_elems + e]; }
        const oracle_material *m = &mats[mat_id ? mat_id[e] : 0];
        for (int q = 0; q < 4; ++q) {
            ld l[4] = {qb, qb, qb, qb}, dN[10][3], J0[3][3], J0i[3][3];
            l[q] = qa;
            p2_shape(l, dN);
            for (int I = 0; I < 3; ++I)
                for (int d = 0; d < 3; ++d) {
                    ld s2 = 0.0L;
                    for (int a = 0; a < 10; ++a) s2 += Xe[a][I] * dN[a][d];
                    J0[I][d] = s2;
                }
            ld dj = inv3(J0, J0i);
            if (!(dj > 0.0L)) { rc = 1; if (first_bad) *first_bad = e; break; }
            ld w = dj / 24.0L;
            ld G[10][3];
            for (int a = 0; a < 10; ++a)
                for (int I = 0; I < 3; ++I) {
                    ld s2 = 0.0L;
                    for (int d = 0; d < 3; ++d) s2 += J0i[d][I] * dN[a][d];
                    G[a][I] = s2;
                }
            ld F[3][3], P[3][3], W;
            for (int c = 0; c < 3; ++c)
                for (int I = 0; I < 3; ++I) {
                    ld s2 = 0.0L;
                    for (int a = 0; a < 10; ++a) s2 += xe[a][c] * G[a][I];
                    F[c][I] = s2;
                }
            if (pk1_l(m, F, ef, es, P, &W)) { rc = 1; if (first_bad) *first_bad = e; break; }
            ld J = det3(F);
            if (J < mj) mj = J;
            E += W * w;
            for (int a = 0; a < 10; ++a) {
                int64_t n = conn[e * 10 + a];
                for (int c = 0; c < 3; ++c) {
                    ld s2 = 0.0L;
                    for (int I = 0; I < 3; ++I) s2 += P[c][I] * G[a][I];
                    Bl[c * n_nodes + n] -= s2 * w;
                }
            }
        }
    }
    for (int64_t i = 0; i < 3 * n_nodes; ++i) B[i] = (double)Bl[i];
    if (energy) *energy = (double)E;
    if (minJ) *minJ = (double)mj;
    free(Bl);
    return rc;
}

/* ------------------------------------------------------------------------------------------
 * O9  solid boundary loads (NEXT-4; Table 3 row "Solid boundary" L398).  All ADD to B [3][n_nodes].
 *  tethers (L263 "fixed left face ... penalty parameter kappa = 10^6", L425): the paper gives only the
 *    parameter; reading A24: a penalty spring to the reference position, B_a += kappa (X_a - x_a),
 *    energy kappa/2 sum |x_a - X_a|^2.
 *  traction (L263): dead load q t0 per unit REFERENCE area on boundary faces, B_a += q t0 int N_a dA.
 *  pressure (L303, L315 "uniform pressure applied to the endocardial surface"): follower load -p n per
 *    unit CURRENT area, n the outward normal of the face as oriented, B_a -= p int N_a n da.
 * Faces: npf = 4 bilinear quads (nodes in cyclic order; 2x2 Gauss, exact for these integrands) or
 * npf = 3 linear triangles (one point).  n da = d x/d xi x d x/d eta d xi d eta.
 * ---------------------------------------------------------------------------------------- */
void oracle_tethers(int64_t n_nodes, int64_t n_t, const int32_t *ids, const double *X, const double *x,
                    double kappa, double *B, double *energy)
{
    ld E = 0.0L;
    for (int64_t k = 0; k < n_t; ++k)
        for (int c = 0; c < 3; ++c) {
            ld d = (ld)x[c * n_nodes + ids[k]] - (ld)X[c * n_nodes + ids[k]];
            B[c * n_nodes + ids[k]] = (double)((ld)B[c * n_nodes + ids[k]] - (ld)kappa * d);
            E += 0.5L * (ld)kappa * d * d;
        }
    if (energy) *energy = (double)E;
}

void oracle_surface_loads(int64_t n_nodes, int64_t n_faces, int32_t npf, const int32_t *faces,
                          const double *X, const double *x, const double *qt0, double p, double *B)
{
    const ld g = 0.57735026918962576450914878050196L;
    /* reading A27: 6-node (quadratic) triangles take the symmetric 6-point rule of degree 4,
     *   a,b = (8 - sqrt10 +- sqrt(38 - 44 sqrt(2/5)))/18,  w = (620 +- sqrt(213125 - 53320 sqrt10))/3720,
     * points (t,t), (t,1-2t), (1-2t,t) for t = a (weight w+) and t = b (weight w-), times the area 1/2 of
     * the reference triangle: exact for the follower pressure (N_a (t1 x t2) has degree 4). */
    const ld s10 = sqrtl(10.0L), rr = sqrtl(38.0L - 44.0L * sqrtl(0.4L)), tt = sqrtl(213125.0L - 53320.0L * s10);
    const ld qa = (8.0L - s10 + rr) / 18.0L, qb = (8.0L - s10 - rr) / 18.0L;
    const ld wa = (620.0L + tt) / 3720.0L, wb = (620.0L - tt) / 3720.0L;
    for (int64_t f = 0; f < n_faces; ++f) {
        ld add[6][3] = {{0}};
        int nq = npf == 4 ? 4 : (npf == 6 ? 6 : 1);
        for (int q = 0; q < nq; ++q) {
            ld N[6] = {0}, dNx[6] = {0}, dNe[6] = {0}, wq;
            if (npf == 4) {                          /* cyclic node order (-1,-1),(1,-1),(1,1),(-1,1) */
                ld xi = (q & 1) ? g : -g, et = (q & 2) ? g : -g;
                const ld sx[4] = {-1, 1, 1, -1}, se[4] = {-1, -1, 1, 1};
                for (int a = 0; a < 4; ++a) {
                    N[a] = 0.25L * (1 + sx[a] * xi) * (1 + se[a] * et);
                    dNx[a] = 0.25L * sx[a] * (1 + se[a] * et);
                    dNe[a] = 0.25L * (1 + sx[a] * xi) * se[a];
                }
                wq = 1.0L;
            } else if (npf == 6) {                   /* nodes: vertices 0,1,2, then the middles of 01, 12, 20 */
                ld t = q < 3 ? qa : qb;
                int k = q % 3;
                ld xi = k == 2 ? 1.0L - 2.0L * t : t, et = k == 1 ? 1.0L - 2.0L * t : t;
                ld l0 = 1.0L - xi - et, l1 = xi, l2 = et;
                N[0] = l0 * (2 * l0 - 1); N[1] = l1 * (2 * l1 - 1); N[2] = l2 * (2 * l2 - 1);
                N[3] = 4 * l0 * l1; N[4] = 4 * l1 * l2; N[5] = 4 * l2 * l0;
                dNx[0] = -(4 * l0 - 1); dNx[1] = 4 * l1 - 1; dNx[2] = 0;
                dNx[3] = 4 * (l0 - l1); dNx[4] = 4 * l2; dNx[5] = -4 * l2;
                dNe[0] = -(4 * l0 - 1); dNe[1] = 0; dNe[2] = 4 * l2 - 1;
                dNe[3] = -4 * l1; dNe[4] = 4 * l1; dNe[5] = 4 * (l0 - l2);
                wq = 0.5L * (q < 3 ? wa : wb);
            } else {                                 /* N = (1-xi-eta, xi, eta) at the centroid, weight 1/2 */
                N[0] = N[1] = N[2] = 1.0L / 3.0L;
                dNx[0] = -1; dNx[1] = 1; dNx[2] = 0;
                dNe[0] = -1; dNe[1] = 0; dNe[2] = 1;
                wq = 0.5L;
            }
            ld tX[2][3] = {{0}}, tx[2][3] = {{0}};
            for (int a = 0; a < npf; ++a)
                for (int c = 0; c < 3; ++c) {
                    int64_t n = faces[f * npf + a];
                    tX[0][c] += dNx[a] * X[c * n_nodes + n]; tX[1][c] += dNe[a] * X[c * n_nodes + n];
                    tx[0][c] += dNx[a] * x[c * n_nodes + n]; tx[1][c] += dNe[a] * x[c * n_nodes + n];
                }
            ld NX[3] = {tX[0][1] * tX[1][2] - tX[0][2] * tX[1][1], tX[0][2] * tX[1][0] - tX[0][0] * tX[1][2],
                        tX[0][0] * tX[1][1] - tX[0][1] * tX[1][0]};
            ld nx[3] = {tx[0][1] * tx[1][2] - tx[0][2] * tx[1][1], tx[0][2] * tx[1][0] - tx[0][0] * tx[1][2],
                        tx[0][0] * tx[1][1] - tx[0][1] * tx[1][0]};
            ld dA = sqrtl(NX[0] * NX[0] + NX[1] * NX[1] + NX[2] * NX[2]);
            for (int a = 0; a < npf; ++a)
                for (int c = 0; c < 3; ++c)
                    add[a][c] += wq * N[a] * ((qt0 ? (ld)qt0[c] : 0.0L) * dA - (ld)p * nx[c]);
        }
        for (int a = 0; a < npf; ++a)
            for (int c = 0; c < 3; ++c) {
                int64_t n = faces[f * npf + a];
                B[c * n_nodes + n] = (double)((ld)B[c * n_nodes + n] + add[a][c]);
            }
    }
}

/* ------------------------------------------------------------------------------------------
 * O4  force points, lumped weights, prolongation; O7 restriction.
 * Reading A13 (Griffith-Luo style quadrature coupling; PAPER.md L233-237 projection, L241 nodal
 * weights w_q = int phi_q): with sub-point rule {xi_s, W_s} per element,
 *   w_a  = sum_{e contains a} sum_s W_s N_a(xi_s)                (lumped mass, same rule)
 *   x_s  = sum_a N_a(xi_s) x_a                                   (chi_h at the point)
 *   Fhat_a = B_a / w_a ;  G_s = W_s sum_a N_a(xi_s) Fhat_a       (force carried by the point)
 *   U_a  = (1/w_a) sum_{e,s} W_s N_a(xi_s) U_s                   (lumped L2 projection, L235)
 * ---------------------------------------------------------------------------------------- */
int64_t oracle_num_points(int64_t n_nodes, int64_t n_elems, const int32_t *nsub)
{
    if (!nsub) return n_nodes;
    int64_t P = 0;
    for (int64_t e = 0; e < n_elems; ++e) P += (int64_t)nsub[3 * e] * nsub[3 * e + 1] * nsub[3 * e + 2];
    return P;
}

static void sub_xi(const int32_t *ns, int64_t s, ld xi[3])
{
    int64_t m1 = s % ns[0], m2 = (s / ns[0]) % ns[1], m3 = s / ((int64_t)ns[0] * ns[1]);
    xi[0] = -1.0L + (ld)(2 * m1 + 1) / (ld)ns[0];
    xi[1] = -1.0L + (ld)(2 * m2 + 1) / (ld)ns[1];
    xi[2] = -1.0L + (ld)(2 * m3 + 1) / (ld)ns[2];
}

/* xp [3][P] from x; Wp [P] and w_a [n_nodes] from X.  Any output may be NULL. */
int oracle_points(int64_t n_nodes, int64_t n_elems, const int32_t *conn, const double *X,
                  const double *x, const int32_t *nsub, double *xp, double *Wp, double *w_a)
{
    int64_t P = oracle_num_points(n_nodes, n_elems, nsub);
    ld *wl = w_a ? (ld *)calloc((size_t)n_nodes, sizeof(ld)) : NULL;
    int64_t p = 0;
    int rc = 0;
    for (int64_t e = 0; e < n_elems; ++e) {
        ld Xe[8][3], xe[8][3];
        for (int a = 0; a < 8; ++a) {
            int64_t n = conn[e * 8 + a];
            for (int c = 0; c < 3; ++c) { Xe[a][c] = X[c * n_nodes + n]; xe[a][c] = x ? x[c * n_nodes + n] : 0.0L; }
        }
        const int32_t *ns = &nsub[3 * e];
        int64_t S = (int64_t)ns[0] * ns[1] * ns[2];
        for (int64_t s = 0; s < S; ++s, ++p) {
            ld xi[3], N[8], dN[8][3], J0[3][3];
            sub_xi(ns, s, xi);
            shape(xi, N, dN);
            ref_jacobian(Xe, dN, J0);
            ld dj = det3(J0);
            if (!(dj > 0.0L)) rc = 1;
            ld W = dj * 8.0L / (ld)S;
            if (Wp) Wp[p] = (double)W;
            if (xp)
                for (int c = 0; c < 3; ++c) {
                    ld v = 0.0L;
                    for (int a = 0; a < 8; ++a) v += N[a] * xe[a][c];
                    xp[c * P + p] = (double)v;
                }
            if (wl)
                for (int a = 0; a < 8; ++a) wl[conn[e * 8 + a]] += W * N[a];
        }
    }
    if (wl) { for (int64_t n = 0; n < n_nodes; ++n) w_a[n] = (double)wl[n]; free(wl); }
    return rc;
}

/* nodal rule of PAPER.md L241: w_q = int phi_q dX, by 2x2x2 Gauss quadrature (exact for Q1
 * on parallelepipeds, the standard rule otherwise). */
void oracle_nodal_weights(int64_t n_nodes, int64_t n_elems, const int32_t *conn, const double *X,
                          double *w_q)
{
    ld *wl = (ld *)calloc((size_t)n_nodes, sizeof(ld));
    const ld g = 1.0L / sqrtl(3.0L);
    for (int64_t e = 0; e < n_elems; ++e) {
        ld Xe[8][3];
        for (int a = 0; a < 8; ++a)
            for (int c = 0; c < 3; ++c) Xe[a][c] = X[c * n_nodes + conn[e * 8 + a]];
        for (int q = 0; q < 8; ++q) {
            ld xi[3] = {(q & 1) ? g : -g, (q & 2) ? g : -g, (q & 4) ? g : -g};
            ld N[8], dN[8][3], J0[3][3];
            shape(xi, N, dN);
            ref_jacobian(Xe, dN, J0);
            ld dj = det3(J0);
            for (int a = 0; a < 8; ++a) wl[conn[e * 8 + a]] += N[a] * dj;
        }
    }
    for (int64_t n = 0; n < n_nodes; ++n) w_q[n] = (double)wl[n];
    free(wl);
}

void oracle_prolong(int64_t n_nodes, int64_t n_elems, const int32_t *conn, const int32_t *nsub,
                    const double *w_a, const double *Wp, const double *B, double *Gp)
{
    int64_t P = oracle_num_points(n_nodes, n_elems, nsub), p = 0;
    for (int64_t e = 0; e < n_elems; ++e) {
        const int32_t *ns = &nsub[3 * e];
        int64_t S = (int64_t)ns[0] * ns[1] * ns[2];
        for (int64_t s = 0; s < S; ++s, ++p) {
            ld xi[3], N[8], dN[8][3];
            sub_xi(ns, s, xi);
            shape(xi, N, dN);
            for (int c = 0; c < 3; ++c) {
                ld v = 0.0L;
                for (int a = 0; a < 8; ++a) {
                    int64_t n = conn[e * 8 + a];
                    v += N[a] * ((ld)B[c * n_nodes + n] / (ld)w_a[n]);
                }
                Gp[c * P + p] = (double)((ld)Wp[p] * v);
            }
        }
    }
}

void oracle_restrict(int64_t n_nodes, int64_t n_elems, const int32_t *conn, const int32_t *nsub,
                     const double *w_a, const double *Wp, const double *Up, double *Un)
{
    int64_t P = oracle_num_points(n_nodes, n_elems, nsub), p = 0;
    ld *acc = (ld *)calloc((size_t)(3 * n_nodes), sizeof(ld));
    for (int64_t e = 0; e < n_elems; ++e) {
        const int32_t *ns = &nsub[3 * e];
        int64_t S = (int64_t)ns[0] * ns[1] * ns[2];
        for (int64_t s = 0; s < S; ++s, ++p) {
            ld xi[3], N[8], dN[8][3];
            sub_xi(ns, s, xi);
            shape(xi, N, dN);
            for (int a = 0; a < 8; ++a) {
                int64_t n = conn[e * 8 + a];
                for (int c = 0; c < 3; ++c) acc[c * n_nodes + n] += (ld)Wp[p] * N[a] * (ld)Up[c * P + p];
            }
        }
    }
    for (int c = 0; c < 3; ++c)
        for (int64_t n = 0; n < n_nodes; ++n) Un[c * n_nodes + n] = (double)(acc[c * n_nodes + n] / (ld)w_a[n]);
    free(acc);
}

/* ------------------------------------------------------------------------------------------
 * O5 spread (Eq.(24)-(26) L211-217; nodal form L253-257) and O6 interpolation
 * (Eq.(27)-(29) L222-229; L243-247).  Reading A14: spread carries a force G_s (density times
 * weight) through delta_h (which contains h^-3) -> f is force per volume; interpolation weight is
 * delta_h * dx^3 = phi phi phi.  Component c lives on its own staggered lattice with offset o_c:
 * u (0,1/2,1/2), v (1/2,0,1/2), w (1/2,1/2,0):
 *   s_d = (x_d - x0_d)/h - o_{c,d};  i0_d = floor(s_d) - 1;
 *   f_c[wrap(i0+m)] += G_{s,c} phi(s_1-i0_1-m_1) phi(s_2-..) phi(s_3-..) / h^3,  m in {0..3}^3
 *   U_{s,c} = sum_m u_c[wrap(i0+m)] phi phi phi
 * ---------------------------------------------------------------------------------------- */
static const ld OFFS[3][3] = {{0.0L, 0.5L, 0.5L}, {0.5L, 0.0L, 0.5L}, {0.5L, 0.5L, 0.0L}};

static int64_t wrapi(int64_t i, int64_t n) { i %= n; return i < 0 ? i + n : i; }
/* index of a support face: wrapped (periodic) or -1 if it lies outside a bounded grid */
static int64_t facei(const oracle_grid *g, int64_t i, int64_t n)
{
    if (g->periodic) return wrapi(i, n);
    return (i < 0 || i >= n) ? -1 : i;
}

static void support(const oracle_grid *g, int c, const ld xpt[3], int64_t i0[3], ld wt[3][4])
{
    const ld org[3] = {g->x0, g->y0, g->z0};
    for (int d = 0; d < 3; ++d) {
        ld s = (xpt[d] - org[d]) / (ld)g->h - OFFS[c][d];
        ld fl = floorl(s);
        i0[d] = (int64_t)fl - 1;
        for (int m = 0; m < 4; ++m) wt[d][m] = phi_l(s - (ld)(i0[d] + m));
    }
}

/* one point's share of component c, Eq.(24)-(26): acc[face] += G_c phi phi phi / h^3 over its 4x4x4 support */
static void spread_point(const oracle_grid *g, int c, int64_t P, int64_t p, const double *xp, const double *Gp, ld h3, ld *acc)
{
    ld xpt[3] = {xp[p], xp[P + p], xp[2 * P + p]}, wt[3][4];
    int64_t i0[3];
    support(g, c, xpt, i0, wt);
    ld G = Gp[c * P + p];
    for (int m3 = 0; m3 < 4; ++m3)
        for (int m2 = 0; m2 < 4; ++m2)
            for (int m1 = 0; m1 < 4; ++m1) {
                int64_t i = facei(g, i0[0] + m1, g->nx), j = facei(g, i0[1] + m2, g->ny), k = facei(g, i0[2] + m3, g->nz);
                if (i < 0 || j < 0 || k < 0) continue;
                acc[(k * g->ny + j) * g->nx + i] += G * wt[0][m1] * wt[1][m2] * wt[2][m3] / h3;
            }
}

void oracle_spread(const oracle_grid *g, int64_t P, const double *xp, const double *Gp,
                   double *fu, double *fv, double *fw, int32_t accumulate)
{
    int64_t ncell = (int64_t)g->nx * g->ny * g->nz;
    double *f[3] = {fu, fv, fw};
    ld h3 = (ld)g->h * (ld)g->h * (ld)g->h;
    for (int c = 0; c < 3; ++c) {
        ld *acc = (ld *)calloc((size_t)ncell, sizeof(ld));
        if (accumulate) for (int64_t i = 0; i < ncell; ++i) acc[i] = f[c][i];
#ifdef _OPENMP            /* timing leg only (liboracle_omp.so): one private grid per thread, summed at the end */
#pragma omp parallel
        {
            ld *mine = (ld *)calloc((size_t)ncell, sizeof(ld));
#pragma omp for schedule(static)
            for (int64_t p = 0; p < P; ++p) spread_point(g, c, P, p, xp, Gp, h3, mine);
#pragma omp critical
            for (int64_t i = 0; i < ncell; ++i) acc[i] += mine[i];
            free(mine);
        }
#else
        for (int64_t p = 0; p < P; ++p) spread_point(g, c, P, p, xp, Gp, h3, acc);
#endif
        for (int64_t i = 0; i < ncell; ++i) f[c][i] = (double)acc[i];
        free(acc);
    }
}

void oracle_interp(const oracle_grid *g, int64_t P, const double *xp, const double *u,
                   const double *v, const double *w, double *Up)
{
    const double *f[3] = {u, v, w};
    for (int c = 0; c < 3; ++c)
#ifdef _OPENMP            /* timing leg only (liboracle_omp.so): points are independent */
#pragma omp parallel for schedule(static)
#endif
        for (int64_t p = 0; p < P; ++p) {
            ld xpt[3] = {xp[p], xp[P + p], xp[2 * P + p]}, wt[3][4];
            int64_t i0[3];
            support(g, c, xpt, i0, wt);
            ld s = 0.0L;
            for (int m3 = 0; m3 < 4; ++m3)
                for (int m2 = 0; m2 < 4; ++m2)
                    for (int m1 = 0; m1 < 4; ++m1) {
                        int64_t i = facei(g, i0[0] + m1, g->nx), j = facei(g, i0[1] + m2, g->ny), k = facei(g, i0[2] + m3, g->nz);
                        if (i < 0 || j < 0 || k < 0) continue;
                        s += (ld)f[c][(k * g->ny + j) * g->nx + i] * wt[0][m1] * wt[1][m2] * wt[2][m3];
                    }
            Up[c * P + p] = (double)s;
        }
}

/* Brute-force variants: every face of the grid, minimum-image distance computed from the face
 * COORDINATES (not from index arithmetic), same phi.  For grids <= 16^3 only. */
static ld min_image(ld d, ld L) { d -= L * roundl(d / L); return d; }

static void face_coord(const oracle_grid *g, int c, int64_t i, int64_t j, int64_t k, ld xf[3])
{
    xf[0] = (ld)g->x0 + ((ld)i + OFFS[c][0]) * (ld)g->h;
    xf[1] = (ld)g->y0 + ((ld)j + OFFS[c][1]) * (ld)g->h;
    xf[2] = (ld)g->z0 + ((ld)k + OFFS[c][2]) * (ld)g->h;
}

void oracle_spread_brute(const oracle_grid *g, int64_t P, const double *xp, const double *Gp,
                         double *fu, double *fv, double *fw)
{
    double *f[3] = {fu, fv, fw};
    ld h = g->h, L[3] = {g->nx * h, g->ny * h, g->nz * h};
    for (int c = 0; c < 3; ++c)
        for (int64_t k = 0; k < g->nz; ++k)
            for (int64_t j = 0; j < g->ny; ++j)
                for (int64_t i = 0; i < g->nx; ++i) {
                    ld xf[3], s = 0.0L;
                    face_coord(g, c, i, j, k, xf);
                    for (int64_t p = 0; p < P; ++p) {
                        ld wgt = 1.0L;
                        for (int d = 0; d < 3; ++d)
                            wgt *= phi_l((g->periodic ? min_image(xf[d] - (ld)xp[d * P + p], L[d]) : xf[d] - (ld)xp[d * P + p]) / h);
                        s += (ld)Gp[c * P + p] * wgt / (h * h * h);
                    }
                    f[c][(k * g->ny + j) * g->nx + i] = (double)s;
                }
}

void oracle_interp_brute(const oracle_grid *g, int64_t P, const double *xp, const double *u,
                         const double *v, const double *w, double *Up)
{
    const double *f[3] = {u, v, w};
    ld h = g->h, L[3] = {g->nx * h, g->ny * h, g->nz * h};
    for (int c = 0; c < 3; ++c)
        for (int64_t p = 0; p < P; ++p) {
            ld s = 0.0L;
            for (int64_t k = 0; k < g->nz; ++k)
                for (int64_t j = 0; j < g->ny; ++j)
                    for (int64_t i = 0; i < g->nx; ++i) {
                        ld xf[3], wgt = 1.0L;
                        face_coord(g, c, i, j, k, xf);
                        for (int d = 0; d < 3; ++d)
                            wgt *= phi_l((g->periodic ? min_image(xf[d] - (ld)xp[d * P + p], L[d]) : xf[d] - (ld)xp[d * P + p]) / h);
                        s += (ld)f[c][(k * g->ny + j) * g->nx + i] * wgt;
                    }
            Up[c * P + p] = (double)s;
        }
}

/* ------------------------------------------------------------------------------------------
 * O8  bin + stable sort by Eulerian cell (not in the paper; north_star requirement; A21).
 * In plain IEEE double, no contraction: c_d = (int64)floor((x_d - x0_d) * inv_h) mod n_d,
 * tile edge T=8, key = ((tz*nty+ty)*ntx+tx)*512 + ((lz*8+ly)*8+lx); perm = stable sort of ids.
 * ---------------------------------------------------------------------------------------- */
typedef struct { int64_t key; int32_t id; } kv_t;

static void merge_sort(kv_t *a, kv_t *tmp, int64_t n)
{
    if (n < 2) return;
    int64_t h = n / 2;
    merge_sort(a, tmp, h);
    merge_sort(a + h, tmp, n - h);
    int64_t i = 0, j = h, k = 0;
    while (i < h && j < n) tmp[k++] = (a[j].key < a[i].key) ? a[j++] : a[i++];   /* ties: left first */
    while (i < h) tmp[k++] = a[i++];
    while (j < n) tmp[k++] = a[j++];
    memcpy(a, tmp, (size_t)n * sizeof(kv_t));
}

void oracle_bin_sort(const oracle_grid *g, double inv_h, int64_t P, const double *xp,
                     int64_t *key_out, int32_t *perm_out)
{
    kv_t *kv = (kv_t *)malloc((size_t)(P > 0 ? P : 1) * sizeof(kv_t));
    kv_t *tmp = (kv_t *)malloc((size_t)(P > 0 ? P : 1) * sizeof(kv_t));
    const double org[3] = {g->x0, g->y0, g->z0};
    const int64_t n[3] = {g->nx, g->ny, g->nz};
    int64_t ntx = g->nx / 8, nty = g->ny / 8;
    for (int64_t p = 0; p < P; ++p) {
        int64_t c[3];
        for (int d = 0; d < 3; ++d) {
            volatile double diff = xp[d * P + p] - org[d];      /* volatile: forbid contraction */
            volatile double sc = diff * inv_h;
            c[d] = wrapi((int64_t)floor(sc), n[d]);
        }
        int64_t t = ((c[2] / 8) * nty + (c[1] / 8)) * ntx + (c[0] / 8);
        int64_t l = ((c[2] % 8) * 8 + (c[1] % 8)) * 8 + (c[0] % 8);
        kv[p].key = t * 512 + l;
        kv[p].id = (int32_t)p;
        key_out[p] = kv[p].key;
    }
    merge_sort(kv, tmp, P);
    for (int64_t p = 0; p < P; ++p) perm_out[p] = kv[p].id;
    free(kv);
    free(tmp);
}

/* ------------------------------------------------------------------------------------------
 * The whole coupling step (BASELINE.json "one coupling step"; reading
 * A16: one position array x for force, spread and interpolation):
 *   B = fe_force(x);  G = prolong(B);  f = spread(x_s, G);  U = interp(x_s, u);  Un = restrict(U)
 * nsub == NULL: the paper's nodal method verbatim (L241-257): points = nodes, G = B, Un = U.
 * ---------------------------------------------------------------------------------------- */
int oracle_coupling_step(const oracle_grid *g, int64_t n_nodes, int64_t n_elems,
                         const int32_t *conn, const double *X, const double *fibers,
                         const int32_t *mat_id, const int32_t *nsub, const oracle_material *mats,
                         const double *x, const double *u, const double *v, const double *w,
                         double *fu, double *fv, double *fw, double *Un, double *B,
                         int64_t *first_bad)
{
    double *Bl = B ? B : (double *)malloc((size_t)(3 * n_nodes) * sizeof(double));
    int rc = oracle_fe_force(n_nodes, n_elems, conn, X, x, fibers, mat_id, mats, Bl, NULL, NULL, first_bad);
    if (rc) { if (!B) free(Bl); return rc; }
    if (!nsub) {
        oracle_spread(g, n_nodes, x, Bl, fu, fv, fw, 0);
        oracle_interp(g, n_nodes, x, u, v, w, Un);
    } else {
        int64_t P = oracle_num_points(n_nodes, n_elems, nsub);
        double *xp = (double *)malloc((size_t)(3 * P) * sizeof(double));
        double *Gp = (double *)malloc((size_t)(3 * P) * sizeof(double));
        double *Up = (double *)malloc((size_t)(3 * P) * sizeof(double));
        double *Wp = (double *)malloc((size_t)P * sizeof(double));
        double *wa = (double *)malloc((size_t)n_nodes * sizeof(double));
        rc = oracle_points(n_nodes, n_elems, conn, X, x, nsub, xp, Wp, wa);
        oracle_prolong(n_nodes, n_elems, conn, nsub, wa, Wp, Bl, Gp);
        oracle_spread(g, P, xp, Gp, fu, fv, fw, 0);
        oracle_interp(g, P, xp, u, v, w, Up);
        oracle_restrict(n_nodes, n_elems, conn, nsub, wa, Wp, Up, Un);
        free(xp); free(Gp); free(Up); free(Wp); free(wa);
    }
    if (!B) free(Bl);
    return rc;
}
