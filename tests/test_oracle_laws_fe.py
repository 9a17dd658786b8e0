"""Pins for the oracle's constitutive laws, FE nodal force, force points and projection (no GPU).

SURVEY.md §8(c) pins 1-4, 11 and readings A2, A3, A6, A9-A13: closed-form stresses, P = dPsi/dF
and B = -dE/dx by central differences, objectivity, HO -> neo-Hookean reduction, fibre terms
switching off in compression, zero force under rigid motion, zero net force/torque, patch test,
single-cube closed form, lumped weights summing to the volume, prolong/restrict transposes.
"""
import os

import numpy as np
import pytest

from helpers import distorted_block, rotation
from paper_2503_22695_b200 import workloads as W

GOLD = os.path.join(os.path.dirname(__file__), "golden")
NH = W.material(W.LAW_NEOHOOKEAN, a=1e4, kappa=1e6)
HO = W.material(W.LAW_HO, **W.HO_LV)
# PAPER.md Table 2 (L351-366) parameter set, dyn/cm^2 -- a free extra test vector (A8)
HO_T2 = W.material(W.LAW_HO, a=2244.87, b=1.6215, af=24267.0, bf=1.8268, as_=5562.38, bs=0.7746,
                   afs=3905.16, bfs=1.695, kappa=1e6)


def _fd_P(orc, mat, F, ef, es, eps=1e-6):
    P = np.zeros((3, 3))
    for c in range(3):
        for K in range(3):
            Fp, Fm = F.copy(), F.copy()
            Fp[c, K] += eps
            Fm[c, K] -= eps
            P[c, K] = (orc.pk1(mat, Fp, ef, es)[1] - orc.pk1(mat, Fm, ef, es)[1]) / (2 * eps)
    return P


def test_neo_hookean_closed_forms(orc):
    rows = {}
    for line in open(os.path.join(GOLD, "nh_closed_form.txt")):
        if not line.startswith("#"):
            p = line.split()
            rows[p[0]] = list(map(float, p[1:]))
    l = 1.2
    P, psi = orc.pk1(W.material(0, a=1e4, kappa=123.0), np.diag([l, l ** -0.5, l ** -0.5]))
    assert np.allclose(np.diag(P), rows["isochoric_uniaxial_l1.2_mu1e4"], rtol=1e-13)
    assert np.max(np.abs(P - np.diag(np.diag(P)))) < 1e-9
    assert abs(psi - 0.5e4 * (l * l + 2 / l - 3)) < 1e-10 * psi          # mu/2 (Ibar1 - 3), J = 1
    P, psi = orc.pk1(NH, np.diag([1.1, 1.0, 1.0]))
    assert np.allclose(np.diag(P), rows["diag_1.1_1_1_mu1e4_kappa1e6"], rtol=1e-13)
    # pure dilation: Ibar1 = 3 -> only U(J) = kappa/2 (ln J)^2; P = kappa lnJ / lam I
    lam = 1.05
    P, psi = orc.pk1(NH, lam * np.eye(3))
    assert abs(psi - 0.5e6 * (3 * np.log(lam)) ** 2) < 1e-12 * psi
    assert np.allclose(P, 1e6 * 3 * np.log(lam) / lam * np.eye(3), rtol=1e-12, atol=1e-7)
    # identity is stress free
    P, psi = orc.pk1(NH, np.eye(3))
    assert np.max(np.abs(P)) < 1e-9 and abs(psi) < 1e-12


def test_ho_closed_forms(orc):
    m = HO
    ex, ey = np.array([1.0, 0, 0]), np.array([0, 1.0, 0])
    # isochoric uniaxial stretch along the fibre: I4f = l^2, I4s = 1/l < 1 (switched off, A9), I8 = 0
    l = 1.15
    F = np.diag([l, l ** -0.5, l ** -0.5])
    I1 = l * l + 2 / l
    P, psi = orc.pk1(m, F, ex, ey)
    e_iso = np.exp(m["b"] * (I1 - 3))
    e_f = np.exp(m["bf"] * (l * l - 1) ** 2)
    assert abs(psi - (m["a"] / (2 * m["b"]) * e_iso + m["af"] / (2 * m["bf"]) * (e_f - 1))) < 1e-14 * psi
    P11 = m["a"] * e_iso * (l - I1 / (3 * l)) + 2 * m["af"] * (l * l - 1) * e_f * l
    P22 = m["a"] * e_iso * (l ** -0.5 - I1 / 3 * l ** 0.5)
    assert np.allclose(np.diag(P), [P11, P22, P22], rtol=1e-13)
    # simple shear F = I + g ex (x) ey: F ef = ex, F es = g ex + ey -> I8 = g, I4s = 1 + g^2, J = 1
    gam = 0.3
    F = np.eye(3)
    F[0, 1] = gam
    P, psi = orc.pk1(m, F, ex, ey)
    I1 = 3 + gam * gam
    e_iso = np.exp(m["b"] * gam * gam)
    e_s = np.exp(m["bs"] * gam ** 4)
    e_fs = np.exp(m["bfs"] * gam * gam)
    psi_exp = (m["a"] / (2 * m["b"]) * e_iso + m["as_"] / (2 * m["bs"]) * (e_s - 1)
               + m["afs"] / (2 * m["bfs"]) * (e_fs - 1))
    assert abs(psi - psi_exp) < 1e-14 * psi
    Finv_T = np.eye(3)
    Finv_T[1, 0] = -gam
    Fs = np.array([gam, 1.0, 0])
    P_exp = (m["a"] * e_iso * (F - I1 / 3 * Finv_T) + 2 * m["as_"] * gam * gam * e_s * np.outer(Fs, ey)
             + m["afs"] * gam * e_fs * (np.outer(ex, ey) + np.outer(Fs, ex)))
    assert np.allclose(P, P_exp, rtol=1e-13, atol=1e-15)


@pytest.mark.parametrize("mat", [NH, HO, HO_T2], ids=["NH", "HO", "HO_table2"])
def test_P_is_dPsi_dF_and_objective(orc, mat):
    rng = np.random.default_rng(0)
    for trial in range(6):
        F = np.eye(3) + 0.25 * rng.normal(size=(3, 3))
        if np.linalg.det(F) < 0.3:
            continue
        ef = rng.normal(size=3)
        ef /= np.linalg.norm(ef)
        es = np.cross(ef, rng.normal(size=3))
        es /= np.linalg.norm(es)
        P, psi = orc.pk1(mat, F, ef, es)
        Pfd = _fd_P(orc, mat, F, ef, es)
        assert np.max(np.abs(P - Pfd)) < 2e-8 * np.max(np.abs(P)), trial        # A2, A3
        # P F^T symmetric (Cauchy stress symmetric; fails for the cross term as printed, A3)
        S = P @ F.T
        assert np.max(np.abs(S - S.T)) < 1e-13 * np.max(np.abs(S))
        # spatial objectivity: Psi(QF) = Psi(F), P(QF) = Q P(F)
        Q = rotation(trial)
        Pq, psiq = orc.pk1(mat, Q @ F, ef, es)
        assert abs(psiq - psi) < 1e-13 * abs(psi)
        assert np.max(np.abs(Pq - Q @ P)) < 1e-12 * np.max(np.abs(P))
        # material frame (A11): rotating F and the fibres together leaves Psi unchanged
        R = rotation(trial + 100)
        _, psir = orc.pk1(mat, F @ R.T, R @ ef, R @ es)
        assert abs(psir - psi) < 1e-13 * abs(psi)


def test_ho_reduces_to_neo_hookean_and_compression_switch(orc):
    rng = np.random.default_rng(1)
    F = np.eye(3) + 0.2 * rng.normal(size=(3, 3))
    ef, es = np.array([0, 0, 1.0]), np.array([1.0, 0, 0])
    # A6: HO with b=0 and no fibre constants == NH
    P1, w1 = orc.pk1(W.material(W.LAW_HO, a=1e4, b=0.0, kappa=1e6), F, ef, es)
    P0, w0 = orc.pk1(NH, F)
    assert np.array_equal(P1, P0) and w1 == w0
    # b -> 0 limit is continuous
    P2, _ = orc.pk1(W.material(W.LAW_HO, a=1e4, b=1e-9, kappa=1e6), F, ef, es)
    assert np.max(np.abs(P2 - P0)) < 1e-7 * np.max(np.abs(P0))
    # A9: fibres in compression (I4 < 1) contribute exactly nothing
    Fc = np.diag([1.3, 1.0, 0.7])                    # ef = ez compressed, es = ex stretched
    m_f = W.material(W.LAW_HO, a=0.24, b=5.08, af=1.46, bf=4.15, kappa=1e3)
    m_0 = W.material(W.LAW_HO, a=0.24, b=5.08, kappa=1e3)
    Pf, wf = orc.pk1(m_f, Fc, ef, es)
    Pn, wn = orc.pk1(m_0, Fc, ef, es)
    assert np.array_equal(Pf, Pn) and wf == wn
    # inverted element is an error (A10)
    with pytest.raises(ValueError):
        orc.pk1(NH, np.diag([1.0, 1.0, -1.0]))


def test_single_cube_element_closed_form(orc):
    # one unit-cube element under homogeneous x = F0 X: B_a,c = -sum_I P_cI xi_a,I / 4
    conn = np.arange(8, dtype=np.int32).reshape(1, 8)
    X = np.array([[a & 1, (a >> 1) & 1, (a >> 2) & 1] for a in range(8)], dtype=np.float64).T
    F0 = np.array([[1.1, 0.3, 0.0], [0.0, 0.9, -0.2], [0.1, 0.0, 1.05]])
    x = F0 @ X + np.array([[0.3], [0.1], [-0.2]])
    ef, es = np.array([0.6, 0.8, 0.0]), np.array([-0.8, 0.6, 0.0])
    fib = np.concatenate([ef, es]).reshape(6, 1)
    for mat in (NH, HO):
        r = orc.fe_force(conn, X, x, fib, np.zeros(1, np.int32), [mat])
        P, psi = orc.pk1(mat, F0, ef, es)
        xi = 2 * X - 1
        Bexp = -(P @ xi) / 4
        assert np.max(np.abs(r["B"] - Bexp)) < 1e-13 * np.max(np.abs(Bexp))
        assert abs(r["energy"] - psi) < 1e-13 * abs(psi)
        assert abs(r["minJ"] - np.linalg.det(F0)) < 1e-14


@pytest.mark.parametrize("mat", [NH, HO], ids=["NH", "HO"])
def test_force_is_minus_energy_gradient(orc, mat):
    # pin 1: B = -dE/dx by central differences on a distorted mesh
    conn, X, x, fib = distorted_block(3, 3, 2, seed=1)
    mid = np.zeros(conn.shape[0], np.int32)
    B = orc.fe_force(conn, X, x, fib, mid, [mat])["B"]
    d = 0.1 * 1e-6
    rng = np.random.default_rng(0)
    nn = X.shape[1]
    worst = 0.0
    for _ in range(25):
        c, n = int(rng.integers(3)), int(rng.integers(nn))
        xp_, xm_ = x.copy(), x.copy()
        xp_[c, n] += d
        xm_[c, n] -= d
        Ep = orc.fe_force(conn, X, xp_, fib, mid, [mat])["energy"]
        Em = orc.fe_force(conn, X, xm_, fib, mid, [mat])["energy"]
        fd = -(Ep - Em) / (2 * d)
        worst = max(worst, abs(fd - B[c, n]) / np.max(np.abs(B)))
    assert worst < 5e-8, worst


def test_rigid_motion_balance_and_patch(orc):
    conn, X, x, fib = distorted_block(4, 3, 3, seed=2)
    ne, nn = conn.shape[0], X.shape[1]
    mid = np.zeros(ne, np.int32)
    h = 0.1
    for mat in (NH, HO):
        kappa = mat["kappa"]
        # pin 2: rigid translation + rotation of the reference -> no force
        Q = rotation(5)
        xr = Q @ X + np.array([[0.4], [-0.2], [0.7]])
        # fibres are material vectors, they do not rotate with the body
        B = orc.fe_force(conn, X, xr, fib, mid, [mat])["B"]
        assert np.max(np.abs(B)) < 1e-12 * kappa * h * h
        # zero net force and torque for ANY deformation (internal forces)
        B = orc.fe_force(conn, X, x, fib, mid, [mat])["B"]
        scale = np.abs(B).sum()
        assert np.max(np.abs(B.sum(axis=1))) < 1e-14 * scale
        tq = np.cross(x.T, B.T).sum(axis=0)
        assert np.max(np.abs(tq)) < 1e-14 * scale
    # pin 4 (A12): homogeneous x = F0 X on a distorted mesh, homogeneous material (constant fibres)
    # -> interior nodal forces vanish
    F0 = np.array([[1.2, 0.1, 0.0], [0.05, 0.95, 0.1], [0.0, -0.1, 1.1]])
    fibc = np.tile(np.array([[0.6], [0.0], [0.8], [0.0], [1.0], [0.0]]), (1, ne))
    B = orc.fe_force(conn, X, F0 @ X, fibc, mid, [HO])["B"]
    cnt = np.bincount(conn.ravel(), minlength=nn)
    interior = cnt == 8
    assert interior.sum() > 0
    assert np.max(np.abs(B[:, interior])) < 1e-12 * np.max(np.abs(B[:, ~interior]))
    # A10: an inverted element is reported with its id
    xi = x.copy()
    n0 = conn[7, 0]
    xi[:, n0] = x[:, conn[7, 7]] + (x[:, conn[7, 7]] - x[:, n0])       # push node 0 through node 7
    r = orc.fe_force(conn, X, xi, fib, mid, [NH])
    assert r["rc"] == 1 and r["first_bad"] >= 0


def test_points_weights_prolong_restrict(orc):
    conn, X, x, fib = distorted_block(3, 2, 2, seed=3)
    ne, nn = conn.shape[0], X.shape[1]
    rng = np.random.default_rng(0)
    nsub = rng.integers(1, 5, size=(ne, 3)).astype(np.int32)
    xp, Wp, wa = orc.points(conn, X, x, nsub)
    P = int(np.prod(nsub, axis=1).sum())
    assert xp.shape == (3, P) and orc.num_points(nn, ne, nsub) == P
    # pin 11: sum w_a = sum W_s; with a 2x2x2 midpoint-free check on an undistorted box it is the volume
    assert abs(wa.sum() - Wp.sum()) < 1e-14 * Wp.sum()
    cb, Xb, _, _ = distorted_block(3, 2, 2, seed=3, ref_noise=0.0, cur_noise=0.0)
    _, Wb, wb = orc.points(cb, Xb, Xb, nsub)
    assert abs(Wb.sum() - 0.3 * 0.3 * 0.2) < 1e-15
    interior_w = wb[np.bincount(cb.ravel(), minlength=nn) == 8]
    assert interior_w.size == 0 or np.allclose(interior_w, 0.1 * 0.15 * 0.1)
    # affine map is reproduced at every sub-point: x_s = A X_s + c  (X_s from the same routine)
    A = np.array([[1.1, 0.2, 0.0], [0.0, 0.9, 0.1], [0.3, 0.0, 1.2]])
    Xs, _, _ = orc.points(conn, X, X, nsub)
    xs, _, _ = orc.points(conn, X, A @ X + 0.5, nsub)
    assert np.max(np.abs(xs - (A @ Xs + 0.5))) < 1e-15
    # sub-point ordering s = m1 + n1 (m2 + n2 m3) on the unit cube: X_s is the cell midpoint
    c1 = np.arange(8, dtype=np.int32).reshape(1, 8)
    X1 = np.array([[a & 1, (a >> 1) & 1, (a >> 2) & 1] for a in range(8)], dtype=np.float64).T
    ns = np.array([[2, 3, 4]], dtype=np.int32)
    Xs1, W1, _ = orc.points(c1, X1, X1, ns)
    m3, m2, m1 = np.meshgrid(np.arange(4), np.arange(3), np.arange(2), indexing="ij")
    exp = np.stack([(m1.ravel() + .5) / 2, (m2.ravel() + .5) / 3, (m3.ravel() + .5) / 4])
    assert np.max(np.abs(Xs1 - exp)) < 1e-16 and np.allclose(W1, 1 / 24, rtol=1e-15)
    # prolongation conserves the total force (partition of unity); a constant force density is exact
    B = rng.normal(size=(3, nn))
    Gp = orc.prolong(conn, nsub, wa, Wp, B)
    assert np.max(np.abs(Gp.sum(axis=1) - B.sum(axis=1))) < 1e-13 * np.abs(B).sum()
    Gc = orc.prolong(conn, nsub, wa, Wp, wa[None, :] * np.array([[2.0], [-1.0], [0.5]]))
    assert np.max(np.abs(Gc - Wp[None, :] * np.array([[2.0], [-1.0], [0.5]]))) < 1e-15
    # restriction is the transpose: sum_s G_s.U_s = sum_a B_a.U_a ; constants are preserved
    Up = rng.normal(size=(3, P))
    Un = orc.restrict(conn, nsub, wa, Wp, Up)
    assert abs(np.sum(Gp * Up) - np.sum(B * Un)) < 1e-13 * abs(np.sum(B * Un))
    Uc = orc.restrict(conn, nsub, wa, Wp, np.tile(np.array([[1.5], [0.0], [-2.0]]), (1, P)))
    assert np.max(np.abs(Uc - np.array([[1.5], [0.0], [-2.0]]))) < 1e-15
    # nodal rule of PAPER.md L241: w_q = int phi_q, sums to the volume of the mesh
    wq = orc.nodal_weights(cb, Xb)
    assert abs(wq.sum() - 0.3 * 0.3 * 0.2) < 1e-15


def test_nodal_weights_node_by_node_on_a_regular_block(orc):
    """w_q = int phi_q dX on an undistorted n1 x n2 x n3 block of bricks d1 x d2 x d3: the
    trilinear hat of a node integrates to d1 d2 d3 / 8 over each brick it belongs to, so w_q = V_brick
    k_q / 8 with k_q = number of bricks at the node: 8 inside, 4 on a face, 2 on an edge, 1 at a corner.
    A weight assigned to the wrong node fails this; the sum alone would not."""
    n1, n2, n3 = 3, 4, 2
    conn, (N1, N2, N3) = W.block_connectivity(n1, n2, n3)
    d = np.array([0.11, 0.07, 0.13])
    k, j, i = np.meshgrid(np.arange(N3), np.arange(N2), np.arange(N1), indexing="ij")
    X = np.stack([0.2 + i.ravel() * d[0], 0.3 + j.ravel() * d[1], 0.1 + k.ravel() * d[2]])
    wq = orc.nodal_weights(conn.astype(np.int32), X)
    per_axis = lambda idx, n: np.where((idx == 0) | (idx == n), 1, 2)          # bricks along one axis at the node
    kq = per_axis(i.ravel(), n1) * per_axis(j.ravel(), n2) * per_axis(k.ravel(), n3)
    assert np.max(np.abs(wq - d.prod() * kq / 8.0)) < 1e-16
    # and on a sheared block (affine map A): every weight scales by det A, node by node
    A = np.array([[1.0, 0.3, -0.1], [0.0, 0.9, 0.2], [0.05, 0.0, 1.1]])
    assert np.max(np.abs(orc.nodal_weights(conn.astype(np.int32), A @ X) - np.linalg.det(A) * wq)) < 1e-16


def test_coupling_step_composition_and_node_level_adjointness(orc):
    conn, X, x, fib = distorted_block(3, 3, 2, size=(0.3, 0.3, 0.2), origin=(0.35, 0.3, 0.4), seed=4)
    ne, nn = conn.shape[0], X.shape[1]
    nsub = np.tile(np.array([[2, 3, 2]], np.int32), (ne, 1))
    mid = np.zeros(ne, np.int32)
    n, h = 16, 1.0 / 16
    g = orc.make_grid(n, n, n, h)
    rng = np.random.default_rng(0)
    u, v, w = rng.normal(size=(3, n ** 3))
    out = orc.coupling_step(g, conn, X, fib, mid, nsub, [HO], x, u, v, w)
    # pieces
    B = orc.fe_force(conn, X, x, fib, mid, [HO])["B"]
    assert np.array_equal(out["B"], B)
    # pin 7: total spread force = total Lagrangian force = 0 for internal forces
    for f in (out["fu"], out["fv"], out["fw"]):
        assert abs(h ** 3 * f.sum()) < 1e-12 * np.abs(B).sum()
    # pin 6 (node level, A13): h^3 sum f.u = sum_a B_a . Un_a
    lhs = h ** 3 * (out["fu"] @ u + out["fv"] @ v + out["fw"] @ w)
    rhs = np.sum(B * out["Un"])
    assert abs(lhs - rhs) < 1e-12 * abs(rhs)
    # nodal mode reproduces PAPER.md L253-257 literally: points = nodes, spread B itself
    outn = orc.coupling_step(g, conn, X, fib, mid, None, [HO], x, u, v, w)
    fN = orc.spread(g, x, B)
    UN = orc.interp(g, x, u, v, w)
    assert np.array_equal(outn["fu"], fN[0]) and np.array_equal(outn["Un"], UN)


def test_generated_configs_are_valid(orc):
    # every synthetic config has positive Jacobians and moderate deformation
    for wl in (W.config1(), W.config2(), W.lv_small()):
        r = orc.fe_force(wl.conn, wl.X, wl.x, wl.fibers, wl.mat_id, wl.mats)
        assert r["rc"] == 0 and r["minJ"] > 0.2, (wl.name, r["minJ"])
        ef, es = wl.fibers[:3], wl.fibers[3:]
        assert np.allclose(np.linalg.norm(ef, axis=0), 1) and np.allclose(np.linalg.norm(es, axis=0), 1)
        assert np.max(np.abs(np.sum(ef * es, axis=0))) < 1e-9
        lo = np.array(wl.origin) + 4 * wl.h   # full-size 6h margins: tests/test_workloads.py
        hi = np.array(wl.origin) + (np.array([wl.nx, wl.ny, wl.nz]) - 4) * wl.h
        assert np.all(wl.x.min(axis=1) > lo) and np.all(wl.x.max(axis=1) < hi)


# ---- NEXT-2: the paper's other constitutive laws and the active stress ------------------------------
# Table 1 (L273-285)-like magnitudes for Eq.(7); Table 4 (L410-421) recast for Eq.(10)-(11)
MSR = W.material(W.LAW_MSR, a=8e4, af=1.6e5, bf=2.0e6, kappa=4e6)          # G_T, G_L, E_L
FR2 = W.material(W.LAW_FR2, a=2 * 1.21 * 7.99, b=7.99, af=24.23, bf=57.62, kappa=1e3)


@pytest.mark.parametrize("mat", [MSR, FR2], ids=["MSR_eq7", "FR2_eq10"])
def test_next2_laws_P_is_dPsi_dF_and_objective(orc, mat):
    rng = np.random.default_rng(5)
    for trial in range(6):
        F = np.eye(3) + 0.12 * rng.normal(size=(3, 3))
        ef = rng.normal(size=3)
        ef /= np.linalg.norm(ef)
        es = np.cross(ef, rng.normal(size=3))
        es /= np.linalg.norm(es)
        P, psi = orc.pk1(mat, F, ef, es)
        Pfd = _fd_P(orc, mat, F, ef, es)
        assert np.max(np.abs(P - Pfd)) < 2e-8 * np.max(np.abs(P)), trial       # Eq.(7) / Eq.(11) with A4
        S = P @ F.T
        assert np.max(np.abs(S - S.T)) < 1e-12 * np.max(np.abs(S))
        Q = rotation(trial)
        Pq, psiq = orc.pk1(mat, Q @ F, ef, es)
        assert abs(psiq - psi) < 1e-12 * max(abs(psi), 1e-30)
        assert np.max(np.abs(Pq - Q @ P)) < 1e-12 * np.max(np.abs(P))
    P, psi = orc.pk1(mat, np.eye(3), np.array([1.0, 0, 0]), np.array([0, 1.0, 0]))
    assert np.max(np.abs(P)) < 1e-9 * mat["kappa"] and abs(psi) < 1e-12          # stress-free reference


def test_next2_closed_forms(orc):
    ex, ey = np.array([1.0, 0, 0]), np.array([0, 1.0, 0])
    # Eq.(7) on F = diag(l, 1, 1), fibre along x: I4 = l^2, I5 = l^4;
    # P11 = iso11 + (G_T-G_L)(2l - 2l^3) + (E_L+G_T-4G_L)/2 (l^2-1) l, other entries = isotropic part
    l = 1.07
    F = np.diag([l, 1.0, 1.0])
    P, psi = orc.pk1(MSR, F, ex, ey)
    P_iso, psi_iso = orc.pk1(W.material(W.LAW_NEOHOOKEAN, a=MSR["a"], kappa=MSR["kappa"]), F)
    GT, GL, EL = MSR["a"], MSR["af"], MSR["bf"]
    add = (GT - GL) * (2 * l - 2 * l ** 3) + 0.5 * (EL + GT - 4 * GL) * (l * l - 1) * l
    expect = P_iso.copy()
    expect[0, 0] += add
    assert np.allclose(P, expect, rtol=1e-13, atol=1e-9)
    assert abs(psi - psi_iso - (0.5 * (GT - GL) * (2 * l * l - l ** 4 - 1) + 0.125 * (EL + GT - 4 * GL) * (l * l - 1) ** 2)) < 1e-9
    # Eq.(8)-(9) is the HO law with a = 2 C1, b = 0 and only the fibre family: same numbers as Eq.(9) typed out
    C1, af, bf, kap = 17.0, 31.0, 4.0, 1e3
    m = W.material(W.LAW_HO, a=2 * C1, b=0.0, af=af, bf=bf, kappa=kap)
    P, _ = orc.pk1(m, F, ex, ey)
    J, I1 = l, l * l + 2
    Fit = np.diag([1 / l, 1.0, 1.0])
    P9 = 2 * C1 * J ** (-2 / 3) * (F - I1 / 3 * Fit) + 2 * af * (l * l - 1) * np.exp(bf * (l * l - 1) ** 2) * l * np.outer(ex, ex) \
        + kap * np.log(J) * Fit
    assert np.allclose(P, P9, rtol=1e-13, atol=1e-12)
    # Eq.(11) has no tension switch: a compressed fibre pushes back (HO's I4* would give exactly zero)
    lc = 0.9
    Fc = np.diag([lc, 1.0, 1.0])
    Pc, _ = orc.pk1(FR2, Fc, ex, ey)
    Pc0, _ = orc.pk1(W.material(W.LAW_FR2, a=FR2["a"], b=FR2["b"], kappa=FR2["kappa"]), Fc, ex, ey)
    d = lc * lc - 1
    assert abs((Pc - Pc0)[0, 0] - 2 * FR2["af"] * d * np.exp(FR2["bf"] * d * d) * lc) < 1e-12
    assert (Pc - Pc0)[0, 0] < 0 and np.count_nonzero(Pc - Pc0) == 1


def test_active_stress_closed_form(orc):
    """L317-331: P^a = F S_a, S_a = T e_f (x) e_f, T = T_a (1 + 4.9 (sqrt(I4f) - 1))."""
    ex, ey = np.array([1.0, 0, 0]), np.array([0, 1.0, 0])
    Ta, l = 60.0, 1.15
    F = np.diag([l, 0.95, 1.0])
    passive = dict(HO)
    active = dict(HO, Ta=Ta)
    P0, w0 = orc.pk1(passive, F, ex, ey)
    P1, w1 = orc.pk1(active, F, ex, ey)
    expect = np.zeros((3, 3))
    expect[0, 0] = Ta * (1 + 4.9 * (l - 1)) * l
    assert np.allclose(P1 - P0, expect, rtol=0, atol=1e-12) and w1 == w0
    # general F and fibre: the added first Piola stress is T (F ef)(x)ef and keeps P F^T symmetric
    rng = np.random.default_rng(2)
    F = np.eye(3) + 0.2 * rng.normal(size=(3, 3))
    ef = rng.normal(size=3)
    ef /= np.linalg.norm(ef)
    es = np.cross(ef, rng.normal(size=3))
    es /= np.linalg.norm(es)
    dP = orc.pk1(active, F, ef, es)[0] - orc.pk1(passive, F, ef, es)[0]
    S = np.linalg.solve(F, dP)                                  # second Piola-Kirchhoff S_a = F^-1 P^a
    T = Ta * (1 + 4.9 * (np.linalg.norm(F @ ef) - 1))
    assert np.allclose(S, T * np.outer(ef, ef), rtol=1e-11, atol=1e-11)
    # at the reference configuration the active tension is T_a along the fibre
    assert np.allclose(orc.pk1(active, np.eye(3), ex, ey)[0], Ta * np.outer(ex, ex), atol=1e-10)


# ---- NEXT-3: P1 tetrahedra (the paper's valve meshes are tetrahedral, L372 / L447) ------------------
def _tet_block(seed=3):
    conn, X, x, fib = distorted_block(3, 3, 2, seed=seed, ref_noise=0.12, cur_noise=0.06)
    tets = W.tets_from_hexes(conn, X)
    rng = np.random.default_rng(seed)
    ef = rng.normal(size=(3, tets.shape[0]))
    ef /= np.linalg.norm(ef, axis=0)
    es = np.cross(ef.T, rng.normal(size=(tets.shape[0], 3))).T
    es /= np.linalg.norm(es, axis=0)
    return tets, X, x, np.concatenate([ef, es])


def test_tet_single_element_closed_form(orc):
    """Unit right tetrahedron, x = F0 X: the force on node a is -V P(F0) grad N_a with V = 1/6 and
    grad N = (-1,-1,-1), e_x, e_y, e_z."""
    X = np.array([[0.0, 1, 0, 0], [0, 0, 1, 0], [0, 0, 0, 1]])
    conn = np.array([[0, 1, 2, 3]], dtype=np.int32)
    F0 = np.array([[1.1, 0.05, 0.0], [0.0, 0.95, 0.1], [0.02, 0.0, 1.03]])
    x = F0 @ X
    out = orc.fe_force(conn, X, x, None, None, [NH])
    P, psi = orc.pk1(NH, F0)
    G = np.array([[-1.0, -1, -1], [1, 0, 0], [0, 1, 0], [0, 0, 1]]).T          # [I, a]
    assert np.allclose(out["B"], -(P @ G) / 6.0, rtol=1e-13, atol=1e-9)
    assert abs(out["energy"] - psi / 6.0) < 1e-12 * psi and abs(out["minJ"] - np.linalg.det(F0)) < 1e-14
    assert orc.fe_force(conn[:, [0, 2, 1, 3]], X, x, None, None, [NH])["rc"] == 1   # inverted reference


@pytest.mark.parametrize("mat", [NH, HO], ids=["NH", "HO"])
def test_tet_force_is_minus_energy_gradient_and_balances(orc, mat):
    tets, X, x, fib = _tet_block()
    out = orc.fe_force(tets, X, x, fib, None, [mat])
    assert out["rc"] == 0 and out["minJ"] > 0.3
    B = out["B"]
    rng = np.random.default_rng(0)
    eps = 1e-6 * 0.1
    for _ in range(12):
        c, n = rng.integers(0, 3), rng.integers(0, X.shape[1])
        xp, xm = x.copy(), x.copy()
        xp[c, n] += eps
        xm[c, n] -= eps
        fd = -(orc.fe_force(tets, X, xp, fib, None, [mat])["energy"]
               - orc.fe_force(tets, X, xm, fib, None, [mat])["energy"]) / (2 * eps)
        assert abs(fd - B[c, n]) < 2e-7 * np.max(np.abs(B)), (c, n)
    assert np.max(np.abs(B.sum(axis=1))) < 1e-12 * np.max(np.abs(B))                       # no net force
    assert np.max(np.abs(np.cross(x.T, B.T).sum(axis=0))) < 1e-11 * np.max(np.abs(B))      # no net torque


def test_tet_rigid_motion_patch_and_volume(orc):
    tets, X, x, fib = _tet_block(seed=4)
    # total volume of the 6-tet split against the hex oracle's lumped weights of the same block
    conn_hex, Xh, _, _ = distorted_block(3, 3, 2, seed=4, ref_noise=0.12, cur_noise=0.06)
    vol_hex = orc.nodal_weights(conn_hex, Xh).sum()
    P = X[:, tets]
    vol_tet = np.einsum("in,in->n", np.cross((P[:, :, 1] - P[:, :, 0]).T, (P[:, :, 2] - P[:, :, 0]).T).T,
                        P[:, :, 3] - P[:, :, 0]).sum() / 6.0
    assert vol_tet > 0 and abs(vol_tet - vol_hex) < 0.02 * vol_hex   # planar-face split vs trilinear faces: close, not equal
    # rigid motion: zero force
    Q, t = rotation(5), np.array([[0.3], [-0.2], [0.1]])
    B = orc.fe_force(tets, X, Q @ X + t, fib, None, [HO])["B"]
    assert np.max(np.abs(B)) < 1e-12 * HO["kappa"] * 0.1 ** 2
    # patch test: homogeneous deformation -> every node not on the boundary of the block is in balance
    F0 = np.array([[1.05, 0.08, -0.02], [0.01, 0.97, 0.05], [-0.03, 0.02, 1.04]])
    B = orc.fe_force(tets, X, F0 @ X, None, None, [NH])["B"]
    N1, N2, N3 = 4, 4, 3
    k, j, i = np.meshgrid(np.arange(N3), np.arange(N2), np.arange(N1), indexing="ij")
    interior = ((i > 0) & (i < N1 - 1) & (j > 0) & (j < N2 - 1) & (k > 0) & (k < N3 - 1)).ravel()
    assert interior.sum() == 4
    assert np.max(np.abs(B[:, interior])) < 1e-11 * np.max(np.abs(B[:, ~interior]))


# ---- NEXT-4: solid boundary loads (Table 3 "Solid boundary", L263, L303, L315, L425) ----------------
def _enclosed_volume(faces, x):
    """(1/3) closed-surface integral of x.n da, 2x2 Gauss per bilinear quad / centroid rule per triangle
    -- a formula of its own (divergence theorem), not the oracle's load integral."""
    V = 0.0
    g = 1 / np.sqrt(3)
    for f in faces:
        P = x[:, f]
        if len(f) == 3:
            n = np.cross(P[:, 1] - P[:, 0], P[:, 2] - P[:, 0])
            V += np.dot(P.mean(axis=1), n) / 2 / 3
        else:
            for xi in (-g, g):
                for et in (-g, g):
                    sx, se = np.array([-1, 1, 1, -1]), np.array([-1, -1, 1, 1])
                    N = 0.25 * (1 + sx * xi) * (1 + se * et)
                    tx = P @ (0.25 * sx * (1 + se * et))
                    te = P @ (0.25 * (1 + sx * xi) * se)
                    V += np.dot(P @ N, np.cross(tx, te)) / 3
    return V


@pytest.mark.parametrize("kind", ["hex", "tet"])
def test_boundary_loads_pins(orc, kind):
    conn, X, x, _ = distorted_block(3, 3, 2, seed=12, ref_noise=0.1, cur_noise=0.06)
    if kind == "tet":
        conn = W.tets_from_hexes(conn, X)
    faces = W.boundary_faces(conn)
    assert faces.shape == ((2 * (9 + 6 + 6), 4) if kind == "hex" else (4 * (9 + 6 + 6), 3))
    nn = X.shape[1]
    zero = np.zeros((3, nn))
    # closed surface: the enclosed volume is the element volume (orientation is outward)
    vol = orc.nodal_weights(*distorted_block(3, 3, 2, seed=12, ref_noise=0.1, cur_noise=0.06)[:2]).sum()
    if kind == "tet":
        Pt = X[:, conn]
        vol = np.einsum("in,in->n", np.cross((Pt[:, :, 1] - Pt[:, :, 0]).T, (Pt[:, :, 2] - Pt[:, :, 0]).T).T,
                        Pt[:, :, 3] - Pt[:, :, 0]).sum() / 6
    assert abs(_enclosed_volume(faces, X) - vol) < 1e-12 * vol
    # pressure: follower load -p n da on a closed surface = -p dV/dx, no net force, no net torque
    p = 3.7
    Bp = orc.surface_loads(faces, X, x, None, p, zero)
    rng = np.random.default_rng(1)
    eps = 1e-6 * 0.1
    for _ in range(10):
        c, n = rng.integers(0, 3), rng.integers(0, nn)
        xp, xm = x.copy(), x.copy()
        xp[c, n] += eps
        xm[c, n] -= eps
        fd = -p * (_enclosed_volume(faces, xp) - _enclosed_volume(faces, xm)) / (2 * eps)
        assert abs(fd - Bp[c, n]) < 1e-7 * np.max(np.abs(Bp)), (c, n)
    assert np.max(np.abs(Bp.sum(axis=1))) < 1e-13 * np.max(np.abs(Bp)) * nn
    assert np.max(np.abs(np.cross(x.T, Bp.T).sum(axis=0))) < 1e-12 * np.max(np.abs(Bp)) * nn
    # traction: dead load q t0 per unit reference area: total = q t0 * area; on the flat undistorted block the
    # face x = const has area 0.3 x 0.2 and each of its 4 x 3 nodes gets its lumped share
    conn0, X0, _, _ = distorted_block(3, 3, 2, seed=12, ref_noise=0.0, cur_noise=0.0)
    if kind == "tet":
        conn0 = W.tets_from_hexes(conn0, X0)
    f0 = W.boundary_faces(conn0)
    right = f0[np.all(np.abs(X0[0, f0] - X0[0].max()) < 1e-12, axis=1)]
    qt0 = np.array([0.0, 6.25, 0.0])
    Bt = orc.surface_loads(right, X0, X0 * 1.3, qt0, 0.0, np.zeros_like(X0))       # current config is irrelevant
    assert np.allclose(Bt.sum(axis=1), qt0 * 0.3 * 0.2, rtol=1e-13, atol=1e-15)
    assert np.count_nonzero(Bt[1]) == 12 and np.all(Bt[[0, 2]] == 0)
    # tethers: penalty spring to the reference position, B = -dE/dx with E = kappa/2 sum |x-X|^2
    ids = np.unique(faces[np.all(np.abs(X[0, faces] - X[0].min()) < 0.05, axis=1)])[:7]
    Bk, E = orc.tethers(ids, X, x, 1e6, zero)
    assert np.allclose(Bk[:, ids], 1e6 * (X - x)[:, ids], rtol=1e-14) and np.count_nonzero(Bk) == 3 * ids.size
    assert abs(E - 0.5e6 * np.sum((x - X)[:, ids] ** 2)) < 1e-12 * E
    assert np.array_equal(orc.tethers(ids, X, X, 1e6, zero)[0], zero)


# ---- NEXT-3, second half: P2 tetrahedra (Cook's membrane is discretised with P2 elements, L265) -----
def _p2_block(seed=6, bend=0.0):
    conn, X, x, _ = distorted_block(3, 2, 2, seed=seed, ref_noise=0.1, cur_noise=0.0)
    tets = W.tets_from_hexes(conn, X)
    c10, X10 = W.p2_from_tets(tets, X)
    rng = np.random.default_rng(seed)
    if bend:                                              # curved edges: move the mid-edge nodes a little
        X10[:, X.shape[1]:] += bend * rng.uniform(-1, 1, (3, X10.shape[1] - X.shape[1]))
    x10 = X10 + 0.006 * rng.uniform(-1, 1, X10.shape)
    return c10, X10, x10


def test_p2_single_element_closed_form(orc):
    """Straight-sided P2 tetrahedron under x = F0 X: int grad N_vertex = 0 and int grad N_(ab) =
    V (grad l_a + grad l_b), so the vertices carry no force and edge (ab) carries -V P (grad l_a + grad l_b)."""
    X4 = np.array([[0.0, 1.2, 0.1, 0.2], [0.0, 0.1, 0.9, 0.3], [0.0, 0.0, 0.2, 1.1]])
    c10, X10 = W.p2_from_tets(np.array([[0, 1, 2, 3]], dtype=np.int32), X4)
    F0 = np.array([[1.1, 0.05, 0.0], [0.0, 0.95, 0.1], [0.02, 0.0, 1.03]])
    out = orc.fe_force(c10, X10, F0 @ X10, None, None, [NH])
    P, psi = orc.pk1(NH, F0)
    D = np.stack([X4[:, 1] - X4[:, 0], X4[:, 2] - X4[:, 0], X4[:, 3] - X4[:, 0]], axis=1)
    V = np.linalg.det(D) / 6
    gl = np.linalg.inv(D)                                  # rows: grad l_1, grad l_2, grad l_3
    gl = np.vstack([-gl.sum(axis=0), gl])                  # grad l_0 = -(sum)
    B = out["B"]
    assert np.max(np.abs(B[:, :4])) < 1e-10 * np.max(np.abs(B))
    for k, (a, b) in enumerate([(0, 1), (1, 2), (0, 2), (0, 3), (1, 3), (2, 3)]):
        assert np.allclose(B[:, c10[0, 4 + k]], -V * P @ (gl[a] + gl[b]), rtol=1e-12, atol=1e-9)
    assert abs(out["energy"] - psi * V) < 1e-12 * psi * V


@pytest.mark.parametrize("mat", [NH, HO], ids=["NH", "HO"])
def test_p2_force_is_minus_energy_gradient_and_balances(orc, mat):
    c10, X10, x10 = _p2_block(bend=0.004)
    ne = c10.shape[0]
    rng = np.random.default_rng(3)
    ef = rng.normal(size=(3, ne))
    ef /= np.linalg.norm(ef, axis=0)
    es = np.cross(ef.T, rng.normal(size=(ne, 3))).T
    es /= np.linalg.norm(es, axis=0)
    fib = np.concatenate([ef, es])
    out = orc.fe_force(c10, X10, x10, fib, None, [mat])
    assert out["rc"] == 0 and out["minJ"] > 0.5
    B = out["B"]
    eps = 1e-7
    for _ in range(12):
        c, n = rng.integers(0, 3), rng.integers(0, X10.shape[1])
        xp, xm = x10.copy(), x10.copy()
        xp[c, n] += eps
        xm[c, n] -= eps
        fd = -(orc.fe_force(c10, X10, xp, fib, None, [mat])["energy"]
               - orc.fe_force(c10, X10, xm, fib, None, [mat])["energy"]) / (2 * eps)
        assert abs(fd - B[c, n]) < 5e-7 * np.max(np.abs(B)), (c, n)
    assert np.max(np.abs(B.sum(axis=1))) < 1e-11 * np.max(np.abs(B))
    assert np.max(np.abs(np.cross(x10.T, B.T).sum(axis=0))) < 1e-10 * np.max(np.abs(B))


def test_p2_rigid_motion_and_patch(orc):
    c10, X10, _ = _p2_block(seed=9)
    Q, t = rotation(6), np.array([[0.1], [0.4], [-0.3]])
    B = orc.fe_force(c10, X10, Q @ X10 + t, None, None, [HO])["B"]
    assert np.max(np.abs(B)) < 1e-12 * HO["kappa"] * 0.1 ** 2
    F0 = np.array([[1.04, 0.06, -0.02], [0.01, 0.98, 0.04], [-0.03, 0.02, 1.03]])
    B = orc.fe_force(c10, X10, F0 @ X10, None, None, [NH])["B"]
    # nodes strictly inside the block (vertices and mid-edge nodes): in balance under a homogeneous deformation
    lo, hi = X10.min(axis=1, keepdims=True), X10.max(axis=1, keepdims=True)
    conn_hex, Xh, _, _ = distorted_block(3, 2, 2, seed=9, ref_noise=0.1, cur_noise=0.0)
    faces = W.boundary_faces(W.tets_from_hexes(conn_hex, Xh))
    on_bnd = np.zeros(X10.shape[1], bool)
    on_bnd[np.unique(faces)] = True
    tets = c10[:, :4]
    pairs = np.array([[0, 1], [1, 2], [0, 2], [0, 3], [1, 3], [2, 3]])
    fe = {tuple(sorted(p)) for f in faces for p in ((f[0], f[1]), (f[1], f[2]), (f[0], f[2]))}
    for t_, row in zip(tets, c10):
        for k, (a, b) in enumerate(pairs):
            if tuple(sorted((t_[a], t_[b]))) in fe:
                on_bnd[row[4 + k]] = True
    assert (~on_bnd).sum() >= 5
    assert np.max(np.abs(B[:, ~on_bnd])) < 1e-10 * np.max(np.abs(B[:, on_bnd]))


# ---- NEXT-4 on P2 meshes: loads on 6-node (quadratic) faces, reading A27 ------------------------------
_T6_MONO = np.zeros((6, 3, 3))                            # N_a = sum_ij c[a,i,j] xi^i eta^j
_T6_MONO[0, 0, 0], _T6_MONO[0, 1, 0], _T6_MONO[0, 0, 1] = 1, -3, -3
_T6_MONO[0, 2, 0], _T6_MONO[0, 1, 1], _T6_MONO[0, 0, 2] = 2, 4, 2
_T6_MONO[1, 1, 0], _T6_MONO[1, 2, 0] = -1, 2
_T6_MONO[2, 0, 1], _T6_MONO[2, 0, 2] = -1, 2
_T6_MONO[3, 1, 0], _T6_MONO[3, 2, 0], _T6_MONO[3, 1, 1] = 4, -4, -4
_T6_MONO[4, 1, 1] = 4
_T6_MONO[5, 0, 1], _T6_MONO[5, 1, 1], _T6_MONO[5, 0, 2] = 4, -4, -4


def _pmul(a, b):
    out = np.zeros((a.shape[0] + b.shape[0] - 1, a.shape[1] + b.shape[1] - 1))
    for i in range(a.shape[0]):
        for j in range(a.shape[1]):
            out[i:i + b.shape[0], j:j + b.shape[1]] += a[i, j] * b
    return out


def _pint(a):
    """integral over the unit triangle: xi^i eta^j -> i! j! / (i + j + 2)!"""
    from math import factorial as f
    return sum(a[i, j] * f(i) * f(j) / f(i + j + 2) for i in range(a.shape[0]) for j in range(a.shape[1]))


def _t6_volume_exact(faces, x):
    """(1/3) closed-surface integral of x.(x_xi x x_eta) over quadratic triangles, integrated exactly by
    polynomial algebra (the integrand has degree 4) -- no quadrature rule involved."""
    V = 0.0
    for f in faces:
        X3 = [np.tensordot(x[c, f], _T6_MONO, axes=(0, 0)) for c in range(3)]           # 3 polynomials [3,3]
        dxi = [np.pad(q[1:, :] * np.arange(1, 3)[:, None], ((0, 1), (0, 0))) for q in X3]
        det = [np.pad(q[:, 1:] * np.arange(1, 3)[None, :], ((0, 0), (0, 1))) for q in X3]
        cr = [_pmul(dxi[1], det[2]) - _pmul(dxi[2], det[1]), _pmul(dxi[2], det[0]) - _pmul(dxi[0], det[2]),
              _pmul(dxi[0], det[1]) - _pmul(dxi[1], det[0])]
        V += sum(_pint(_pmul(X3[c], cr[c])) for c in range(3)) / 3
    return V


def test_p2_face_loads_pins(orc):
    c10, X10, x10 = _p2_block(seed=8, bend=0.012)
    faces = W.boundary_faces(c10)
    assert faces.shape == (2 * 2 * (6 + 6 + 4), 6)
    nn = X10.shape[1]
    zero = np.zeros((3, nn))
    # orientation and bookkeeping: with straight edges the closed surface encloses the volume of the tetrahedra
    c10s, X10s, _ = _p2_block(seed=8, bend=0.0)
    Pt = X10s[:, c10s[:, :4]]
    vol = np.einsum("in,in->n", np.cross((Pt[:, :, 1] - Pt[:, :, 0]).T, (Pt[:, :, 2] - Pt[:, :, 0]).T).T,
                    Pt[:, :, 3] - Pt[:, :, 0]).sum() / 6
    assert abs(_t6_volume_exact(W.boundary_faces(c10s), X10s) - vol) < 1e-13 * vol
    # follower pressure on the curved closed surface: B = -p dV/dx (vertex and mid-edge nodes), no net force or torque
    p = 2.9
    Bp = orc.surface_loads(faces, X10, x10, None, p, zero)
    on_surf = np.unique(faces)
    rng = np.random.default_rng(4)
    eps = 1e-6
    for n in rng.choice(on_surf, 12, replace=False):
        c = rng.integers(0, 3)
        xp, xm = x10.copy(), x10.copy()
        xp[c, n] += eps
        xm[c, n] -= eps
        fd = -p * (_t6_volume_exact(faces, xp) - _t6_volume_exact(faces, xm)) / (2 * eps)
        assert abs(fd - Bp[c, n]) < 1e-8 * np.max(np.abs(Bp)), (c, n)
    assert np.max(np.abs(Bp.sum(axis=1))) < 1e-13 * np.max(np.abs(Bp)) * nn
    assert np.max(np.abs(np.cross(x10.T, Bp.T).sum(axis=0))) < 1e-12 * np.max(np.abs(Bp)) * nn
    interior = np.setdiff1d(np.arange(nn), on_surf)
    assert np.all(Bp[:, interior] == 0)
    # one flat straight-sided face, closed form: int N_vertex = 0 and int N_mid = A/3, so the vertices carry
    # nothing and every mid-edge node a third of the load -- pressure along the normal, traction along t0
    V3 = np.array([[0.1, 1.3, 0.4], [0.2, 0.3, 1.5], [0.0, 0.4, 0.1]])
    Xf = np.concatenate([V3, 0.5 * (V3[:, [0, 1, 2]] + V3[:, [1, 2, 0]])], axis=1)
    one = np.arange(6, dtype=np.int32)[None, :]
    nA = 0.5 * np.cross(V3[:, 1] - V3[:, 0], V3[:, 2] - V3[:, 0])                 # area vector
    Bf = orc.surface_loads(one, Xf, Xf, None, p, np.zeros((3, 6)))
    assert np.max(np.abs(Bf[:, :3])) < 1e-15
    assert np.allclose(Bf[:, 3:], np.repeat((-p * nA / 3)[:, None], 3, axis=1), rtol=1e-14, atol=1e-16)
    qt0 = np.array([0.5, -2.0, 1.25])
    Bq = orc.surface_loads(one, Xf, 1.7 * Xf, qt0, 0.0, np.zeros((3, 6)))          # current configuration is irrelevant
    assert np.max(np.abs(Bq[:, :3])) < 1e-15
    assert np.allclose(Bq[:, 3:], np.repeat((qt0 * np.linalg.norm(nA) / 3)[:, None], 3, axis=1), rtol=1e-14)
