"""Pins for the oracle's delta kernel, spread, interpolation and bin/sort (no GPU).

What the paper and the mathematics fix (pins 5-10, W1):
closed-form phi values, Peskin's moment identities, the worked example W1, brute force over all
faces with minimum-image distances, adjointness, force conservation,
constant/linear reproduction, periodic-shift equivariance, tie on a cell boundary.
"""
import os

import numpy as np
import pytest

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def test_phi_closed_form_values(orc):
    for line in open(os.path.join(GOLD, "phi_closed_form.txt")):
        if line.startswith("#"):
            continue
        r, val = map(float, line.split())
        assert abs(orc.phi(r) - val) < 1e-16, (r, orc.phi(r), val)


def test_phi_peskin_identities(orc):
    # A1: sum_j phi(r-j)=1; sum_j (r-j)phi(r-j)=0; sum_j phi^2 = 3/8; even-j sum = odd-j sum = 1/2
    rng = np.random.default_rng(1)
    for r in np.concatenate([rng.uniform(-1, 1, 200), [0.0, 0.5, -0.5, 0.999999, 1e-12]]):
        js = np.arange(-4, 5)
        ph = np.array([orc.phi(r - j) for j in js])
        assert abs(ph.sum() - 1.0) < 4e-16
        assert abs(((r - js) * ph).sum()) < 4e-16
        assert abs((ph ** 2).sum() - 0.375) < 4e-16
        assert abs(ph[js % 2 == 0].sum() - 0.5) < 4e-16
        assert abs(ph[js % 2 == 1].sum() - 0.5) < 4e-16
    assert orc.phi(2.0000001) == 0.0 and orc.phi(-3.0) == 0.0
    # even and compactly supported, continuous at |r|=1 and |r|=2
    assert abs(orc.phi(0.3) - orc.phi(-0.3)) == 0.0
    assert abs(orc.phi(1 - 1e-9) - orc.phi(1 + 1e-9)) < 1e-8
    assert orc.phi(2 - 1e-9) < 1e-8


def test_worked_example_w1(orc):
    g = orc.make_grid(8, 8, 8, 0.125)
    xp = np.full((3, 1), 3.5 * 0.125)
    G = np.array([[1.0], [2.0], [-3.0]])
    f = orc.spread(g, xp, G)
    names = dict(fu=0, fv=1, fw=2)
    for line in open(os.path.join(GOLD, "w1_single_point.txt")):
        if line.startswith("#"):
            continue
        c, i, j, k, val = line.split()
        got = f[names[c]][(int(k) * 8 + int(j)) * 8 + int(i)]
        assert abs(got - float(val)) < 1e-13 * 512, (line, got)
    for c in range(3):
        assert np.count_nonzero(f[c]) == 36          # 4 x 3 x 3 (phi(2)=0 kills the fourth centre weight)
        assert abs(f[c].sum() * 0.125 ** 3 - G[c, 0]) < 1e-14
    # interpolating the field u[i,j,k] = i*h (x-coordinate of the u faces) returns x_p = 3.5h
    i = np.arange(8)
    u = np.broadcast_to(i * 0.125, (8, 8, 8)).reshape(-1).copy()
    U = orc.interp(g, xp, u, np.zeros(512), np.zeros(512))
    assert abs(U[0, 0] - 0.4375) < 1e-15


@pytest.mark.parametrize("n,origin", [((8, 8, 8), (0.0, 0.0, 0.0)), ((12, 8, 16), (-0.3, 0.2, 1.0))])
def test_spread_interp_match_brute_force(orc, n, origin):
    h = 0.1
    g = orc.make_grid(*n, h, origin)
    rng = np.random.default_rng(5)
    L = np.array(n) * h
    P = 23
    # points anywhere in the periodic box, including next to the wrap and outside [0,L)
    xp = np.asarray(origin)[:, None] + rng.uniform(-0.3, 1.3, (3, P)) * L[:, None]
    xp[:, 0] = np.asarray(origin) + 1e-9
    xp[:, 1] = np.asarray(origin) + L - 1e-9
    G = rng.normal(size=(3, P))
    f = orc.spread(g, xp, G)
    fb = orc.spread(g, xp, G, brute=True)
    for c in range(3):
        assert np.max(np.abs(f[c] - fb[c])) < 1e-13 * np.max(np.abs(fb[c]))
    ncell = n[0] * n[1] * n[2]
    u, v, w = rng.normal(size=(3, ncell))
    U = orc.interp(g, xp, u, v, w)
    Ub = orc.interp(g, xp, u, v, w, brute=True)
    assert np.max(np.abs(U - Ub)) < 1e-14 * np.max(np.abs(Ub))


def test_adjointness_and_conservation(orc):
    # <S G, u>_h = <G, S* u>;  A14: h^3 sum f = sum G
    n, h = (16, 8, 8), 0.05
    g = orc.make_grid(*n, h, (0.1, -0.2, 0.3))
    rng = np.random.default_rng(9)
    P = 300
    xp = rng.uniform(-1, 2, (3, P))
    G = rng.normal(size=(3, P))
    ncell = n[0] * n[1] * n[2]
    uvw = rng.normal(size=(3, ncell))
    f = orc.spread(g, xp, G)
    U = orc.interp(g, xp, *uvw)
    lhs = h ** 3 * sum(np.dot(f[c], uvw[c]) for c in range(3))
    rhs = np.sum(G * U)
    assert abs(lhs - rhs) < 1e-13 * abs(rhs)
    for c in range(3):
        assert abs(h ** 3 * f[c].sum() - G[c].sum()) < 1e-13 * np.abs(G[c]).sum()
    # accumulate flag adds to the existing field
    f2 = orc.spread(g, xp, G, f0=f)
    for c in range(3):
        assert np.max(np.abs(f2[c] - 2 * f[c])) < 1e-13 * np.max(np.abs(f[c]))


def test_constant_and_linear_reproduction(orc):
    n, h, org = (16, 16, 16), 0.0625, (0.0, 0.0, 0.0)
    g = orc.make_grid(*n, h, org)
    rng = np.random.default_rng(2)
    xp = rng.uniform(0.3, 0.7, (3, 50))             # away from the wrap
    k, j, i = np.meshgrid(np.arange(16), np.arange(16), np.arange(16), indexing="ij")
    # constant
    one = np.ones(16 ** 3)
    U = orc.interp(g, xp, 3.0 * one, -2.0 * one, 0.5 * one)
    assert np.max(np.abs(U - np.array([[3.0], [-2.0], [0.5]]))) < 1e-15
    # linear field a.x + b sampled at EACH component's own face locations (A17: a wrong staggering
    # offset or index origin breaks this)
    a = np.array([1.3, -0.7, 2.1])
    offs = [(0, .5, .5), (.5, 0, .5), (.5, .5, 0)]
    fld = []
    for c in range(3):
        xf = (i + offs[c][0]) * h
        yf = (j + offs[c][1]) * h
        zf = (k + offs[c][2]) * h
        fld.append((a[0] * xf + a[1] * yf + a[2] * zf + 0.25 * c).reshape(-1))
    U = orc.interp(g, xp, *fld)
    for c in range(3):
        assert np.max(np.abs(U[c] - (a @ xp + 0.25 * c))) < 2e-15


def test_periodic_shift_equivariance_and_boundary_tie(orc):
    n, h = (8, 8, 8), 0.125
    g = orc.make_grid(*n, h)
    rng = np.random.default_rng(3)
    xp = rng.uniform(0.2, 0.8, (3, 40))
    G = rng.normal(size=(3, 40))
    uvw = rng.normal(size=(3, 512))
    f = orc.spread(g, xp, G)
    U = orc.interp(g, xp, *uvw)
    sh = np.array([3, 5, 6])
    xs = xp + (sh * h)[:, None]                       # straddles the wrap
    fs = orc.spread(g, xs, G)
    for c in range(3):
        rolled = np.roll(f[c].reshape(8, 8, 8), shift=(sh[2], sh[1], sh[0]), axis=(0, 1, 2)).reshape(-1)
        assert np.max(np.abs(fs[c] - rolled)) < 1e-12 * np.max(np.abs(rolled))
    uvs = [np.roll(a.reshape(8, 8, 8), shift=(sh[2], sh[1], sh[0]), axis=(0, 1, 2)).reshape(-1) for a in uvw]
    Us = orc.interp(g, xs, *uvs)
    assert np.max(np.abs(Us - U)) < 1e-13
    # A19: a point exactly on a face/cell boundary -- nudging it either way changes nothing
    x0 = np.array([[0.25], [0.375], [0.5]])
    fa = orc.spread(g, x0 - 1e-13, np.ones((3, 1)))
    fb = orc.spread(g, x0 + 1e-13, np.ones((3, 1)))
    fc = orc.spread(g, x0, np.ones((3, 1)))
    for c in range(3):
        assert np.max(np.abs(fa[c] - fb[c])) < 1e-9 * np.max(np.abs(fc[c]))
        assert np.max(np.abs(fa[c] - fc[c])) < 1e-9 * np.max(np.abs(fc[c]))


def test_bin_sort_keys_and_stability(orc):
    # A21: key=((tz*nty+ty)*ntx+tx)*512+((lz*8+ly)*8+lx); stable sort (ties keep ascending id)
    n, h, org = (16, 8, 24), 0.25, (-1.0, 0.5, 2.0)
    g = orc.make_grid(*n, h, org)
    # points at the centres of known cells -> expected keys by integer construction
    cells = [(0, 0, 0), (15, 7, 23), (8, 0, 9), (7, 7, 7), (9, 1, 16), (8, 0, 9), (0, 0, 0)]
    xp = np.array([[org[d] + (c[d] + 0.5) * h for c in cells] for d in range(3)])
    key, perm = orc.bin_sort(g, xp)
    ntx, nty = n[0] // 8, n[1] // 8
    exp = [(((c[2] // 8) * nty + c[1] // 8) * ntx + c[0] // 8) * 512 + ((c[2] % 8) * 8 + c[1] % 8) * 8 + c[0] % 8
           for c in cells]
    assert key.tolist() == exp
    assert sorted(perm.tolist()) == list(range(len(cells)))
    ks = key[perm]
    assert np.all(np.diff(ks) >= 0)
    for a, b in zip(perm[:-1], perm[1:]):
        if key[a] == key[b]:
            assert a < b
    # periodic wrap: a point one box length away lands in the same cell
    xq = xp + (np.array(n) * h)[:, None] * np.array([[1], [-1], [2]])
    key2, _ = orc.bin_sort(g, xq)
    assert key2.tolist() == exp
    # random cloud vs numpy's stable argsort of the oracle's own keys (checks the sort, not the key)
    rng = np.random.default_rng(4)
    xr = np.asarray(org)[:, None] + rng.uniform(0, 1, (3, 5000)) * (np.array(n) * h)[:, None]
    k3, p3 = orc.bin_sort(g, xr)
    assert np.array_equal(p3, np.argsort(k3, kind="stable").astype(np.int32))
    # empty input
    k0, p0 = orc.bin_sort(g, np.zeros((3, 0)))
    assert k0.size == 0 and p0.size == 0


# ---- NEXT-4, second half: bounded (non-periodic) grid, reading A26 --------------------------------
def test_bounded_grid_truncates_supports(orc):
    """periodic=0: faces 0..n-1 exist, a support reaching outside is cut.  Pins: brute force over all
    faces with plain (not minimum-image) distances; identical to the periodic result away from the walls;
    a point half a cell from the wall keeps exactly the in-box share of its force (closed form)."""
    n, h, org = (8, 12, 8), 0.125, (-0.5, 0.0, 1.0)
    gb, gp = orc.make_grid(*n, h, org, periodic=0), orc.make_grid(*n, h, org, periodic=1)
    rng = np.random.default_rng(4)
    L = np.array(n) * h
    P = 60
    xp = np.asarray(org)[:, None] + rng.uniform(0.0, 1.0, (3, P)) * L[:, None]      # anywhere in the box, walls included
    G = rng.normal(size=(3, P))
    uvw = rng.normal(size=(3, n[0] * n[1] * n[2]))
    f, fb = orc.spread(gb, xp, G), orc.spread(gb, xp, G, brute=True)
    for c in range(3):
        assert np.max(np.abs(f[c] - fb[c])) < 1e-13 * np.max(np.abs(fb[c]))
    U, Ub = orc.interp(gb, xp, *uvw), orc.interp(gb, xp, *uvw, brute=True)
    assert np.max(np.abs(U - Ub)) < 1e-14 * np.max(np.abs(Ub))
    # adjointness survives the truncation (the same faces are dropped on both sides)
    lhs = h ** 3 * sum(np.dot(f[c], uvw[c]) for c in range(3))
    assert abs(lhs - np.sum(G * U)) < 1e-13 * np.sum(np.abs(G * U))
    # interior points (>= 2.5 h from every wall): same as periodic
    inner = np.asarray(org)[:, None] + 2.5 * h + rng.uniform(0, 1, (3, P)) * (L - 5 * h)[:, None]
    for a, b in zip(orc.spread(gb, inner, G), orc.spread(gp, inner, G)):
        assert np.array_equal(a, b)
    assert np.array_equal(orc.interp(gb, inner, *uvw), orc.interp(gp, inner, *uvw))
    # closed form: point at the centre of the corner cell (0,0,0), force (1,1,1).
    # face-aligned weights [a,b,b,a] at faces -1..2 -> the face -1 is outside: share 1-a, a = (2-sqrt2)/8;
    # centre-aligned weights [1/4,1/2,1/4,0] at -1..2 -> share 3/4
    x1 = (np.asarray(org) + 0.5 * h)[:, None]
    f1 = orc.spread(gb, x1, np.ones((3, 1)))
    al = (2 - np.sqrt(2)) / 8
    for c in range(3):
        assert abs(h ** 3 * f1[c].sum() - (1 - al) * 0.75 * 0.75) < 1e-15
    assert abs(h ** 3 * orc.spread(gp, x1, np.ones((3, 1)))[0].sum() - 1.0) < 1e-15       # periodic keeps all of it
