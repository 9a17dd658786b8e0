"""Seeded synthetic workloads: the five configs of BASELINE.json as fixed in SURVEY.md §8(d).

This module serves both the CUDA path and the CPU oracle with *inputs only*.  It holds none of
the method's arithmetic (no shape-function evaluation of sub-points, no deformation gradient,
no stress, no delta kernel, no binning): it builds structured Q1-hex connectivity, node
coordinates from closed-form parametrisations, per-element fibre frames, material tables,
seeded perturbations and a seeded Fourier velocity field sampled at the MAC face locations
(the face locations are the storage convention of SURVEY.md §8 "Conventions", realising
PAPER.md L205, L211-217).

The paper's own workloads (image-based LV L301, porcine AV L349/L372, human MV L447, P2-tet
Cook's membrane L265) are not available; these stand in for them with the same shapes, sizes
and parameter magnitudes.

RNG recipe: numpy.random.default_rng([250322695, cfg, stream]); streams: 0 node noise,
1 smooth deformation, 2/3/4 Fourier modes of u/v/w.
"""
from __future__ import annotations

import hashlib
from dataclasses import dataclass, field

import numpy as np

SEED_ROOT = 250322695

LAW_NEOHOOKEAN = 0
LAW_HO = 1
LAW_MSR = 2          # modified standard reinforcing model, Eq.(7): a=G_T, af=G_L, bf=E_L
LAW_FR2 = 3          # fibre-reinforced model 2, Eq.(10)-(11): a=2 C10 C01, b=C01, af, bf (no tension switch)

# local node a = ia + 2*ja + 4*ka  (SURVEY.md §8 "Mesh")
_LOCAL = np.array([[a & 1, (a >> 1) & 1, (a >> 2) & 1] for a in range(8)], dtype=np.int64)


def material(law, a=0.0, b=0.0, af=0.0, bf=0.0, as_=0.0, bs=0.0, afs=0.0, bfs=0.0, kappa=0.0, Ta=0.0):
    """One row of the material table (ib_material in include/ibcouple.h). NH: a=mu, b=0."""
    return dict(law=int(law), a=float(a), b=float(b), af=float(af), bf=float(bf), as_=float(as_),
                bs=float(bs), afs=float(afs), bfs=float(bfs), kappa=float(kappa), Ta=float(Ta))


@dataclass
class Workload:
    name: str
    nx: int
    ny: int
    nz: int
    h: float
    origin: tuple
    conn: np.ndarray      # int32 [n_elems, 8]
    X: np.ndarray         # float64 [3, n_nodes] reference
    x: np.ndarray         # float64 [3, n_nodes] current
    fibers: np.ndarray    # float64 [6, n_elems] (e_f, e_s)
    mat_id: np.ndarray    # int32 [n_elems]
    nsub: np.ndarray      # int32 [n_elems, 3]
    mats: list
    u: np.ndarray         # float64 [nz*ny*nx], idx=(k*ny+j)*nx+i
    v: np.ndarray
    w: np.ndarray
    notes: dict = field(default_factory=dict)

    @property
    def n_nodes(self):
        return self.X.shape[1]

    @property
    def n_elems(self):
        return self.conn.shape[0]

    @property
    def n_points(self):
        return int(np.prod(self.nsub.astype(np.int64), axis=1).sum())

    @property
    def n_cells(self):
        return self.nx * self.ny * self.nz

    def sha256(self):
        """SHA-256 of every array, so oracle and GPU provably saw the same bytes."""
        out = {}
        for k in ("conn", "X", "x", "fibers", "mat_id", "nsub", "u", "v", "w"):
            out[k] = hashlib.sha256(np.ascontiguousarray(getattr(self, k)).tobytes()).hexdigest()[:16]
        return out


# --------------------------------------------------------------------------------------------
# structured blocks
# --------------------------------------------------------------------------------------------
def block_connectivity(n1, n2, n3, periodic2=False):
    """Structured n1 x n2 x n3 hex block. Node id (k*N2+j)*N1+i; direction 2 may wrap.
    Returns (conn [ne,8] int64, node index grids shape (N3,N2,N1))."""
    N1, N2, N3 = n1 + 1, (n2 if periodic2 else n2 + 1), n3 + 1
    ek, ej, ei = np.meshgrid(np.arange(n3), np.arange(n2), np.arange(n1), indexing="ij")
    ei, ej, ek = ei.ravel(), ej.ravel(), ek.ravel()
    conn = np.empty((ei.size, 8), dtype=np.int64)
    for a in range(8):
        ia, ja, ka = _LOCAL[a]
        jj = (ej + ja) % N2 if periodic2 else (ej + ja)
        conn[:, a] = ((ek + ka) * N2 + jj) * N1 + (ei + ia)
    return conn, (N1, N2, N3)


def tets_from_hexes(conn_hex, X):
    """Kuhn split of every hexahedron into 6 tetrahedra along the diagonal (local nodes 0-7), each
    ordered so that det [X1-X0, X2-X0, X3-X0] > 0.  Inputs only: the P1 meshes of NEXT-3 stand in for the
    paper's tetrahedral valve meshes (L372, L447)."""
    loc = np.array([[0, 1, 3, 7], [0, 3, 2, 7], [0, 2, 6, 7], [0, 6, 4, 7], [0, 4, 5, 7], [0, 5, 1, 7]])
    tets = conn_hex[:, loc].reshape(-1, 4).astype(np.int64)
    P = X[:, tets]                                   # [3, nt, 4]
    d = np.einsum("in,in->n", np.cross((P[:, :, 1] - P[:, :, 0]).T, (P[:, :, 2] - P[:, :, 0]).T).T,
                  P[:, :, 3] - P[:, :, 0])
    neg = d < 0
    tets[neg] = tets[neg][:, [0, 2, 1, 3]]
    return tets.astype(np.int32)


def p2_from_tets(tets, X):
    """Quadratic (10-node) tetrahedra from linear ones: one new node at the middle of every edge, local
    order 0-3 vertices, 4-9 edges (01, 12, 02, 03, 13, 23).  Returns (conn10 [nt,10], X10 [3, nn + n_edges]).
    Stands in for the paper's P2 Cook-membrane mesh (L265)."""
    pairs = np.array([[0, 1], [1, 2], [0, 2], [0, 3], [1, 3], [2, 3]])
    e = np.sort(tets[:, pairs].reshape(-1, 2), axis=1)
    uniq, inv = np.unique(e, axis=0, return_inverse=True)
    nn = X.shape[1]
    Xm = 0.5 * (X[:, uniq[:, 0]] + X[:, uniq[:, 1]])
    conn10 = np.concatenate([tets, nn + inv.reshape(-1, 6)], axis=1).astype(np.int32)
    return conn10, np.ascontiguousarray(np.concatenate([X, Xm], axis=1))


_HEX_FACES = np.array([[0, 4, 6, 2], [1, 3, 7, 5], [0, 1, 5, 4], [2, 6, 7, 3], [0, 2, 3, 1], [4, 5, 7, 6]])
_TET_FACES = np.array([[1, 2, 3], [0, 3, 2], [0, 1, 3], [0, 2, 1]])
# the same faces of a 10-node tetrahedron (p2_from_tets order): 3 vertices, then the middles of the edges
# (v0 v1), (v1 v2), (v2 v0) of the face
_TET10_FACES = np.array([[1, 2, 3, 5, 9, 8], [0, 3, 2, 7, 9, 6], [0, 1, 3, 4, 8, 7], [0, 2, 1, 6, 5, 4]])


def boundary_faces(conn):
    """Faces that belong to exactly one element, nodes in cyclic order with the normal pointing out of the
    element (right-handed elements): [nf,4] for hexahedra, [nf,3] for linear and [nf,6] for quadratic
    tetrahedra.  Inputs for the surface loads of NEXT-4 (pressure on the endocardium L303, traction on the
    Cook membrane's face L263)."""
    loc = {8: _HEX_FACES, 4: _TET_FACES, 10: _TET10_FACES}[conn.shape[1]]
    faces = conn[:, loc].reshape(-1, loc.shape[1])
    key = np.sort(faces[:, :3] if conn.shape[1] == 10 else faces, axis=1)
    _, inv, cnt = np.unique(key, axis=0, return_inverse=True, return_counts=True)
    return np.ascontiguousarray(faces[cnt[inv.ravel()] == 1]).astype(np.int32)


def _orient(conn, X):
    """Make every element right-handed (positive reference Jacobian at the centroid) by
    swapping the local xi_1 direction when the mean-edge triple product is negative."""
    P = X[:, conn]                                   # [3, ne, 8]
    e1 = sum(P[:, :, a] * (2 * _LOCAL[a, 0] - 1) for a in range(8))
    e2 = sum(P[:, :, a] * (2 * _LOCAL[a, 1] - 1) for a in range(8))
    e3 = sum(P[:, :, a] * (2 * _LOCAL[a, 2] - 1) for a in range(8))
    vol = np.einsum("in,in->n", np.cross(e1.T, e2.T).T, e3)
    neg = vol < 0
    conn = conn.copy()
    conn[neg] = conn[neg][:, [1, 0, 3, 2, 5, 4, 7, 6]]
    return conn, neg


def _unit(v):
    return v / np.linalg.norm(v, axis=0, keepdims=True)


# --------------------------------------------------------------------------------------------
# velocity field
# --------------------------------------------------------------------------------------------
def fourier_velocity(cfg, nx, ny, nz, h, M, K=4):
    """u,v,w = sum_m cos(2 pi k_m.(x-x0)/L + theta_m) at each component's face locations
    (u at (i, j+1/2, k+1/2)h etc.). Amplitude 1, integer k_m in [-K,K]^3 \\ {0}."""
    out = []
    offs = [(0.0, 0.5, 0.5), (0.5, 0.0, 0.5), (0.5, 0.5, 0.0)]
    for c in range(3):
        rng = np.random.default_rng([SEED_ROOT, cfg, 2 + c])
        km = np.zeros((M, 3), dtype=np.int64)
        for m in range(M):
            while True:
                k = rng.integers(-K, K + 1, size=3)
                if np.any(k != 0):
                    break
            km[m] = k
        theta = rng.uniform(0.0, 2 * np.pi, size=M)
        # separable evaluation: exp(i(kx X + ky Y + kz Z + theta))
        fx = (np.arange(nx) + offs[c][0]) / nx
        fy = (np.arange(ny) + offs[c][1]) / ny
        fz = (np.arange(nz) + offs[c][2]) / nz
        ks = np.arange(-K, K + 1)
        Ex = np.exp(2j * np.pi * np.outer(ks, fx))   # [2K+1, nx]
        Ey = np.exp(2j * np.pi * np.outer(ks, fy))
        Ez = np.exp(2j * np.pi * np.outer(ks, fz))
        C = np.zeros((2 * K + 1,) * 3, dtype=np.complex128)     # [kz, ky, kx]
        for m in range(M):
            C[km[m, 2] + K, km[m, 1] + K, km[m, 0] + K] += np.exp(1j * theta[m])
        A = np.einsum("zyx,xi->zyi", C, Ex)
        Bm = np.einsum("zyi,yj->zji", A, Ey)
        F = np.einsum("zji,zk->kji", Bm, Ez).real
        out.append(np.ascontiguousarray(F.reshape(-1)))
    return out


def _noise(cfg, shape, amp):
    rng = np.random.default_rng([SEED_ROOT, cfg, 0])
    return rng.uniform(-amp, amp, size=shape)


def _finish(name, cfg, n, h, origin, parts, mats, x, M, notes=None):
    """parts: list of (conn, X, fibers, mat_id, nsub) already with global node numbering in X order."""
    conn = np.concatenate([p[0] for p in parts]).astype(np.int32)
    X = np.concatenate([p[1] for p in parts], axis=1)
    fib = np.concatenate([p[2] for p in parts], axis=1)
    mat = np.concatenate([p[3] for p in parts]).astype(np.int32)
    nsub = np.concatenate([p[4] for p in parts]).astype(np.int32)
    u, v, w = fourier_velocity(cfg, n[0], n[1], n[2], h, M)
    return Workload(name, n[0], n[1], n[2], float(h), tuple(float(o) for o in origin),
                    np.ascontiguousarray(conn), np.ascontiguousarray(X), np.ascontiguousarray(x),
                    np.ascontiguousarray(fib), mat, np.ascontiguousarray(nsub), mats, u, v, w,
                    notes or {})


def _const_fibers(ne, ef=(1.0, 0.0, 0.0), es=(0.0, 1.0, 0.0)):
    f = np.empty((6, ne))
    f[0:3] = np.asarray(ef)[:, None]
    f[3:6] = np.asarray(es)[:, None]
    return f


# --------------------------------------------------------------------------------------------
# config 1: tiny slab
# --------------------------------------------------------------------------------------------
def config1(shift_cells=(0, 0, 0), nsub=(4, 4, 4)):
    cfg, n, h = 1, 32, 1.0 / 32
    conn, (N1, N2, N3) = block_connectivity(8, 8, 2)
    k, j, i = np.meshgrid(np.arange(N3), np.arange(N2), np.arange(N1), indexing="ij")
    X = np.stack([0.375 + i.ravel() * h, 0.375 + j.ravel() * h, 0.46875 + k.ravel() * h])
    X = X + (np.asarray(shift_cells, dtype=np.float64) * h)[:, None]
    x = X + _noise(cfg, X.shape, 0.1 * h)
    conn, _ = _orient(conn, X)
    ne = conn.shape[0]
    mats = [material(LAW_NEOHOOKEAN, a=1e4, kappa=1e6)]
    part = (conn, X, _const_fibers(ne), np.zeros(ne), np.tile(np.asarray(nsub), (ne, 1)))
    return _finish("C1-slab", cfg, (n, n, n), h, (0.0, 0.0, 0.0), [part], mats, x, M=8)


# --------------------------------------------------------------------------------------------
# config 2: Cook's-membrane-shaped plate
# --------------------------------------------------------------------------------------------
def config2():
    cfg, n, h = 2, 64, 1.0 / 64
    n1, n2, n3 = 32, 32, 4
    conn, (N1, N2, N3) = block_connectivity(n1, n2, n3)
    k, j, i = np.meshgrid(np.arange(N3), np.arange(N2), np.arange(N1), indexing="ij")
    r, s, q = i.ravel() / n1, j.ravel() / n2, k.ravel() / n3
    X = np.stack([0.48 * r, 0.44 * r + (0.44 - 0.28 * r) * s, 0.1 * q])
    lo, hi = X.min(axis=1), X.max(axis=1)
    X = X + (0.5 - 0.5 * (lo + hi))[:, None]          # centre the bounding box in [0,1]^3
    x = X + _noise(cfg, X.shape, 0.05 * h)
    conn, _ = _orient(conn, X)
    ne = conn.shape[0]
    mats = [material(LAW_NEOHOOKEAN, a=80.0, kappa=4e4)]
    part = (conn, X, _const_fibers(ne), np.zeros(ne), np.tile([2, 2, 4], (ne, 1)))
    return _finish("C2-cook", cfg, (n, n, n), h, (0.0, 0.0, 0.0), [part], mats, x, M=16)


# --------------------------------------------------------------------------------------------
# config 3 / 5: LV-shaped prolate shell
# --------------------------------------------------------------------------------------------
HO_LV = dict(a=0.24, b=5.08, af=1.46, bf=4.15, as_=0.87, bs=1.6, afs=0.3, bfs=1.3, kappa=1e3)
HO_LEAFLET = dict(a=19.336, b=7.99, af=24.23, bf=57.62, as_=0.0, bs=0.0, afs=0.0, bfs=0.0, kappa=1e3)


def _lv_shell(nt, nth, nnu):
    """Truncated prolate ellipsoidal shell, layer t in [0,1]: a=2.5+t, c=7+t (cm);
    x=a sin(nu) cos(th), y=a sin(nu) sin(th), z=-c cos(nu); nu from 0.05 pi to the z=+0.5 cut."""
    conn, (N1, N2, N3) = block_connectivity(nt, nth, nnu, periodic2=True)
    k, j, i = np.meshgrid(np.arange(N3), np.arange(N2), np.arange(N1), indexing="ij")
    t = i.ravel() / nt
    th = 2 * np.pi * j.ravel() / nth
    zeta = k.ravel() / nnu

    def pos(t, th, zeta):
        a, c = 2.5 + t, 7.0 + t
        nu0, nu1 = 0.05 * np.pi, np.arccos(-0.5 / c)
        nu = nu0 + (nu1 - nu0) * zeta
        return np.stack([a * np.sin(nu) * np.cos(th), a * np.sin(nu) * np.sin(th), -c * np.cos(nu)])

    X = pos(t, th, zeta)
    # fibres at element centroids (analytic frame from central differences of the closed form)
    ek, ej, ei = np.meshgrid(np.arange(nnu), np.arange(nth), np.arange(nt), indexing="ij")
    tc = (ei.ravel() + 0.5) / nt
    thc = 2 * np.pi * (ej.ravel() + 0.5) / nth
    zc = (ek.ravel() + 0.5) / nnu
    d = 1e-6
    dt = (pos(tc + d, thc, zc) - pos(tc - d, thc, zc)) / (2 * d)
    dth = (pos(tc, thc + d, zc) - pos(tc, thc - d, zc)) / (2 * d)
    e_t = _unit(dt)
    e_c = _unit(dth - np.sum(dth * e_t, axis=0) * e_t)
    e_l = np.cross(e_t.T, e_c.T).T
    alpha = np.deg2rad(60.0 - 120.0 * tc)            # +60 deg endo (t=0) -> -60 deg epi (t=1)
    e_f = np.cos(alpha) * e_c + np.sin(alpha) * e_l
    fib = np.concatenate([_unit(e_f), e_t])
    return conn, X, fib, (t, th, zeta)


def _lv_deform(cfg, X, params, h):
    t, th, zeta = params
    rng = np.random.default_rng([SEED_ROOT, cfg, 1])
    m = int(rng.integers(1, 4))
    nn = int(rng.integers(1, 3))
    th1, th2 = rng.uniform(0, 2 * np.pi, size=2)
    s = 1.0 + 0.05 * (1.0 + np.cos(m * th + th1) * np.cos(nn * np.pi * zeta + th2))
    x = X.copy()
    x[0] *= s
    x[1] *= s
    return x


def config3(nt=8, nth=128, nnu=96, n=128, nsub=(4, 4, 4), cfg=3, M=16):
    h = 10.0 / n
    origin = (-5.0, -5.0, -8.75)
    conn, X, fib, params = _lv_shell(nt, nth, nnu)
    x = _lv_deform(cfg, X, params, h) + _noise(cfg, X.shape, 0.05 * h)
    conn, _ = _orient(conn, X)
    ne = conn.shape[0]
    mats = [material(LAW_HO, **HO_LV)]
    part = (conn, X, fib, np.zeros(ne), np.tile(np.asarray(nsub), (ne, 1)))
    return _finish("C3-lv-shell", cfg, (n, n, n), h, origin, [part], mats, x, M=M)


# --------------------------------------------------------------------------------------------
# config 4: aortic-valve-like leaflets + root
# --------------------------------------------------------------------------------------------
def _leaflet(idx, n1=64, n2=48, n3=2, thick=0.05, x_base=3.3, height=1.4, r_wall=1.2,
             yc=2.0, zc=2.0):
    """Curved leaflet patch in the 120-degree sector idx around the x axis. (r,s,q) in [0,1]^3:
    r circumferential, s from the attachment on the wall to the free edge, q through thickness."""
    conn, (N1, N2, N3) = block_connectivity(n1, n2, n3)
    k, j, i = np.meshgrid(np.arange(N3), np.arange(N2), np.arange(N1), indexing="ij")
    r, s, q = i.ravel() / n1, j.ravel() / n2, k.ravel() / n3

    def mid(r, s):
        # attachment arc on the wall and a free edge that is a quadratic Bezier curve from
        # commissure to commissure dipping to 0.15 cm from the axis, blended by g(s) = s^1.5;
        # element sizes stay ~uniform (a polar parametrisation would shrink them near the axis)
        rw = r_wall - 0.02
        phi0 = np.deg2rad(120.0 * idx + 6.0)
        phi1 = phi0 + np.deg2rad(108.0)
        phim = 0.5 * (phi0 + phi1)
        A = rw * np.array([np.cos(phi0), np.sin(phi0)])
        Bp = rw * np.array([np.cos(phi1), np.sin(phi1)])
        em = np.array([np.cos(phim), np.sin(phim)])
        Cc = 2.0 * (0.15 * em - 0.25 * (A + Bp))
        phi = phi0 + (phi1 - phi0) * r
        att = rw * np.stack([np.cos(phi), np.sin(phi)])
        free = ((1 - r) ** 2)[None] * A[:, None] + (2 * r * (1 - r))[None] * Cc[:, None] + (r ** 2)[None] * Bp[:, None]
        gs = s ** 1.5
        yz = (1 - gs)[None] * att + gs[None] * free
        xx = x_base + height * s * (0.55 + 0.45 * np.sin(np.pi * r))
        return np.stack([xx, yc + yz[0], zc + yz[1]]), phi

    P, _ = mid(r, s)
    d = 1e-6
    dr = (mid(np.clip(r + d, 0, 1), s)[0] - mid(np.clip(r - d, 0, 1), s)[0])
    ds = (mid(r, np.clip(s + d, 0, 1))[0] - mid(r, np.clip(s - d, 0, 1))[0])
    # at s=0 the bulge derivative in s vanishes smoothly; both tangents stay non-degenerate
    nrm = _unit(np.cross(_unit(dr).T, _unit(ds).T).T)
    X = P + nrm * (thick * (q - 0.5))
    # fibres: circumferential (r) parameter direction at the element centroid
    ek, ej, ei = np.meshgrid(np.arange(n3), np.arange(n2), np.arange(n1), indexing="ij")
    rc, sc = (ei.ravel() + 0.5) / n1, (ej.ravel() + 0.5) / n2
    drc = mid(rc + d, sc)[0] - mid(rc - d, sc)[0]
    dsc = mid(rc, sc + d)[0] - mid(rc, sc - d)[0]
    e_f = _unit(drc)
    e_n = _unit(np.cross(e_f.T, _unit(dsc).T).T)
    e_s = np.cross(e_n.T, e_f.T).T
    return conn, X, np.concatenate([e_f, _unit(e_s)])


def _root(n1=4, n2=192, n3=64, r0=1.2, r1=1.35, x_lo=2.5, length=3.0, yc=2.0, zc=2.0):
    conn, (N1, N2, N3) = block_connectivity(n1, n2, n3, periodic2=True)
    k, j, i = np.meshgrid(np.arange(N3), np.arange(N2), np.arange(N1), indexing="ij")
    rad = r0 + (r1 - r0) * i.ravel() / n1
    th = 2 * np.pi * j.ravel() / n2
    X = np.stack([x_lo + length * k.ravel() / n3, yc + rad * np.cos(th), zc + rad * np.sin(th)])
    return conn, X


def config4():
    cfg, h = 4, 1.0 / 32
    n = (256, 128, 128)
    parts, off = [], 0
    mats = [material(LAW_HO, **HO_LEAFLET), material(LAW_NEOHOOKEAN, a=100.0, kappa=1e3)]
    Xs = []
    for l in range(3):
        conn, X, fib = _leaflet(l)
        conn, _ = _orient(conn, X)
        ne = conn.shape[0]
        parts.append((conn + off, X, fib, np.zeros(ne), np.tile([4, 2, 2], (ne, 1))))
        off += X.shape[1]
        Xs.append(X)
    conn, X = _root()
    conn, _ = _orient(conn, X)
    ne = conn.shape[0]
    parts.append((conn + off, X, _const_fibers(ne), np.ones(ne), np.tile([2, 1, 1], (ne, 1))))
    Xs.append(X)
    Xall = np.concatenate(Xs, axis=1)
    x = Xall + _noise(cfg, Xall.shape, 0.05 * h)
    return _finish("C4-av", cfg, n, h, (0.0, 0.0, 0.0), parts, mats, x, M=32)


# --------------------------------------------------------------------------------------------
# config 5: scaling sweep
# --------------------------------------------------------------------------------------------
def _annular_leaflet(idx, n1=128, n2=64, n3=2, thick=0.1):
    """Cone sector of 170 degrees hanging from r~2.2 at z~0.4 to r~1.0 at z~-1.0."""
    conn, (N1, N2, N3) = block_connectivity(n1, n2, n3)
    k, j, i = np.meshgrid(np.arange(N3), np.arange(N2), np.arange(N1), indexing="ij")
    r, s, q = i.ravel() / n1, j.ravel() / n2, k.ravel() / n3

    def mid(r, s):
        phi = np.deg2rad(180.0 * idx + 5.0 + 170.0 * r)
        rho = 2.2 - 1.2 * s
        z = 0.4 - 1.4 * s
        return np.stack([rho * np.cos(phi), rho * np.sin(phi), z])

    d = 1e-6
    P = mid(r, s)
    dr = mid(r + d, s) - mid(r - d, s)
    ds = mid(r, s + d) - mid(r, s - d)
    nrm = _unit(np.cross(_unit(dr).T, _unit(ds).T).T)
    X = P + nrm * (thick * (q - 0.5))
    ek, ej, ei = np.meshgrid(np.arange(n3), np.arange(n2), np.arange(n1), indexing="ij")
    rc, sc = (ei.ravel() + 0.5) / n1, (ej.ravel() + 0.5) / n2
    e_f = _unit(mid(rc + d, sc) - mid(rc - d, sc))
    e_s = _unit(mid(rc, sc + d) - mid(rc, sc - d))
    e_s = _unit(e_s - np.sum(e_s * e_f, axis=0) * e_f)
    return conn, X, np.concatenate([e_f, e_s])


def config5(level=3, sub=4, leaflets=None, n=256):
    """level 1: 4x64x48, 2: 8x128x96, 3: 16x256x192 (+ two annular leaflets at level 3)."""
    cfg = 5
    h = 10.0 / n
    origin = (-5.0, -5.0, -8.75)
    nt, nth, nnu = {1: (4, 64, 48), 2: (8, 128, 96), 3: (16, 256, 192)}[level]
    if leaflets is None:
        leaflets = (level == 3)
    conn, X, fib, params = _lv_shell(nt, nth, nnu)
    xs = _lv_deform(cfg, X, params, h)
    conn, _ = _orient(conn, X)
    ne = conn.shape[0]
    mats = [material(LAW_HO, **HO_LV), material(LAW_HO, **HO_LEAFLET)]
    parts = [(conn, X, fib, np.zeros(ne), np.tile([sub, sub, sub], (ne, 1)))]
    xparts = [xs]
    off = X.shape[1]
    if leaflets:
        for l in range(2):
            c2, X2, f2 = _annular_leaflet(l)
            c2, _ = _orient(c2, X2)
            ne2 = c2.shape[0]
            parts.append((c2 + off, X2, f2, np.ones(ne2), np.tile([sub, sub, sub], (ne2, 1))))
            xparts.append(X2.copy())
            off += X2.shape[1]
    x = np.concatenate(xparts, axis=1)
    x = x + _noise(cfg, x.shape, 0.05 * h)
    return _finish(f"C5-sweep-L{level}-s{sub}", cfg, (n, n, n), h, origin, parts, mats, x, M=64)


def make(cfg, **kw):
    return {1: config1, 2: config2, 3: config3, 4: config4, 5: config5}[int(cfg)](**kw)


def lv_small(nt=4, nth=32, nnu=24, n=64, nsub=(3, 2, 4)):
    """Reduced LV shell (HO law, curved geometry, periodic theta) sized for seconds-long oracle runs;
    ragged nsub so sub-point indexing is exercised with n1 != n2 != n3."""
    return config3(nt=nt, nth=nth, nnu=nnu, n=n, nsub=nsub, cfg=3, M=16)
