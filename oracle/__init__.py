"""CPU oracle (test infrastructure -- see the header of ib_oracle.c).

ctypes binding of oracle/ib_oracle.c.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package; the CUDA package never does.
It imports nothing from paper_2503_22695_b200.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ib_oracle.c")
_SO = os.path.join(_HERE, "liboracle.so")
_SO_OMP = os.path.join(_HERE, "liboracle_omp.so")      # same source with -fopenmp: bench.py's all-core timing leg only
_lib = None
_lib_omp = None


class Material(C.Structure):
    _fields_ = [("law", C.c_int32)] + [(k, C.c_double) for k in
                                       ("a", "b", "af", "bf", "as_", "bs", "afs", "bfs", "kappa", "Ta")]


class Grid(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
                ("h", C.c_double), ("x0", C.c_double), ("y0", C.c_double), ("z0", C.c_double),
                ("periodic", C.c_int32)]


def build(force=False):
    """gcc -O2, no -ffast-math, no FMA contraction (the binning formula must round like IEEE)."""
    if force or (not os.path.exists(_SO)) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-ffp-contract=off", "-fno-fast-math",
               "-o", _SO, _SRC, "-lm"]
        subprocess.check_call(cmd)
    return _SO


def build_omp(force=False):
    """The same source with -fopenmp (spreading with one private grid per thread, interpolation over the
    points): the all-core timing leg of bench.py.  Parity always uses the single-thread build."""
    if force or (not os.path.exists(_SO_OMP)) or os.path.getmtime(_SO_OMP) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-ffp-contract=off", "-fno-fast-math", "-fopenmp",
               "-o", _SO_OMP, _SRC, "-lm"]
        subprocess.check_call(cmd)
    return _SO_OMP


def _declare(L):
    L.oracle_phi.restype = C.c_double
    L.oracle_phi.argtypes = [C.c_double]
    L.oracle_num_points.restype = C.c_int64
    return L


def lib(omp=False):
    global _lib, _lib_omp
    if omp:
        if _lib_omp is None:
            build_omp()
            _lib_omp = _declare(C.CDLL(_SO_OMP))
        return _lib_omp
    if _lib is None:
        build()
        _lib = _declare(C.CDLL(_SO))
    return _lib


def _p(a, t=C.c_double):
    if a is None:
        return None
    return a.ctypes.data_as(C.POINTER(t))


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i32(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.int32)


def make_materials(mats):
    arr = (Material * len(mats))()
    for i, m in enumerate(mats):
        arr[i].law = int(m["law"])
        for k in ("a", "b", "af", "bf", "as_", "bs", "afs", "bfs", "kappa"):
            setattr(arr[i], k, float(m[k]))
        arr[i].Ta = float(m.get("Ta", 0.0))
    return arr


def make_grid(nx, ny, nz, h, origin=(0.0, 0.0, 0.0), periodic=1):
    return Grid(int(nx), int(ny), int(nz), float(h), float(origin[0]), float(origin[1]), float(origin[2]),
                int(periodic))


def phi(r):
    return lib().oracle_phi(float(r))


def pk1(mat, F, ef=None, es=None):
    """P (3x3) and Psi for one deformation gradient F (3x3, F[c,J] = dx_c/dX_J)."""
    F = _f64(F).reshape(9)
    P = np.empty(9)
    psi = C.c_double(0.0)
    m = make_materials([mat])
    ef = None if ef is None else _f64(ef)
    es = None if es is None else _f64(es)
    rc = lib().oracle_pk1(m, _p(F), _p(ef), _p(es), _p(P), C.byref(psi))
    if rc:
        raise ValueError("J <= 0")
    return P.reshape(3, 3), psi.value


def fe_force(conn, X, x, fibers, mat_id, mats, want=("B", "energy", "minJ")):
    conn = _i32(conn)
    X, x = _f64(X), _f64(x)
    nn, ne = X.shape[1], conn.shape[0]
    fibers = None if fibers is None else _f64(fibers)
    mat_id = _i32(mat_id)
    B = np.empty((3, nn))
    E, mj, bad = C.c_double(0), C.c_double(0), C.c_int64(-1)
    # conn [ne,8]: Q1 hexahedra; conn [ne,4]: P1 tetrahedra; conn [ne,10]: P2 tetrahedra (NEXT-3)
    fn = {4: lib().oracle_fe_force_tet, 10: lib().oracle_fe_force_tet10}.get(conn.shape[1], lib().oracle_fe_force)
    rc = fn(C.c_int64(nn), C.c_int64(ne), _p(conn, C.c_int32), _p(X), _p(x),
            _p(fibers), _p(mat_id, C.c_int32), make_materials(mats), _p(B),
            C.byref(E), C.byref(mj), C.byref(bad))
    return dict(B=B, energy=E.value, minJ=mj.value, rc=rc, first_bad=bad.value)


def tethers(ids, X, x, kappa, B):
    """B += kappa (X - x) on the nodes `ids`; returns (B, energy)."""
    ids, X, x = _i32(ids), _f64(X), _f64(x)
    B = _f64(B).copy()
    E = C.c_double(0)
    lib().oracle_tethers(C.c_int64(X.shape[1]), C.c_int64(ids.size), _p(ids, C.c_int32), _p(X), _p(x),
                         C.c_double(kappa), _p(B), C.byref(E))
    return B, E.value


def surface_loads(faces, X, x, qt0, p, B):
    """B += q t0 int N dA (reference faces) - p int N n da (current faces); faces [nf,3], [nf,4] or [nf,6] (quadratic triangles)."""
    faces, X, x = _i32(faces), _f64(X), _f64(x)
    B = _f64(B).copy()
    qt0 = None if qt0 is None else _f64(qt0)
    lib().oracle_surface_loads(C.c_int64(X.shape[1]), C.c_int64(faces.shape[0]), C.c_int32(faces.shape[1]),
                               _p(faces, C.c_int32), _p(X), _p(x), _p(qt0), C.c_double(p), _p(B))
    return B


def num_points(n_nodes, n_elems, nsub):
    nsub = _i32(nsub)
    return int(lib().oracle_num_points(C.c_int64(n_nodes), C.c_int64(n_elems), _p(nsub, C.c_int32)))


def points(conn, X, x, nsub):
    """(xp [3,P], Wp [P], w_a [n_nodes])."""
    conn, nsub = _i32(conn), _i32(nsub)
    X, x = _f64(X), _f64(x)
    nn, ne = X.shape[1], conn.shape[0]
    P = num_points(nn, ne, nsub)
    xp, Wp, wa = np.empty((3, P)), np.empty(P), np.empty(nn)
    rc = lib().oracle_points(C.c_int64(nn), C.c_int64(ne), _p(conn, C.c_int32), _p(X), _p(x),
                             _p(nsub, C.c_int32), _p(xp), _p(Wp), _p(wa))
    if rc:
        raise ValueError("det J0 <= 0 at a sub-point")
    return xp, Wp, wa


def nodal_weights(conn, X):
    conn, X = _i32(conn), _f64(X)
    nn, ne = X.shape[1], conn.shape[0]
    wq = np.empty(nn)
    lib().oracle_nodal_weights(C.c_int64(nn), C.c_int64(ne), _p(conn, C.c_int32), _p(X), _p(wq))
    return wq


def prolong(conn, nsub, w_a, Wp, B):
    conn, nsub = _i32(conn), _i32(nsub)
    w_a, Wp, B = _f64(w_a), _f64(Wp), _f64(B)
    nn, ne = B.shape[1], conn.shape[0]
    Gp = np.empty((3, Wp.shape[0]))
    lib().oracle_prolong(C.c_int64(nn), C.c_int64(ne), _p(conn, C.c_int32), _p(nsub, C.c_int32),
                         _p(w_a), _p(Wp), _p(B), _p(Gp))
    return Gp


def restrict(conn, nsub, w_a, Wp, Up):
    conn, nsub = _i32(conn), _i32(nsub)
    w_a, Wp, Up = _f64(w_a), _f64(Wp), _f64(Up)
    nn, ne = w_a.shape[0], conn.shape[0]
    Un = np.empty((3, nn))
    lib().oracle_restrict(C.c_int64(nn), C.c_int64(ne), _p(conn, C.c_int32), _p(nsub, C.c_int32),
                          _p(w_a), _p(Wp), _p(Up), _p(Un))
    return Un


def spread(grid, xp, Gp, f0=None, brute=False):
    xp, Gp = _f64(xp), _f64(Gp)
    P = xp.shape[1]
    n = grid.nx * grid.ny * grid.nz
    if f0 is None:
        f = [np.zeros(n) for _ in range(3)]
        acc = 0
    else:
        f = [np.array(a, dtype=np.float64, copy=True) for a in f0]
        acc = 1
    if brute:
        lib().oracle_spread_brute(C.byref(grid), C.c_int64(P), _p(xp), _p(Gp), _p(f[0]), _p(f[1]), _p(f[2]))
    else:
        lib().oracle_spread(C.byref(grid), C.c_int64(P), _p(xp), _p(Gp), _p(f[0]), _p(f[1]), _p(f[2]),
                            C.c_int32(acc))
    return f


def interp(grid, xp, u, v, w, brute=False):
    xp, u, v, w = _f64(xp), _f64(u), _f64(v), _f64(w)
    P = xp.shape[1]
    Up = np.empty((3, P))
    fn = lib().oracle_interp_brute if brute else lib().oracle_interp
    fn(C.byref(grid), C.c_int64(P), _p(xp), _p(u), _p(v), _p(w), _p(Up))
    return Up


def bin_sort(grid, xp, inv_h=None):
    xp = _f64(xp)
    P = xp.shape[1]
    if inv_h is None:
        inv_h = 1.0 / grid.h
    key = np.empty(P, dtype=np.int64)
    perm = np.empty(P, dtype=np.int32)
    lib().oracle_bin_sort(C.byref(grid), C.c_double(inv_h), C.c_int64(P), _p(xp), _p(key, C.c_int64),
                          _p(perm, C.c_int32))
    return key, perm


def coupling_step(grid, conn, X, fibers, mat_id, nsub, mats, x, u, v, w, omp=False):
    """dict(fu, fv, fw, Un, B).  omp=True: the OpenMP build (timing only; sums in another order)."""
    conn, nsub, mat_id = _i32(conn), _i32(nsub), _i32(mat_id)
    X, x, u, v, w = _f64(X), _f64(x), _f64(u), _f64(v), _f64(w)
    fibers = None if fibers is None else _f64(fibers)
    nn, ne = X.shape[1], conn.shape[0]
    n = grid.nx * grid.ny * grid.nz
    fu, fv, fw = np.zeros(n), np.zeros(n), np.zeros(n)
    Un, B = np.empty((3, nn)), np.empty((3, nn))
    bad = C.c_int64(-1)
    rc = lib(omp).oracle_coupling_step(C.byref(grid), C.c_int64(nn), C.c_int64(ne), _p(conn, C.c_int32),
                                    _p(X), _p(fibers), _p(mat_id, C.c_int32), _p(nsub, C.c_int32),
                                    make_materials(mats), _p(x), _p(u), _p(v), _p(w),
                                    _p(fu), _p(fv), _p(fw), _p(Un), _p(B), C.byref(bad))
    if rc:
        raise ValueError(f"inverted element {bad.value}")
    return dict(fu=fu, fv=fv, fw=fw, Un=Un, B=B)
