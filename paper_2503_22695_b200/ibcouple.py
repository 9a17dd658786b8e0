"""Thin Python binding of libibcouple.so (include/ibcouple.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI; torch is used for device
memory and streams.  There is no CPU fallback: if the shared library is missing or a call
fails, this module raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libibcouple.so")
_lib = None

STATUS = {0: "IB_OK", 1: "IB_ERR_INVALID_ARG", 2: "IB_ERR_UNSUPPORTED", 3: "IB_ERR_ALLOC", 4: "IB_ERR_CUDA",
          5: "IB_ERR_INVERTED_ELEMENT", 6: "IB_ERR_NONFINITE", 7: "IB_ERR_OUT_OF_DOMAIN", 8: "IB_ERR_TOO_LARGE"}

EXPORTS = ["ib_create", "ib_destroy", "ib_num_points", "ib_num_nodes", "ib_num_elems", "ib_fe_force",
           "ib_points", "ib_restrict", "ib_bin_sort", "ib_bin_sort_static", "ib_spread", "ib_interp", "ib_coupling_step",
           "ib_coupling_step_host", "ib_coupling_step_host3", "ib_step_eq16", "ib_check", "ib_launch_count", "ib_set_variant", "ib_set_graph", "ib_set_tethers", "ib_set_surface", "ib_set_loads", "ib_probe_dfma",
           "ib_profile_enable", "ib_profile_read",
           "ib_status_string"]


class IbError(RuntimeError):
    def __init__(self, code, where):
        self.code = int(code)
        super().__init__(f"{where}: {STATUS.get(int(code), code)}")


class GridDesc(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32), ("h", C.c_double),
                ("x0", C.c_double), ("y0", C.c_double), ("z0", C.c_double), ("periodic", C.c_int32)]


class Material(C.Structure):
    _fields_ = [("law", C.c_int32)] + [(k, C.c_double) for k in
                                       ("a", "b", "af", "bf", "as_", "bs", "afs", "bfs", "kappa", "Ta")]


class MeshDesc(C.Structure):
    _fields_ = [("n_nodes", C.c_int64), ("n_elems", C.c_int64), ("conn", C.c_void_p), ("X_ref", C.c_void_p),
                ("fibers", C.c_void_p), ("mat_id", C.c_void_p), ("nsub", C.c_void_p), ("mats", C.c_void_p),
                ("n_mats", C.c_int32), ("elem_type", C.c_int32)]


def lib():
    """Load libibcouple.so (built in-tree by paper_2503_22695_b200.build). Fails loudly."""
    global _lib
    if _lib is None:
        if not os.path.exists(_SO):
            raise ImportError(f"{_SO} is missing: run `python -m paper_2503_22695_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(_SO)
        vp, i32, i64 = C.c_void_p, C.c_int32, C.c_int64
        L.ib_create.argtypes = [C.POINTER(vp), C.POINTER(GridDesc), C.POINTER(MeshDesc), i32]
        L.ib_destroy.argtypes = [vp]
        for n in ("ib_num_points", "ib_num_nodes", "ib_num_elems", "ib_launch_count"):
            getattr(L, n).argtypes = [vp]
            getattr(L, n).restype = i64
        L.ib_fe_force.argtypes = [vp, vp, vp, vp]
        L.ib_points.argtypes = [vp, vp, vp, vp, vp, vp]
        L.ib_restrict.argtypes = [vp, vp, vp, vp]
        L.ib_bin_sort.argtypes = [vp, vp, i64, vp, vp, vp]
        L.ib_bin_sort_static.argtypes = [C.POINTER(GridDesc), vp, i64, vp, vp, i32, vp]
        L.ib_spread.argtypes = [vp, vp, vp, i64, vp, vp, vp, i32, vp]
        L.ib_interp.argtypes = [vp, vp, i64, vp, vp, vp, vp, vp]
        L.ib_coupling_step.argtypes = [vp] * 11
        L.ib_coupling_step_host.argtypes = [vp] * 11
        L.ib_coupling_step_host3.argtypes = [vp] * 7
        L.ib_step_eq16.argtypes = [vp] * 5 + [C.c_double] + [vp] * 7
        L.ib_check.argtypes = [vp, C.POINTER(i64)]
        L.ib_set_variant.argtypes = [vp, i32]
        L.ib_set_graph.argtypes = [vp, i32]
        L.ib_set_tethers.argtypes = [vp, i64, vp, C.c_double]
        L.ib_set_surface.argtypes = [vp, i64, i32, vp]
        L.ib_set_loads.argtypes = [vp, vp, C.c_double]
        L.ib_profile_enable.argtypes = [vp, i32]
        L.ib_profile_read.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(i64)]
        L.ib_probe_dfma.argtypes = [i32, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.ib_status_string.argtypes = [i32]
        L.ib_status_string.restype = C.c_char_p
        _lib = L
    return _lib


def _chk(code, where):
    if code != 0:
        raise IbError(code, where)


def _dp(t):
    """device (or pinned host) pointer of a torch tensor, or None."""
    if t is None:
        return None
    assert t.is_contiguous()
    return C.c_void_p(t.data_ptr())


def _stream(stream):
    import torch
    if stream is None:
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream)


BIN_SORT_STATIC_MAX_POINTS = 262144      # IB_BIN_SORT_STATIC_MAX_POINTS of include/ibcouple.h


def ib_bin_sort_static(grid, xp, P, key_out, perm_out, check=0, stream=None):
    """ib_bin_sort without a context and without any allocation (fixed scratch area inside the library);
    grid = (nx, ny, nz, h, (x0, y0, z0), periodic).  Raises IbError (IB_ERR_TOO_LARGE beyond the limit)."""
    nx, ny, nz, h, org, periodic = grid
    g = GridDesc(int(nx), int(ny), int(nz), float(h), float(org[0]), float(org[1]), float(org[2]), int(periodic))
    _chk(lib().ib_bin_sort_static(C.byref(g), _dp(xp), int(P), _dp(key_out), _dp(perm_out), int(check), _stream(stream)),
         "ib_bin_sort_static")


def probe_dfma(device=0):
    d, ms = C.c_double(0), C.c_double(0)
    _chk(lib().ib_probe_dfma(int(device), C.byref(d), C.byref(ms)), "ib_probe_dfma")
    return d.value, ms.value


class Context:
    """ib_ctx wrapper. Static mesh arrays are numpy (host); per-step arrays are torch CUDA tensors."""

    def __init__(self, nx, ny, nz, h, origin, conn, X, fibers, mat_id, nsub, mats, device=0, periodic=1):
        L = lib()
        self._h = C.c_void_p(None)
        self.device = int(device)
        conn = np.ascontiguousarray(conn, dtype=np.int32)
        X = np.ascontiguousarray(X, dtype=np.float64)
        fibers = None if fibers is None else np.ascontiguousarray(fibers, dtype=np.float64)
        mat_id = None if mat_id is None else np.ascontiguousarray(mat_id, dtype=np.int32)
        nsub = None if nsub is None else np.ascontiguousarray(nsub, dtype=np.int32)
        marr = (Material * max(len(mats), 1))()
        for i, m in enumerate(mats):
            marr[i].law = int(m["law"])
            for k in ("a", "b", "af", "bf", "as_", "bs", "afs", "bfs", "kappa"):
                setattr(marr[i], k, float(m[k]))
            marr[i].Ta = float(m.get("Ta", 0.0))
        g = GridDesc(int(nx), int(ny), int(nz), float(h), float(origin[0]), float(origin[1]), float(origin[2]),
                     int(periodic))
        md = MeshDesc(X.shape[1] if X.ndim == 2 else 0, conn.shape[0],
                      conn.ctypes.data if conn.size else None, X.ctypes.data if X.size else None,
                      None if fibers is None else fibers.ctypes.data,
                      None if mat_id is None else mat_id.ctypes.data,
                      None if nsub is None else nsub.ctypes.data,
                      C.cast(marr, C.c_void_p), len(mats), {4: 1, 10: 2}.get(conn.shape[1] if conn.ndim == 2 else 8, 0))
        _chk(L.ib_create(C.byref(self._h), C.byref(g), C.byref(md), self.device), "ib_create")
        self.nx, self.ny, self.nz, self.h = int(nx), int(ny), int(nz), float(h)
        self.n_cells = self.nx * self.ny * self.nz
        self.n_nodes = int(L.ib_num_nodes(self._h))
        self.n_elems = int(L.ib_num_elems(self._h))
        self.n_points = int(L.ib_num_points(self._h))

    @classmethod
    def from_workload(cls, wl, device=0, nodal=False):
        return cls(wl.nx, wl.ny, wl.nz, wl.h, wl.origin, wl.conn, wl.X, wl.fibers, wl.mat_id,
                   None if nodal else wl.nsub, wl.mats, device=device)

    def close(self):
        if self._h:
            lib().ib_destroy(self._h)
            self._h = C.c_void_p(None)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- the C ABI, same names ---------------------------------------------------------------
    def ib_set_variant(self, variant):
        _chk(lib().ib_set_variant(self._h, int(variant)), "ib_set_variant")

    def ib_set_tethers(self, node_ids, kappa):
        ids = np.ascontiguousarray(node_ids, dtype=np.int32)
        _chk(lib().ib_set_tethers(self._h, ids.size, ids.ctypes.data if ids.size else None, float(kappa)), "ib_set_tethers")

    def ib_set_surface(self, faces):
        f = np.ascontiguousarray(faces, dtype=np.int32)
        npf = f.shape[1] if f.ndim == 2 and f.size else 4
        _chk(lib().ib_set_surface(self._h, f.shape[0] if f.size else 0, npf, f.ctypes.data if f.size else None), "ib_set_surface")

    def ib_set_loads(self, qt0=None, p=0.0):
        q = None if qt0 is None else np.ascontiguousarray(qt0, dtype=np.float64)
        _chk(lib().ib_set_loads(self._h, None if q is None else q.ctypes.data, float(p)), "ib_set_loads")

    def ib_set_graph(self, on=True):
        _chk(lib().ib_set_graph(self._h, int(bool(on))), "ib_set_graph")

    PHASES = ("fe_force", "points", "sort", "spread_interp", "restrict", "zero")

    def ib_profile_enable(self, on=True):
        _chk(lib().ib_profile_enable(self._h, int(bool(on))), "ib_profile_enable")

    def ib_profile_read(self):
        """{phase: (ms_sum, calls)} since the last read."""
        ms = (C.c_double * len(self.PHASES))()
        n = (C.c_int64 * len(self.PHASES))()
        _chk(lib().ib_profile_read(self._h, ms, n), "ib_profile_read")
        return {k: (ms[i], int(n[i])) for i, k in enumerate(self.PHASES)}

    def ib_launch_count(self):
        return int(lib().ib_launch_count(self._h))

    def ib_fe_force(self, x, B, stream=None):
        _chk(lib().ib_fe_force(self._h, _dp(x), _dp(B), _stream(stream)), "ib_fe_force")

    def ib_points(self, x, B, xp, Gp, stream=None):
        _chk(lib().ib_points(self._h, _dp(x), _dp(B), _dp(xp), _dp(Gp), _stream(stream)), "ib_points")

    def ib_restrict(self, Up, Un, stream=None):
        _chk(lib().ib_restrict(self._h, _dp(Up), _dp(Un), _stream(stream)), "ib_restrict")

    def ib_bin_sort(self, xp, P, key_out, perm_out, stream=None):
        _chk(lib().ib_bin_sort(self._h, _dp(xp), int(P), _dp(key_out), _dp(perm_out), _stream(stream)), "ib_bin_sort")

    def ib_spread(self, xp, Gp, P, fu, fv, fw, accumulate=0, stream=None):
        _chk(lib().ib_spread(self._h, _dp(xp), _dp(Gp), int(P), _dp(fu), _dp(fv), _dp(fw), int(accumulate),
                             _stream(stream)), "ib_spread")

    def ib_interp(self, xp, P, u, v, w, Up, stream=None):
        _chk(lib().ib_interp(self._h, _dp(xp), int(P), _dp(u), _dp(v), _dp(w), _dp(Up), _stream(stream)), "ib_interp")

    def ib_coupling_step(self, x, u, v, w, fu, fv, fw, Un, B=None, stream=None):
        _chk(lib().ib_coupling_step(self._h, _dp(x), _dp(u), _dp(v), _dp(w), _dp(fu), _dp(fv), _dp(fw), _dp(Un),
                                    _dp(B), _stream(stream)), "ib_coupling_step")

    def ib_step_eq16(self, x, u, v, w, dt, x_new, fu, fv, fw, Un, B=None, stream=None):
        _chk(lib().ib_step_eq16(self._h, _dp(x), _dp(u), _dp(v), _dp(w), float(dt), _dp(x_new), _dp(fu), _dp(fv),
                                _dp(fw), _dp(Un), _dp(B), _stream(stream)), "ib_step_eq16")

    def ib_coupling_step_host(self, x, u, v, w, fu, fv, fw, Un, B=None, stream=None):
        """All tensors are (pinned) HOST tensors."""
        _chk(lib().ib_coupling_step_host(self._h, _dp(x), _dp(u), _dp(v), _dp(w), _dp(fu), _dp(fv), _dp(fw),
                                         _dp(Un), _dp(B), _stream(stream)), "ib_coupling_step_host")

    def ib_coupling_step_host3(self, x, uvw, f, Un, B=None, stream=None):
        """All tensors are (pinned) HOST tensors; uvw and f are [3][n_cells]."""
        _chk(lib().ib_coupling_step_host3(self._h, _dp(x), _dp(uvw), _dp(f), _dp(Un), _dp(B), _stream(stream)),
             "ib_coupling_step_host3")

    def ib_check(self):
        """Synchronise and return (status code, first bad id)."""
        bad = C.c_int64(-1)
        code = lib().ib_check(self._h, C.byref(bad))
        return int(code), int(bad.value)

    def check(self):
        code, bad = self.ib_check()
        if code != 0:
            raise IbError(code, f"ib_check (first bad id {bad})")
