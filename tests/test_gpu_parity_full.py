"""Full-size parity of the CUDA path against the CPU oracle, in the launch configurations bench.py times.

Bar (BASELINE.json north_star): fp64 rel-L2 <= 1e-12 and max-abs <= 1e-10 x ||oracle||_inf per output
array (A20).  Configs 3 and 4 and the low and middle points of the config-5 ladder are compared element
by element over the whole step; at the top of config 5 (52 M force points, minutes of oracle time) the
Eulerian force is compared element by element inside boxes (Eq.(24)-(26) L211-217: a face only
sees the points within two cells, so the oracle needs only the elements near the box), together with
sampled B, U^IB and Un and the invariants that hold at any size (L237-239).
"""
import numpy as np
import pytest

from helpers import max_abs_scaled
from paper_2503_22695_b200 import workloads as W
from test_gpu_parity import _close, _grid, _run_step, _t, ib  # noqa: F401  (ib is a fixture)

pytestmark = pytest.mark.gpu

_WL, _REF = {}, {}


def _workload(name):
    if name not in _WL:
        _WL[name] = {"C3": W.config3, "C4": W.config4,
                     "C5-L1-s2": lambda: W.config5(level=1, sub=2),
                     "C5-L2-s3": lambda: W.config5(level=2, sub=3),
                     "C5-L3-s4": lambda: W.config5(level=3, sub=4)}[name]()
    return _WL[name]


def _oracle_step(orc, name):
    """whole oracle step of a workload, computed once per test session (C3 takes ~20 s)"""
    if name not in _REF:
        wl = _workload(name)
        _REF[name] = orc.coupling_step(_grid(orc, wl), wl.conn, wl.X, wl.fibers, wl.mat_id, wl.nsub, wl.mats,
                                       wl.x, wl.u, wl.v, wl.w)
    return _REF[name]


# C3 = the bench workload; C4 = thin leaflets, non-uniform nsub; C5-L1-s2 / C5-L2-s3 = the sparse end of the
# sweep (about one point per cell on the 256^3 grid: most points take the direct path of the sparse tiles)
@pytest.mark.parametrize("name", ["C3", "C4", "C5-L1-s2", "C5-L2-s3"])
def test_full_size_step_matches_oracle(ib, orc, name):
    wl = _workload(name)
    ref = _oracle_step(orc, name)
    got = _run_step(ib, wl, 1)
    for k in ("B", "fu", "fv", "fw", "Un"):
        _close(got[k], ref[k], f"{name} full {k}")
    # runs of the same step differ only by the order of the atomic sums
    again = _run_step(ib, wl, 1)
    for k in ("fu", "fv", "fw", "Un"):
        assert max_abs_scaled(again[k], got[k]) <= 1e-12, k
    assert np.array_equal(again["B"], got["B"])                 # node-gathered: bit-reproducible


def test_c3_graph_replay_on_private_stream_matches_oracle(ib, orc):
    """What bench.py times: ib_coupling_step on a private stream, replayed as a CUDA graph from the third
    call on.  Every call is compared with the oracle (the first two run eagerly, the rest are replays)."""
    import torch
    wl, ref = _workload("C3"), _oracle_step(orc, "C3")
    ctx = ib.Context.from_workload(wl)
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        x, u, v, w = _t(wl.x), _t(wl.u), _t(wl.v), _t(wl.w)
        fu, fv, fw = (torch.empty(wl.n_cells, dtype=torch.float64, device="cuda") for _ in range(3))
        Un = torch.empty((3, wl.n_nodes), dtype=torch.float64, device="cuda")
        B = torch.empty((3, wl.n_nodes), dtype=torch.float64, device="cuda")
        for it in range(5):
            for t in (fu, fv, fw, Un, B):
                t.fill_(5.0 + it)                                 # stale values must not survive a replay
            ctx.ib_coupling_step(x, u, v, w, fu, fv, fw, Un, B, st)
            ctx.check()
            for k, t in (("B", B), ("fu", fu), ("fv", fv), ("fw", fw), ("Un", Un)):
                _close(t, ref[k], f"C3 private stream call {it} {k}")
    st.synchronize()
    ctx.close()


@pytest.mark.parametrize("name", ["C3", "C5-L2-s3"])
def test_step_is_stable_over_many_replays(ib, orc, name):
    """The tile kernel's two warp groups hand record buffers to each other through mbarriers, and no race
    detector is available on this pool (profiles/r02_sanitizer.md): replay the captured step 300 times and
    compare every result on the device with the first one -- B and Un bit for bit (no atomics feed them
    except through Up, which is written once per point), f to the order of its REDs -- and the last one
    with the oracle.  A lost update, a stale record or a buffer handed over too early shows at 1e-3."""
    import torch
    wl, ref = _workload(name), _oracle_step(orc, name)
    ctx = ib.Context.from_workload(wl)
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        x, u, v, w = _t(wl.x), _t(wl.u), _t(wl.v), _t(wl.w)
        out = [torch.empty(wl.n_cells, dtype=torch.float64, device="cuda") for _ in range(3)]
        out += [torch.empty((3, wl.n_nodes), dtype=torch.float64, device="cuda") for _ in range(2)]     # Un, B
        first, worst = None, 0.0
        for it in range(300):
            ctx.ib_coupling_step(x, u, v, w, *out, st)
            if first is None:
                ctx.check()
                first = [t.clone() for t in out]
                scale = [float(t.abs().max()) for t in first]
                continue
            assert torch.equal(out[3], first[3]) and torch.equal(out[4], first[4]), f"replay {it}: Un or B changed"
            for c in range(3):
                worst = max(worst, float((out[c] - first[c]).abs().max()) / scale[c])
        ctx.check()
        assert worst <= 1e-12, worst
        for k, t in zip(("fu", "fv", "fw", "Un", "B"), out):
            _close(t, ref[k], f"{name} after 300 replays {k}")
    st.synchronize()
    ctx.close()


def test_c3_host_step_matches_oracle(ib, orc):
    """The end-to-end number of bench.py: ib_coupling_step_host at C3 (8 z-slabs of 4 tile layers, the band
    shortcut for the layers the shell cannot reach), pinned host buffers, against the oracle."""
    import torch
    wl, ref = _workload("C3"), _oracle_step(orc, "C3")
    ctx = ib.Context.from_workload(wl)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    x, u, v, w = pin(wl.x), pin(wl.u), pin(wl.v), pin(wl.w)
    outs = [torch.full((wl.n_cells,), 9.0, dtype=torch.float64).pin_memory() for _ in range(3)]
    Un = torch.empty((3, wl.n_nodes), dtype=torch.float64).pin_memory()
    B = torch.empty((3, wl.n_nodes), dtype=torch.float64).pin_memory()
    for it in range(3):
        for t in outs:
            t.fill_(9.0 + it)
        ctx.ib_coupling_step_host(x, u, v, w, *outs, Un, B)
        ctx.check()
        for k, t in (("B", B), ("fu", outs[0]), ("fv", outs[1]), ("fw", outs[2]), ("Un", Un)):
            _close(t.numpy(), ref[k], f"C3 host step call {it} {k}")
    # the packed entry point bench.py times: one [3][n_cells] host array per direction
    uvw = pin(np.stack([wl.u, wl.v, wl.w]))
    f3 = torch.full((3, wl.n_cells), 7.0, dtype=torch.float64).pin_memory()
    for it in range(2):
        f3.fill_(7.0 + it)
        ctx.ib_coupling_step_host3(x, uvw, f3, Un, B)
        ctx.check()
        for c, k in enumerate(("fu", "fv", "fw")):
            _close(f3[c].numpy(), ref[k], f"C3 host3 call {it} {k}")
        _close(Un.numpy(), ref["Un"], f"C3 host3 call {it} Un")
        _close(B.numpy(), ref["B"], f"C3 host3 call {it} B")
    ctx.close()


# ---- top of the config-5 sweep -------------------------------------------------------------------------
def _submesh(wl, elems):
    """the elements `elems` as a mesh of their own: (conn, X, x, fibers, mat_id, nsub, node ids)"""
    conn = wl.conn[elems]
    used = np.unique(conn)
    remap = -np.ones(wl.n_nodes, dtype=np.int64)
    remap[used] = np.arange(used.size)
    return (remap[conn].astype(np.int32), np.ascontiguousarray(wl.X[:, used]), np.ascontiguousarray(wl.x[:, used]),
            np.ascontiguousarray(wl.fibers[:, elems]), np.ascontiguousarray(wl.mat_id[elems]),
            np.ascontiguousarray(wl.nsub[elems]), used)


def _box_case(orc, wl, centre_elem, half):
    """Oracle values of f on the faces [c-half, c+half)^3 around the cell c of an element's centroid, and of
    Un on the nodes next to it.  S1 = elements whose bounding box comes within 2.5 h of the box (sub-points
    are convex combinations of the nodes, a support reaches 2 h, staggering half a cell); S2 = S1 and every
    element sharing a node with it, so that B and the lumped weights w_a are complete on the nodes of S1."""
    org, h = np.asarray(wl.origin, dtype=np.float64), wl.h
    xe = wl.x[:, wl.conn]                                         # [3, ne, 8]
    c = np.floor((xe[:, centre_elem].mean(axis=1) - org) / h).astype(int)
    lo_i, hi_i = c - half, c + half
    assert np.all(lo_i >= 3) and np.all(hi_i <= np.array([wl.nx, wl.ny, wl.nz]) - 3), "box must not touch the wrap"
    lo, hi = org + lo_i * h - 2.5 * h, org + hi_i * h + 2.5 * h
    emin, emax = xe.min(axis=2), xe.max(axis=2)
    s1 = np.all((emax >= lo[:, None]) & (emin <= hi[:, None]), axis=0)
    node_s1 = np.zeros(wl.n_nodes, dtype=bool)
    node_s1[wl.conn[s1].ravel()] = True
    s2 = np.any(node_s1[wl.conn], axis=1)
    e2 = np.flatnonzero(s2)
    conn2, X2, x2, fib2, mid2, nsub2, used = _submesh(wl, e2)
    complete = np.bincount(wl.conn.ravel(), minlength=wl.n_nodes)[used] == np.bincount(conn2.ravel(), minlength=used.size)
    assert np.all(complete[np.unique(conn2[s1[e2]])])            # every node of S1 has all its elements in S2
    B2 = orc.fe_force(conn2, X2, x2, fib2, mid2, wl.mats)["B"]
    xp2, Wp2, wa2 = orc.points(conn2, X2, x2, nsub2)
    Gp2 = orc.prolong(conn2, nsub2, wa2, Wp2, B2)
    npts = nsub2.prod(axis=1)
    in_s1 = np.repeat(s1[e2], npts)                               # points are numbered element by element
    g = _grid(orc, wl)
    f = orc.spread(g, np.ascontiguousarray(xp2[:, in_s1]), np.ascontiguousarray(Gp2[:, in_s1]))
    Up2 = orc.interp(g, xp2, wl.u, wl.v, wl.w)
    Un2 = orc.restrict(conn2, nsub2, wa2, Wp2, Up2)
    box = np.s_[lo_i[2]:hi_i[2], lo_i[1]:hi_i[1], lo_i[0]:hi_i[0]]
    return dict(box=box, f=[np.asarray(a).reshape(wl.nz, wl.ny, wl.nx)[box] for a in f], nodes=used[complete],
                B=B2[:, complete], Un=Un2[:, complete], n_points=int(in_s1.sum()))


def test_c5_top_of_sweep_boxes_samples_and_invariants(ib, orc):
    """C5 level 3 x 4^3 (52 M force points): f element by element inside two boxes (one across the shell
    wall, one around a leaflet), B and Un on the nodes around them, U^IB at the sub-points of a band, and
    the properties that hold at any size (adjointness L237-239, total force)."""
    import torch
    wl = _workload("C5-L3-s4")
    got = _run_step(ib, wl, 1)
    h3 = wl.h ** 3
    # total Eulerian force = total Lagrangian force (A14), per component
    for c, k in enumerate(("fu", "fv", "fw")):
        tot_f, tot_B = h3 * np.sum(got[k]), np.sum(got["B"][c])
        scale = h3 * np.sum(np.abs(got[k]))
        assert abs(tot_f - tot_B) <= 1e-11 * scale, (k, tot_f, tot_B)
    # node-level adjointness  h^3 sum f.u = sum_a B_a . Un_a
    lhs = h3 * (np.dot(got["fu"], wl.u) + np.dot(got["fv"], wl.v) + np.dot(got["fw"], wl.w))
    rhs = float(np.sum(got["B"] * got["Un"]))
    scale = h3 * (np.dot(np.abs(got["fu"]), np.abs(wl.u)) + np.dot(np.abs(got["fv"]), np.abs(wl.v))
                  + np.dot(np.abs(got["fw"]), np.abs(wl.w)))
    assert abs(lhs - rhs) <= 1e-11 * scale, (lhs, rhs)
    # boxes: shell wall (element in the middle of the shell block) and a leaflet (mat_id 1)
    layer = 16 * 256                                          # elements per longitudinal layer of the shell
    leaf = np.flatnonzero(wl.mat_id == 1)
    assert leaf.size == 2 * 128 * 64 * 2
    for what, ce, half in (("shell", 100 * layer + 64 * 16 + 8, 8), ("leaflet", int(leaf[leaf.size // 4]), 8)):
        case = _box_case(orc, wl, ce, half)
        assert case["n_points"] > 20000, (what, case["n_points"])
        for k, fr in zip(("fu", "fv", "fw"), case["f"]):
            assert np.max(np.abs(fr)) > 0
            _close(got[k].reshape(wl.nz, wl.ny, wl.nx)[case["box"]], fr, f"C5 top {what} box {k}")
        assert case["nodes"].size > 500
        _close(got["B"][:, case["nodes"]], case["B"], f"C5 top {what} B")
        _close(got["Un"][:, case["nodes"]], case["Un"], f"C5 top {what} Un")
    # sampled U^IB at the sub-points of one layer of shell elements, through the exported point generator
    e0 = 60 * layer
    conn1, X1, x1, _, _, nsub1, _ = _submesh(wl, np.arange(e0, e0 + layer))
    ctx = ib.Context.from_workload(wl)
    P = ctx.n_points
    xp = torch.empty((3, P), dtype=torch.float64, device="cuda")
    ctx.ib_points(_t(wl.x), None, xp, None)
    p0 = e0 * 64
    xs = xp[:, p0:p0 + layer * 64].contiguous()
    Up = torch.empty_like(xs)
    ctx.ib_interp(xs, xs.shape[1], _t(wl.u), _t(wl.v), _t(wl.w), Up)
    ctx.check()
    xp_ref, _, _ = orc.points(conn1, X1, x1, nsub1)
    _close(xs, xp_ref, "C5 sampled xp")
    _close(Up, orc.interp(_grid(orc, wl), xp_ref, wl.u, wl.v, wl.w), "C5 sampled U")
    ctx.close()
