"""Parity of the CUDA path (through the C ABI) against the CPU oracle on identical seeded inputs.

Bar (BASELINE.json north_star): fp64 rel-L2 <= 1e-12 and max-abs <= 1e-10 x ||oracle||_inf per output
array (A20); bit-exact for the integer binning/sort permutation.
"""
import numpy as np
import pytest

from helpers import distorted_block, max_abs_scaled, rel_l2, rotation
from paper_2503_22695_b200 import workloads as W

pytestmark = pytest.mark.gpu

REL, MAXABS = 1e-12, 1e-10


@pytest.fixture(scope="module")
def ib():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_2503_22695_b200 import build, ibcouple
    build.build()
    ibcouple.lib()
    return ibcouple


def _t(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _close(got, exp, what):
    got = got.cpu().numpy() if hasattr(got, "cpu") else got
    r, m = rel_l2(got, exp), max_abs_scaled(got, exp)
    assert r <= REL and m <= MAXABS, f"{what}: rel-L2 {r:.3e} max-abs/scale {m:.3e}"
    return r, m


def _grid(orc, wl):
    return orc.make_grid(wl.nx, wl.ny, wl.nz, wl.h, wl.origin)


def _run_step(ib, wl, variant, nodal=False):
    import torch
    ctx = ib.Context.from_workload(wl, nodal=nodal)
    ctx.ib_set_variant(variant)
    x, u, v, w = _t(wl.x), _t(wl.u), _t(wl.v), _t(wl.w)
    fu, fv, fw = (torch.full((wl.n_cells,), 7.0, dtype=torch.float64, device="cuda") for _ in range(3))
    Un = torch.empty((3, wl.n_nodes), dtype=torch.float64, device="cuda")
    B = torch.empty((3, wl.n_nodes), dtype=torch.float64, device="cuda")
    ctx.ib_coupling_step(x, u, v, w, fu, fv, fw, Un, B)
    ctx.check()
    out = dict(fu=fu.cpu().numpy(), fv=fv.cpu().numpy(), fw=fw.cpu().numpy(), Un=Un.cpu().numpy(), B=B.cpu().numpy())
    ctx.close()
    return out


CONFIGS = {
    "C1": lambda: W.config1(),
    "C1-wrap": lambda: W.config1(shift_cells=(14, 15, 17)),      # block straddles the periodic wrap (A18)
    "C2": lambda: W.config2(),
    "LV-small": lambda: W.lv_small(),
}


@pytest.mark.parametrize("variant", [0, 1])
@pytest.mark.parametrize("name", list(CONFIGS))
def test_coupling_step_matches_oracle(ib, orc, name, variant):
    wl = CONFIGS[name]()
    ref = orc.coupling_step(_grid(orc, wl), wl.conn, wl.X, wl.fibers, wl.mat_id, wl.nsub, wl.mats, wl.x, wl.u, wl.v, wl.w)
    got = _run_step(ib, wl, variant)
    for k in ("B", "fu", "fv", "fw", "Un"):
        _close(got[k], ref[k], f"{name} v{variant} {k}")


@pytest.mark.parametrize("variant", [0, 1])
def test_nodal_mode_matches_oracle(ib, orc, variant):
    wl = W.config1()
    ref = orc.coupling_step(_grid(orc, wl), wl.conn, wl.X, wl.fibers, wl.mat_id, None, wl.mats, wl.x, wl.u, wl.v, wl.w)
    got = _run_step(ib, wl, variant, nodal=True)
    for k in ("B", "fu", "fv", "fw", "Un"):
        _close(got[k], ref[k], f"nodal v{variant} {k}")


def test_fe_force_pieces_and_determinism(ib, orc):
    import torch
    conn, X, x, fib = distorted_block(5, 4, 3, seed=8)
    ne, nn = conn.shape[0], X.shape[1]
    rng = np.random.default_rng(0)
    mats = [W.material(W.LAW_NEOHOOKEAN, a=1e4, kappa=1e6), W.material(W.LAW_HO, **W.HO_LV)]
    mid = rng.integers(0, 2, ne).astype(np.int32)
    nsub = rng.integers(1, 5, (ne, 3)).astype(np.int32)        # ragged sub-point counts
    ctx = ib.Context(16, 16, 16, 1 / 16, (0, 0, 0), conn, X, fib, mid, nsub, mats)
    xd = _t(x)
    B = torch.empty((3, nn), dtype=torch.float64, device="cuda")
    ctx.ib_fe_force(xd, B)
    ctx.check()
    ref = orc.fe_force(conn, X, x, fib, mid, mats)
    _close(B, ref["B"], "fe_force B")
    B2 = torch.empty_like(B)
    ctx.ib_fe_force(xd, B2)
    assert torch.equal(B, B2)                                     # node-gathered: bit-reproducible
    # points / prolongation / restriction
    P = ctx.n_points
    xp_r, Wp_r, wa_r = orc.points(conn, X, x, nsub)
    assert P == xp_r.shape[1]
    xp = torch.empty((3, P), dtype=torch.float64, device="cuda")
    Gp = torch.empty((3, P), dtype=torch.float64, device="cuda")
    ctx.ib_points(xd, B, xp, Gp)
    _close(xp, xp_r, "xp")
    _close(Gp, orc.prolong(conn, nsub, wa_r, Wp_r, ref["B"]), "Gp")
    Up = rng.normal(size=(3, P))
    Un = torch.empty((3, nn), dtype=torch.float64, device="cuda")
    ctx.ib_restrict(_t(Up), Un)
    ctx.check()
    _close(Un, orc.restrict(conn, nsub, wa_r, Wp_r, Up), "Un")
    ctx.close()


@pytest.mark.parametrize("sub", [(3, 3, 3), (5, 5, 5), (6, 6, 6), (2, 3, 5), (7, 8, 8), (4, 4, 4), (3, 4, 2), (1, 1, 1)])
def test_restrict_uniform_subpoint_counts(ib, orc, sub):
    """ib_restrict takes one of three kernels by the sub-point rule: rows-per-element a power of
    two (shuffles), any other uniform rule (rows meet in shared memory; CTAs of 256 / (n2 n3) elements -- 59 elements
    leave a ragged last CTA for every rule here), ragged rules (test_fe_force_pieces_and_determinism)."""
    import torch
    conn, X, x, fib = distorted_block(5, 4, 3, seed=21)
    conn, fib = conn[:59], fib[:, :59]                           # 59 elements: not a multiple of any CTA's element count
    ne, nn = conn.shape[0], X.shape[1]
    used = np.unique(conn)
    remap = -np.ones(nn, np.int64); remap[used] = np.arange(used.size)
    conn, X, x = remap[conn].astype(np.int32), X[:, used], x[:, used]
    nn = X.shape[1]
    nsub = np.tile(np.array(sub, np.int32), (ne, 1))
    mats = [W.material(W.LAW_NEOHOOKEAN, a=1e4, kappa=1e6)]
    ctx = ib.Context(16, 16, 16, 1 / 16, (0, 0, 0), conn, X, fib, np.zeros(ne, np.int32), nsub, mats)
    xp_r, Wp_r, wa_r = orc.points(conn, X, x, nsub)
    P = ctx.n_points
    assert P == ne * sub[0] * sub[1] * sub[2]
    rng = np.random.default_rng(5)
    Up = rng.normal(size=(3, P))
    Un = torch.empty((3, nn), dtype=torch.float64, device="cuda")
    ctx.ib_restrict(_t(Up), Un)
    ctx.check()
    _close(Un, orc.restrict(conn, nsub, wa_r, Wp_r, Up), f"Un {sub}")
    Un2 = torch.empty_like(Un)
    ctx.ib_restrict(_t(Up), Un2)
    assert torch.equal(Un, Un2)                                   # fixed summation order: bit-reproducible
    ctx.close()


@pytest.mark.parametrize("variant", [0, 1])
def test_spread_interp_generic_cloud(ib, orc, variant):
    import torch
    n, h, org = (24, 16, 32), 0.05, (-0.4, 0.1, 0.3)
    ctx = ib.Context(*n, h, org, np.zeros((0, 8), np.int32), np.zeros((3, 0)), None, None, None, [])
    ctx.ib_set_variant(variant)
    g = orc.make_grid(*n, h, org)
    rng = np.random.default_rng(3)
    L = np.array(n) * h
    P = 20011                                                  # ragged tail
    xp = np.asarray(org)[:, None] + rng.uniform(-0.5, 1.5, (3, P)) * L[:, None]     # outside the box too
    xp[:, :64] = np.asarray(org)[:, None] + (rng.integers(0, 24, (3, 64)) * h)      # exactly on cell boundaries
    G = rng.normal(size=(3, P))
    ncell = n[0] * n[1] * n[2]
    uvw = rng.normal(size=(3, ncell))
    f = [torch.full((ncell,), 3.0, dtype=torch.float64, device="cuda") for _ in range(3)]
    ctx.ib_spread(_t(xp), _t(G), P, *f, accumulate=0)
    Up = torch.empty((3, P), dtype=torch.float64, device="cuda")
    ctx.ib_interp(_t(xp), P, _t(uvw[0]), _t(uvw[1]), _t(uvw[2]), Up)
    ctx.check()
    fr = orc.spread(g, xp, G)
    for c in range(3):
        _close(f[c], fr[c], f"spread c{c}")
    _close(Up, orc.interp(g, xp, *uvw), "interp")
    # accumulate=1 adds to what is there
    ctx.ib_spread(_t(xp), _t(G), P, *f, accumulate=1)
    for c in range(3):
        _close(f[c], 2 * fr[c], f"spread accumulate c{c}")
    # empty cloud: zero-fill only
    ctx.ib_spread(None, None, 0, *f, accumulate=0)
    assert all(float(t.abs().max()) == 0.0 for t in f)
    # GPU-vs-GPU adjointness
    ctx.ib_spread(_t(xp), _t(G), P, *f, accumulate=0)
    lhs = h ** 3 * sum(float(torch.dot(f[c], _t(uvw[c]))) for c in range(3))
    rhs = float((Up * _t(G)).sum())
    assert abs(lhs - rhs) < 1e-11 * abs(rhs)
    ctx.close()


@pytest.mark.parametrize("periodic", [1, 0])
def test_interp_halo_by_tma_and_by_copies_agree(ib, orc, periodic):
    """The tile kernel loads the 8^3 velocity halo of a tile by TMA box loads (zero fill outside a bounded grid)
    and falls back to element copies for tiles at the wrap of a periodic grid and for arrays that are not
    16-byte aligned: both must give the same bits, and the oracle's values."""
    import torch
    n, h, org = (32, 24, 40), 0.1, (0.3, -0.2, 1.0)
    ctx = ib.Context(*n, h, org, np.zeros((0, 8), np.int32), np.zeros((3, 0)), None, None, None, [], periodic=periodic)
    g = orc.make_grid(*n, h, org, periodic=periodic)
    rng = np.random.default_rng(77 + periodic)
    L = np.array(n) * h
    P = 150001                                                 # ~5 points per cell: every tile goes through the tile kernel
    lo, hi = (-0.1, 1.1) if periodic else (0.0, 1.0)
    xp = np.asarray(org)[:, None] + rng.uniform(lo, hi, (3, P)) * L[:, None]
    if not periodic:
        xp = np.minimum(xp, (np.asarray(org) + L * (1 - 1e-12))[:, None])
    ncell = n[0] * n[1] * n[2]
    uvw = rng.normal(size=(3, ncell))
    x_d = _t(xp)
    Up = torch.empty((3, P), dtype=torch.float64, device="cuda")
    ctx.ib_interp(x_d, P, _t(uvw[0]), _t(uvw[1]), _t(uvw[2]), Up)                   # aligned arrays: TMA where the tile allows
    ctx.check()
    _close(Up, orc.interp(g, xp, *uvw), "interp, aligned arrays")
    shifted = []
    for c in range(3):                                                              # the same values at an address = 8 mod 16
        big = torch.empty(ncell + 1, dtype=torch.float64, device="cuda")
        big[1:] = _t(uvw[c])
        assert big[1:].data_ptr() % 16 == 8
        shifted.append(big[1:])
    Up2 = torch.empty((3, P), dtype=torch.float64, device="cuda")
    ctx.ib_interp(x_d, P, *shifted, Up2)
    ctx.check()
    assert torch.equal(Up, Up2)
    ctx.close()


def test_bin_sort_bit_exact(ib, orc):
    import torch
    for n, P in (((16, 8, 24), 0), ((16, 8, 24), 1), ((16, 8, 24), 5000), ((64, 64, 64), 300007)):
        h, org = 0.25, (-1.0, 0.5, 2.0)
        ctx = ib.Context(*n, h, org, np.zeros((0, 8), np.int32), np.zeros((3, 0)), None, None, None, [])
        rng = np.random.default_rng(P)
        xp = np.asarray(org)[:, None] + rng.uniform(-0.2, 1.2, (3, P)) * (np.array(n) * h)[:, None]
        if P > 100:
            xp[:, :50] = np.asarray(org)[:, None] + rng.integers(0, 8, (3, 50)) * h     # exact boundaries
            xp[:, 50:100] = xp[:, 100:101]                                              # many ties
        key = torch.empty(P, dtype=torch.int64, device="cuda")
        perm = torch.empty(P, dtype=torch.int32, device="cuda")
        ctx.ib_bin_sort(_t(xp) if P else None, P, key, perm)
        ctx.check()
        k_ref, p_ref = orc.bin_sort(orc.make_grid(*n, h, org), xp)
        assert np.array_equal(key.cpu().numpy(), k_ref)
        assert np.array_equal(perm.cpu().numpy(), p_ref)
        ctx.close()


def test_error_latch_inverted_element_and_nan(ib):
    import torch
    conn, X, x, fib = distorted_block(3, 3, 2, seed=9)
    nn = X.shape[1]
    ctx = ib.Context(16, 16, 16, 1 / 16, (0, 0, 0), conn, X, fib, None, None, [W.material(0, a=1.0, kappa=10.0)])
    B = torch.empty((3, nn), dtype=torch.float64, device="cuda")
    xi = x.copy()
    n0, n7 = conn[7, 0], conn[7, 7]
    xi[:, n0] = x[:, n7] + (x[:, n7] - x[:, n0])
    ctx.ib_fe_force(_t(xi), B)
    code, bad = ctx.ib_check()
    assert code == 5 and bad >= 0
    xn = x.copy()
    xn[1, 3] = np.nan
    ctx.ib_fe_force(_t(xn), B)
    code, bad = ctx.ib_check()
    assert code == 6
    ctx.ib_fe_force(_t(x), B)                                    # latch was cleared
    assert ctx.ib_check()[0] == 0
    ctx.close()


@pytest.mark.parametrize("variant", [0, 1])
def test_step_with_nonfinite_node_latches_and_recovers(ib, orc, variant):
    """A NaN node position inside the whole step (FE force, on-the-fly sub-points, binning, tile kernel): the step
    ends, the latch reads IB_ERR_NONFINITE, nothing hangs or faults; the same context then gives the oracle's
    result for clean positions, on the default stream and on a private one (graph replay)."""
    import torch
    wl = W.config1()
    ctx = ib.Context.from_workload(wl)
    ctx.ib_set_variant(variant)
    u, v, w = _t(wl.u), _t(wl.v), _t(wl.w)
    fu, fv, fw = (torch.empty((wl.n_cells,), dtype=torch.float64, device="cuda") for _ in range(3))
    Un = torch.empty((3, wl.n_nodes), dtype=torch.float64, device="cuda")
    B = torch.empty((3, wl.n_nodes), dtype=torch.float64, device="cuda")
    xn = wl.x.copy()
    xn[2, wl.n_nodes // 2] = np.nan
    ctx.ib_coupling_step(_t(xn), u, v, w, fu, fv, fw, Un, B)
    code, bad = ctx.ib_check()
    assert code == 6 and bad >= 0
    ref = orc.coupling_step(_grid(orc, wl), wl.conn, wl.X, wl.fibers, wl.mat_id, wl.nsub, wl.mats, wl.x, wl.u, wl.v, wl.w)
    x = _t(wl.x)
    st = torch.cuda.Stream()
    for stream in (None, st, st, st):
        for t in (fu, fv, fw, Un, B):
            t.fill_(3.0)
        torch.cuda.synchronize()
        if stream is None:
            ctx.ib_coupling_step(x, u, v, w, fu, fv, fw, Un, B)
        else:
            with torch.cuda.stream(stream):
                ctx.ib_coupling_step(x, u, v, w, fu, fv, fw, Un, B, stream)
        assert ctx.ib_check()[0] == 0                                # latch was cleared
        torch.cuda.synchronize()
        _close(B, ref["B"], "B after a non-finite step")
        for k, t in zip(("fu", "fv", "fw"), (fu, fv, fw)):
            _close(t, ref[k], f"{k} after a non-finite step")
        _close(Un, ref["Un"], "Un after a non-finite step")
    ctx.close()


@pytest.mark.parametrize("variant", [0, 1])
@pytest.mark.parametrize("name", ["C1", "LV-small"])
def test_host_entry_point_matches_device_path(ib, name, variant):
    """ib_coupling_step_host (variant 1: spread and interpolation pipelined around the host copies on two
    streams) gives what the device-pointer step gives."""
    import torch
    wl = CONFIGS[name]()
    ctx = ib.Context.from_workload(wl)
    dev = _run_step(ib, wl, variant)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    outs = [torch.full((wl.n_cells,), 9.0, dtype=torch.float64).pin_memory() for _ in range(3)]
    Un = torch.empty((3, wl.n_nodes), dtype=torch.float64).pin_memory()
    B = torch.empty((3, wl.n_nodes), dtype=torch.float64).pin_memory()
    ctx.ib_set_variant(variant)
    for _ in range(2):                                            # twice: buffers and events are reused
        ctx.ib_coupling_step_host(pin(wl.x), pin(wl.u), pin(wl.v), pin(wl.w), *outs, Un, B)
    ctx.check()
    assert np.array_equal(B.numpy(), dev["B"])
    for k, o in zip(("fu", "fv", "fw"), outs):
        _close(o.numpy(), dev[k], f"host {k}")
    _close(Un.numpy(), dev["Un"], "host Un")
    ctx.close()


@pytest.mark.parametrize("case", ["wrap", "bounded", "one-slab", "pageable", "non-cubic", "packed"])
def test_host_step_slabs_against_oracle(ib, orc, case):
    """ib_coupling_step_host cuts the step into z-slabs (copies of u,v,w and f overlap the tile kernel):
    a structure across the periodic z wrap (first and last slab share points), a bounded grid with the
    structure in a corner, and a grid too thin for more than one slab, each against the oracle."""
    import torch
    wl = W.config1()
    nz, periodic = wl.nz, 1
    org = np.asarray(wl.origin, dtype=np.float64).copy()
    if case == "wrap":
        shift = np.array([0.0, 0.0, 0.5 * wl.nz * wl.h + 0.37 * wl.h])      # the slab sits on the z wrap
    elif case == "bounded":
        shift = org - wl.X.min(axis=1) + 0.3 * wl.h
        periodic = 0
    elif case in ("pageable", "packed"):          # plain (unpinned) host memory: slower copies, same answer;
        shift = np.zeros(3)                       # packed: ib_coupling_step_host3, one [3][n_cells] array per direction
    elif case == "non-cubic":                     # 24 x 16 x 40 cells: 5 slabs of 2 tile layers, the slab tilted across them
        shift = np.zeros(3)
    else:
        nz = 8
        shift = np.zeros(3)
        org[2] = 0.5 * (wl.X[2].min() + wl.X[2].max()) - 4 * wl.h + 0.21 * wl.h
    X, x = wl.X + shift[:, None], wl.x + shift[:, None]
    nx, ny = wl.nx, wl.ny
    if case == "non-cubic":
        nx, ny, nz = 24, 16, 40
        org = np.array([0.125, 0.25, -0.125])
        c0 = 0.5 * (wl.X.min(axis=1) + wl.X.max(axis=1))
        R = rotation(5)                                       # the slab turned out of its plane: it spans several z-slabs
        X, x = c0[:, None] + R @ (wl.X - c0[:, None]), c0[:, None] + R @ (wl.x - c0[:, None])
    ncell = nx * ny * nz
    if case == "non-cubic":
        u, v, w = np.random.default_rng(77).normal(size=(3, ncell))
    else:
        u, v, w = (np.ascontiguousarray(a.reshape(wl.nz, wl.ny, wl.nx)[:nz].reshape(-1)) for a in (wl.u, wl.v, wl.w))
    g = orc.make_grid(nx, ny, nz, wl.h, tuple(org), periodic=periodic)
    ref = orc.coupling_step(g, wl.conn, X, wl.fibers, wl.mat_id, wl.nsub, wl.mats, x, u, v, w)
    ctx = ib.Context(nx, ny, nz, wl.h, tuple(org), wl.conn, X, wl.fibers, wl.mat_id, wl.nsub, wl.mats, periodic=periodic)
    pin = (lambda a: torch.from_numpy(np.array(a, order="C"))) if case == "pageable" else \
          (lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory())
    outs = [pin(np.full(ncell, 9.0)) for _ in range(3)]
    Un, B = pin(np.empty((3, wl.n_nodes))), pin(np.empty((3, wl.n_nodes)))
    if case == "packed":
        f3 = pin(np.full((3, ncell), 9.0))
        outs = [f3[0], f3[1], f3[2]]
        for _ in range(2):
            ctx.ib_coupling_step_host3(pin(x), pin(np.stack([u, v, w])), f3, Un, B)
    else:
        for _ in range(2):
            ctx.ib_coupling_step_host(pin(x), pin(u), pin(v), pin(w), *outs, Un, B)
    ctx.check()
    for k, t in (("B", B), ("fu", outs[0]), ("fv", outs[1]), ("fw", outs[2]), ("Un", Un)):
        _close(t.numpy(), ref[k], f"host slabs {case} {k}")
    ctx.close()


# ---- NEXT-1: the paper's explicit coupling order, Eq.(16) L165-173 --------------------------------
@pytest.mark.parametrize("variant", [0, 1])
@pytest.mark.parametrize("name,nodal", [("C1", False), ("LV-small", False), ("C1", True)])
def test_step_eq16_matches_oracle_composition(ib, orc, name, nodal, variant):
    """U = I(X^n,u^n) -> nodes; x_new = x + dt U; B = fe_force(x_new); f = E(X^n, F^{n+1}) with the
    deltas at the OLD positions.  The oracle side composes its own operators in that order."""
    import torch
    wl = CONFIGS[name]()
    dt = 2e-3 * wl.h                                       # |u| <= 16: moves nodes by a few % of h
    g = _grid(orc, wl)
    nsub = None if nodal else wl.nsub
    if nodal:
        Un_r = orc.interp(g, wl.x, wl.u, wl.v, wl.w)
    else:
        xp, Wp, wa = orc.points(wl.conn, wl.X, wl.x, wl.nsub)
        Un_r = orc.restrict(wl.conn, wl.nsub, wa, Wp, orc.interp(g, xp, wl.u, wl.v, wl.w))
    x_new_r = wl.x + dt * Un_r
    B_r = orc.fe_force(wl.conn, wl.X, x_new_r, wl.fibers, wl.mat_id, wl.mats)["B"]
    f_r = orc.spread(g, wl.x, B_r) if nodal else orc.spread(g, xp, orc.prolong(wl.conn, wl.nsub, wa, Wp, B_r))

    ctx = ib.Context.from_workload(wl, nodal=nodal)
    ctx.ib_set_variant(variant)
    f = [torch.full((wl.n_cells,), 5.0, dtype=torch.float64, device="cuda") for _ in range(3)]
    Un, B, x_new = (torch.empty((3, wl.n_nodes), dtype=torch.float64, device="cuda") for _ in range(3))
    ctx.ib_step_eq16(_t(wl.x), _t(wl.u), _t(wl.v), _t(wl.w), dt, x_new, *f, Un, B)
    ctx.check()
    _close(Un, Un_r, "eq16 Un")
    _close(x_new, x_new_r, "eq16 x_new")
    # B is compared at matching positions: feed the oracle the GPU's own x_new so that the comparison
    # does not amplify the 1e-16 differences of x_new by the stiffness kappa
    B_g = orc.fe_force(wl.conn, wl.X, x_new.cpu().numpy(), wl.fibers, wl.mat_id, wl.mats)["B"]
    _close(B, B_g, "eq16 B")
    f_g = orc.spread(g, wl.x, B_g) if nodal else orc.spread(g, xp, orc.prolong(wl.conn, wl.nsub, wa, Wp, B_g))
    for c in range(3):
        _close(f[c], f_g[c], f"eq16 f{c}")
        assert rel_l2(f_g[c], f_r[c]) < 1e-8              # and the two oracle runs agree to conditioning
    ctx.close()


@pytest.mark.parametrize("name,nodal", [("LV-small", False), ("C1", True)])
def test_step_eq16_three_steps_with_positions_fed_back(ib, orc, name, nodal):
    """NEXT-1's multi-step driver (Eq.(16)) with a frozen velocity field: three calls of
    ib_step_eq16, x_new of one step being x of the next, against the oracle's operators composed in the
    same order over the same three steps (the oracle advances its own positions)."""
    import torch
    wl = CONFIGS[name]()
    dt = 2e-3 * wl.h
    g = _grid(orc, wl)

    def oracle_step(x):
        if nodal:
            Un = orc.interp(g, x, wl.u, wl.v, wl.w)
            xn = x + dt * Un
            B = orc.fe_force(wl.conn, wl.X, xn, wl.fibers, wl.mat_id, wl.mats)["B"]
            return xn, Un, B, orc.spread(g, x, B)
        xp, Wp, wa = orc.points(wl.conn, wl.X, x, wl.nsub)
        Un = orc.restrict(wl.conn, wl.nsub, wa, Wp, orc.interp(g, xp, wl.u, wl.v, wl.w))
        xn = x + dt * Un
        B = orc.fe_force(wl.conn, wl.X, xn, wl.fibers, wl.mat_id, wl.mats)["B"]
        return xn, Un, B, orc.spread(g, xp, orc.prolong(wl.conn, wl.nsub, wa, Wp, B))

    ctx = ib.Context.from_workload(wl, nodal=nodal)
    f = [torch.full((wl.n_cells,), 5.0, dtype=torch.float64, device="cuda") for _ in range(3)]
    Un, B = (torch.empty((3, wl.n_nodes), dtype=torch.float64, device="cuda") for _ in range(2))
    xa, xb = _t(wl.x), torch.empty((3, wl.n_nodes), dtype=torch.float64, device="cuda")
    u, v, w = _t(wl.u), _t(wl.v), _t(wl.w)
    x_r = wl.x.copy()
    for step in range(3):
        ctx.ib_step_eq16(xa, u, v, w, dt, xb, *f, Un, B)
        ctx.check()
        x_r, Un_r, B_r, f_r = oracle_step(x_r)
        _close(xb, x_r, f"step {step} x_new")
        _close(Un, Un_r, f"step {step} Un")
        # the stiffness kappa amplifies the 1e-16 differences of the positions in B and f: compare those
        # with the oracle at the GPU's own positions, and the two oracle runs to conditioning
        B_g = orc.fe_force(wl.conn, wl.X, xb.cpu().numpy(), wl.fibers, wl.mat_id, wl.mats)["B"]
        _close(B, B_g, f"step {step} B")
        assert rel_l2(B_g, B_r) < 1e-8
        x_old = xa.cpu().numpy()
        if nodal:
            f_g = orc.spread(g, x_old, B_g)
        else:
            xp_g, Wp_g, wa_g = orc.points(wl.conn, wl.X, x_old, wl.nsub)
            f_g = orc.spread(g, xp_g, orc.prolong(wl.conn, wl.nsub, wa_g, Wp_g, B_g))
        for c in range(3):
            _close(f[c], f_g[c], f"step {step} f{c}")
            assert rel_l2(f_g[c], f_r[c]) < 1e-8, (step, c)
        xa, xb = xb, xa                                            # x_new becomes x
    assert np.max(np.abs(x_r - wl.x)) > 1e-4 * wl.h                # the structure did move
    ctx.close()


def test_fe_force_next2_laws_and_active_stress(ib, orc):
    """NEXT-2: Eq.(7), Eq.(8)-(9) as an HO special case, Eq.(10)-(11), and the active stress of L317-331,
    mixed element by element on a distorted block."""
    import torch
    conn, X, x, fib = distorted_block(5, 4, 3, seed=21, cur_noise=0.04)
    ne, nn = conn.shape[0], X.shape[1]
    mats = [W.material(W.LAW_MSR, a=8e4, af=1.6e5, bf=2.0e6, kappa=4e6),
            W.material(W.LAW_HO, a=34.0, b=0.0, af=31.0, bf=4.0, kappa=1e3),                  # Eq.(8)-(9)
            W.material(W.LAW_FR2, a=2 * 1.21 * 7.99, b=7.99, af=24.23, bf=57.62, kappa=1e3),
            W.material(W.LAW_HO, Ta=60.0, **W.HO_LV),                                          # active myocardium
            W.material(W.LAW_NEOHOOKEAN, a=100.0, kappa=1e3, Ta=5.0)]
    mid = (np.arange(ne) % len(mats)).astype(np.int32)
    ctx = ib.Context(16, 16, 16, 1 / 16, (0, 0, 0), conn, X, fib, mid, None, mats)
    B = torch.empty((3, nn), dtype=torch.float64, device="cuda")
    ctx.ib_fe_force(_t(x), B)
    ctx.check()
    ref = orc.fe_force(conn, X, x, fib, mid, mats)
    _close(B, ref["B"], "NEXT-2 laws B")
    # each law alone, so that a wrong branch cannot hide behind the stiffest material
    for k, m in enumerate(mats):
        c1 = ib.Context(16, 16, 16, 1 / 16, (0, 0, 0), conn, X, fib, None, None, [m])
        c1.ib_fe_force(_t(x), B)
        c1.check()
        _close(B, orc.fe_force(conn, X, x, fib, np.zeros(ne, np.int32), [m])["B"], f"law {k} B")
        c1.close()
    ctx.close()


# ---- NEXT-3: P1 tetrahedra with the paper's nodal coupling (L241-257, L372, L447) -------------------
def test_tet_mesh_force_and_nodal_coupling_step(ib, orc):
    import torch
    conn_hex, X, x, _ = distorted_block(6, 5, 4, size=(0.3, 0.25, 0.2), seed=31, ref_noise=0.1, cur_noise=0.05)
    tets = W.tets_from_hexes(conn_hex, X)
    ne, nn = tets.shape[0], X.shape[1]
    assert np.bincount(tets.ravel()).max() > 8                   # valence beyond the hex ELL width
    rng = np.random.default_rng(7)
    ef = rng.normal(size=(3, ne))
    ef /= np.linalg.norm(ef, axis=0)
    es = np.cross(ef.T, rng.normal(size=(ne, 3))).T
    es /= np.linalg.norm(es, axis=0)
    fib = np.concatenate([ef, es])
    mats = [W.material(W.LAW_NEOHOOKEAN, a=1e4, kappa=1e6), W.material(W.LAW_HO, Ta=20.0, **W.HO_LV),
            W.material(W.LAW_FR2, a=2 * 1.21 * 7.99, b=7.99, af=24.23, bf=57.62, kappa=1e3)]
    mid = (np.arange(ne) % 3).astype(np.int32)
    n, h, org = (32, 32, 32), 1 / 32, (0.0, 0.0, 0.0)
    g = orc.make_grid(*n, h, org)
    uvw = np.random.default_rng(8).normal(size=(3, n[0] * n[1] * n[2]))
    ref_B = orc.fe_force(tets, X, x, fib, mid, mats)["B"]
    ref_f = orc.spread(g, x, ref_B)
    ref_U = orc.interp(g, x, *uvw)
    for variant in (0, 1):
        ctx = ib.Context(*n, h, org, tets, X, fib, mid, None, mats)
        ctx.ib_set_variant(variant)
        B = torch.empty((3, nn), dtype=torch.float64, device="cuda")
        ctx.ib_fe_force(_t(x), B)
        ctx.check()
        _close(B, ref_B, "tet B")
        B2 = torch.empty_like(B)
        ctx.ib_fe_force(_t(x), B2)
        assert torch.equal(B, B2)                                 # CSR node gather: bit-reproducible
        f = [torch.full((g.nx * g.ny * g.nz,), 2.0, dtype=torch.float64, device="cuda") for _ in range(3)]
        Un = torch.empty((3, nn), dtype=torch.float64, device="cuda")
        ctx.ib_coupling_step(_t(x), _t(uvw[0]), _t(uvw[1]), _t(uvw[2]), *f, Un, B)
        ctx.check()
        for c in range(3):
            _close(f[c], ref_f[c], f"tet v{variant} f{c}")
        _close(Un, ref_U, f"tet v{variant} Un")
        # inverted tetrahedron is latched
        xi = x.copy()
        t0 = tets[5]
        xi[:, t0[3]] = 2 * x[:, t0[0]] - x[:, t0[3]] + (x[:, t0[1]] - x[:, t0[0]])
        ctx.ib_fe_force(_t(xi), B)
        assert ctx.ib_check()[0] == 5
        ctx.close()
    # sub-point coupling is not defined for tetrahedra
    with pytest.raises(ib.IbError):
        ib.Context(*n, h, org, tets, X, fib, mid, np.ones((ne, 3), np.int32), mats)


def test_graph_replay_matches_eager_step(ib, orc):
    """On a non-default stream the third call with the same pointers replays a captured CUDA graph
    (two side streams inside); results equal the eager step's to the order of the atomic sums, B bit for bit."""
    import torch
    for name, nodal in (("C1", False), ("LV-small", False), ("C1", True)):
        wl = CONFIGS[name]()
        eager = _run_step(ib, wl, 1, nodal=nodal)                       # default stream: never captured
        ctx = ib.Context.from_workload(wl, nodal=nodal)
        st = torch.cuda.Stream()
        with torch.cuda.stream(st):
            x, u, v, w = _t(wl.x), _t(wl.u), _t(wl.v), _t(wl.w)
            fu, fv, fw = (torch.full((wl.n_cells,), 7.0, dtype=torch.float64, device="cuda") for _ in range(3))
            Un = torch.empty((3, wl.n_nodes), dtype=torch.float64, device="cuda")
            B = torch.empty((3, wl.n_nodes), dtype=torch.float64, device="cuda")
            counts = []
            for it in range(4):
                fu.fill_(3.0 + it)
                l0 = ctx.ib_launch_count()
                ctx.ib_coupling_step(x, u, v, w, fu, fv, fw, Un, B, st)
                counts.append(ctx.ib_launch_count() - l0)
                ctx.check()
                assert np.array_equal(B.cpu().numpy(), eager["B"])
                for k, t in (("fu", fu), ("fv", fv), ("fw", fw), ("Un", Un)):
                    assert max_abs_scaled(t.cpu().numpy(), eager[k]) <= 1e-12, (name, it, k)
            assert len(set(counts)) == 1                                # replay reports the same launches
            # new pointers: falls back to eager, then captures again
            Un2 = torch.empty_like(Un)
            for it in range(3):
                ctx.ib_coupling_step(x, u, v, w, fu, fv, fw, Un2, B, st)
            ctx.check()
            assert max_abs_scaled(Un2.cpu().numpy(), eager["Un"]) <= 1e-12
        st.synchronize()
        ctx.close()


# ---- NEXT-4: solid boundary loads ---------------------------------------------------------------------
@pytest.mark.parametrize("kind", ["hex-sub", "hex-nodal", "tet", "tet10"])
def test_boundary_loads_enter_force_and_step(ib, orc, kind):
    """Tethers (L263, L425), dead traction (L263) and follower pressure (L303, L315) are added to B by
    ib_fe_force and reach the grid through the step (Fhat = B / w_a includes them)."""
    import torch
    conn, X, x, fib = distorted_block(5, 4, 3, size=(0.3, 0.25, 0.2), seed=41, ref_noise=0.1, cur_noise=0.05)
    if kind in ("tet", "tet10"):
        conn = W.tets_from_hexes(conn, X)
        fib = None
    if kind == "tet10":                                           # 6-node faces with curved edges (reading A27)
        nv = X.shape[1]
        conn, X = W.p2_from_tets(conn, X)
        rng = np.random.default_rng(43)
        X[:, nv:] += 0.004 * rng.uniform(-1, 1, (3, X.shape[1] - nv))
        x = X + 0.004 * rng.uniform(-1, 1, X.shape)
    ne, nn = conn.shape[0], X.shape[1]
    nsub = np.tile([3, 2, 2], (ne, 1)).astype(np.int32) if kind == "hex-sub" else None
    mats = [W.material(W.LAW_NEOHOOKEAN, a=80.0, kappa=4e4)]
    faces = W.boundary_faces(conn)
    left = np.unique(faces[np.all(X[0, faces] < X[0].min() + 0.03, axis=1)])
    qt0, p, kap = np.array([0.0, 6.25, -1.0]), 14.53, 1e6
    B_r = orc.fe_force(conn, X, x, fib, None, mats)["B"]
    B_r, _ = orc.tethers(left, X, x, kap, B_r)
    B_r = orc.surface_loads(faces, X, x, qt0, p, B_r)
    n, h, org = (32, 32, 32), 1 / 32, (0.0, 0.0, 0.0)
    g = orc.make_grid(*n, h, org)
    if nsub is None:
        f_r = orc.spread(g, x, B_r)
    else:
        xp, Wp, wa = orc.points(conn, X, x, nsub)
        f_r = orc.spread(g, xp, orc.prolong(conn, nsub, wa, Wp, B_r))
    ctx = ib.Context(*n, h, org, conn, X, fib, None, nsub, mats)
    ctx.ib_set_tethers(left, kap)
    ctx.ib_set_surface(faces)
    ctx.ib_set_loads(qt0, p)
    B = torch.empty((3, nn), dtype=torch.float64, device="cuda")
    ctx.ib_fe_force(_t(x), B)
    ctx.check()
    _close(B, B_r, f"{kind} loaded B")
    ncell = n[0] * n[1] * n[2]
    uvw = np.random.default_rng(2).normal(size=(3, ncell))
    f = [torch.empty(ncell, dtype=torch.float64, device="cuda") for _ in range(3)]
    Un = torch.empty((3, nn), dtype=torch.float64, device="cuda")
    ctx.ib_coupling_step(_t(x), _t(uvw[0]), _t(uvw[1]), _t(uvw[2]), *f, Un, B)
    ctx.check()
    for c in range(3):
        _close(f[c], f_r[c], f"{kind} loaded f{c}")
    # loads off again: back to the plain elastic force
    ctx.ib_set_tethers([], 0.0)
    ctx.ib_set_loads(None, 0.0)
    ctx.ib_fe_force(_t(x), B)
    _close(B, orc.fe_force(conn, X, x, fib, None, mats)["B"], f"{kind} unloaded B")
    ctx.close()


@pytest.mark.parametrize("variant", [0, 1])
def test_spread_interp_heavy_contention(ib, orc, variant):
    """Degenerate clouds: 60,000 points inside ONE cell (32 chunks of one tile, every item crowded, all
    atomics on the same 3 x 64 faces), many exactly coincident points, and a cloud of exactly one point."""
    import torch
    n, h, org = (16, 16, 24), 0.1, (0.0, -0.5, 1.0)
    ctx = ib.Context(*n, h, org, np.zeros((0, 8), np.int32), np.zeros((3, 0)), None, None, None, [])
    ctx.ib_set_variant(variant)
    g = orc.make_grid(*n, h, org)
    rng = np.random.default_rng(11)
    ncell = n[0] * n[1] * n[2]
    uvw = rng.normal(size=(3, ncell))
    for P, where in ((60000, "cell"), (4096, "same"), (1, "same")):
        base = np.asarray(org) + h * np.array([15.0, 0.0, 23.0])            # a corner cell: supports wrap in x, y and z
        xp = base[:, None] + (rng.uniform(0, h, (3, P)) if where == "cell" else np.full((3, P), 0.37 * h))
        G = rng.normal(size=(3, P))
        f = [torch.empty(ncell, dtype=torch.float64, device="cuda") for _ in range(3)]
        Up = torch.empty((3, P), dtype=torch.float64, device="cuda")
        ctx.ib_spread(_t(xp), _t(G), P, *f, accumulate=0)
        ctx.ib_interp(_t(xp), P, _t(uvw[0]), _t(uvw[1]), _t(uvw[2]), Up)
        ctx.check()
        fr = orc.spread(g, xp, G)
        for c in range(3):
            _close(f[c], fr[c], f"contention {where} {P} f{c}")
            assert abs(h ** 3 * float(f[c].sum()) - G[c].sum()) <= 1e-11 * np.abs(G[c]).sum()
        _close(Up, orc.interp(g, xp, *uvw), f"contention {where} {P} U")
    ctx.close()


def test_p2_tet_mesh_force_and_nodal_step(ib, orc):
    """NEXT-3, second half: P2 tetrahedra (L265) with curved edges, mixed laws, nodal coupling."""
    import torch
    conn_hex, X, _, _ = distorted_block(5, 4, 3, size=(0.3, 0.25, 0.2), seed=51, ref_noise=0.1, cur_noise=0.0)
    c10, X10 = W.p2_from_tets(W.tets_from_hexes(conn_hex, X), X)
    rng = np.random.default_rng(5)
    X10[:, X.shape[1]:] += 0.003 * rng.uniform(-1, 1, (3, X10.shape[1] - X.shape[1]))      # curved edges
    x10 = X10 + 0.004 * rng.uniform(-1, 1, X10.shape)
    ne, nn = c10.shape[0], X10.shape[1]
    ef = rng.normal(size=(3, ne))
    ef /= np.linalg.norm(ef, axis=0)
    es = np.cross(ef.T, rng.normal(size=(ne, 3))).T
    es /= np.linalg.norm(es, axis=0)
    fib = np.concatenate([ef, es])
    mats = [W.material(W.LAW_MSR, a=8e4, af=1.6e5, bf=2.0e6, kappa=4e6),                    # Cook's membrane law
            W.material(W.LAW_HO, Ta=20.0, **W.HO_LV), W.material(W.LAW_NEOHOOKEAN, a=1e4, kappa=1e6)]
    mid = (np.arange(ne) % 3).astype(np.int32)
    n, h, org = (32, 32, 32), 1 / 32, (0.0, 0.0, 0.0)
    g = orc.make_grid(*n, h, org)
    uvw = rng.normal(size=(3, n[0] * n[1] * n[2]))
    ref_B = orc.fe_force(c10, X10, x10, fib, mid, mats)["B"]
    ctx = ib.Context(*n, h, org, c10, X10, fib, mid, None, mats)
    B = torch.empty((3, nn), dtype=torch.float64, device="cuda")
    ctx.ib_fe_force(_t(x10), B)
    ctx.check()
    _close(B, ref_B, "P2 B")
    f = [torch.empty(n[0] * n[1] * n[2], dtype=torch.float64, device="cuda") for _ in range(3)]
    Un = torch.empty((3, nn), dtype=torch.float64, device="cuda")
    ctx.ib_coupling_step(_t(x10), _t(uvw[0]), _t(uvw[1]), _t(uvw[2]), *f, Un, B)
    ctx.check()
    ref_f = orc.spread(g, x10, ref_B)
    for c in range(3):
        _close(f[c], ref_f[c], f"P2 f{c}")
    _close(Un, orc.interp(g, x10, *uvw), "P2 Un")
    ctx.close()


# ---- NEXT-4, second half: bounded (non-periodic) grid, supports truncated at the walls (A26) -------
@pytest.mark.parametrize("variant", [0, 1])
def test_bounded_grid_cloud_and_mesh(ib, orc, variant):
    import torch
    n, h, org = (24, 16, 32), 0.05, (-0.4, 0.1, 0.3)
    L = np.array(n) * h
    g = orc.make_grid(*n, h, org, periodic=0)
    rng = np.random.default_rng(13)
    ncell = n[0] * n[1] * n[2]
    uvw = rng.normal(size=(3, ncell))
    # a cloud filling the box right up to the walls (dense near two corners), one point outside
    P = 30011
    xp = np.asarray(org)[:, None] + rng.uniform(0.0, 1.0, (3, P)) * L[:, None]
    xp[:, :4000] = np.asarray(org)[:, None] + rng.uniform(0.0, 1.9 * h, (3, 4000))
    xp[:, 4000:8000] = (np.asarray(org) + L)[:, None] - rng.uniform(1e-9, 1.9 * h, (3, 4000))
    G = rng.normal(size=(3, P))
    ctx = ib.Context(*n, h, org, np.zeros((0, 8), np.int32), np.zeros((3, 0)), None, None, None, [], periodic=0)
    ctx.ib_set_variant(variant)
    f = [torch.empty(ncell, dtype=torch.float64, device="cuda") for _ in range(3)]
    Up = torch.empty((3, P), dtype=torch.float64, device="cuda")
    ctx.ib_spread(_t(xp), _t(G), P, *f, accumulate=0)
    ctx.ib_interp(_t(xp), P, _t(uvw[0]), _t(uvw[1]), _t(uvw[2]), Up)
    ctx.check()
    fr = orc.spread(g, xp, G)
    for c in range(3):
        _close(f[c], fr[c], f"bounded v{variant} f{c}")
    _close(Up, orc.interp(g, xp, *uvw), f"bounded v{variant} U")
    xo = xp.copy()
    xo[0, 17] = org[0] - 0.3 * h                                  # outside the box: latched, skipped, U = 0
    ctx.ib_interp(_t(xo), P, _t(uvw[0]), _t(uvw[1]), _t(uvw[2]), Up)
    code, bad = ctx.ib_check()
    assert code == 7 and bad == 17 and float(Up[:, 17].abs().max()) == 0.0
    ctx.close()
    # a structure pushed into the corner of the box: sub-point coupling through the whole step
    wl = W.config1()
    shift = np.asarray(wl.origin) - wl.X.min(axis=1) + 0.3 * wl.h         # 0.3 h from three walls
    X, x = wl.X + shift[:, None], wl.x + shift[:, None]
    gb = orc.make_grid(wl.nx, wl.ny, wl.nz, wl.h, wl.origin, periodic=0)
    ref = orc.coupling_step(gb, wl.conn, X, wl.fibers, wl.mat_id, wl.nsub, wl.mats, x, wl.u, wl.v, wl.w)
    ctx = ib.Context(wl.nx, wl.ny, wl.nz, wl.h, wl.origin, wl.conn, X, wl.fibers, wl.mat_id, wl.nsub, wl.mats, periodic=0)
    ctx.ib_set_variant(variant)
    fo = [torch.empty(wl.n_cells, dtype=torch.float64, device="cuda") for _ in range(3)]
    Un, B = (torch.empty((3, wl.n_nodes), dtype=torch.float64, device="cuda") for _ in range(2))
    ctx.ib_coupling_step(_t(x), _t(wl.u), _t(wl.v), _t(wl.w), *fo, Un, B)
    ctx.check()
    for k, t in (("B", B), ("fu", fo[0]), ("fv", fo[1]), ("fw", fo[2]), ("Un", Un)):
        _close(t, ref[k], f"bounded step v{variant} {k}")
    ctx.close()


def test_create_and_setters_reject_bad_input(ib):
    """What ib_create and the setters refuse (include/ibcouple.h: error behaviour): each case names the status code
    the header states, and a refused creation leaves no context behind."""
    conn, X, x, fib = distorted_block(3, 3, 2, seed=3)
    ne, nn = conn.shape[0], X.shape[1]
    mats = [W.material(0, a=1.0, kappa=10.0)]
    sub = np.full((ne, 3), 2, np.int32)
    good = lambda **kw: dict(dict(nx=16, ny=16, nz=16, h=1 / 16, origin=(0, 0, 0), conn=conn, X=X, fibers=fib,
                                  mat_id=None, nsub=sub, mats=mats), **kw)
    ib.Context(**good()).close()                                            # the unmodified case is accepted
    INVALID, UNSUPPORTED = 1, 2

    def refused(code, **kw):
        with pytest.raises(ib.IbError) as e:
            ib.Context(**good(**kw))
        assert e.value.code == code, (kw.keys(), e.value)

    refused(INVALID, nx=12)                                                 # grid edge not a multiple of the tile edge
    refused(INVALID, h=0.0)
    refused(INVALID, h=float("nan"))
    refused(UNSUPPORTED, nx=4104, ny=8, nz=8)                               # tile coordinates are packed in 10 + 10 + 11 bits
    bad = conn.copy(); bad[2, 5] = nn
    refused(INVALID, conn=bad)                                              # node id out of range
    bad = conn.copy(); bad[2, 5] = -1
    refused(INVALID, conn=bad)
    s9 = sub.copy(); s9[1, 2] = 9
    refused(INVALID, nsub=s9)                                               # at most 8 sub-points per direction
    s0 = sub.copy(); s0[0, 0] = 0
    refused(INVALID, nsub=s0)
    refused(INVALID, mat_id=np.full(ne, 1, np.int32))                       # material index beyond the table
    Xo = np.concatenate([X, X[:, :1] + 5.0], axis=1)
    refused(INVALID, X=Xo)                                                  # a node of no element has lumped weight 0 (A13)
    ib.Context(**good(X=Xo, nsub=None)).close()                             # ... which the nodal rule does not need
    law9 = [dict(mats[0], law=9)]
    refused(INVALID, mats=law9)
    # nine elements at one node: the ELL adjacency holds eight
    star = np.concatenate([conn, conn[:1]], axis=0)
    refused(UNSUPPORTED, conn=star, nsub=np.full((ne + 1, 3), 2, np.int32),
            fibers=None if fib is None else np.concatenate([fib, fib[:, :1]], axis=1))

    ctx = ib.Context(**good())
    for call, args in ((ctx.ib_set_variant, (2,)), (ctx.ib_set_tethers, ([0, 1, 1], 10.0)),
                       (ctx.ib_set_tethers, ([nn], 10.0)), (ctx.ib_set_tethers, ([0], float("inf"))),
                       (ctx.ib_set_surface, (np.array([[0, 1, 2, nn]], np.int32),))):
        with pytest.raises(ib.IbError) as e:
            call(*args)
        assert e.value.code == INVALID, (call.__name__, args)
    ctx.ib_set_tethers([0, 1, 2], 10.0)                                     # and the context still works
    ctx.close()
