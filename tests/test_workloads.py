"""Input generators: sizes of SURVEY.md §8(d), determinism, wall margins (no GPU, no oracle)."""
import numpy as np

from paper_2503_22695_b200 import workloads as W


def _margin_ok(wl, cells=6):
    lo = np.array(wl.origin) + cells * wl.h
    hi = np.array(wl.origin) + (np.array([wl.nx, wl.ny, wl.nz]) - cells) * wl.h
    return np.all(wl.x.min(axis=1) > lo) and np.all(wl.x.max(axis=1) < hi)


def test_config_sizes_match_survey_table():
    c1, c2, c3, c4 = W.config1(), W.config2(), W.config3(), W.config4()
    assert (c1.n_elems, c1.n_nodes, c1.n_points, c1.n_cells) == (128, 243, 8192, 32 ** 3)
    assert (c2.n_elems, c2.n_nodes, c2.n_points, c2.n_cells) == (4096, 5445, 65536, 64 ** 3)
    assert (c3.n_elems, c3.n_nodes, c3.n_points, c3.n_cells) == (98304, 111744, 6291456, 128 ** 3)
    assert (c4.n_elems, c4.n_nodes, c4.n_points, c4.n_cells) == (67584, 91065, 393216, 256 * 128 * 128)
    for wl in (c1, c2, c3, c4):
        assert _margin_ok(wl), wl.name
        assert wl.conn.dtype == np.int32 and wl.conn.min() == 0 and wl.conn.max() == wl.n_nodes - 1
        assert wl.u.shape == (wl.n_cells,) and np.isfinite(wl.u).all()
        # every node belongs to at most 8 elements (ELL adjacency bound used by the CUDA path)
        assert np.bincount(wl.conn.ravel()).max() <= 8
    assert abs(c3.h - 0.078125) < 1e-15 and abs(c4.h - 0.03125) < 1e-15
    # determinism: same seed -> same bytes
    assert W.config2().sha256() == c2.sha256()


def test_config5_ladder_counts():
    l1 = W.config5(level=1, sub=2)
    assert (l1.n_elems, l1.n_points) == (12288, 98304)
    l2 = W.config5(level=2, sub=3)
    assert (l2.n_elems, l2.n_points) == (98304, 98304 * 27)
    assert _margin_ok(l2)


def test_velocity_field_is_the_stated_fourier_sum():
    # u at face (i, j+1/2, k+1/2)h is sum_m cos(2 pi k_m.(x-x0)/L + theta_m): check by direct evaluation
    wl = W.config1()
    rng = np.random.default_rng([W.SEED_ROOT, 1, 2])
    km = []
    for m in range(8):
        while True:
            k = rng.integers(-4, 5, size=3)
            if np.any(k != 0):
                break
        km.append(k)
    th = rng.uniform(0, 2 * np.pi, size=8)
    for (i, j, k) in [(0, 0, 0), (5, 17, 30), (31, 31, 31)]:
        fx, fy, fz = i / 32, (j + .5) / 32, (k + .5) / 32
        val = sum(np.cos(2 * np.pi * (q[0] * fx + q[1] * fy + q[2] * fz) + t) for q, t in zip(km, th))
        assert abs(wl.u[(k * 32 + j) * 32 + i] - val) < 1e-12
