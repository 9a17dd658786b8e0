"""Small seeded meshes and comparison helpers shared by the tests (inputs only, no method arithmetic)."""
import numpy as np

from paper_2503_22695_b200 import workloads as W


def distorted_block(n1=3, n2=3, n3=2, size=(0.3, 0.3, 0.2), origin=(0.35, 0.35, 0.4), seed=0,
                    ref_noise=0.15, cur_noise=0.08):
    """Structured hex block whose REFERENCE nodes are perturbed (distorted elements) and whose
    current nodes are perturbed again. Returns conn [ne,8], X [3,nn], x [3,nn], fibers [6,ne]."""
    rng = np.random.default_rng([7, seed])
    conn, (N1, N2, N3) = W.block_connectivity(n1, n2, n3)
    k, j, i = np.meshgrid(np.arange(N3), np.arange(N2), np.arange(N1), indexing="ij")
    d = np.array([size[0] / n1, size[1] / n2, size[2] / n3])
    X = np.stack([origin[0] + i.ravel() * d[0], origin[1] + j.ravel() * d[1], origin[2] + k.ravel() * d[2]])
    X = X + rng.uniform(-ref_noise, ref_noise, X.shape) * d[:, None]
    x = X + rng.uniform(-cur_noise, cur_noise, X.shape) * d[:, None]
    ne = conn.shape[0]
    ef = rng.normal(size=(3, ne))
    ef /= np.linalg.norm(ef, axis=0)
    es = rng.normal(size=(3, ne))
    es -= np.sum(es * ef, axis=0) * ef
    es /= np.linalg.norm(es, axis=0)
    return conn.astype(np.int32), X, x, np.concatenate([ef, es])


def rel_l2(a, b):
    a, b = np.asarray(a, dtype=np.float64).ravel(), np.asarray(b, dtype=np.float64).ravel()
    nb = np.linalg.norm(b)
    return np.linalg.norm(a - b) / (nb if nb > 0 else 1.0)


def max_abs_scaled(a, b):
    a, b = np.asarray(a, dtype=np.float64).ravel(), np.asarray(b, dtype=np.float64).ravel()
    s = np.max(np.abs(b)) if b.size else 0.0
    return (np.max(np.abs(a - b)) if a.size else 0.0) / (s if s > 0 else 1.0)


def rotation(seed=0):
    rng = np.random.default_rng([11, seed])
    Q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
    if np.linalg.det(Q) < 0:
        Q[:, 0] *= -1
    return Q
