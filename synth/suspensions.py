"""Seeded particle placements: monodisperse spheres of radius a in a cubic periodic box of edge L.

No hydrodynamics here — only geometry.  scipy's periodic KD-tree is used for overlap queries.
"""
import numpy as np
from scipy.spatial import cKDTree


def box_length(N, phi, a=1.0):
    """L = (4 pi N a^3 / (3 phi))^(1/3)  (BASELINE.json configs)."""
    return float((4.0 * np.pi * N * a**3 / (3.0 * phi)) ** (1.0 / 3.0))


def _greedy_keep(cand, L, dmin):
    """Sequential acceptance among candidates (in proposal order): keep j iff no kept i < j within dmin."""
    if len(cand) < 2:
        return np.ones(len(cand), bool)
    pairs = cKDTree(cand, boxsize=L).query_pairs(dmin, output_type='ndarray')
    keep = np.ones(len(cand), bool)
    if len(pairs):
        lo, hi = pairs.min(axis=1), pairs.max(axis=1)
        order = np.argsort(hi, kind='stable')
        for i, j in zip(lo[order], hi[order]):
            if keep[i] and keep[j]:
                # all conflicts of j with lower indices are visited before any pair whose larger index exceeds j
                keep[j] = False
    return keep


def rsa(N, phi, seed=0, a=1.0, max_rounds=100000):
    """Random sequential addition: uniform proposals in [0,L)^3 from Philox(seed), accepted iff the
    minimum-image distance to every earlier accepted centre exceeds 2a.  Returns (x (N,3) fp64, L)."""
    L = box_length(N, phi, a)
    g = np.random.Generator(np.random.Philox(seed))
    dmin = 2.0 * a * (1.0 + 1e-9)
    acc = np.empty((N, 3))
    n = 0
    rate = 1.0
    for _ in range(max_rounds):
        if n >= N:
            break
        K = int(min(max(256, 1.5 * (N - n) / max(rate, 1e-4)), 400_000))
        cand = g.random((K, 3)) * L
        if n:
            d, _ = cKDTree(acc[:n], boxsize=L).query(cand, k=1, distance_upper_bound=dmin)
            cand = cand[np.isinf(d)]
        cand = cand[_greedy_keep(cand, L, dmin)]
        take = min(len(cand), N - n)
        acc[n:n + take] = cand[:take]
        n += take
        rate = 0.5 * rate + 0.5 * max(take / K, 1e-4)
    if n < N:
        raise RuntimeError(f'RSA stalled at {n}/{N} (phi={phi})')
    return acc, L


def relax_overlaps(x, L, a=1.0, sweeps=10, kick=0.05, seed=0, max_push=200):
    """Equilibration sweeps for config 3: Gaussian kick of std `kick`*a on every centre, then symmetric
    push-apart of every overlapping pair to contact, repeated until overlap-free."""
    g = np.random.Generator(np.random.Philox(seed + 7919))
    x = np.array(x, dtype=np.float64)
    dmin = 2.0 * a
    for _ in range(sweeps):
        x = (x + kick * a * g.standard_normal(x.shape)) % L
        for _ in range(max_push):
            pairs = cKDTree(x, boxsize=L).query_pairs(dmin, output_type='ndarray')
            if len(pairs) == 0:
                break
            d = x[pairs[:, 0]] - x[pairs[:, 1]]
            d -= L * np.round(d / L)
            r = np.linalg.norm(d, axis=1)
            push = 0.5 * (dmin * (1 + 1e-6) - r)[:, None] * d / r[:, None]
            np.add.at(x, pairs[:, 0], push)
            np.add.at(x, pairs[:, 1], -push)
            x %= L
        else:
            raise RuntimeError('relax_overlaps did not converge')
    return x


def min_separation(x, L):
    d, _ = cKDTree(x, boxsize=L).query(x, k=2)
    return float(d[:, 1].min())


def _random_rotation(g):
    q = g.standard_normal(4)
    q /= np.linalg.norm(q)
    w, x, y, z = q
    return np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)],
                     [2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)],
                     [2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)]])


def _stick(PA, PB, g, a):
    """Cluster-cluster sticking: B (randomly rotated) approaches A along a random line with a random impact
    offset and stops at first contact r = 2a(1+1e-6).  Returns the merged, re-centred cluster."""
    dc = 2.0 * a * (1.0 + 1e-6)
    RA = np.linalg.norm(PA, axis=1).max() + a
    while True:
        B = PB @ _random_rotation(g).T
        RB = np.linalg.norm(B, axis=1).max() + a
        u = g.standard_normal(3)
        u /= np.linalg.norm(u)
        p = np.cross(u, g.standard_normal(3))
        p /= np.linalg.norm(p)
        q = np.cross(u, p)
        rho, th = (RA + RB) * np.sqrt(g.random()), 2 * np.pi * g.random()
        c0 = (RA + RB + dc) * u + rho * (np.cos(th) * p + np.sin(th) * q)
        w = (B + c0)[None, :, :] - PA[:, None, :]                  # (nA, nB, 3)
        wu = w @ u
        disc = dc * dc - (np.einsum('abi,abi->ab', w, w) - wu * wu)
        hit = disc >= 0
        if not hit.any():
            continue
        s = (wu - np.sqrt(np.where(hit, disc, 0.0)))[hit].min()
        merged = np.concatenate([PA, B + c0 - s * u])
        return merged - merged.mean(axis=0)


def cluster(n, g, a=1.0):
    """One aggregate of n = 2^k spheres by hierarchical cluster-cluster aggregation (equal sizes merge)."""
    if n == 1:
        return np.zeros((1, 3))
    return _stick(cluster(n // 2, g, a), cluster(n - n // 2, g, a), g, a)


def radius_of_gyration(P):
    return float(np.sqrt(((P - P.mean(axis=0))**2).sum(axis=1).mean()))


def fractal_aggregates(N, phi, seed=0, a=1.0, cluster_size=32, pool=32, max_tries=2000000):
    """Config 5 stand-in: N spheres as N/cluster_size fractal aggregates (hierarchical cluster-cluster
    aggregation, mass fractal dimension measured ~1.8-1.9 from R_g ~ n^(1/d_f)), placed at random positions and
    orientations without sphere overlap at overall volume fraction phi.  A pool of `pool` distinct aggregates
    is built from Philox(seed) and re-used with fresh rotations.  Returns (x (N,3), L)."""
    assert N % cluster_size == 0
    L = box_length(N, phi, a)
    g = np.random.Generator(np.random.Philox(seed))
    shapes = [cluster(cluster_size, g, a) for _ in range(pool)]
    x = np.empty((N, 3))
    n = 0
    dmin = 2.0 * a * (1.0 + 1e-9)
    tree, n_tree = None, 0                       # k-d tree over x[:n_tree]; x[n_tree:n] is checked directly until the next rebuild
    for _ in range(max_tries):
        if n >= N:
            break
        P = (shapes[int(g.integers(pool))] @ _random_rotation(g).T + g.random(3) * L) % L
        if tree is not None:
            d, _ = tree.query(P, k=1, distance_upper_bound=dmin)
            if not np.all(np.isinf(d)):
                continue
        if n > n_tree:
            dd = P[:, None, :] - x[None, n_tree:n, :]
            dd -= L * np.round(dd / L)
            if np.einsum('ijk,ijk->ij', dd, dd).min() < dmin * dmin:
                continue
        x[n:n + cluster_size] = P
        n += cluster_size
        if n - n_tree >= max(cluster_size, n_tree // 16):
            tree, n_tree = cKDTree(x[:n], boxsize=L), n
    if n < N:
        raise RuntimeError(f'aggregate placement stalled at {n}/{N}')
    return x, L
