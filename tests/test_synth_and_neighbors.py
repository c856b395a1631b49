"""Input generators and the brute-force neighbour oracle (CPU only)."""
import numpy as np

import synth
from oracle import neighbors as nbo


def test_rsa_no_overlap_and_seeded():
    x, L = synth.rsa(512, 0.20, seed=3)
    assert abs(L - (4 * np.pi * 512 / (3 * 0.20)) ** (1 / 3)) < 1e-12
    assert x.shape == (512, 3) and x.min() >= 0 and x.max() < L
    assert synth.suspensions.min_separation(x, L) > 2.0
    x2, _ = synth.rsa(512, 0.20, seed=3)
    assert np.array_equal(x, x2)
    x3, _ = synth.rsa(512, 0.20, seed=4)
    assert not np.array_equal(x, x3)


def test_relax_keeps_hard_spheres():
    x, L = synth.rsa(256, 0.30, seed=1)
    y = synth.relax_overlaps(x, L, sweeps=3, seed=1)
    assert synth.suspensions.min_separation(y, L) >= 2.0
    assert np.abs(y - x).max() > 0


def test_noise_shapes_and_determinism():
    F, S = synth.gaussian_inputs(64, 0)
    assert F.dtype == np.float32 and F.shape == (64, 3) and S.shape == (64, 5)
    w1, w2 = synth.brownian_noise(64, 32, 0)
    assert w1.shape == (512,) and w2.shape == (3, 32, 32, 17, 2) and w2.dtype == np.float32
    assert np.array_equal(w1, synth.brownian_noise(64, 32, 0)[0])
    assert abs(float(w2.std()) - 1) < 0.01


def test_neighbor_oracle_against_fp64_brute_force():
    """Away from the fp32 decision boundary the fp32 sets equal the exact ones; they are symmetric; wrap works."""
    x, L = synth.rsa(200, 0.15, seed=2)
    rc = 5.0
    sets = nbo.neighbor_sets(x.astype(np.float32), L, rc)
    d = x[:, None] - x[None]
    d -= L * np.round(d / L)
    r = np.linalg.norm(d, axis=2)
    for a in range(200):
        exact = set(np.nonzero((r[a] < rc) & (np.arange(200) != a))[0])
        fuzzy = set(np.nonzero(np.abs(r[a] - rc) < 1e-4)[0])
        assert set(sets[a]) - fuzzy == exact - fuzzy
        for b in sets[a]:
            assert a in sets[b]
    shifted = (x + L * np.array([1, -2, 3])).astype(np.float32)
    w = nbo.wrap32(shifted, L)
    assert w.min() >= 0 and w.max() < np.float32(L)
