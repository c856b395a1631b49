"""Philox Gaussian vectors, generated on the host and handed to both the oracle and the GPU path."""
import numpy as np


def gaussian_inputs(N, seed=0):
    """F (N,3) and S (N,5), i.i.d. N(0,1) drawn in fp64 from Philox(seed) and rounded once to fp32; both the
    oracle (which widens them back to fp64) and the GPU consume the rounded values."""
    g = np.random.Generator(np.random.Philox(seed))
    F = g.standard_normal((N, 3)).astype(np.float32)
    S = g.standard_normal((N, 5)).astype(np.float32)
    return F, S


def brownian_noise(N, Mg, seed=0):
    """w1 (8N,) then the wave buffer [3][Mg][Mg][Mg/2+1][2], fp32 N(0,1) from Philox(seed)."""
    g = np.random.Generator(np.random.Philox(seed))
    w1 = g.standard_normal(8 * N).astype(np.float32)
    w2 = g.standard_normal((3, Mg, Mg, Mg // 2 + 1, 2), dtype=np.float32)
    return w1, w2
