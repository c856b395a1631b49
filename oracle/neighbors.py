"""Brute-force neighbour sets in the GPU's own fp32 arithmetic (reading R16).  Test infrastructure only.

The paper only says "linked-cell lists ... sub-cells of size r_cut"; which pairs are inside the
cutoff is decided by an fp32 comparison, so both sides must take it in the same precision and operation order:
    wrap:  x' = x - L * floorf(x * (1/L))   (each op rounded to fp32; x' := 0 if x' >= L or x' < 0)
    d = x'_a - x'_b ;  d -= L * rintf(d * (1/L)) ;  r2 = (dx*dx + dy*dy) + dz*dz ;  neighbour iff r2 < rcut*rcut
"""
import numpy as np

f32 = np.float32


def wrap32(pos, L):
    x = np.asarray(pos, dtype=f32)[:, :3]
    L32 = f32(L)
    invL = f32(1.0) / L32
    w = (x - (L32 * np.floor(x * invL).astype(f32)).astype(f32)).astype(f32)
    w[(w >= L32) | (w < 0)] = f32(0)
    return w


def neighbor_sets(pos, L, rcut, rows=None):
    """List (length N, or len(rows)) of sorted int arrays: all beta != alpha with minimum-image fp32 r2 < rcut^2."""
    x = wrap32(pos, L)
    L32 = f32(L)
    invL = f32(1.0) / L32
    rc2 = f32(rcut) * f32(rcut)
    out = []
    for a in (range(x.shape[0]) if rows is None else rows):
        d = (x[a][None, :] - x).astype(f32)
        d = (d - (L32 * np.rint((d * invL).astype(f32)).astype(f32)).astype(f32)).astype(f32)
        sq = (d * d).astype(f32)
        r2 = ((sq[:, 0] + sq[:, 1]).astype(f32) + sq[:, 2]).astype(f32)
        m = r2 < rc2
        m[a] = False
        out.append(np.nonzero(m)[0].astype(np.int64))
    return out
