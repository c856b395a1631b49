"""Deformed periodic lattices: the grand mobility by direct Ewald sums when the
periodic cell is the unit cube of edge L mapped by a volume-preserving linear deformation A, i.e. the lattice vectors are
the columns of L A ("r = A . z").  fp64, test infrastructure only.

    simple shear       A = [[1, g, 0], [0, 1, 0], [0, 0, 1]]          Eq. (56), PAPER.md:318   (Lees-Edwards)
    planar extension   A = diag(e, 1/e, 1)                            Eq. (58), PAPER.md:330   (Kraynik-Reinelt)
    lambda_max(A^T A)  Eqs. (57), (59); Table I
    quadrature bound   Eq. (55):  C [ exp(-pi^2 P^2/(2 m^2 lambda_max)) + erfc(m/sqrt(2 lambda_max)) ]

The sums themselves are those of oracle.mobility with the image vectors L A n and the reciprocal vectors
k = (2 pi/L) A^{-T} n, n in Z^3 (Eq. 14 "reciprocal space lattice vectors"); V = L^3 because det A = 1.
"""
import itertools

import numpy as np

from . import functions as fn
from . import mobility as mob

f32 = np.float32


def shear(gamma):
    """Eq. (56)."""
    return np.array([[1.0, gamma, 0.0], [0.0, 1.0, 0.0], [0.0, 0.0, 1.0]])


def extension(eps):
    """Eq. (58)."""
    return np.array([[eps, 0.0, 0.0], [0.0, 1.0 / eps, 0.0], [0.0, 0.0, 1.0]])


def lambda_max(A):
    """Largest eigenvalue of A^T A."""
    A = np.asarray(A, dtype=np.float64)
    return float(np.linalg.eigvalsh(A.T @ A).max())


def lambda_max_shear(gamma):
    """Eq. (57)."""
    return 1.0 + gamma**2 / 2.0 + gamma * np.sqrt(1.0 + gamma**2 / 4.0)


def lambda_max_extension(eps):
    """Eq. (59)."""
    return eps**2 if eps >= 1.0 else 1.0 / eps**2


def quadrature_bound(P, lam, m=None):
    """Eq. (55) without its unknown constant C; m = sqrt(pi P) unless given."""
    from scipy.special import erfc
    m = np.sqrt(np.pi * P) if m is None else m
    return float(np.exp(-np.pi**2 * P**2 / (2.0 * m**2 * lam)) + erfc(m / np.sqrt(2.0 * lam)))


def to_lattice(x, A):
    """Lattice coordinates s (in length units, period L in every component) of physical points x = A s."""
    return np.asarray(x, dtype=np.float64) @ np.linalg.inv(np.asarray(A, dtype=np.float64)).T


def real_pairs(x, L, A, rmax, rows=None):
    """All (alpha, beta, rvec) with |x_alpha - x_beta + L A n| <= rmax, n in Z^3 (incl. alpha == beta, n = 0): brute force
    over the images within the bound |n_i| <= ||row_i(A^-1)|| rmax/L + 1/2 of the nearest lattice-coordinate image."""
    x = np.asarray(x, dtype=np.float64)
    A = np.asarray(A, dtype=np.float64)
    Ai = np.linalg.inv(A)
    N = x.shape[0]
    rows = np.arange(N) if rows is None else np.asarray(rows)
    s0 = (x[rows][:, None, :] - x[None, :, :]) @ Ai.T / L
    s0 -= np.round(s0)
    nimg = [int(np.ceil(np.linalg.norm(Ai[i]) * rmax / L + 0.5)) for i in range(3)]
    ia, ib, rv = [], [], []
    for n in itertools.product(*(range(-m, m + 1) for m in nimg)):
        d = L * (s0 + np.array(n, dtype=np.float64)) @ A.T
        m = np.einsum('abi,abi->ab', d, d) <= rmax * rmax
        a_, b_ = np.nonzero(m)
        ia.append(rows[a_]); ib.append(b_); rv.append(d[a_, b_])
    return np.concatenate(ia), np.concatenate(ib), np.concatenate(rv)


def wave_vectors(L, A, kmax):
    """k = (2 pi/L) A^{-T} n, n in Z^3 \\ {0}, |k| <= kmax;  |n_i| <= kmax L ||col_i(A)||/(2 pi)."""
    A = np.asarray(A, dtype=np.float64)
    nm = [int(np.floor(kmax * L * np.linalg.norm(A[:, i]) / (2 * np.pi))) for i in range(3)]
    n = np.stack(np.meshgrid(*(np.arange(-m, m + 1) for m in nm), indexing='ij'), -1).reshape(-1, 3)
    k = 2 * np.pi * (n @ np.linalg.inv(A)) / L
    k2 = np.einsum('ki,ki->k', k, k)
    return k[(k2 > 0) & (k2 <= kmax * kmax)]


def real_apply(x, L, A, a, eta, xi, F, S5, rows=None, eps=1e-14, rcut=None):
    """[U;E]_rows = M^(r) [F;S] on the deformed lattice (pair forms: oracle.mobility.pair_apply)."""
    x = np.asarray(x, dtype=np.float64)
    rows = np.arange(x.shape[0]) if rows is None else np.asarray(rows)
    rmax = mob.real_cutoff(xi, a, eps) if rcut is None else rcut
    ia, ib, rv = real_pairs(x, L, A, rmax, rows)
    if rcut is not None:
        keep = np.einsum('ni,ni->n', rv, rv) < rcut * rcut
        ia, ib, rv = ia[keep], ib[keep], rv[keep]
    R = fn.real_space_functions(np.linalg.norm(rv, axis=1), xi, a)
    U, E = mob.pair_apply(rv, np.asarray(F, float)[ib], fn.to_tensor(np.asarray(S5, float)[ib]), R, 1.0 / (6 * np.pi * eta * a))
    lut = {int(r_): i for i, r_ in enumerate(rows)}
    pos = np.array([lut[int(i)] for i in ia], dtype=np.int64)
    Uo, Eo = np.zeros((rows.size, 3)), np.zeros((rows.size, 5))
    np.add.at(Uo, pos, U)
    np.add.at(Eo, pos, fn.to_coords(E))
    return Uo, Eo


def wave_apply(x, L, A, a, eta, xi, F, S5, rows=None, eps=1e-14):
    k = wave_vectors(L, A, mob.wave_cutoff(xi, eps))
    k2 = np.einsum('ki,ki->k', k, k)
    return mob.wave_apply_modes(x, L, a, eta, k, fn.hasimoto_H(np.sqrt(k2), xi) / (eta * L**3 * k2), F, S5, rows)


def mobility_apply(x, L, A, a, eta, xi, F, S5, rows=None, eps=1e-14, part='both'):
    U, E = 0.0, 0.0
    if part in ('both', 'real'):
        Ur, Er = real_apply(x, L, A, a, eta, xi, F, S5, rows, eps)
        U, E = U + Ur, E + Er
    if part in ('both', 'wave'):
        Uw, Ew = wave_apply(x, L, A, a, eta, xi, F, S5, rows, eps)
        U, E = U + Uw, E + Ew
    return U, E


def dense(x, L, A, a, eta, xi, eps=1e-14, part='both'):
    """Dense 8N x 8N grand mobility on the deformed lattice (small N)."""
    x = np.asarray(x, dtype=np.float64)
    N = x.shape[0]
    M = np.zeros((N, 8, N, 8))
    if part in ('both', 'real'):
        ia, ib, rv = real_pairs(x, L, A, mob.real_cutoff(xi, a, eps))
        R = fn.real_space_functions(np.linalg.norm(rv, axis=1), xi, a)
        for c in range(8):
            v = np.zeros((rv.shape[0], 8)); v[:, c] = 1.0
            U, E = mob.pair_apply(rv, v[:, :3], fn.to_tensor(v[:, 3:]), R, 1.0 / (6 * np.pi * eta * a))
            np.add.at(M[:, :, :, c], (ia, slice(None), ib), np.concatenate([U, fn.to_coords(E)], axis=1))
    M = M.reshape(8 * N, 8 * N)
    if part in ('both', 'wave'):
        k = wave_vectors(L, A, mob.wave_cutoff(xi, eps))
        k2 = np.einsum('ki,ki->k', k, k)
        M = M + mob.dense_wave_modes(x, a, k, fn.hasimoto_H(np.sqrt(k2), xi) / (eta * L**3 * k2))
    return M


def neighbor_sets(pos, L, a11, a12, a22, rcut, rows=None):
    """Neighbour sets on the lattice A = [[a11, a12, 0], [0, a22, 0], [0, 0, 1]] in the GPU's fp32 operation order
    (reading R16 extended by R22): s = A^-1 x with every product and sum rounded, wrapped into [0, L);
    d = s_a - s_b, d -= L rintf(d/L);  r = (a11 dx + a12 dy, a22 dy, dz);  r2 = (rx^2 + ry^2) + rz^2 < rcut^2."""
    x = np.asarray(pos, dtype=f32)[:, :3]
    i11, i12, i22 = f32(1.0 / a11), f32(-a12 / (a11 * a22)), f32(1.0 / a22)
    b11, b12, b22 = f32(a11), f32(a12), f32(a22)
    L32 = f32(L)
    invL = f32(1.0) / L32
    s = np.empty_like(x)
    s[:, 0] = ((i11 * x[:, 0]).astype(f32) + (i12 * x[:, 1]).astype(f32)).astype(f32)
    s[:, 1] = (i22 * x[:, 1]).astype(f32)
    s[:, 2] = x[:, 2]
    w = (s - (L32 * np.floor((s * invL).astype(f32)).astype(f32)).astype(f32)).astype(f32)
    w[(w >= L32) | (w < 0)] = f32(0)
    rc2 = f32(rcut) * f32(rcut)
    out = []
    for al in (range(w.shape[0]) if rows is None else rows):
        d = (w[al][None, :] - w).astype(f32)
        d = (d - (L32 * np.rint((d * invL).astype(f32)).astype(f32)).astype(f32)).astype(f32)
        rx = ((b11 * d[:, 0]).astype(f32) + (b12 * d[:, 1]).astype(f32)).astype(f32)
        ry = (b22 * d[:, 1]).astype(f32)
        rz = d[:, 2]
        r2 = (((rx * rx).astype(f32) + (ry * ry).astype(f32)).astype(f32) + (rz * rz).astype(f32)).astype(f32)
        m = r2 < rc2
        m[al] = False
        out.append(np.nonzero(m)[0].astype(np.int64))
    return out


def brownian(x, L, A, a, eta, kT, xi, dt, Mg, w1, wbuf, eps=1e-14):
    """Eq. (76) on the deformed lattice: principal square root of the dense real-space matrix plus the wave-space
    factor over the modes of the Mg^3 grid (oracle.brownian.wave_sqrt_apply with k = (2 pi/L) A^{-T} n)."""
    from . import brownian as brn
    N = np.asarray(x).shape[0]
    yr = (brn.sqrtm_psd(dense(x, L, A, a, eta, xi, eps, part='real')) @ np.asarray(w1, dtype=np.float64).ravel()).reshape(N, 8)
    Uw, Ew = brn.wave_sqrt_apply(x, L, a, eta, xi, Mg, wbuf, A=A)
    amp = np.sqrt(2.0 * kT / dt)
    return amp * (yr[:, :3] + Uw), amp * (yr[:, 3:] + Ew)


class LatticeReference:
    """Second tier on a deformed lattice, for sizes the direct sums cannot reach (pinned against them in
    tests/test_oracle_lattice.py): the fp64 NUFFT of oracle.pse_reference carried out in LATTICE coordinates s = A^-1 x, where the
    cell is the cube, with the Green's function at the physical wave vector k = (2 pi/L) A^-T n; the Gaussian of the quadrature then
    is one of the lattice coordinates and its transform exp(-eta_g kappa^2/4 xi^2), kappa = 2 pi n/L, is what is divided out.
    Real space: pairs from a periodic k-d tree in lattice coordinates within ||A^-1|| r_cut, kept if |A d| < r_cut, scalar
    functions by quadrature."""

    def __init__(self, L, A, a, eta, xi, tol=1e-8):
        import scipy.fft as sfft
        from . import pse_reference as pr
        self.A = np.asarray(A, dtype=np.float64)
        self.Ai = np.linalg.inv(self.A)
        s = np.sqrt(-np.log(tol))
        rcut = s / xi + 2.0 * a
        self.reach = float(np.linalg.norm(self.Ai, 2))
        if rcut * self.reach > 0.5 * L:
            raise ValueError('LatticeReference: r_cut ||A^-1|| > L/2; raise xi')
        gfac = max(np.linalg.norm(self.A[:, i]) for i in range(3))
        M = int(np.ceil(1.1 * 2.0 * xi * s * L / np.pi * gfac))
        M = max(8, M + (M & 1))
        while sfft.next_fast_len(M, real=True) != M or (M & 1):
            M += 1
        self.ref = pr.PSEReference(L, a, eta, xi, tol, M=M, rcut=rcut)
        self.L, self.a, self.eta, self.xi, self.rcut = float(L), float(a), float(eta), float(xi), rcut

    def real_apply(self, x, F, S5, rows):
        from scipy.spatial import cKDTree
        s = to_lattice(x, self.A) % self.L
        rows = np.asarray(rows, dtype=np.int64)
        F, S5 = np.asarray(F, float), np.asarray(S5, float)
        nb = cKDTree(s, boxsize=self.L).query_ball_point(s[rows], self.reach * self.rcut)
        ia = np.concatenate([np.full(len(b), i, dtype=np.int64) for i, b in enumerate(nb)])
        ib = np.concatenate([np.asarray(b, dtype=np.int64) for b in nb])
        keep = rows[ia] != ib
        ia, ib = ia[keep], ib[keep]
        d = s[rows[ia]] - s[ib]
        d -= self.L * np.round(d / self.L)
        rv = d @ self.A.T
        r = np.linalg.norm(rv, axis=1)
        m = r < self.rcut
        ia, ib, rv, r = ia[m], ib[m], rv[m], r[m]
        R = fn.real_space_functions(r, self.xi, self.a)
        pref = 1.0 / (6 * np.pi * self.eta * self.a)
        Up, Ep = mob.pair_apply(rv, F[ib], fn.to_tensor(S5[ib]), R, pref)
        U, E = np.zeros((rows.size, 3)), np.zeros((rows.size, 5))
        np.add.at(U, ia, Up)
        np.add.at(E, ia, fn.to_coords(Ep))
        R0 = fn.real_space_functions(np.zeros(1), self.xi, self.a)
        return U + pref * R0['F1'][0] * F[rows], E + pref * R0['Z0'][0] / 5.0 * S5[rows]

    def wave_apply(self, x, F, S5, rows):
        import os
        import scipy.fft as sfft
        ref = self.ref
        s = to_lattice(x, self.A) % self.L
        rows = np.ascontiguousarray(rows, dtype=np.int64)
        M, V = ref.M, self.L ** 3
        nw = os.cpu_count() or 1
        gh = sfft.rfftn(ref.spread(s, np.hstack([np.asarray(F, float), np.asarray(S5, float)])), axes=(1, 2, 3), workers=nw)
        qx, qy, qz, live = ref._kvec()                                  # kappa = 2 pi n/L, the wave vector of the cube
        kap2 = qx * qx + qy * qy + qz * qz
        Ai = self.Ai                                                    # k_i = sum_j kappa_j (A^-1)_ji
        kx = qx * Ai[0, 0] + qy * Ai[1, 0] + qz * Ai[2, 0]
        ky = qx * Ai[0, 1] + qy * Ai[1, 1] + qz * Ai[2, 1]
        kz = qx * Ai[0, 2] + qy * Ai[1, 2] + qz * Ai[2, 2]
        k2 = kx * kx + ky * ky + kz * kz
        k2 = np.where(k2 > 0, k2, 1.0)
        kn = np.sqrt(k2)
        c0, c1 = fn.s0(kn * self.a), fn.s1(kn * self.a)
        e = fn.basis()
        kk = (kx, ky, kz)
        fh = []
        for i in range(3):
            Sk = 0.0
            for q in range(5):
                for j in range(3):
                    if e[q, i, j] != 0.0:
                        Sk = Sk + e[q, i, j] * kk[j] * gh[3 + q]
            fh.append(c0 * gh[i] - 1j * c1 * Sk)
        del gh
        Bt = np.where(live, (ref.h ** 3 / V) * fn.hasimoto_H(kn, self.xi) * np.exp(ref.eta_g * kap2 / (4.0 * self.xi ** 2)) / (self.eta * k2), 0.0)
        kf = (kx * fh[0] + ky * fh[1] + kz * fh[2]) / k2
        uh = [Bt * (fh[i] - kk[i] * kf) for i in range(3)]
        del fh
        oh = np.stack(ref._outputs(uh, kx, ky, kz, c0, c1))
        del uh
        go = sfft.irfftn(oh, s=(M, M, M), axes=(1, 2, 3), workers=nw) * float(M) ** 3
        del oh
        out = ref.interpolate(s, go, rows)
        return out[:, :3], out[:, 3:]

    def apply(self, x, F, S5, rows):
        Ur, Er = self.real_apply(x, F, S5, rows)
        Uw, Ew = self.wave_apply(x, F, S5, rows)
        return Ur + Uw, Er + Ew
