"""PSE Brownian sample and the mid-point constrained step (fp64, dense, small N).  Test infrastructure only.

    [U^B; E^B] = sqrt(2 kT / dt) ( M_r^{1/2} w1 + A_w w2 )          Eqs. (71), (76), (B4)

M_r^{1/2} is the principal square root of the dense real-space matrix (what Lanczos converges to);
A_w = D^H P^H B^{1/2} is the specific wave-space factor of Eq. (74) evaluated by direct
non-uniform sums over exactly the wave vectors of an Mg^3 FFT grid (readings R8, R10).
"""
import numpy as np
from . import functions as fn
from . import mobility as mob


def signed(i, Mg):
    """FFT index -> signed wave number."""
    return np.where(i <= (Mg - 1) // 2, i, i - Mg) if Mg % 2 else np.where(i < Mg // 2, i, i - Mg)


def canonical_modes(Mg):
    """Half-spectrum storage indices (ix, iy, iz), iz in [0, Mg/2], of the modes that carry their own noise
    entry (reading R8): every mode with 0 < kz; in the plane kz = 0 the member of each +-k pair with signed
    ky > 0, or ky = 0 and kx > 0.  k = 0 and Nyquist modes (any index == Mg/2, Mg even) are excluded: their
    weight is set to zero in both the mobility product and the Brownian sample.
    Returns idx (n,3) int and n (n,3) signed wave numbers."""
    ix, iy, iz = np.meshgrid(np.arange(Mg), np.arange(Mg), np.arange(Mg // 2 + 1), indexing='ij')
    idx = np.stack([ix, iy, iz], -1).reshape(-1, 3)
    n = np.stack([signed(idx[:, 0], Mg), signed(idx[:, 1], Mg), idx[:, 2]], -1)
    nyq = np.zeros(len(idx), bool) if Mg % 2 else np.any(idx == Mg // 2, axis=1)
    canon = (n[:, 2] > 0) | ((n[:, 2] == 0) & ((n[:, 1] > 0) | ((n[:, 1] == 0) & (n[:, 0] > 0))))
    keep = canon & ~nyq
    return idx[keep], n[keep]


def grid_modes(Mg, L):
    """All signed wave vectors of the Mg^3 grid except k = 0 and Nyquist: the canonical ones and their negatives."""
    _, n = canonical_modes(Mg)
    return 2 * np.pi * np.concatenate([n, -n]) / L


def wave_sqrt_apply(x, L, a, eta, xi, Mg, wbuf, chunk=None, rows=None, A=None):
    """A_w w2.  wbuf: real array [3][Mg][Mg][Mg/2+1][2] of i.i.d. N(0,1).  For each canonical mode
    W(k) = (g_re + i g_im)/sqrt2, W(-k) = conj W(k), so the pair contributes 2 Re[...]:
        uh = sqrt(H/(eta V k^2)) (I - kh kh) W ;  U_a = sum_k e^{ik.x_a} s0 uh ;  E^q_a = sum_k e^{ik.x_a} i s1 (e^q k).uh
    rows restricts the particles a the sum is evaluated at (the noise field does not depend on the particles).
    A (3x3, det 1): deformed lattice with vectors = columns of L A; the mode of integer indices n is then
    k = (2 pi/L) A^{-T} n instead of 2 pi n/L, everything else unchanged (V = L^3).
    """
    x = np.asarray(x, dtype=np.float64)
    if rows is not None:
        x = x[np.asarray(rows)]
    N = x.shape[0]
    wbuf = np.asarray(wbuf, dtype=np.float64).reshape(3, Mg, Mg, Mg // 2 + 1, 2)
    idx, n = canonical_modes(Mg)
    k = 2 * np.pi * n / L if A is None else 2 * np.pi * (n @ np.linalg.inv(np.asarray(A, dtype=np.float64))) / L
    W = (wbuf[:, idx[:, 0], idx[:, 1], idx[:, 2], 0] + 1j * wbuf[:, idx[:, 0], idx[:, 1], idx[:, 2], 1]).T / np.sqrt(2)
    e = fn.basis()
    U, E = np.zeros((N, 3)), np.zeros((N, 5))
    chunk = chunk or max(1, 4_000_000 // max(N, 1))
    for lo in range(0, k.shape[0], chunk):
        kk, Wk = k[lo:lo + chunk], W[lo:lo + chunk]
        k2 = np.einsum('ki,ki->k', kk, kk)
        kn = np.sqrt(k2)
        kh = kk / kn[:, None]
        uh = np.sqrt(fn.hasimoto_H(kn, xi) / (eta * L**3 * k2))[:, None] * (Wk - kh * np.einsum('ki,ki->k', kh, Wk)[:, None])
        pa = np.exp(1j * (kk @ x.T))
        U += 2 * np.real(np.einsum('ka,ki->ai', pa, fn.s0(kn * a)[:, None] * uh))
        dq = 1j * fn.s1(kn * a)[:, None] * np.einsum('qij,kj,ki->kq', e, kk, uh)
        E += 2 * np.real(np.einsum('ka,kq->aq', pa, dq))
    return U, E


def wave_sqrt_dense(x, L, a, eta, xi, Mg):
    """A_w as a dense (8N) x (3*Mg*Mg*(Mg/2+1)*2) matrix, one unit noise entry at a time (pin P9). Tiny grids."""
    N = np.asarray(x).shape[0]
    ncol = 3 * Mg * Mg * (Mg // 2 + 1) * 2
    A = np.zeros((8 * N, ncol))
    for c in range(ncol):
        w = np.zeros(ncol); w[c] = 1.0
        U, E = wave_sqrt_apply(x, L, a, eta, xi, Mg, w)
        A[:, c] = np.concatenate([U, E], axis=1).ravel()
    return A


def sqrtm_psd(M):
    """Principal square root of a symmetric positive semi-definite matrix."""
    w, V = np.linalg.eigh(0.5 * (M + M.T))
    return (V * np.sqrt(np.clip(w, 0.0, None))) @ V.T


def brownian(x, L, a, eta, kT, xi, dt, Mg, w1, wbuf, eps=1e-14):
    """Eq. (76) with the sqrt(2kT/dt) amplitude of Eq. (B4).  w1: (8N,) in the
    per-particle (Ux,Uy,Uz,e1..e5) ordering."""
    N = np.asarray(x).shape[0]
    yr = (sqrtm_psd(mob.dense_real(x, L, a, eta, xi, eps)) @ np.asarray(w1, dtype=np.float64).ravel()).reshape(N, 8)
    Uw, Ew = wave_sqrt_apply(x, L, a, eta, xi, Mg, wbuf)
    amp = np.sqrt(2.0 * kT / dt)
    return amp * (yr[:, :3] + Uw), amp * (yr[:, 3:] + Ew)


def heyes_melrose(x, L, a, eta, dt):
    """Hard-sphere overlap force, reading R12 (named by BASELINE.json, not in the paper; pinned by the property that defines it:
    a free-draining pair moved by it for one dt ends exactly at contact, tests/test_oracle_pins.py):
    F_i = sum_{j: r_ij < 2a} 3 pi eta a (2a - r_ij)/dt rhat_ij,  rhat_ij = (x_i - x_j)/r_ij (minimum image)."""
    x = np.asarray(x, dtype=np.float64)
    d = x[:, None, :] - x[None, :, :]
    d -= L * np.round(d / L)
    r = np.linalg.norm(d, axis=2)
    np.fill_diagonal(r, np.inf)
    m = r < 2 * a
    coef = np.where(m, 3 * np.pi * eta * a * (2 * a - r) / dt / np.where(m, r, 1.0), 0.0)
    return np.einsum('ab,abi->ai', coef, d)


def bond_forces(x, L, pairs, k, r0):
    """Forces of the pair potential of the paper's equilibrium test, U(r) = k |r - r0|, on the bonded
    pairs `pairs` (n,2): F_i = -dU/dx_i = -k sign(r - r0) rhat_ij, F_j = -F_i, rhat_ij = (x_i - x_j)/r (minimum image)."""
    x = np.asarray(x, dtype=np.float64)
    F = np.zeros_like(x)
    for i, j in np.asarray(pairs, dtype=np.int64).reshape(-1, 2):
        d = x[i] - x[j]
        d -= L * np.round(d / L)
        r = np.linalg.norm(d)
        f = -k * np.sign(r - r0) * d / r
        F[i] += f
        F[j] -= f
    return F


def pair_distance_pdf(r, kt, r0):
    """Eq. (80): Boltzmann density of the centre-to-centre distance of a pair bound by U = k|r - r0|,
    f(r) = kt^3 / (2 (2 + kt^2 r0^2)) r^2 exp(-kt |r - r0|),  kt = k / kT."""
    r = np.asarray(r, dtype=np.float64)
    return kt ** 3 / (2.0 * (2.0 + kt ** 2 * r0 ** 2)) * r ** 2 * np.exp(-kt * np.abs(r - r0))


def constrained_solve(M, N, UB, EB, FP):
    """Eqs. (36)-(38), (78) with deterministic forces (reading R12):
    solve M_ES S = -(E^B + M_EF F^P), then U = U^B + M_UF F^P + M_US S.  M is the dense 8N x 8N matrix."""
    iu = (8 * np.arange(N)[:, None] + np.arange(3)[None, :]).ravel()
    ie = (8 * np.arange(N)[:, None] + 3 + np.arange(5)[None, :]).ravel()
    rhs = -(EB.ravel() + M[np.ix_(ie, iu)] @ FP.ravel())
    S = np.linalg.solve(M[np.ix_(ie, ie)], rhs)
    U = UB.ravel() + M[np.ix_(iu, iu)] @ FP.ravel() + M[np.ix_(iu, ie)] @ S
    return U.reshape(N, 3), S.reshape(N, 5)


def constrained_mobility(M, N):
    """R_FU^{-1} = M_UF - M_US M_ES^{-1} M_EF (Eq. B15), the 3N x 3N mobility of rigid spheres, from the
    dense 8N x 8N grand mobility."""
    iu = (8 * np.arange(N)[:, None] + np.arange(3)[None, :]).ravel()
    ie = (8 * np.arange(N)[:, None] + 3 + np.arange(5)[None, :]).ravel()
    return M[np.ix_(iu, iu)] - M[np.ix_(iu, ie)] @ np.linalg.solve(M[np.ix_(ie, ie)], M[np.ix_(ie, iu)])


def constrained_mobility_divergence(x, L, a, eta, xi, h=1e-4, eps=1e-12):
    """(div R_FU^{-1})_i = sum_l d/dx_l (R_FU^{-1})_{il}, the drift of Eq. (B12) per unit kT dt, by central
    differences of the dense matrix.  Returns (div R_FU^{-1}, div M_UF), each (3N,); the second is zero."""
    x = np.asarray(x, dtype=np.float64)
    N = x.shape[0]
    iu = (8 * np.arange(N)[:, None] + np.arange(3)[None, :]).ravel()
    div_c, div_uf = np.zeros(3 * N), np.zeros(3 * N)
    for l in range(3 * N):
        cols = []
        for sgn in (1.0, -1.0):
            y = x.copy().ravel()
            y[l] += sgn * h
            M = mob.dense(y.reshape(N, 3), L, a, eta, xi, 'both', eps)
            cols.append((constrained_mobility(M, N)[:, l], M[np.ix_(iu, iu)][:, l]))
        div_c += (cols[0][0] - cols[1][0]) / (2 * h)
        div_uf += (cols[0][1] - cols[1][1]) / (2 * h)
    return div_c, div_uf


def step(x, L, a, eta, kT, xi, dt, Mg, w1, wbuf, eps=1e-14, bonds=None):
    """One mid-point step, Eqs. (76)-(79).  Returns x_{k+1} (not wrapped), U_{k+1/2}, S.
    bonds = (pairs, k, r0) adds the forces of U = k|r - r0| at the mid-point to F^P."""
    x = np.asarray(x, dtype=np.float64)
    N = x.shape[0]
    UB, EB = brownian(x, L, a, eta, kT, xi, dt, Mg, w1, wbuf, eps)          # (76)
    xh = x + 0.5 * dt * UB                                                   # (77)
    xh -= L * np.floor(xh / L)
    M = mob.dense(xh, L, a, eta, xi, 'both', eps)
    FP = heyes_melrose(xh, L, a, eta, dt)
    if bonds is not None:
        FP = FP + bond_forces(xh, L, *bonds)
    U, S = constrained_solve(M, N, UB, EB, FP)                               # (78)
    return x + dt * U, U, S                                                  # (79)
