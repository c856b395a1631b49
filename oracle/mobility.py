"""Direct Ewald sums of the grand mobility M [F;S] -> [U;E] (fp64).  Test infrastructure only.

M = M^(r) + M^(w) through the exact Hasimoto split (Eqs. 21-28): the split is an
identity, so carried to convergence this *is* the lattice sum of Eqs. (15)-(18).
Vectors are ordered per particle as (Ux, Uy, Uz, e^1..e^5): index 8*alpha + c.
"""
import itertools
import numpy as np
from . import functions as fn


def pair_apply(rvec, F, S, R, pref):
    """Real-space pair action, Eqs. (25)-(27) in the form of SURVEY.md §8(c) O4.

    rvec (n,3) = x_alpha - x_beta (+ lattice vector), F (n,3) force on beta, S (n,3,3) symmetric traceless
    stresslet of beta, R dict of the seven R_X at |rvec|.  Returns U (n,3), E (n,3,3) at alpha.
      U = R_F1 (F - rh f) + R_F2 rh f + (G1+G2) t - (G1+4G2) rh q
      E = -[(G1+G2) sym(F rh) + G2 f I - (G1+4G2) f rh rh] + A S + B (rh t + t rh) + C q I + D q rh rh
    with f = rh.F, t = S.rh, q = rh.S.rh.  At r = 0 (self term, Eqs. A4/A12 PAPER.md:636, 744) rh := 0.
    """
    r = np.linalg.norm(rvec, axis=1)
    rh = np.where(r[:, None] > 0, rvec / np.where(r > 0, r, 1.0)[:, None], 0.0)
    A, B, C, D = fn.rank4_combinations(R)
    Ga, Gb = R['G1'] + R['G2'], R['G1'] + 4.0 * R['G2']
    f = np.einsum('ni,ni->n', rh, F)
    t = np.einsum('nij,nj->ni', S, rh)
    q = np.einsum('ni,ni->n', rh, t)
    I3 = np.eye(3)
    rr = rh[:, :, None] * rh[:, None, :]
    U = (R['F1'][:, None] * (F - rh * f[:, None]) + R['F2'][:, None] * rh * f[:, None]
         + Ga[:, None] * t - Gb[:, None] * rh * q[:, None])
    symFr = 0.5 * (F[:, :, None] * rh[:, None, :] + rh[:, :, None] * F[:, None, :])
    rt = rh[:, :, None] * t[:, None, :] + t[:, :, None] * rh[:, None, :]
    E = (-(Ga[:, None, None] * symFr + (R['G2'] * f)[:, None, None] * I3 - (Gb * f)[:, None, None] * rr)
         + A[:, None, None] * S + B[:, None, None] * rt + (C * q)[:, None, None] * I3
         + (D * q)[:, None, None] * rr)
    return pref * U, pref * E


def real_cutoff(xi, a, eps=1e-14):
    """r_max with R_X(r_max) < eps (functions decay like exp(-xi^2 (r-2a)^2))."""
    return np.sqrt(-np.log(eps)) / xi + 2.0 * a


def wave_cutoff(xi, eps=1e-14):
    """k_max with H(k) exp-tail < eps."""
    return 2.0 * xi * np.sqrt(-np.log(eps) + 4.0)


def real_pairs(x, L, rmax, rows=None):
    """All (alpha, beta, rvec) with |x_alpha - x_beta + n L| <= rmax, n in Z^3, including alpha == beta, n = 0
    (the self term) and images of a particle with itself.  Brute force.  rows restricts alpha."""
    x = np.asarray(x, dtype=np.float64)
    N = x.shape[0]
    rows = np.arange(N) if rows is None else np.asarray(rows)
    nimg = int(np.ceil(rmax / L + 0.5))
    ia, ib, rv = [], [], []
    d0 = x[rows][:, None, :] - x[None, :, :]
    d0 -= L * np.round(d0 / L)
    for n in itertools.product(range(-nimg, nimg + 1), repeat=3):
        d = d0 + L * np.array(n, dtype=np.float64)
        m = np.einsum('abi,abi->ab', d, d) <= rmax * rmax
        a_, b_ = np.nonzero(m)
        ia.append(rows[a_]); ib.append(b_); rv.append(d[a_, b_])
    return np.concatenate(ia), np.concatenate(ib), np.concatenate(rv)


def real_apply(x, L, a, eta, xi, F, S5, rows=None, eps=1e-14, rcut=None):
    """[U;E]_rows = M^(r) [F;S]: direct lattice sum (SURVEY.md §8(c) O4+O5).  rcut, if given, truncates the
    sum at r < rcut instead of convergence (used only to measure the truncation error itself)."""
    x = np.asarray(x, dtype=np.float64)
    N = x.shape[0]
    rows = np.arange(N) if rows is None else np.asarray(rows)
    rmax = real_cutoff(xi, a, eps) if rcut is None else rcut
    ia, ib, rv = real_pairs(x, L, rmax, rows)
    if rcut is not None:
        keep = np.einsum('ni,ni->n', rv, rv) < rcut * rcut
        ia, ib, rv = ia[keep], ib[keep], rv[keep]
    R = fn.real_space_functions(np.linalg.norm(rv, axis=1), xi, a)
    U, E = pair_apply(rv, np.asarray(F, float)[ib], fn.to_tensor(np.asarray(S5, float)[ib]), R,
                      1.0 / (6 * np.pi * eta * a))
    pos = np.searchsorted(rows, ia) if np.all(np.diff(rows) > 0) else None
    if pos is None:
        lut = {int(r_): i for i, r_ in enumerate(rows)}
        pos = np.array([lut[int(i)] for i in ia], dtype=np.int64)
    Uo, Eo = np.zeros((rows.size, 3)), np.zeros((rows.size, 5))
    np.add.at(Uo, pos, U)
    np.add.at(Eo, pos, fn.to_coords(E))
    return Uo, Eo


def wave_vectors(L, kmax):
    """k = 2 pi n / L, n in Z^3 \\ {0}, |k| <= kmax (the k = 0 mode is dropped)."""
    nmax = int(np.floor(kmax * L / (2 * np.pi)))
    g = np.arange(-nmax, nmax + 1)
    n = np.stack(np.meshgrid(g, g, g, indexing='ij'), -1).reshape(-1, 3)
    k = 2 * np.pi * n / L
    k2 = np.einsum('ki,ki->k', k, k)
    return k[(k2 > 0) & (k2 <= kmax * kmax)]


def wave_apply_modes(x, L, a, eta, k, weight, F, S5, rows=None, chunk=None):
    """Direct wave-space sum over the given modes k (n_k, 3), summand weight(k) in place of H(k)/(eta V k^2)
    (straight from Eqs. 21-24):
        fh(k) = sum_beta exp(-i k.x_beta) [ s0 F_beta - i s1 S_beta.k ]
        uh(k) = weight(k) (I - kh kh) fh(k)
        U_alpha += Re sum_k exp(i k.x_alpha) s0 uh ;  E^q_alpha += Re sum_k exp(i k.x_alpha) i s1 (e^q k).uh
    """
    x = np.asarray(x, dtype=np.float64)
    N = x.shape[0]
    rows = np.arange(N) if rows is None else np.asarray(rows)
    F = np.asarray(F, dtype=np.float64)
    S = fn.to_tensor(np.asarray(S5, dtype=np.float64))
    e = fn.basis()
    U, E = np.zeros((rows.size, 3)), np.zeros((rows.size, 5))
    chunk = chunk or max(1, 8_000_000 // max(N, 1))
    for lo in range(0, k.shape[0], chunk):
        kk, wk = k[lo:lo + chunk], weight[lo:lo + chunk]
        kn = np.linalg.norm(kk, axis=1)
        kh = kk / kn[:, None]
        c0, c1 = fn.s0(kn * a), fn.s1(kn * a)
        ph = np.exp(-1j * (kk @ x.T))                                  # (n_k, N)
        Sk = np.einsum('bij,kj->kbi', S, kk)                           # S_beta . k
        fh = c0[:, None] * (ph @ F) - 1j * c1[:, None] * np.einsum('kb,kbi->ki', ph, Sk)
        uh = wk[:, None] * (fh - kh * np.einsum('ki,ki->k', kh, fh)[:, None])
        pa = np.conj(ph[:, rows])                                      # exp(+i k.x_alpha)
        U += np.real(np.einsum('ka,ki->ai', pa, c0[:, None] * uh))
        ek = np.einsum('qij,kj->kqi', e, kk)                           # e^q . k
        dq = 1j * c1[:, None] * np.einsum('kqi,ki->kq', ek, uh)
        E += np.real(np.einsum('ka,kq->aq', pa, dq))
    return U, E


def wave_apply(x, L, a, eta, xi, F, S5, rows=None, eps=1e-14):
    """[U;E]_rows = M^(w) [F;S] summed to convergence (Eqs. 21-24)."""
    k = wave_vectors(L, wave_cutoff(xi, eps))
    k2 = np.einsum('ki,ki->k', k, k)
    w = fn.hasimoto_H(np.sqrt(k2), xi) / (eta * L**3 * k2)
    return wave_apply_modes(x, L, a, eta, k, w, F, S5, rows)


def mobility_apply(x, L, a, eta, xi, F, S5, rows=None, eps=1e-14):
    """[U;E]_rows = (M^(r) + M^(w)) [F;S]  (Eq. 30)."""
    Ur, Er = real_apply(x, L, a, eta, xi, F, S5, rows, eps)
    Uw, Ew = wave_apply(x, L, a, eta, xi, F, S5, rows, eps)
    return Ur + Uw, Er + Ew


def dense_real(x, L, a, eta, xi, eps=1e-14):
    """Dense 8N x 8N M^(r): pair_apply on the 8 unit inputs of every pair (incl. images and self)."""
    x = np.asarray(x, dtype=np.float64)
    N = x.shape[0]
    ia, ib, rv = real_pairs(x, L, real_cutoff(xi, a, eps))
    R = fn.real_space_functions(np.linalg.norm(rv, axis=1), xi, a)
    M = np.zeros((N, 8, N, 8))
    n = rv.shape[0]
    for c in range(8):
        v = np.zeros((n, 8)); v[:, c] = 1.0
        U, E = pair_apply(rv, v[:, :3], fn.to_tensor(v[:, 3:]), R, 1.0 / (6 * np.pi * eta * a))
        np.add.at(M[:, :, :, c], (ia, slice(None), ib), np.concatenate([U, fn.to_coords(E)], axis=1))
    return M.reshape(8 * N, 8 * N)


def dense_wave_modes(x, a, k, weight):
    """Dense 8N x 8N  Re sum_k weight(k) b_k^H (I - kh kh) b_k, the P^H B P structure of Eqs. (39)-(41)
    (PAPER.md:213-221): b_k[i, (beta,c)] = exp(-i k.x_beta) [ s0 delta_ic | -i s1 (e^q k)_i ]."""
    x = np.asarray(x, dtype=np.float64)
    N = x.shape[0]
    e = fn.basis()
    M = np.zeros((8 * N, 8 * N))
    chunk = max(1, 16_000_000 // (24 * N))
    for lo in range(0, k.shape[0], chunk):
        kk, wk = k[lo:lo + chunk], weight[lo:lo + chunk]
        kn = np.linalg.norm(kk, axis=1)
        kh = kk / kn[:, None]
        c0, c1 = fn.s0(kn * a), fn.s1(kn * a)
        ph = np.exp(-1j * (kk @ x.T))                                     # (n_k, N)
        shape = np.zeros((kk.shape[0], 3, 8), dtype=complex)              # P_ii of Eq. (41)
        shape[:, :, :3] = c0[:, None, None] * np.eye(3)
        shape[:, :, 3:] = -1j * c1[:, None, None] * np.einsum('qij,kj->kiq', e, kk)
        b = (ph[:, None, :, None] * shape[:, :, None, :]).reshape(kk.shape[0], 3, 8 * N)
        Pb = b - kh[:, :, None] * np.einsum('ki,kin->kn', kh, b)[:, None, :]
        nk = kk.shape[0]
        M += np.real((np.conj(b) * wk[:, None, None]).reshape(nk * 3, 8 * N).T @ Pb.reshape(nk * 3, 8 * N))
    return M


def dense_wave(x, L, a, eta, xi, eps=1e-14):
    k = wave_vectors(L, wave_cutoff(xi, eps))
    k2 = np.einsum('ki,ki->k', k, k)
    return dense_wave_modes(x, a, k, fn.hasimoto_H(np.sqrt(k2), xi) / (eta * L**3 * k2))


def dense(x, L, a, eta, xi, part='both', eps=1e-14):
    """Dense grand mobility (Eq. 30) in the 8-per-particle coordinates.  Small N only."""
    M = 0.0
    if part in ('both', 'real'):
        M = M + dense_real(x, L, a, eta, xi, eps)
    if part in ('both', 'wave'):
        M = M + dense_wave(x, L, a, eta, xi, eps)
    return M
