"""Direct Ewald sums of the grand mobility with the FULL couplet: [U; Omega; E] = M [F; L; S]  (Eq. 31, PAPER.md:175;
decomposition Eqs. 32-35).  fp64, test infrastructure only.  SURVEY.md 8(f) NEXT-3.

Conventions (reading R21, which settles SURVEY R1 by the physics, not by the paper's inconsistent indices):
    the torque L on a sphere acts on the fluid as the force density (1/2) curl(L delta)   -> fh = (i/2) s1 (k x L),
    the angular velocity is the sphere average of (1/2) curl u (Eq. 6 with Faxen's law)    -> Omega_h = (i/2) s1 (k x uh),
with the couplet shape factor s1(ka) = 3 j1(ka)/ka of PAPER.md:111.  These two maps are adjoint, so M stays symmetric
positive semi-definite, and an isolated sphere turns with Omega = L/(8 pi eta a^3).  (The paper's Eq. 32 with
D_ij = grad_j u_i would give -Omega.)

Wave space is the definition written out (Eqs. 21-24 with the couplet C = S + antisymmetric part):
    fh(k) = sum_beta exp(-i k.x_beta) [ s0 F + (i/2) s1 k x L - i s1 S.k ]
    uh(k) = H(k)/(eta V k^2) (I - kh kh) fh
    U = s0 uh,   Omega = (i/2) s1 k x uh,   E^q = i s1 (e^q k).uh          (summed over k with exp(+i k.x_alpha))
Real space: the same seven scalar functions R_X of Eqs. (25)-(27) (oracle.functions) serve, because the antisymmetric part of
Eq. (26) contracts to (G1 - G2) and the angular averages of the L and Omega couplings contain only j0, j2 (k^2 s1^2 weights,
i.e. Z0, Z2).  With rh the unit separation x_alpha - x_beta and T = R_G1 - R_G2:
    U     += (T/2) L x rh                                             (rotlet: L x rh/(8 pi eta r^2) for r > 2a)
    Omega += (T/2) F x rh + (1/4) [ (2/3) R_Z0 L + R_Z2 (rh rh.L - L/3) ] + (R_Z2/2) (S rh) x rh
    E     += (R_Z2/2) sym[ rh (x) (rh x L) ]
Vectors are ordered per particle as (Ux,Uy,Uz, Ox,Oy,Oz, e^1..e^5): index 11*alpha + c.
"""
import numpy as np

from . import functions as fn
from . import mobility as mob


def pair_apply_full(rvec, F, Lq, S, R, pref):
    """Real-space pair action on (F, L, S) of beta -> (U, Omega, E) at alpha.  The force/stresslet block is
    oracle.mobility.pair_apply; the rotational couplings are the forms in the module docstring (in units of pref)."""
    U, E = mob.pair_apply(rvec, F, S, R, pref)
    r = np.linalg.norm(rvec, axis=1)
    rh = np.where(r[:, None] > 0, rvec / np.where(r > 0, r, 1.0)[:, None], 0.0)
    T = (R['G1'] - R['G2'])[:, None]
    Z0, Z2 = R['Z0'][:, None], R['Z2'][:, None]
    Lxr = np.cross(Lq, rh)
    t = np.einsum('nij,nj->ni', S, rh)
    U = U + pref * 0.5 * T * Lxr
    W = pref * (0.5 * T * np.cross(F, rh)
                + 0.25 * ((2.0 / 3.0) * Z0 * Lq + Z2 * (rh * np.einsum('ni,ni->n', rh, Lq)[:, None] - Lq / 3.0))
                + 0.5 * Z2 * np.cross(t, rh))
    rxL = -Lxr
    E = E + pref * 0.25 * Z2[:, :, None] * (rh[:, :, None] * rxL[:, None, :] + rxL[:, :, None] * rh[:, None, :])
    return U, W, E


def real_apply_full(x, L, a, eta, xi, F, Lq, S5, rows=None, eps=1e-14, rcut=None, A=None):
    """[U;Omega;E]_rows = M^(r) [F;L;S]: direct lattice sum incl. self term and periodic images (as oracle.mobility.real_apply).
    A (3x3, det 1): deformed lattice, image vectors L A n (oracle.lattice)."""
    x = np.asarray(x, dtype=np.float64)
    N = x.shape[0]
    rows = np.arange(N) if rows is None else np.asarray(rows)
    rmax = mob.real_cutoff(xi, a, eps) if rcut is None else rcut
    if A is None:
        ia, ib, rv = mob.real_pairs(x, L, rmax, rows)
    else:
        from . import lattice as lat
        ia, ib, rv = lat.real_pairs(x, L, A, rmax, rows)
    if rcut is not None:
        keep = np.einsum('ni,ni->n', rv, rv) < rcut * rcut
        ia, ib, rv = ia[keep], ib[keep], rv[keep]
    R = fn.real_space_functions(np.linalg.norm(rv, axis=1), xi, a)
    U, W, E = pair_apply_full(rv, np.asarray(F, float)[ib], np.asarray(Lq, float)[ib], fn.to_tensor(np.asarray(S5, float)[ib]), R,
                              1.0 / (6 * np.pi * eta * a))
    lut = {int(r_): i for i, r_ in enumerate(rows)}
    pos = np.array([lut[int(i)] for i in ia], dtype=np.int64)
    Uo, Wo, Eo = np.zeros((rows.size, 3)), np.zeros((rows.size, 3)), np.zeros((rows.size, 5))
    np.add.at(Uo, pos, U)
    np.add.at(Wo, pos, W)
    np.add.at(Eo, pos, fn.to_coords(E))
    return Uo, Wo, Eo


def wave_apply_modes_full(x, a, k, weight, F, Lq, S5, rows=None, chunk=None):
    """Direct wave-space sum over the modes k (n_k, 3) with summand weight(k) in place of H(k)/(eta V k^2)."""
    x = np.asarray(x, dtype=np.float64)
    N = x.shape[0]
    rows = np.arange(N) if rows is None else np.asarray(rows)
    F, Lq = np.asarray(F, dtype=np.float64), np.asarray(Lq, dtype=np.float64)
    S = fn.to_tensor(np.asarray(S5, dtype=np.float64))
    e = fn.basis()
    U, W, E = np.zeros((rows.size, 3)), np.zeros((rows.size, 3)), np.zeros((rows.size, 5))
    chunk = chunk or max(1, 8_000_000 // max(N, 1))
    for lo in range(0, k.shape[0], chunk):
        kk, wk = k[lo:lo + chunk], weight[lo:lo + chunk]
        kn = np.linalg.norm(kk, axis=1)
        kh = kk / kn[:, None]
        c0, c1 = fn.s0(kn * a), fn.s1(kn * a)
        ph = np.exp(-1j * (kk @ x.T))                                  # (n_k, N)
        Sk = np.einsum('bij,kj->kbi', S, kk)                           # S_beta . k
        fh = (c0[:, None] * (ph @ F) + 0.5j * c1[:, None] * np.cross(kk, ph @ Lq)
              - 1j * c1[:, None] * np.einsum('kb,kbi->ki', ph, Sk))
        uh = wk[:, None] * (fh - kh * np.einsum('ki,ki->k', kh, fh)[:, None])
        pa = np.conj(ph[:, rows])                                      # exp(+i k.x_alpha)
        U += np.real(np.einsum('ka,ki->ai', pa, c0[:, None] * uh))
        W += np.real(np.einsum('ka,ki->ai', pa, 0.5j * c1[:, None] * np.cross(kk, uh)))
        ek = np.einsum('qij,kj->kqi', e, kk)                           # e^q . k
        E += np.real(np.einsum('ka,kq->aq', pa, 1j * c1[:, None] * np.einsum('kqi,ki->kq', ek, uh)))
    return U, W, E


def wave_apply_full(x, L, a, eta, xi, F, Lq, S5, rows=None, eps=1e-14, A=None):
    if A is None:
        k = mob.wave_vectors(L, mob.wave_cutoff(xi, eps))
    else:
        from . import lattice as lat
        k = lat.wave_vectors(L, A, mob.wave_cutoff(xi, eps))
    k2 = np.einsum('ki,ki->k', k, k)
    return wave_apply_modes_full(x, a, k, fn.hasimoto_H(np.sqrt(k2), xi) / (eta * L**3 * k2), F, Lq, S5, rows)


def mobility_apply_full(x, L, a, eta, xi, F, Lq, S5, rows=None, eps=1e-14, part='both', A=None):
    """[U;Omega;E]_rows = (M^(r) + M^(w)) [F;L;S]  (Eqs. 30-31); A: deformed lattice (oracle.lattice)."""
    out = [0.0, 0.0, 0.0]
    if part in ('both', 'real'):
        out = [o + v for o, v in zip(out, real_apply_full(x, L, a, eta, xi, F, Lq, S5, rows, eps, A=A))]
    if part in ('both', 'wave'):
        out = [o + v for o, v in zip(out, wave_apply_full(x, L, a, eta, xi, F, Lq, S5, rows, eps, A=A))]
    return tuple(out)


def dense_full(x, L, a, eta, xi, part='both', eps=1e-14):
    """Dense 11N x 11N grand mobility: the product applied to the 11N unit inputs (small N only)."""
    x = np.asarray(x, dtype=np.float64)
    N = x.shape[0]
    M = np.zeros((N, 11, N, 11))
    if part in ('both', 'real'):                       # pair_apply_full on the 11 unit inputs of every pair (incl. images and self)
        ia, ib, rv = mob.real_pairs(x, L, mob.real_cutoff(xi, a, eps))
        R = fn.real_space_functions(np.linalg.norm(rv, axis=1), xi, a)
        for c in range(11):
            v = np.zeros((rv.shape[0], 11)); v[:, c] = 1.0
            U, W, E = pair_apply_full(rv, v[:, :3], v[:, 3:6], fn.to_tensor(v[:, 6:]), R, 1.0 / (6 * np.pi * eta * a))
            np.add.at(M[:, :, :, c], (ia, slice(None), ib), np.concatenate([U, W, fn.to_coords(E)], axis=1))
    M = M.reshape(11 * N, 11 * N)
    if part in ('both', 'wave'):
        for col in range(11 * N):
            v = np.zeros((N, 11)); v[col // 11, col % 11] = 1.0
            U, W, E = wave_apply_full(x, L, a, eta, xi, v[:, :3], v[:, 3:6], v[:, 6:], eps=eps)
            M[:, col] += np.concatenate([U, W, E], axis=1).ravel()
    return M


def constrained_solve_full(M, N, UB, WB, EB, F, Lq):
    """Eqs. (36)-(38) with torques: solve M_ES S = -(E^B + M_EF F + M_EL L), then
    [U;Omega] = [U^B;Omega^B] + M_{U F} [F;L] + M_{U S} S.  M dense 11N x 11N.  Returns U, Omega, S."""
    idx = np.arange(11 * N).reshape(N, 11)
    iu, ie = idx[:, :6].ravel(), idx[:, 6:].ravel()
    FL = np.concatenate([np.asarray(F, float), np.asarray(Lq, float)], axis=1).ravel()
    rhs = -(np.asarray(EB, float).ravel() + M[np.ix_(ie, iu)] @ FL)
    S = np.linalg.solve(M[np.ix_(ie, ie)], rhs)
    UW = np.concatenate([np.asarray(UB, float), np.asarray(WB, float)], axis=1).ravel() + M[np.ix_(iu, iu)] @ FL + M[np.ix_(iu, ie)] @ S
    UW = UW.reshape(N, 6)
    return UW[:, :3], UW[:, 3:], S.reshape(N, 5)


def wave_sqrt_apply_full(x, L, a, eta, xi, Mg, wbuf, rows=None):
    """A_w w2 of Eq. (75) with the angular-velocity rows: the random field uh = sqrt(H/(eta V k^2)) (I - kh kh) W(k)
    over the modes of the Mg^3 grid is that of oracle.brownian.wave_sqrt_apply (same noise buffer, reading R8); here its moments are
    U = s0 uh, Omega = (i/2) s1 k x uh, E^q = i s1 (e^q k).uh.  Returns U, Omega, E at the particles (rows)."""
    from . import brownian as brn
    x = np.asarray(x, dtype=np.float64)
    if rows is not None:
        x = x[np.asarray(rows)]
    N = x.shape[0]
    wbuf = np.asarray(wbuf, dtype=np.float64).reshape(3, Mg, Mg, Mg // 2 + 1, 2)
    idx, n = brn.canonical_modes(Mg)
    k = 2 * np.pi * n / L
    Wn = (wbuf[:, idx[:, 0], idx[:, 1], idx[:, 2], 0] + 1j * wbuf[:, idx[:, 0], idx[:, 1], idx[:, 2], 1]).T / np.sqrt(2)
    e = fn.basis()
    U, W, E = np.zeros((N, 3)), np.zeros((N, 3)), np.zeros((N, 5))
    chunk = max(1, 4_000_000 // max(N, 1))
    for lo in range(0, k.shape[0], chunk):
        kk, Wk = k[lo:lo + chunk], Wn[lo:lo + chunk]
        k2 = np.einsum('ki,ki->k', kk, kk)
        kn = np.sqrt(k2)
        kh = kk / kn[:, None]
        uh = np.sqrt(fn.hasimoto_H(kn, xi) / (eta * L**3 * k2))[:, None] * (Wk - kh * np.einsum('ki,ki->k', kh, Wk)[:, None])
        pa = np.exp(1j * (kk @ x.T))
        c0, c1 = fn.s0(kn * a), fn.s1(kn * a)
        U += 2 * np.real(np.einsum('ka,ki->ai', pa, c0[:, None] * uh))
        W += 2 * np.real(np.einsum('ka,ki->ai', pa, 0.5j * c1[:, None] * np.cross(kk, uh)))
        E += 2 * np.real(np.einsum('ka,kq->aq', pa, 1j * c1[:, None] * np.einsum('qij,kj,ki->kq', e, kk, uh)))
    return U, W, E


def brownian_full(x, L, a, eta, kT, xi, dt, Mg, w1, wbuf, eps=1e-14):
    """Eq. (76) for the 11 components: sqrt(2kT/dt) ( M_r^{1/2} w1 + A_w w2 ), M_r the dense 11N x 11N real-space
    matrix (principal root), w1 (N, 11) in the (U, Omega, E) ordering.  Returns U^B, Omega^B, E^B."""
    from . import brownian as brn
    N = np.asarray(x).shape[0]
    yr = (brn.sqrtm_psd(dense_full(x, L, a, eta, xi, part='real', eps=eps)) @ np.asarray(w1, dtype=np.float64).ravel()).reshape(N, 11)
    Uw, Ww, Ew = wave_sqrt_apply_full(x, L, a, eta, xi, Mg, wbuf)
    amp = np.sqrt(2.0 * kT / dt)
    return amp * (yr[:, :3] + Uw), amp * (yr[:, 3:6] + Ww), amp * (yr[:, 6:] + Ew)


def step_full(x, L, a, eta, kT, xi, dt, Mg, w1, wbuf, Lq, eps=1e-14):
    """One mid-point step, Eqs. (76)-(79), with external torques Lq in script-F = [F^P; L]: the Brownian slip of
    oracle.brownian.brownian at x_k, the overlap forces, torques and the dense 11N x 11N matrix at x_{k+1/2}.
    Returns x_{k+1} (not wrapped), U_{k+1/2}, Omega_{k+1/2}, S."""
    from . import brownian as brn
    x = np.asarray(x, dtype=np.float64)
    N = x.shape[0]
    UB, EB = brn.brownian(x, L, a, eta, kT, xi, dt, Mg, w1, wbuf, eps)          # (76)
    xh = x + 0.5 * dt * UB                                                   # (77)
    xh -= L * np.floor(xh / L)
    M = dense_full(xh, L, a, eta, xi, eps=eps)
    FP = brn.heyes_melrose(xh, L, a, eta, dt)
    U, W, S = constrained_solve_full(M, N, UB, np.zeros((N, 3)), EB, FP, Lq)   # (78)
    return x + dt * U, U, W, S                                               # (79)
