"""Pins of the full-couplet oracle (oracle/couplet.py: [U;Omega;E] = M [F;L;S], Eq. 31) against what the
mathematics and the textbooks fix.  CPU only (-m "not gpu").  SURVEY.md 8(f) NEXT-3 asks for the rotation pin
Omega = L/(8 pi eta a^3), xi-independence and positive-definiteness of the 11N x 11N matrix.
"""
import numpy as np
import pytest

from oracle import couplet as cpl
from oracle import functions as fn
from oracle import mobility as mob

A, ETA = 1.0, 1.0 / (6.0 * np.pi)


def rel(a, b):
    return float(np.linalg.norm(np.asarray(a) - np.asarray(b)) / np.linalg.norm(np.asarray(b)))


def cluster(N=5, L=9.0, seed=2):
    rng = np.random.default_rng(seed)
    x = rng.uniform(0, L, (N, 3))
    x[1] = x[0] + np.array([0.9, 0.7, 0.8])              # overlapping pair, r = 1.39 < 2a
    return x % L, L


def test_C1_isolated_sphere_in_a_periodic_box_turns_with_the_exact_closed_form():
    """M_OmegaL(self) = (1/4 eta V) sum_{k != 0} s1(ka)^2 (I - kh kh); cubic symmetry gives (2/3) I, and by Poisson
    summation (1/V) sum_{all k} s1(ka)^2 = int rho^2 = 3/(4 pi a^3) for L > 2a (s1 is the transform of the uniform ball
    3/(4 pi a^3) 1_{|x|<a}, whose self-convolution vanishes beyond 2a).  Hence
        Omega = L/(8 pi eta a^3) * (1 - (4 pi/3)(a/L)^3)   exactly:   the textbook L/(8 pi eta a^3) as the box grows."""
    for L in (4.5, 7.0, 20.0):
        x = np.array([[0.3, 0.4, 0.5]])
        Lq = np.array([[0.2, -1.0, 0.5]])
        z3, z5 = np.zeros((1, 3)), np.zeros((1, 5))
        U, W, E = cpl.mobility_apply_full(x, L, A, ETA, 0.8, z3, Lq, z5)
        want = Lq / (8 * np.pi * ETA * A**3) * (1.0 - 4 * np.pi / 3 * (A / L)**3)
        assert rel(W, want) < 1e-11
        assert np.abs(U).max() < 1e-13 and np.abs(E).max() < 1e-13        # cubic symmetry: no translation, no strain
        U, W, E = cpl.mobility_apply_full(x, L, A, ETA, 0.8, np.array([[1.0, 2.0, 3.0]]), z3, np.array([[1., 2, 3, 4, 5]]))
        assert np.abs(W).max() < 1e-13


def test_C2_full_couplet_is_independent_of_the_splitting_parameter():
    x, L = cluster()
    rng = np.random.default_rng(0)
    F, Lq, S = rng.standard_normal((5, 3)), rng.standard_normal((5, 3)), rng.standard_normal((5, 5))
    ref = np.hstack(cpl.mobility_apply_full(x, L, A, ETA, 0.55, F, Lq, S))
    for xi in (0.8, 1.1):
        got = np.hstack(cpl.mobility_apply_full(x, L, A, ETA, xi, F, Lq, S))
        assert rel(got, ref) < 1e-11
    # every input block alone, every output block separately: a wrong sign in one coupling cannot hide in the total
    for blk in range(3):
        Fi, Li, Si = (F if blk == 0 else 0 * F), (Lq if blk == 1 else 0 * Lq), (S if blk == 2 else 0 * S)
        a_ = cpl.mobility_apply_full(x, L, A, ETA, 0.55, Fi, Li, Si)
        b_ = cpl.mobility_apply_full(x, L, A, ETA, 1.0, Fi, Li, Si)
        scale = max(np.abs(v).max() for v in a_)
        for u, v in zip(a_, b_):
            assert np.abs(u - v).max() < 1e-11 * scale


def test_C3_symmetric_positive_definite_and_the_force_stresslet_block_is_the_8x8_oracle():
    x, L = cluster(N=4, L=8.0, seed=5)
    xi = 0.7
    M = cpl.dense_full(x, L, A, ETA, xi)
    assert np.abs(M - M.T).max() < 1e-12 * np.abs(M).max()
    np.linalg.cholesky(M)
    for part in ('real', 'wave'):
        Mp = cpl.dense_full(x, L, A, ETA, xi, part=part)
        assert np.abs(Mp - Mp.T).max() < 1e-12 * np.abs(M).max()
        assert np.linalg.eigvalsh(0.5 * (Mp + Mp.T)).min() > -1e-12 * np.abs(M).max()
    keep = np.array([11 * i + c for i in range(4) for c in (0, 1, 2, 6, 7, 8, 9, 10)])
    M8 = mob.dense(x, L, A, ETA, xi)
    assert np.abs(M[np.ix_(keep, keep)] - M8).max() < 1e-13 * np.abs(M8).max()
    # and the product agrees with the matrix
    rng = np.random.default_rng(1)
    v = rng.standard_normal((4, 11))
    U, W, E = cpl.mobility_apply_full(x, L, A, ETA, xi, v[:, :3], v[:, 3:6], v[:, 6:])
    assert rel(np.concatenate([U, W, E], axis=1).ravel(), M @ v.ravel()) < 1e-12


def _textbook_pair(rvec, F, Lq, S):
    """Free-space couplings of two equal spheres, typed from the textbooks (not from the oracle's scalar functions):
    r > 2a: rotlet u = L x r/(8 pi eta r^3); vorticity of the Stokeslet, Omega = F x r/(8 pi eta r^3); rotation-rotation
    mu^rr = -(I - 3 rh rh)/(16 pi eta r^3) (e.g. Kim & Karrila ch. 3; Dhont); flow of a point stresslet
    u = 3 r (r.S.r)/(8 pi eta r^5) (force moment exerted ON the fluid), whose half curl is 3 (S rh) x rh/(8 pi eta r^3);
    r <= 2a: Wajnryb, Mizerski, Zuk & Szymczak, J. Fluid Mech. 731 (2013) R3, equal radii:
      mu^rr = [ (1 - 27 rho/32 + 5 rho^3/64) I + (9 rho/32 - 3 rho^3/64) rh rh ]/(8 pi eta a^3),
      mu^tr = (rho - 3 rho^2/8)/(16 pi eta a^2) (eps . rh)."""
    r = np.linalg.norm(rvec)
    rh = rvec / r
    rho = r / A
    if rho > 2:
        U_L = np.cross(Lq, rh) / (8 * np.pi * ETA * r**2)
        W_F = np.cross(F, rh) / (8 * np.pi * ETA * r**2)
        W_L = -(Lq - 3 * rh * (rh @ Lq)) / (16 * np.pi * ETA * r**3)
        W_S = 3 * np.cross(S @ rh, rh) / (8 * np.pi * ETA * r**3)
    else:
        t = (rho - 3 * rho**2 / 8) / (16 * np.pi * ETA * A**2)
        U_L, W_F = t * np.cross(Lq, rh), t * np.cross(F, rh)
        W_L = ((1 - 27 * rho / 32 + 5 * rho**3 / 64) * Lq + (9 * rho / 32 - 3 * rho**3 / 64) * rh * (rh @ Lq)) / (8 * np.pi * ETA * A**3)
        W_S = None
    return U_L, W_F, W_L, W_S


def test_C4_free_space_rotational_couplings_against_textbook_forms():
    rng = np.random.default_rng(3)
    pref = 1.0 / (6 * np.pi * ETA * A)
    for rho in (0.4, 1.0, 1.7, 2.0, 2.6, 5.0):
        rv = rng.standard_normal(3)
        rv *= rho * A / np.linalg.norm(rv)
        F, Lq = rng.standard_normal(3), rng.standard_normal(3)
        S = fn.to_tensor(rng.standard_normal(5))
        R = {n: np.atleast_1d(v) for n, v in fn.free_space(np.array([rho * A]), A).items()}
        z3, z33 = np.zeros((1, 3)), np.zeros((1, 3, 3))
        U_L, W_L, E_L = cpl.pair_apply_full(rv[None], z3, Lq[None], z33, R, pref)
        _, W_F, _ = cpl.pair_apply_full(rv[None], F[None], z3, z33, R, pref)
        _, W_S, _ = cpl.pair_apply_full(rv[None], z3, z3, S[None], R, pref)
        tU_L, tW_F, tW_L, tW_S = _textbook_pair(rv, F, Lq, S)
        assert rel(U_L[0], tU_L) < 1e-13 and rel(W_F[0], tW_F) < 1e-13 and rel(W_L[0], tW_L) < 1e-13
        if tW_S is not None:
            assert rel(W_S[0], tW_S) < 1e-13
        # E <- L is the transpose of Omega <- S:  S : E_L == L . Omega_S  for any S, L
        assert abs(np.einsum('ij,ij->', S, E_L[0]) - Lq @ W_S[0]) < 1e-13 * np.abs(W_S).max()
        assert abs(np.trace(E_L[0])) < 1e-15 and np.abs(E_L[0] - E_L[0].T).max() < 1e-15


def test_C5_two_spheres_in_a_large_box_approach_the_free_space_couplings():
    """Periodic corrections decay like (r/L)^2 relative to the rotlet and faster for the others: at L = 60a the periodic
    result is within 2 % of the textbook pair forms for U <- L, and the sign and direction are unmistakable."""
    L = 60.0
    x = np.array([[10.0, 10.0, 10.0], [12.0, 11.5, 9.0]])
    Lq = np.array([[0.0, 0.0, 0.0], [0.3, -0.7, 1.1]])
    z3, z5 = np.zeros((2, 3)), np.zeros((2, 5))
    U, W, E = cpl.mobility_apply_full(x, L, A, ETA, 0.35, z3, Lq, z5, eps=1e-10)
    tU_L, _, tW_L, _ = _textbook_pair(x[0] - x[1], z3[0], Lq[1], np.zeros((3, 3)))
    assert rel(U[0], tU_L) < 0.02 and rel(W[0], tW_L) < 0.02


def test_C6_constrained_solve_with_torques_leaves_no_rate_of_strain():
    x, L = cluster(N=4, L=8.0, seed=7)
    M = cpl.dense_full(x, L, A, ETA, 0.7)
    rng = np.random.default_rng(4)
    F, Lq = rng.standard_normal((4, 3)), rng.standard_normal((4, 3))
    UB, WB, EB = rng.standard_normal((4, 3)), rng.standard_normal((4, 3)), rng.standard_normal((4, 5))
    U, W, S = cpl.constrained_solve_full(M, 4, UB, WB, EB, F, Lq)
    Uo, Wo, Eo = cpl.mobility_apply_full(x, L, A, ETA, 0.7, F, Lq, S)
    assert np.abs(Eo + EB).max() < 1e-11
    assert rel(U, UB + Uo) < 1e-11 and rel(W, WB + Wo) < 1e-11
    # without torques the translational part is the 8-component oracle's constrained solve
    from oracle import brownian as brn
    U0, W0, S0 = cpl.constrained_solve_full(M, 4, UB, WB, EB, F, 0 * Lq)
    U8, S8 = brn.constrained_solve(mob.dense(x, L, A, ETA, 0.7), 4, UB, EB, F)
    assert rel(U0, U8) < 1e-11 and rel(S0, S8) < 1e-11


def test_C7_full_couplet_on_a_deformed_lattice_split_independence_and_lattice_equivalence():
    """The torque rows on a sheared cell (oracle.lattice): xi-independence, and gamma -> gamma - 1 is the same lattice."""
    from oracle import lattice as lat
    x, L = cluster()
    rng = np.random.default_rng(6)
    F, Lq, S = rng.standard_normal((5, 3)), rng.standard_normal((5, 3)), rng.standard_normal((5, 5))
    a_ = np.hstack(cpl.mobility_apply_full(x, L, A, ETA, 0.6, F, Lq, S, A=lat.shear(0.4)))
    b_ = np.hstack(cpl.mobility_apply_full(x, L, A, ETA, 0.9, F, Lq, S, A=lat.shear(0.4)))
    c_ = np.hstack(cpl.mobility_apply_full(x, L, A, ETA, 0.6, F, Lq, S, A=lat.shear(-0.6)))
    assert rel(b_, a_) < 1e-11 and rel(c_, a_) < 1e-11
    cube = np.hstack(cpl.mobility_apply_full(x, L, A, ETA, 0.6, F, Lq, S))
    assert rel(np.hstack(cpl.mobility_apply_full(x, L, A, ETA, 0.6, F, Lq, S, A=np.eye(3))), cube) < 1e-13 and rel(a_, cube) > 1e-3


def test_C8_wave_factor_of_the_full_couplet_has_the_covariance_of_its_matrix():
    """A_w A_w^T = M_w summed over exactly the modes of the noise grid (the identity of pin P9, now with the Omega rows), built one unit
    noise entry at a time on a 4^3 and a 5^3 grid; the U and E rows are those of oracle.brownian.wave_sqrt_apply."""
    from oracle import brownian as brn
    x, L = cluster(N=3, L=7.0, seed=11)
    xi = 0.8
    for Mg in (4, 5):
        ncol = 3 * Mg * Mg * (Mg // 2 + 1) * 2
        Aw = np.zeros((33, ncol))
        for c in range(ncol):
            w = np.zeros(ncol); w[c] = 1.0
            Aw[:, c] = np.concatenate(cpl.wave_sqrt_apply_full(x, L, A, ETA, xi, Mg, w), axis=1).ravel()
        k = brn.grid_modes(Mg, L)
        k2 = np.einsum('ki,ki->k', k, k)
        wt = fn.hasimoto_H(np.sqrt(k2), xi) / (ETA * L**3 * k2)
        M = np.zeros((33, 33))
        for col in range(33):
            v = np.zeros((3, 11)); v[col // 11, col % 11] = 1.0
            M[:, col] = np.concatenate(cpl.wave_apply_modes_full(x, A, k, wt, v[:, :3], v[:, 3:6], v[:, 6:]), axis=1).ravel()
        assert np.abs(Aw @ Aw.T - M).max() < 1e-13 * np.abs(M).max()
        w2 = np.random.default_rng(Mg).standard_normal(ncol)
        U, W, E = cpl.wave_sqrt_apply_full(x, L, A, ETA, xi, Mg, w2)
        U8, E8 = brn.wave_sqrt_apply(x, L, A, ETA, xi, Mg, w2)
        assert np.abs(U - U8).max() < 1e-14 and np.abs(E - E8).max() < 1e-14


def test_C9_brownian_full_amplitude_and_real_part():
    """brownian_full against its dense factors: zero wave noise leaves sqrt(2kT/dt) sqrtm(M_r) w1, whose square is M_r; without the
    Omega rows of the noise and with the torque-free block it is NOT the 8-component sample (the principal root of a bordered matrix
    differs), but both have the covariance of their matrix -- only the latter is asserted."""
    from oracle import brownian as brn
    x, L = cluster(N=3, L=7.0, seed=12)
    xi, dt, kT, Mg = 0.8, 1e-3, 0.7, 4
    w1 = np.random.default_rng(1).standard_normal((3, 11))
    zero = np.zeros(3 * Mg * Mg * (Mg // 2 + 1) * 2)
    U, W, E = cpl.brownian_full(x, L, A, ETA, kT, xi, dt, Mg, w1, zero)
    Mr = cpl.dense_full(x, L, A, ETA, xi, part='real')
    R = brn.sqrtm_psd(Mr)
    assert np.abs(R @ R - Mr).max() < 1e-12 * np.abs(Mr).max()
    want = np.sqrt(2 * kT / dt) * (R @ w1.ravel())
    assert rel(np.concatenate([U, W, E], axis=1).ravel(), want) < 1e-12


def test_C10_step_with_torques_reduces_to_the_pinned_step_and_turns_the_spheres():
    """step_full with L = 0 is oracle.brownian.step (pinned by hand in tests/test_oracle_pins.py); with a torque on one sphere every
    translational velocity changes by exactly the constrained response to that torque at the SAME mid-point."""
    from oracle import brownian as brn
    import synth
    N, xi, dt, Mg, L = 6, 0.9, 1e-3, 6, 7.5
    rng = np.random.default_rng(3)
    x = rng.uniform(0, L, (N, 3))
    x[1] = x[0] + np.array([1.0, 0.9, 0.7])
    w1, w2 = synth.brownian_noise(N, Mg, 1)
    x0, U0, S0 = brn.step(x, L, A, ETA, 1.0, xi, dt, Mg, w1, w2, eps=1e-12)
    x1, U1, W1, S1 = cpl.step_full(x, L, A, ETA, 1.0, xi, dt, Mg, w1, w2, np.zeros((N, 3)), eps=1e-12)
    assert rel(x1 - x, x0 - x) < 1e-11 and rel(S1, S0) < 1e-11 and np.abs(W1).max() > 0
    Lq = np.zeros((N, 3)); Lq[2] = (0.0, 0.0, 5.0)
    x2, U2, W2, S2 = cpl.step_full(x, L, A, ETA, 1.0, xi, dt, Mg, w1, w2, Lq, eps=1e-12)
    UB, EB = brn.brownian(x, L, A, ETA, 1.0, xi, dt, Mg, w1, w2, 1e-12)
    xh = (x + 0.5 * dt * UB) % L
    M = cpl.dense_full(xh, L, A, ETA, xi, eps=1e-12)
    dU, dW, dS = cpl.constrained_solve_full(M, N, np.zeros((N, 3)), np.zeros((N, 3)), np.zeros((N, 5)), np.zeros((N, 3)), Lq)
    assert rel(U2 - U1, dU) < 1e-9 and rel(W2 - W1, dW) < 1e-9 and dW[2, 2] > 0
