"""Pins of the CPU oracle against what the paper and the mathematics fix (CPU only, -m "not gpu").

P1 Hasimoto self-mobility, P2 xi-independence, P3 symmetry + positive-definiteness, P4 limits/continuity of the
scalar functions, P5 free-space forms against the Fourier-space definition, P6 printed closed forms of
Appendix A, P7 single-sphere cubic symmetry, P8 worked example, P9 exact covariance identity, P12 Schur solve.
"""
import os
import sys

import numpy as np
import pytest

sys.path.insert(0, os.path.join(os.path.dirname(__file__), 'golden'))
import paper_appendix_a as app  # noqa: E402
from oracle import brownian as brn  # noqa: E402
from oracle import functions as fn  # noqa: E402
from oracle import mobility as mob  # noqa: E402

A, ETA = 1.0, 1.0 / (6.0 * np.pi)
X4 = np.array([[0.5, 0.6, 0.7], [2.9, 1.0, 0.9], [1.1, 4.0, 5.5], [2.0, 2.0, 2.3]])  # pair 0-3 overlaps (r = 1.942)


def test_basis_orthonormal_and_roundtrip():
    e = fn.basis()
    assert np.allclose(np.einsum('pij,qij->pq', e, e), np.eye(5), atol=1e-15)
    assert np.allclose(np.einsum('qii->q', e), 0) and np.allclose(e, e.transpose(0, 2, 1))
    s = np.random.default_rng(0).standard_normal((7, 5))
    assert np.allclose(fn.to_coords(fn.to_tensor(s)), s, atol=1e-14)


def test_P1_hasimoto_single_sphere():
    """6 pi eta a mu = 1 - 2.8372974795 a/L + (4 pi/3)(a/L)^3 for one sphere per cubic cell."""
    for L, xi in [(7.0, 0.55), (7.0, 0.9), (11.0, 0.4)]:
        M = mob.dense(np.array([[1.0, 2.0, 3.0]]), L, A, ETA, xi)
        want = 1 - app.HASIMOTO_C * A / L + 4 * np.pi / 3 * (A / L)**3
        assert np.allclose(np.diag(M)[:3], want, atol=5e-10), (L, xi, M[0, 0], want)
        assert np.allclose(M[:3, :3], want * np.eye(3), atol=5e-10)


def test_P7_single_sphere_cubic_symmetry():
    """M_EF,self = 0; self M_ES is diagonal with one value for e1,e2 and one for e3..e5 (cubic anisotropy)."""
    M = mob.dense(np.array([[0.3, 0.2, 0.1]]), 7.0, A, ETA, 0.6)
    assert np.abs(M[:3, 3:]).max() < 1e-13 and np.abs(M[3:, :3]).max() < 1e-13
    d = np.diag(M)[3:]
    assert np.abs(M[3:, 3:] - np.diag(d)).max() < 1e-13
    assert abs(d[0] - d[1]) < 1e-12 and abs(d[2] - d[3]) < 1e-12 and abs(d[3] - d[4]) < 1e-12
    assert abs(d[0] - d[2]) > 1e-2     # anisotropic: 0.8604 vs 0.9081 at L = 7a
    assert abs(d[0] - 0.860374496914) < 1e-9 and abs(d[2] - 0.908098677547) < 1e-9


def test_P2_P3_xi_independence_symmetry_spd():
    Ms = [mob.dense(X4, 7.0, A, ETA, xi) for xi in (0.45, 0.7, 1.0)]
    assert np.abs(Ms[0] - Ms[1]).max() < 1e-12 and np.abs(Ms[0] - Ms[2]).max() < 1e-12
    for xi in (0.45, 1.0):
        Mr, Mw = mob.dense(X4, 7.0, A, ETA, xi, 'real'), mob.dense(X4, 7.0, A, ETA, xi, 'wave')
        for M in (Mr, Mw, Mr + Mw):
            assert np.abs(M - M.T).max() < 1e-13
        np.linalg.cholesky(Mr)                                  # strictly PD
        np.linalg.cholesky(Mr + Mw)
        assert np.linalg.eigvalsh(Mw).min() > -1e-13            # PSD
    w = np.linalg.eigvalsh(Ms[0])
    assert abs(w[0] - 0.183962406486) < 1e-9 and abs(w[-1] - 1.331372501993) < 1e-9


def test_P8_worked_example():
    """Entries of M for the 4-sphere example, computed independently during the survey."""
    M = mob.dense(X4, 7.0, A, ETA, 0.55)
    gold = {(0, 0): 0.606884004986, (0, 8): 0.218163662585, (0, 24): 0.027175723339, (0, 26): 0.047217809432,
            (1, 25): 0.016352878862, (0, 27): 0.005564508157, (3, 24): -0.005564508157, (2, 29): -0.046712907241,
            (3, 27): 0.024490765888, (5, 29): -0.026755324780, (7, 25): 0.078638421506, (3, 11): -0.150187216517,
            (4, 4): 0.860374496914, (5, 5): 0.908098677547}
    for ij, v in gold.items():
        assert abs(M[ij] - v) < 2e-11, (ij, M[ij], v)


def test_dense_matches_apply():
    """The P^H B P matrix form (Eqs. 39-41) and the direct sums (Eqs. 21-24) are two codes for one operator."""
    rng = np.random.default_rng(1)
    F, S = rng.standard_normal((4, 3)), rng.standard_normal((4, 5))
    U, E = mob.mobility_apply(X4, 7.0, A, ETA, 0.6, F, S)
    o = (mob.dense(X4, 7.0, A, ETA, 0.6) @ np.concatenate([F, S], 1).ravel()).reshape(4, 8)
    assert np.abs(o[:, :3] - U).max() < 1e-13 and np.abs(o[:, 3:] - E).max() < 1e-13
    U2, E2 = mob.mobility_apply(X4, 7.0, A, ETA, 0.6, F, S, rows=[1, 3])
    assert np.allclose(U2, U[[1, 3]], atol=1e-14) and np.allclose(E2, E[[1, 3]], atol=1e-14)


def test_P4_limits_and_continuity():
    r = np.array([0.0, 0.6, 1.7, 1.999999, 2.000001, 2.6, 4.5])
    fr = fn.free_space(r, A)
    lo = fn.real_space_functions(r, 1e-3, A)       # xi -> 0: everything stays in real space
    hi = fn.real_space_functions(r[1:], 12.0, A)   # xi -> inf: everything moves to wave space (r > 0)
    for n in fn.NAMES:
        assert np.abs(lo[n] - fr[n]).max() < 2e-3, n     # W_X = O(xi a) as xi -> 0 (3 xi a/sqrt(pi) for F1)
        assert np.abs(hi[n][4:]).max() < 1e-9, n    # exponentially small for r > 2a
        assert np.abs(hi[n][:4]).max() < 1e-3, n    # only O(xi^-4) inside the overlap region (kink of the RPY forms)
        assert abs(fr[n][3] - fr[n][4]) < 1e-5, n   # continuous at r = 2a


def test_P5_free_space_is_the_unsplit_fourier_integral():
    """Free_X(r) = W_X(r; xi -> inf): the closed forms are the inverse transforms of Eqs. (15)-(18); the
    quadrature (with H -> 1 on the resolved band) reproduces them independently of the algebra."""
    r = np.array([0.6, 1.2, 1.9, 2.6, 3.3, 4.5, 6.0])   # (r - 2a) xi >= 7 for the r > 2a points
    fr, wv, wv2 = fn.free_space(r, A), fn.wave_integrals(r, 12.0, A), fn.wave_integrals(r, 24.0, A)
    for n in fn.NAMES:
        assert np.abs(fr[n] - wv[n])[3:].max() < 1e-9, (n, fr[n] - wv[n])        # r > 2a: exact
        d1, d2 = np.abs(fr[n] - wv[n])[:3], np.abs(fr[n] - wv2[n])[:3]
        assert d1.max() < 1e-3 and np.all(d2 < d1 / 8), (n, d1, d2)              # r < 2a: O(xi^-4) approach


def test_P5_rpy_textbook_values():
    """Rotne-Prager-Yamakawa numbers everyone knows: touching spheres and complete overlap."""
    fr = fn.free_space(np.array([2.0, 0.0, 4.0]), A)
    assert abs(fr['F1'][0] - (3 / 8 + 1 / 16)) < 1e-15 and abs(fr['F2'][0] - (3 / 4 - 1 / 8)) < 1e-15
    assert fr['F1'][1] == 1.0 and fr['F2'][1] == 1.0
    assert abs(fr['F2'][2] - (3 / 8 - 1 / 64)) < 1e-15       # (3a/2r)(1 - 2a^2/3r^2) at r = 4a
    assert abs(fr['Z0'][1] - 4.5) < 1e-15                    # 6 pi eta a / (20/3 pi eta a^3) * ... = 9/(2 a^2) -> E = S/(20/3 pi eta a^3)


@pytest.mark.parametrize('xi', [0.3, 0.45, 0.8])
def test_P6_printed_closed_forms(xi):
    r = np.array([0.6, 1.7, 1.999, 2.001, 2.6, 4.5])
    R = fn.real_space_functions(r, xi, A)
    for i, ri in enumerate(r):
        assert abs(R['F1'][i] - app.F1(ri, A, xi)) < 1e-10
        assert abs(R['F2'][i] - app.F2(ri, A, xi)) < 1e-10
        assert abs(2 * R['G2'][i] - app.G2(ri, A, xi)) < 1e-9
    assert abs(fn.real_space_functions(np.array([0.0]), xi, A)['F1'][0] - app.self_UF(A, xi)) < 1e-12


def test_P9_exact_covariance_identity():
    """A_w A_w^T = M_w restricted to the grid's wave vectors, for unit-variance noise (Eq. 73)."""
    x = np.array([[0.3, 0.4, 0.5], [2.2, 1.0, 0.9], [1.1, 3.0, 2.5]])
    L, xi = 5.0, 0.7
    for Mg in (6, 5):
        Aw = brn.wave_sqrt_dense(x, L, A, ETA, xi, Mg)
        k = brn.grid_modes(Mg, L)
        k2 = np.einsum('ki,ki->k', k, k)
        Mw = mob.dense_wave_modes(x, A, k, fn.hasimoto_H(np.sqrt(k2), xi) / (ETA * L**3 * k2))
        assert np.abs(Aw @ Aw.T - Mw).max() < 1e-13
        # conjugate partners and Nyquist / k = 0 entries carry no weight
        used = (np.abs(Aw).sum(axis=0) > 0).reshape(3, Mg, Mg, Mg // 2 + 1, 2)
        idx, _ = brn.canonical_modes(Mg)
        canon = np.zeros((Mg, Mg, Mg // 2 + 1), bool)
        canon[idx[:, 0], idx[:, 1], idx[:, 2]] = True
        assert not used[:, ~canon, :].any() and used[:, canon, :].mean() > 0.9


def test_P10_statistical_covariance_small():
    """<u u^T> -> (2kT/dt) M over many seeds (Eq. B4); M_r^{1/2} part exact by construction."""
    x = X4[:2]
    L, xi, Mg, kT, dt = 7.0, 0.6, 6, 1.3, 0.5
    Mr = mob.dense_real(x, L, A, ETA, xi)
    Sr = brn.sqrtm_psd(Mr)
    assert np.abs(Sr @ Sr - Mr).max() < 1e-13
    Aw = brn.wave_sqrt_dense(x, L, A, ETA, xi, Mg)
    g = np.random.default_rng(5)
    n = 20000
    u = np.sqrt(2 * kT / dt) * (g.standard_normal((n, 16)) @ Sr.T + g.standard_normal((n, Aw.shape[1])) @ Aw.T)
    C = u.T @ u / n
    want = 2 * kT / dt * (Mr + Aw @ Aw.T)
    assert np.abs(C - want).max() < 6 * np.abs(want).max() / np.sqrt(n)


def test_P12_schur_complement_solve():
    """Constraint solve gives E = 0 exactly and U = (M_UF - M_US M_ES^-1 M_EF) F (Eqs. 36-38)."""
    N = 4
    M = mob.dense(X4, 7.0, A, ETA, 0.6)
    rng = np.random.default_rng(2)
    FP = rng.standard_normal((N, 3))
    U, S = brn.constrained_solve(M, N, np.zeros((N, 3)), np.zeros((N, 5)), FP)
    out = (M @ np.concatenate([FP, S], 1).ravel()).reshape(N, 8)
    assert np.abs(out[:, 3:]).max() < 1e-13 and np.abs(out[:, :3] - U).max() < 1e-13
    # the constrained mobility is symmetric positive definite and smaller than M_UF (rigidity adds dissipation)
    iu = (8 * np.arange(N)[:, None] + np.arange(3)).ravel()
    ie = (8 * np.arange(N)[:, None] + 3 + np.arange(5)).ravel()
    Mc = M[np.ix_(iu, iu)] - M[np.ix_(iu, ie)] @ np.linalg.solve(M[np.ix_(ie, ie)], M[np.ix_(ie, iu)])
    assert np.abs(Mc - Mc.T).max() < 1e-13
    assert np.linalg.eigvalsh(Mc).min() > 0 and np.linalg.eigvalsh(M[np.ix_(iu, iu)] - Mc).min() > -1e-13


def test_P13_bond_force_is_minus_gradient_of_the_test_potential():
    """U(r) = k |r - r0|: F = -grad U by central differences, including a bond through the periodic
    boundary and particles in several bonds; the forces of a bond sum to zero."""
    L, k, r0 = 9.0, 2.5, 3.0
    x = np.array([[0.5, 0.6, 0.7], [8.6, 1.0, 0.9], [1.1, 4.0, 5.5], [2.0, 2.0, 2.3], [5.0, 5.5, 2.0]])
    pairs = np.array([[0, 1], [2, 3], [3, 0], [4, 2]])

    def energy(y):
        d = y[pairs[:, 0]] - y[pairs[:, 1]]
        d -= L * np.round(d / L)
        return k * np.abs(np.linalg.norm(d, axis=1) - r0).sum()
    F = brn.bond_forces(x, L, pairs, k, r0)
    h = 1e-6
    for i in range(5):
        for c in range(3):
            xp, xm = x.copy(), x.copy()
            xp[i, c] += h
            xm[i, c] -= h
            assert abs(F[i, c] + (energy(xp) - energy(xm)) / (2 * h)) < 1e-8
    assert np.abs(F.sum(axis=0)).max() < 1e-14
    # bond 0-1 passes through the boundary (minimum-image distance 1.97 < r0: repulsive, 0 pushed towards +x)
    F01 = brn.bond_forces(x, L, pairs[:1], k, r0)
    assert F01[0, 0] > 0 and np.isclose(np.linalg.norm(F01[0]), k)


def test_P14_eq80_is_the_normalised_boltzmann_density_of_the_pair_distance():
    """Eq. (80) as printed: integrates to one and equals r^2 exp(-U/kT) up to that constant."""
    for kt, r0 in [(3.0, 5.0), (1.0, 2.5), (6.0, 4.0)]:
        r = np.linspace(0.0, r0 + 60.0 / kt, 400001)
        f = brn.pair_distance_pdf(r, kt, r0)
        tail = np.exp(-kt * r0) * (2 / kt**3 - 0)      # part of the r^2 e^{-kt|r-r0|} integral that a formula on (-inf, inf) would add
        assert abs(np.trapezoid(f, r) - 1.0) < 2e-3 + tail
        w = r[1:]**2 * np.exp(-kt * np.abs(r[1:] - r0))
        assert np.allclose(f[1:] / w, f[1000] / (r[1000]**2 * np.exp(-kt * abs(r[1000] - r0))), rtol=1e-12)


def test_P15_oracle_midpoint_steps_sample_eq80():
    """Two bonded spheres, 1 500 oracle mid-point steps (Eqs. 76-79) with fresh noise: <|r - r0|> of Eq. (80) within the
    statistical error of ~35 independent samples (a wrong noise amplitude or a missing factor 2 in kT fails it; the
    sharp version of this test runs on the GPU, tests/test_gpu_equilibrium.py)."""
    L, xi, Mg, dt, k, r0, kT = 12.0, 0.3, 8, 4e-3, 6.0, 4.0, 1.0
    x = np.array([[4.0, 4.0, 4.0], [8.0, 4.0, 4.0]])
    g = np.random.Generator(np.random.Philox(7))
    bonds = (np.array([[0, 1]]), k, r0)
    rs = []
    for s in range(1500):
        w1, w2 = g.standard_normal(16), g.standard_normal((3, Mg, Mg, Mg // 2 + 1, 2))
        x, _, _ = brn.step(x, L, A, ETA, kT, xi, dt, Mg, w1, w2, eps=1e-6, bonds=bonds)
        d = x[0] - x[1]
        d -= L * np.round(d / L)
        rs.append(np.linalg.norm(d))
    rs = np.array(rs[60:])
    r = np.linspace(0.0, L / 2, 60001)
    f = brn.pair_distance_pdf(r, k / kT, r0)
    want = np.trapezoid(f * np.abs(r - r0), r)
    got = np.abs(rs - r0).mean()
    assert 0.6 * want < got < 1.5 * want, (got, want)
    assert abs(rs.mean() - np.trapezoid(f * r, r)) < 0.12


def test_P16_divergence_of_M_UF_vanishes_and_constrained_drift_is_antisymmetric():
    """'because div M_UF = 0': the RPY block of the periodic grand mobility is divergence-free, also for an
    overlapping pair; the divergence of the constrained mobility R_FU^-1 (the drift of Eq. B12) is not,
    and for two spheres it is equal and opposite along the line of centres."""
    L, xi = 16.0, 0.5
    for r in (1.7, 2.5):
        x = np.array([[4.0, 4.0, 4.0], [4.0 + r, 4.0, 4.0]])
        div_c, div_uf = brn.constrained_mobility_divergence(x, L, A, ETA, xi)
        assert np.abs(div_uf).max() < 2e-9
        assert abs(div_c[0]) > 5e-3 and abs(div_c[0] + div_c[3]) < 1e-9
        assert np.abs(div_c[[1, 2, 4, 5]]).max() < 1e-9
    M = mob.dense(x, L, A, ETA, xi)
    Mc = brn.constrained_mobility(M, 2)
    U, _ = brn.constrained_solve(M, 2, np.zeros((2, 3)), np.zeros((2, 5)), np.eye(6)[2].reshape(2, 3))
    assert np.abs(Mc[:, 2] - U.ravel()).max() < 1e-14


@pytest.mark.parametrize('xi', [0.3, 0.45, 0.8])
def test_P6_printed_closed_forms_of_the_dipole_couplings(xi):
    """The other printed forms of Appendix A that survive the extraction (SURVEY.md 8(c) errata): K3 in both cases
     pins (Z2 + Z4)/7, G1 for r > 2a pins G1 (printed = -2 R_G1 at a = 1), and the self term
    (A12) pins Z0(0)/5 = -3 x its bracket."""
    r = np.array([0.6, 1.7, 1.999, 2.001, 2.6, 4.5])
    R = fn.real_space_functions(r, xi, A)
    _, _, C, _ = fn.rank4_combinations(R)
    for i, ri in enumerate(r):
        assert abs(C[i] - app.K3(ri, A, xi)) < 1e-10
        if ri > 2 * A:
            assert abs(-2 * R['G1'][i] - app.G1_case1(ri, A, xi)) < 1e-10
    R0 = fn.real_space_functions(np.zeros(1), xi, A)
    assert abs(R0['Z0'][0] / 5 + 3 * app.self_DC_bracket(A, xi)) < 1e-12


def test_heyes_melrose_moves_a_free_draining_pair_exactly_to_contact():
    """What the force is FOR (reading R12): a free-draining pair (mobility 1/(6 pi eta a) each) at separation r < 2a
    moved for one dt by its Heyes-Melrose forces ends at r = 2a exactly; separated pairs feel nothing; pairs through the
    periodic boundary are found; forces sum to zero."""
    L, dt = 11.0, 3e-3
    for a, eta in [(1.0, ETA), (0.7, 0.31)]:
        for r in (1.2 * a, 1.7 * a, 1.999 * a):
            d = np.array([0.3, -0.5, 0.81]); d *= r / np.linalg.norm(d)
            x = np.array([[10.8, 0.2, 5.0], [10.8, 0.2, 5.0] + d]) % L            # pair straddles the boundary
            F = brn.heyes_melrose(x, L, a, eta, dt)
            xn = x + dt * F / (6 * np.pi * eta * a)
            dn = xn[0] - xn[1]
            dn -= L * np.round(dn / L)
            assert abs(np.linalg.norm(dn) - 2 * a) < 1e-13 and np.abs(F.sum(axis=0)).max() < 1e-12
    x = np.array([[1.0, 1.0, 1.0], [3.001, 1.0, 1.0], [1.0, 2.5, 1.0]])            # 0-1 apart, 0-2 overlapping
    F = brn.heyes_melrose(x, L, 1.0, ETA, dt)
    assert np.all(F[1] == 0) and F[0, 1] < 0 < F[2, 1] and F[0, 0] == 0


def test_brownian_amplitude_and_composition_against_its_dense_factors():
    """oracle.brownian.brownian = sqrt(2kT/dt) (sqrtm(M_r) w1 + A_w w2) with exactly that amplitude (Eq. B4) and
    the per-particle (U, e1..e5) ordering of w1."""
    x, L, xi, Mg, kT, dt = X4[:3], 7.0, 0.6, 6, 1.7, 0.02
    g = np.random.default_rng(3)
    w1, w2 = g.standard_normal(24), g.standard_normal((3, Mg, Mg, Mg // 2 + 1, 2))
    U, E = brn.brownian(x, L, A, ETA, kT, xi, dt, Mg, w1, w2)
    want = np.sqrt(2 * kT / dt) * (brn.sqrtm_psd(mob.dense_real(x, L, A, ETA, xi)) @ w1 + brn.wave_sqrt_dense(x, L, A, ETA, xi, Mg) @ w2.ravel())
    assert np.abs(np.hstack([U, E]).ravel() - want).max() < 1e-11
    U4, _ = brn.brownian(x, L, A, ETA, 4 * kT, xi, dt / 4, Mg, w1, w2)
    assert np.allclose(U4, 4 * U, rtol=1e-13)


def test_midpoint_step_structure_written_out_by_hand():
    """Eqs. (76)-(79) for two spheres with a fixed noise vector, every line written out from the dense
    matrices: the half step uses dt/2 (Eq. 77), the matrix of the solve is the one at x_{k+1/2} (Eq. 78), the full step
    starts again from x_k (Eq. 79), and E = 0 holds for the returned S."""
    L, xi, Mg, kT, dt = 9.0, 0.6, 6, 1.0, 0.05
    x = np.array([[3.0, 3.0, 3.0], [5.3, 3.4, 2.8]])
    g = np.random.default_rng(11)
    w1, w2 = g.standard_normal(16), g.standard_normal((3, Mg, Mg, Mg // 2 + 1, 2))
    xn, U, S = brn.step(x, L, A, ETA, kT, xi, dt, Mg, w1, w2)
    ub = (np.sqrt(2 * kT / dt) * (brn.sqrtm_psd(mob.dense_real(x, L, A, ETA, xi)) @ w1
                                  + brn.wave_sqrt_dense(x, L, A, ETA, xi, Mg) @ w2.ravel())).reshape(2, 8)
    xh = x + 0.5 * dt * ub[:, :3]                                         # (77)
    Mh = mob.dense(xh, L, A, ETA, xi)                                     # matrix at the mid-point
    iu, ie = np.array([0, 1, 2, 8, 9, 10]), np.array([3, 4, 5, 6, 7, 11, 12, 13, 14, 15])
    Sh = np.linalg.solve(Mh[np.ix_(ie, ie)], -ub[:, 3:].ravel())          # (78) with F^P = 0 (no overlap, no bonds)
    Uh = ub[:, :3].ravel() + Mh[np.ix_(iu, ie)] @ Sh
    assert np.abs(brn.heyes_melrose(xh, L, A, ETA, dt)).max() == 0
    assert np.abs(U.ravel() - Uh).max() < 1e-12 and np.abs(S.ravel() - Sh).max() < 1e-11
    assert np.abs(xn - (x + dt * Uh.reshape(2, 3))).max() < 1e-13       # (79)
    # a full-dt half step, or the matrix at x_k, is a different (wrong) scheme and is told apart
    Mk = mob.dense(x, L, A, ETA, xi)
    Uk = ub[:, :3].ravel() + Mk[np.ix_(iu, ie)] @ np.linalg.solve(Mk[np.ix_(ie, ie)], -ub[:, 3:].ravel())
    assert np.abs(Uk - Uh).max() > 1e-4
