"""Pins of the fp64 CPU PSE reference (oracle/pse_reference.py, oracle/krylov.py) against the direct O(N^2) oracle and dense
linear algebra (CPU only, -m "not gpu").  SURVEY.md 8(c) pin P11: the NUFFT pipeline equals the direct k-sum to the
tolerance it was built for, and the error falls with that tolerance.
"""
import numpy as np
import pytest

import synth
from oracle import brownian as brn
from oracle import krylov
from oracle import mobility as mob
from oracle import pse_reference as pr

A, ETA, KT = 1.0, 1.0 / (6.0 * np.pi), 1.0


def rel(a, b):
    return float(np.linalg.norm(np.asarray(a) - np.asarray(b)) / np.linalg.norm(np.asarray(b)))


@pytest.fixture(scope='module')
def small():
    x, L = synth.rsa(300, 0.20, seed=3)
    x[7] = x[3] + np.array([1.1, 0.9, 0.6])             # one overlapping pair (r = 1.54 < 2a): the regularised branch
    F, S = synth.gaussian_inputs(300, 1)
    return x % L, L, F.astype(np.float64), S.astype(np.float64)


def test_real_space_cells_and_table_against_direct_sum(small):
    """Linked cells + fine table (C) and k-d tree + per-pair quadrature (numpy) against the brute-force image sum truncated at
    the same r_cut; a box with 2 cells per side (every cell visited once) and one with more."""
    x, L, F, S = small
    for xi in (0.9, 1.6):
        ref = pr.PSEReference(L, A, ETA, xi, tol=1e-8)
        Uo, Eo = mob.real_apply(x, L, A, ETA, xi, F, S, rcut=ref.rcut)
        U, E = ref.real_apply(x, F, S)
        assert rel(np.hstack([U, E]), np.hstack([Uo, Eo])) < 2e-9
        rows = np.array([0, 3, 7, 150, 299])
        Ux, Ex = ref.real_apply(x, F, S, rows=rows, exact=True)
        assert rel(np.hstack([Ux, Ex]), np.hstack([Uo, Eo])[rows]) < 1e-13
        Ur, Er = ref.real_apply(x, F, S, rows=rows)
        assert np.allclose(Ur, U[rows], rtol=0, atol=0) and np.allclose(Er, E[rows], rtol=0, atol=0)


def test_P11_wave_space_nufft_against_direct_k_sum_error_falls_with_tol(small):
    x, L, F, S = small
    xi = 0.9
    Uo, Eo = mob.wave_apply(x, L, A, ETA, xi, F, S)
    want = np.hstack([Uo, Eo])
    errs = []
    for tol in (1e-2, 1e-4, 1e-6, 1e-8):
        ref = pr.PSEReference(L, A, ETA, xi, tol=tol)
        U, E = ref.wave_apply(x, F, S)
        errs.append(rel(np.hstack([U, E]), want))
        assert errs[-1] < 3 * tol, (tol, errs)
    assert errs[3] < 1e-7 and all(errs[i + 1] < 0.1 * errs[i] for i in range(3)), errs
    rows = np.array([5, 17, 200])
    Ur, Er = ref.wave_apply(x, F, S, rows=rows)
    assert np.array_equal(Ur, U[rows]) and np.array_equal(Er, E[rows])


def test_full_product_sampled_rows_mid_size_other_xi():
    """N = 2 500 at phi = 0.3: reference at its own xi against the direct sums at another xi, on sampled rows, U and E."""
    x, L = synth.rsa(2500, 0.30, seed=22)
    F, S = synth.gaussian_inputs(2500, 22)
    rows = np.sort(np.random.default_rng(1).choice(2500, 16, replace=False))
    Uo, Eo = mob.mobility_apply(x, L, A, ETA, 0.6, F, S, rows=rows, eps=1e-11)
    ref = pr.PSEReference(L, A, ETA, 0.45, tol=1e-8)
    U, E = ref.apply(x, F, S, rows=rows)
    assert rel(U, Uo) < 1e-7 and rel(E, Eo) < 1e-7
    Ux, Ex = ref.apply(x, F, S, rows=rows, exact_real=True)
    assert rel(Ux, Uo) < 1e-7 and rel(Ex, Eo) < 1e-7


def test_wave_square_root_on_finer_grid_equals_direct_sum_over_noise_grid_modes(small):
    x, L, _, _ = small
    xi = 0.7
    for Mg in (12, 15):
        _, w2 = synth.brownian_noise(300, Mg, seed=Mg)
        Uo, Eo = brn.wave_sqrt_apply(x, L, A, ETA, xi, Mg, w2)
        ref = pr.PSEReference(L, A, ETA, xi, tol=1e-8)
        assert ref.M >= Mg
        U, E = ref.wave_sqrt_apply(x, Mg, w2)
        assert rel(np.hstack([U, E]), np.hstack([Uo, Eo])) < 1e-7


def test_lanczos_square_root_and_gmres_against_dense_algebra():
    rng = np.random.default_rng(5)
    B = rng.standard_normal((60, 60))
    Aspd = B @ B.T + 0.5 * np.eye(60)
    w = rng.standard_normal(60)
    y, m = krylov.lanczos_sqrt(lambda v: Aspd @ v, w, tol=1e-12)
    assert rel(y, brn.sqrtm_psd(Aspd) @ w) < 1e-10 and m <= 60
    C = Aspd + 0.3 * rng.standard_normal((60, 60))          # non-symmetric
    b = rng.standard_normal(60)
    s, m = krylov.gmres(lambda v: C @ v, b, tol=1e-12)
    assert rel(s, np.linalg.solve(C, b)) < 1e-10 and m <= 60
    assert krylov.gmres(lambda v: C @ v, np.zeros(60))[1] == 0 and krylov.lanczos_sqrt(lambda v: Aspd @ v, np.zeros(60))[1] == 0


def test_reference_step_against_dense_oracle_step():
    """Eqs. (76)-(79) on the fast operators (Lanczos, NUFFT, GMRES) against the dense oracle (eigh, direct sums, LU) at N = 60
    with overlapping pairs (F^P != 0)."""
    N, xi, dt, Mg = 60, 1.1, 1e-3, 14
    x, L = synth.rsa(N, 0.10, seed=6)
    x, L = x * 0.9, L * 0.9
    w1, w2 = synth.brownian_noise(N, Mg, 2)
    xo, Uo, So = brn.step(x, L, A, ETA, KT, xi, dt, Mg, w1, w2, eps=1e-12)
    xr, Ur, Sr, (li, gi) = pr.step(x, L, A, ETA, KT, xi, dt, Mg, w1, w2, tol=1e-8)
    assert np.abs(brn.heyes_melrose(x, L, A, ETA, dt)).max() > 0
    assert rel(Ur, Uo) < 1e-6 and rel(Sr, So) < 1e-6
    assert rel(xr - x, xo - x) < 1e-6 and 2 <= li <= 60 and 2 <= gi <= 60


def test_tree_based_overlap_force_equals_the_dense_one():
    x, L = synth.rsa(400, 0.30, seed=2)
    x, L = x * 0.93, L * 0.93
    Fd = brn.heyes_melrose(x, L, A, ETA, 1e-3)
    assert np.abs(Fd).max() > 0 and np.abs(Fd - pr.heyes_melrose(x, L, A, ETA, 1e-3)).max() < 1e-11


def test_full_couplet_reference_against_direct_sums(small):
    """Torque in, angular velocity out (oracle/couplet.py) through the reference's NUFFT and cut-off pair sum: every output block
    against the direct Ewald sums at another xi, all rows at N = 300 (one overlapping pair) and sampled rows at N = 600."""
    from oracle import couplet as cpl
    x, L, F, S = small
    Lq = np.random.default_rng(8).standard_normal((300, 3))
    want = cpl.mobility_apply_full(x, L, A, ETA, 0.7, F, Lq, S, eps=1e-12)
    ref = pr.PSEReference(L, A, ETA, 0.9, tol=1e-8)
    got = ref.apply_full(x, F, Lq, S)
    for g, w in zip(got, want):
        assert rel(g, w) < 1e-7
    wr = cpl.mobility_apply_full(x, L, A, ETA, 0.9, F, Lq, S, eps=1e-12, part='wave')
    for g, w, t in zip(ref.wave_apply_full(x, F, Lq, S), wr, want):
        assert np.linalg.norm(g - w) < 1e-7 * np.linalg.norm(t)
    x, L = synth.rsa(600, 0.30, seed=22)
    F, S = synth.gaussian_inputs(600, 22)
    Lq = np.random.default_rng(9).standard_normal((600, 3))
    rows = np.sort(np.random.default_rng(1).choice(600, 8, replace=False))
    want = cpl.mobility_apply_full(x, L, A, ETA, 0.75, F, Lq, S, rows=rows, eps=1e-11)
    got = pr.PSEReference(L, A, ETA, 0.6, tol=1e-8).apply_full(x, F, Lq, S, rows=rows)
    for g, w in zip(got, want):
        assert rel(g, w) < 1e-7
