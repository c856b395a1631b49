"""GPU parity: libpse (through its C ABI / ctypes binding) against the CPU fp64 oracle on the same seeded inputs.

Tolerance (BASELINE.json north_star): neighbour lists bit-exact as sets; fp32 product and Brownian sample within
relative L2 error max(2*tol, 1e-5) of the fp64 oracle, tol = configured Ewald tolerance.
"""
import numpy as np
import pytest

import synth
from oracle import brownian as brn
from oracle import functions as fn
from oracle import mobility as mob
from oracle import neighbors as nbo

pytestmark = pytest.mark.gpu
torch = pytest.importorskip('torch')

A, ETA, KT = 1.0, 1.0 / (6.0 * np.pi), 1.0


def rel(a, b):
    return float(np.linalg.norm(np.asarray(a, float) - np.asarray(b, float)) / np.linalg.norm(np.asarray(b, float)))


def bar(tol):
    return max(2 * tol, 1e-5)


def dev(x, dtype=torch.float32):
    return torch.as_tensor(np.ascontiguousarray(x), dtype=dtype).cuda().contiguous()


def pos4(x):
    p = np.zeros((x.shape[0], 4), np.float32)
    p[:, :3] = x
    return p


def make_ctx(N, L, xi, grid, P, rcut, tol):
    import paper_1709_06946_b200 as pse
    return pse.pse_create(N, L, A, ETA, KT, xi, grid, P, rcut, tol)


@pytest.fixture(scope='module')
def config1():
    """BASELINE.json configs[0]: N=64, phi=0.10, tol=1e-3, grid 32^3, P=8, xi=0.6 (R7)."""
    import paper_1709_06946_b200 as pse
    x, L = synth.rsa(64, 0.10, seed=1)
    x32 = x.astype(np.float32)
    xi, grid, P, tol = 0.6, 32, 8, 1e-3
    st, _, _, rcut = pse.pse_suggest_params(64, L, A, tol, xi)
    assert st == 0 and rcut <= L / 2
    ctx = make_ctx(64, L, xi, grid, P, rcut, tol)
    ctx.pse_neighbors(dev(pos4(x32)))
    F, S = synth.gaussian_inputs(64, 0)
    return dict(ctx=ctx, x=x32.astype(np.float64), x32=x32, L=L, xi=xi, grid=grid, P=P, tol=tol, rcut=rcut, F=F, S=S)


def gpu_apply(ctx, F, S, which):
    N = F.shape[0]
    U, E = torch.empty(N, 3, device='cuda'), torch.empty(N, 5, device='cuda')
    ctx.pse_mobility_apply(dev(F), dev(S), U, E, which)
    torch.cuda.synchronize()
    return U.cpu().numpy(), E.cpu().numpy()


def nbr_sets_from_gpu(ctx):
    count, index = ctx.pse_get_neighbors()
    count, index = count.cpu().numpy(), index.cpu().numpy()
    off = np.concatenate([[0], np.cumsum(count)])
    return [np.sort(index[off[i]:off[i + 1]]) for i in range(len(count))]


def test_neighbors_bit_exact_config1(config1):
    got = nbr_sets_from_gpu(config1['ctx'])
    want = nbo.neighbor_sets(config1['x32'], config1['L'], config1['rcut'])
    for g, w in zip(got, want):
        assert np.array_equal(g, w)


@pytest.mark.parametrize('N,phi,xi,seed,shift', [(500, 0.30, 0.9, 3, False), (777, 0.05, 0.5, 4, True), (30, 0.02, 0.35, 5, True),
                                                 (1500, 0.30, 0.23, 6, False)])
def test_neighbors_bit_exact_other(N, phi, xi, seed, shift):
    """Ragged sizes, dense and dilute, unwrapped inputs, a box with fewer than 3 cells per side, and (last case) cells
    with more than 1024 candidates, which take the two-pass fallback of the neighbour build."""
    import paper_1709_06946_b200 as pse
    x, L = synth.rsa(N, phi, seed=seed)
    if shift:
        x = x + L * np.random.default_rng(seed).integers(-2, 3, size=x.shape)
    x32 = x.astype(np.float32)
    rcut = min(pse.pse_suggest_params(N, L, A, 1e-3, xi)[3], 0.5 * L)
    ctx = make_ctx(N, L, xi, 32, 6, rcut, 1e-3)
    ctx.pse_neighbors(dev(pos4(x32)))
    got, want = nbr_sets_from_gpu(ctx), nbo.neighbor_sets(x32, L, rcut)
    assert sum(len(w) for w in want) > 0
    for g, w in zip(got, want):
        assert np.array_equal(g, w)


def test_table_matches_oracle_functions(config1):
    tab, dr = config1['ctx'].pse_get_table()
    r = np.arange(tab.shape[0]) * dr
    R = fn.real_space_functions(r, config1['xi'], A)
    Aa, B, C, D = fn.rank4_combinations(R)
    want = np.stack([R['F1'], R['F2'], R['G1'] + R['G2'], R['G1'] + 4 * R['G2'], Aa, B, D], 1) / (6 * np.pi * ETA * A)
    assert np.abs(tab[:, :7] - want).max() < 2e-6
    assert abs(r[-2] - config1['rcut']) < 1e-9


def test_real_space_product(config1):
    c = config1
    U, E = gpu_apply(c['ctx'], c['F'], c['S'], 1)
    # same truncated sum in fp64: isolates kernel arithmetic + table interpolation
    Ut, Et = mob.real_apply(c['x'], c['L'], A, ETA, c['xi'], c['F'], c['S'], rcut=c['rcut'])
    assert rel(np.hstack([U, E]), np.hstack([Ut, Et])) < 2e-5
    # converged real-space sum: adds the truncation error, must stay inside the Ewald tolerance
    Uc, Ec = mob.real_apply(c['x'], c['L'], A, ETA, c['xi'], c['F'], c['S'], eps=1e-12)
    assert rel(np.hstack([U, E]), np.hstack([Uc, Ec])) < c['tol']


def test_wave_space_product(config1):
    c = config1
    U, E = gpu_apply(c['ctx'], c['F'], c['S'], 2)
    # direct sum over exactly the grid's modes: isolates the NUFFT quadrature (P, Gaussian) + fp32 error
    k = brn.grid_modes(c['grid'], c['L'])
    k2 = np.einsum('ki,ki->k', k, k)
    w = fn.hasimoto_H(np.sqrt(k2), c['xi']) / (ETA * c['L']**3 * k2)
    Ug, Eg = mob.wave_apply_modes(c['x'], c['L'], A, ETA, k, w, c['F'], c['S'])
    assert rel(np.hstack([U, E]), np.hstack([Ug, Eg])) < c['tol']
    Uc, Ec = mob.wave_apply(c['x'], c['L'], A, ETA, c['xi'], c['F'], c['S'], eps=1e-12)
    assert rel(np.hstack([U, E]), np.hstack([Uc, Ec])) < c['tol']


def test_full_product_config1(config1):
    c = config1
    U, E = gpu_apply(c['ctx'], c['F'], c['S'], 3)
    Uo, Eo = mob.mobility_apply(c['x'], c['L'], A, ETA, c['xi'], c['F'], c['S'], eps=1e-12)
    assert rel(U, Uo) < bar(c['tol']) and rel(E, Eo) < bar(c['tol'])
    assert rel(np.hstack([U, E]), np.hstack([Uo, Eo])) < bar(c['tol'])


def test_product_is_linear_and_symmetric(config1):
    """x.(M y) = y.(M x) within fp32 + tolerance; M(ax+by) = aMx + bMy."""
    c = config1
    F2, S2 = synth.gaussian_inputs(64, 11)
    U1, E1 = gpu_apply(c['ctx'], c['F'], c['S'], 3)
    U2, E2 = gpu_apply(c['ctx'], F2, S2, 3)
    d12 = float((c['F'] * U2).sum() + (c['S'] * E2).sum())
    d21 = float((F2 * U1).sum() + (S2 * E1).sum())
    assert abs(d12 - d21) < 1e-3 * max(abs(d12), abs(d21), 1.0)
    U3, E3 = gpu_apply(c['ctx'], 2 * c['F'] - 3 * F2, 2 * c['S'] - 3 * S2, 3)
    assert rel(U3, 2 * U1 - 3 * U2) < 1e-5 and rel(E3, 2 * E1 - 3 * E2) < 1e-5
    assert float((c['F'] * U1).sum() + (c['S'] * E1).sum()) > 0


def test_brownian_sample_config1(config1):
    c = config1
    w1, w2 = synth.brownian_noise(64, c['grid'], 0)
    dt = 1e-3
    UB, EB = torch.empty(64, 3, device='cuda'), torch.empty(64, 5, device='cuda')
    it = c['ctx'].pse_brownian(dt, dev(w1.reshape(64, 8)), dev(w2), UB, EB)
    torch.cuda.synchronize()
    Uo, Eo = brn.brownian(c['x'], c['L'], A, ETA, KT, c['xi'], dt, c['grid'], w1, w2, eps=1e-12)
    assert 2 <= it <= 30
    assert rel(np.hstack([UB.cpu().numpy(), EB.cpu().numpy()]), np.hstack([Uo, Eo])) < bar(c['tol'])


def test_brownian_wave_part_alone(config1):
    """Zero real-space noise: the sample is sqrt(2kT/dt) A_w w2 exactly as the oracle's direct sum over grid modes."""
    c = config1
    _, w2 = synth.brownian_noise(64, c['grid'], 3)
    UB, EB = torch.empty(64, 3, device='cuda'), torch.empty(64, 5, device='cuda')
    c['ctx'].pse_brownian(0.5, torch.zeros(64, 8, device='cuda'), dev(w2), UB, EB)
    Uw, Ew = brn.wave_sqrt_apply(c['x'], c['L'], A, ETA, c['xi'], c['grid'], w2)
    amp = np.sqrt(2 * KT / 0.5)
    assert rel(np.hstack([UB.cpu().numpy(), EB.cpu().numpy()]), amp * np.hstack([Uw, Ew])) < c['tol']


def test_brownian_wave_part_at_a_large_grid_with_an_odd_finer_grid():
    """The wave half of the sample at tol 1e-4 on a 192^3 product grid (config 5's size at that tolerance), whose finer grid
    (reading R19) is the odd 243^3: sqrt(2kT/dt) A_w w2 on sampled particles against the oracle's direct sum over the grid's modes."""
    import paper_1709_06946_b200 as pse
    N, tol, xi, dt, Lbox = 3000, 1e-4, 0.30, 0.5, 300.0
    x, L = synth.rsa(N, N * 4 * np.pi / 3 / Lbox**3, seed=9)
    x32 = x.astype(np.float32)
    st, grid, P, rcut = pse.pse_suggest_params(N, L, A, tol, xi)
    assert st == 0 and (grid, P) == (192, 5)
    ctx = make_ctx(N, L, xi, grid, P, rcut, tol)
    ctx.pse_neighbors(dev(pos4(x32)))
    _, w2 = synth.brownian_noise(N, grid, 3)
    UB, EB = torch.empty(N, 3, device='cuda'), torch.empty(N, 5, device='cuda')
    ctx.pse_brownian(dt, torch.zeros(N, 8, device='cuda'), dev(w2), UB, EB)
    rows = np.sort(np.random.default_rng(1).choice(N, 16, replace=False))
    Uw, Ew = brn.wave_sqrt_apply(x32.astype(np.float64), L, A, ETA, xi, grid, w2, rows=rows)
    amp = np.sqrt(2 * KT / dt)
    assert rel(UB.cpu().numpy()[rows], amp * Uw) < bar(tol) and rel(EB.cpu().numpy()[rows], amp * Ew) < bar(tol)
    ctx.close()


def test_constrained_solve_and_hard_sphere_forces(config1):
    c = config1
    ctx, N = c['ctx'], 64
    # overlapping configuration: shrink the box coordinates so that some pairs overlap
    M = mob.dense(c['x'], c['L'], A, ETA, c['xi'], eps=1e-10)
    rng = np.random.default_rng(7)
    FP = rng.standard_normal((N, 3)).astype(np.float32)
    UBh = rng.standard_normal((N, 3)).astype(np.float32)
    EBh = rng.standard_normal((N, 5)).astype(np.float32)
    U, S = torch.empty(N, 3, device='cuda'), torch.empty(N, 5, device='cuda')
    it = ctx.pse_constrained_solve(dev(FP), dev(UBh), dev(EBh), U, S)
    Uo, So = brn.constrained_solve(M, N, UBh.astype(float), EBh.astype(float), FP.astype(float))
    assert 2 <= it <= 25
    assert rel(S.cpu().numpy(), So) < 5 * c['tol'] and rel(U.cpu().numpy(), Uo) < bar(c['tol'])


def test_hard_sphere_forces_match_oracle():
    x, L = synth.rsa(200, 0.25, seed=9)
    x = x * 0.93                      # compress: creates overlaps
    L2 = L * 0.93
    x32 = x.astype(np.float32)
    ctx = make_ctx(200, L2, 0.6, 32, 6, min(6.0, L2 / 2), 1e-3)
    ctx.pse_neighbors(dev(pos4(x32)))
    F = torch.empty(200, 3, device='cuda')
    ctx.pse_hard_sphere_forces(1e-3, F)
    Fo = brn.heyes_melrose(x32.astype(np.float64), L2, A, ETA, 1e-3)
    assert np.abs(Fo).max() > 0
    assert rel(F.cpu().numpy(), Fo) < 1e-4


def test_step_small_against_dense_oracle():
    """One mid-point step (Eqs. 76-79) on N=48 at phi=0.2, fp32 GPU vs dense fp64 oracle."""
    import paper_1709_06946_b200 as pse
    N, tol, xi, grid, P, dt = 48, 1e-4, 1.1, 32, 9, 1e-3
    x, L = synth.rsa(N, 0.20, seed=6)
    x32 = x.astype(np.float32)
    st, _, _, rcut = pse.pse_suggest_params(N, L, A, tol, xi)
    assert st == 0
    ctx = make_ctx(N, L, xi, grid, P, rcut, tol)
    w1, w2 = synth.brownian_noise(N, grid, 2)
    pos = dev(pos4(x32))
    gi, li = ctx.pse_step(pos, dt, dev(w1.reshape(N, 8)), dev(w2))
    xn, Uo, So = brn.step(x32.astype(np.float64), L, A, ETA, KT, xi, dt, grid, w1, w2, eps=1e-10)
    got = pos.cpu().numpy()[:, :3].astype(np.float64)
    d = got - xn
    d -= L * np.round(d / L)
    disp = xn - x32.astype(np.float64)
    assert 2 <= gi <= 30 and 2 <= li <= 40
    assert np.linalg.norm(d) / np.linalg.norm(disp) < 5 * tol


@pytest.mark.parametrize('N,phi,tol,xi,seed', [(3000, 0.20, 1e-3, 0.5, 21), (2500, 0.30, 1e-4, 0.6, 22), (3500, 0.10, 1e-2, 0.45, 23)])
def test_product_mid_size_sampled_rows(N, phi, tol, xi, seed):
    """Several cells and tiles per side, grid size not a multiple of the tile edge (ragged tail), parameters from
    pse_suggest_params; oracle on sampled output rows."""
    import paper_1709_06946_b200 as pse
    x, L = synth.rsa(N, phi, seed=seed)
    x32 = x.astype(np.float32)
    st, grid, P, rcut = pse.pse_suggest_params(N, L, A, tol, xi)
    assert st == 0
    ctx = make_ctx(N, L, xi, grid, P, rcut, tol)
    ctx.pse_neighbors(dev(pos4(x32)))
    F, S = synth.gaussian_inputs(N, seed)
    U, E = gpu_apply(ctx, F, S, 3)
    rows = np.sort(np.random.default_rng(seed).choice(N, 24, replace=False))
    Uo, Eo = mob.mobility_apply(x32.astype(np.float64), L, A, ETA, xi, F, S, rows=rows, eps=min(1e-7, tol * 1e-3))
    assert rel(U[rows], Uo) < bar(tol) and rel(E[rows], Eo) < bar(tol)


def full_size_checks(x, L, tol, xi_bench, xi_other, bench_params, seed):
    """Checks that hold at any size, for the workloads the O(N^2) oracle cannot finish: (i) neighbour sets of sampled
    particles bit-exact against the fp32 brute force; (ii) the real-space product exactly on sampled rows; (iii) the full
    product independent of xi (other r_cut, grid, tables) and symmetric.  Returns the mean neighbour count at xi_bench."""
    import paper_1709_06946_b200 as pse
    N = x.shape[0]
    x32 = x.astype(np.float32)
    F, S = synth.gaussian_inputs(N, 1)
    F2, S2 = synth.gaussian_inputs(N, 2)
    rows = np.sort(np.random.default_rng(seed).choice(N, 12, replace=False))
    res, nb_mean = {}, None
    for xi in (xi_bench, xi_other):
        st, grid, P, rcut = pse.pse_suggest_params(N, L, A, tol, xi)
        assert st == 0 and (xi != xi_bench or (grid, P) == bench_params)
        ctx = make_ctx(N, L, xi, grid, P, rcut, tol)
        ctx.pse_neighbors(dev(pos4(x32)))
        if xi == xi_bench:
            count, index = ctx.pse_get_neighbors()
            count = count.cpu().numpy()
            off = np.concatenate([[0], np.cumsum(count)])
            want = nbo.neighbor_sets(pos4(x32), L, rcut, rows=rows)
            for r, w in zip(rows, want):
                assert np.array_equal(np.sort(index[off[r]:off[r + 1]].cpu().numpy()), w)
            nb_mean = count.mean()
        res[xi] = dict(full=np.hstack(gpu_apply(ctx, F, S, 3)), real=np.hstack(gpu_apply(ctx, F, S, 1)), rcut=rcut,
                       full2=np.hstack(gpu_apply(ctx, F2, S2, 3)))
        ctx.close()
    assert rel(res[xi_bench]['full'], res[xi_other]['full']) < bar(tol)
    v1, v2 = np.hstack([F, S]).astype(np.float64), np.hstack([F2, S2]).astype(np.float64)
    a, b = res[xi_bench]['full'].astype(np.float64), res[xi_bench]['full2'].astype(np.float64)
    d12, d21 = float((v1 * b).sum()), float((v2 * a).sum())
    assert abs(d12 - d21) < bar(tol) * np.sqrt(float((v1 * a).sum()) * float((v2 * b).sum()))
    assert float((v1 * a).sum()) > 0
    Ur, Er = mob.real_apply(x32.astype(np.float64), L, A, ETA, xi_bench, F, S, rows=rows[:6], rcut=res[xi_bench]['rcut'])
    assert rel(res[xi_bench]['real'][rows[:6]], np.hstack([Ur, Er])) < 2e-5
    return nb_mean


def test_config4_full_size_sampled_neighbors_rows_and_properties():
    """BASELINE.json configs[3] (N=1 048 576, phi=0.10, tol=1e-3) with bench.py's parameters (xi=0.34, grid 216, P=4),
    against xi = 0.42."""
    x, L = synth.rsa(1048576, 0.10, seed=4)
    nb = full_size_checks(x, L, 1e-3, 0.34, 0.42, (216, 4), seed=4)
    assert abs(nb - 65.9) < 1.0


def test_config5_full_size_sampled_neighbors_rows_and_properties():
    """BASELINE.json configs[4] (N=262 144 in 32-sphere fractal aggregates, phi=0.05, tol=1e-3) with bench.py's parameters
    (xi=0.28, grid 144, P=4), against xi = 0.36."""
    x, L = synth.fractal_aggregates(262144, 0.05, seed=5)
    nb = full_size_checks(x, L, 1e-3, 0.28, 0.36, (144, 4), seed=5)
    assert 56.0 < nb < 66.0          # bench.py reports 60; uniform suspension at the same phi: phi r_cut^3 = 56


@pytest.mark.parametrize('grid', [35, 45])
def test_odd_grid_component_masks(grid):
    """Odd M: M^3 is odd, so the S / E planes (first plane 3) of a packed [8][M^3] array would start 4-byte aligned only
    and cuFFT rejects them; the planes are pse_plane_stride(M) apart instead.  S -> E, F -> U and full products."""
    N, xi, tol = 400, 0.5, 1e-3
    x, L = synth.rsa(N, 0.15, seed=41)
    x32 = x.astype(np.float32)
    rcut = np.sqrt(-np.log(tol)) / xi + 1.0
    ctx = make_ctx(N, L, xi, grid, 6, rcut, tol)
    ctx.pse_neighbors(dev(pos4(x32)))
    F, S = synth.gaussian_inputs(N, 41)
    k = brn.grid_modes(grid, L)
    k2 = np.einsum('ki,ki->k', k, k)
    w = fn.hasimoto_H(np.sqrt(k2), xi) / (ETA * L**3 * k2)
    Ug, Eg = mob.wave_apply_modes(x32.astype(np.float64), L, A, ETA, k, w, F, S)
    U, E = gpu_apply(ctx, F, S, 2)
    assert rel(U, Ug) < 1e-3 and rel(E, Eg) < 1e-3
    Us, Es = mob.wave_apply_modes(x32.astype(np.float64), L, A, ETA, k, w, np.zeros_like(F), S)
    E2 = torch.empty(N, 5, device='cuda')
    ctx.pse_mobility_apply(None, dev(S), None, E2, 2)         # S -> E: planes 3-7 both ways
    assert rel(E2.cpu().numpy(), Es) < 1e-3
    Uf, Ef = mob.wave_apply_modes(x32.astype(np.float64), L, A, ETA, k, w, F, np.zeros_like(S))
    U2 = torch.empty(N, 3, device='cuda')
    ctx.pse_mobility_apply(dev(F), None, U2, None, 2)         # F -> U: planes 0-2
    assert rel(U2.cpu().numpy(), Uf) < 1e-3
    ctx.pse_mobility_apply(dev(F), None, None, E2, 2)         # F -> E: planes 0-2 in, 3-7 out
    assert rel(E2.cpu().numpy(), Ef) < 1e-3


def test_large_support_uses_global_interpolation_path():
    """P = 14 exceeds the shared-memory staging budget of the tiled interpolation: fallback kernel, same result."""
    x, L = synth.rsa(200, 0.10, seed=31)
    x32 = x.astype(np.float32)
    xi, grid, tol = 0.6, 36, 1e-3
    rcut = np.sqrt(-np.log(tol)) / xi + 1.0
    F, S = synth.gaussian_inputs(200, 5)
    outs = []
    for P in (8, 14):
        ctx = make_ctx(200, L, xi, grid, P, rcut, tol)
        ctx.pse_neighbors(dev(pos4(x32)))
        outs.append(np.hstack(gpu_apply(ctx, F, S, 2)))
    k = brn.grid_modes(grid, L)
    k2 = np.einsum('ki,ki->k', k, k)
    w = fn.hasimoto_H(np.sqrt(k2), xi) / (ETA * L**3 * k2)
    Ug, Eg = mob.wave_apply_modes(x32.astype(np.float64), L, A, ETA, k, w, F, S)
    assert rel(outs[0], np.hstack([Ug, Eg])) < 1e-3
    assert rel(outs[1], np.hstack([Ug, Eg])) < 2e-5      # P = 14: quadrature error ~1e-9, what is left is fp32


def test_config2_constrained_step_pieces_at_full_size():
    """BASELINE.json configs[1] (N=4096, phi=0.20, tol=1e-4): Brownian slip, hard-sphere forces and the GMRES
    stresslet solve at full size; the oracle checks, on sampled rows, that the solution really satisfies
    Eq. (78): E-rows of M [F;S] + E^B = 0 and U = U^B + U-rows of M [F;S]."""
    import paper_1709_06946_b200 as pse
    N, phi, tol, xi, dt = 4096, 0.20, 1e-4, 0.5, 1e-3
    x, L = synth.rsa(N, phi, seed=2)
    x32 = (x * 0.995).astype(np.float32)          # slight compression: a few overlapping pairs, so F^P != 0
    L = L * 0.995
    st, grid, P, rcut = pse.pse_suggest_params(N, L, A, tol, xi)
    assert st == 0
    ctx = make_ctx(N, L, xi, grid, P, rcut, tol)
    ctx.pse_neighbors(dev(pos4(x32)))
    w1, w2 = synth.brownian_noise(N, grid, 2)
    UB, EB = torch.empty(N, 3, device='cuda'), torch.empty(N, 5, device='cuda')
    li = ctx.pse_brownian(dt, dev(w1.reshape(N, 8)), dev(w2), UB, EB)
    F = torch.empty(N, 3, device='cuda')
    ctx.pse_hard_sphere_forces(dt, F)
    U, S = torch.empty(N, 3, device='cuda'), torch.empty(N, 5, device='cuda')
    gi = ctx.pse_constrained_solve(F, UB, EB, U, S)
    assert 3 <= li <= 30 and 3 <= gi <= 20        # the paper reports 8-10 constraint iterations at 1e-3
    Fh, Sh, UBh, EBh, Uh = (t.cpu().numpy().astype(np.float64) for t in (F, S, UB, EB, U))
    assert np.abs(Fh).max() > 0
    rows = np.sort(np.random.default_rng(4).choice(N, 12, replace=False))
    Uo, Eo = mob.mobility_apply(x32.astype(np.float64), L, A, ETA, xi, Fh, Sh, rows=rows, eps=1e-8)
    # constraint residual relative to the driving term, and the velocity relation
    assert np.linalg.norm(Eo + EBh[rows]) / np.linalg.norm(EBh[rows]) < 3 * bar(tol)     # GMRES tol + product tol
    assert rel(Uh[rows] - UBh[rows], Uo) < 3 * bar(tol)


def test_fractal_aggregates_neighbors_and_product():
    """BASELINE.json configs[4] stand-in at reduced N: clustered particles (very uneven cell and tile occupancy)."""
    import paper_1709_06946_b200 as pse
    N, tol, xi = 2048, 1e-3, 0.4
    x, L = synth.fractal_aggregates(N, 0.05, seed=3)
    x32 = x.astype(np.float32)
    st, grid, P, rcut = pse.pse_suggest_params(N, L, A, tol, xi)
    assert st == 0
    ctx = make_ctx(N, L, xi, grid, P, rcut, tol)
    ctx.pse_neighbors(dev(pos4(x32)))
    got, want = nbr_sets_from_gpu(ctx), nbo.neighbor_sets(x32, L, rcut)
    for g, w in zip(got, want):
        assert np.array_equal(g, w)
    counts = np.array([len(w) for w in want])
    uniform = 0.05 * rcut**3                       # phi r_cut^3 neighbours for a homogeneous suspension
    assert counts.mean() > 1.15 * uniform          # aggregates: more neighbours than a uniform suspension at the same phi
    F, S = synth.gaussian_inputs(N, 9)
    U, E = gpu_apply(ctx, F, S, 3)
    rows = np.sort(np.random.default_rng(9).choice(N, 24, replace=False))
    Uo, Eo = mob.mobility_apply(x32.astype(np.float64), L, A, ETA, xi, F, S, rows=rows, eps=1e-7)
    assert rel(U[rows], Uo) < bar(tol) and rel(E[rows], Eo) < bar(tol)


def test_config3_full_size_properties_and_sampled_rows():
    """bench.py's workload (N=65536, phi=0.30, tol=1e-3) in its launch configuration.  The O(N^2) oracle cannot
    finish here, so: (i) the real-space product is checked exactly on sampled rows; (ii) the full product must not
    depend on the splitting parameter (xi = 0.5, 0.575 = bench.py's value, the largest that keeps the 100^3 grid, and 0.6:
    different r_cut, grid, tables) and must be symmetric."""
    import paper_1709_06946_b200 as pse
    N, phi, tol = 65536, 0.30, 1e-3
    x, L = synth.rsa(N, phi, seed=100)
    x32 = x.astype(np.float32)
    F, S = synth.gaussian_inputs(N, 1)
    F2, S2 = synth.gaussian_inputs(N, 2)
    res = {}
    for xi in (0.5, 0.575, 0.6):
        st, grid, P, rcut = pse.pse_suggest_params(N, L, A, tol, xi)
        assert st == 0 and (xi != 0.575 or grid == 100)
        ctx = make_ctx(N, L, xi, grid, P, rcut, tol)
        ctx.pse_neighbors(dev(pos4(x32)))
        res[xi] = dict(full=np.hstack(gpu_apply(ctx, F, S, 3)), real=np.hstack(gpu_apply(ctx, F, S, 1)), rcut=rcut,
                       full2=np.hstack(gpu_apply(ctx, F2, S2, 3)))
        ctx.close()
    assert rel(res[0.5]['full'], res[0.6]['full']) < bar(tol)
    assert rel(res[0.575]['full'], res[0.5]['full']) < bar(tol)
    assert rel(res[0.575]['full'], res[0.6]['full']) < bar(tol)
    v1, v2 = np.hstack([F, S]).astype(np.float64), np.hstack([F2, S2]).astype(np.float64)
    d12, d21 = float((v1 * res[0.5]['full2']).sum()), float((v2 * res[0.5]['full']).sum())
    assert abs(d12 - d21) < bar(tol) * np.sqrt(float((v1 * res[0.5]['full']).sum()) * float((v2 * res[0.5]['full2']).sum()))
    assert float((v1 * res[0.5]['full']).sum()) > 0
    rows = np.sort(np.random.default_rng(5).choice(N, 8, replace=False))
    Ur, Er = mob.real_apply(x32.astype(np.float64), L, A, ETA, 0.5, F, S, rows=rows, rcut=res[0.5]['rcut'])
    assert rel(res[0.5]['real'][rows], np.hstack([Ur, Er])) < 2e-5


@pytest.mark.parametrize('N,sep', [(1, None), (2, 1.6), (2, 2.5), (3, 9.0)])
def test_degenerate_sizes_against_oracle(N, sep):
    """One particle (only self terms and its own periodic images: the Hasimoto lattice), an overlapping pair (r < 2a,
    the regularised branch of the real-space functions), a separated pair, and three particles none of
    which has a neighbour inside r_cut (empty lists): product and Brownian sample against the oracle."""
    import paper_1709_06946_b200 as pse
    L, xi, tol, grid, P = 16.0, 0.6, 1e-3, 36, 8
    _, _, _, rcut = pse.pse_suggest_params(max(N, 2), L, A, tol, xi)
    rng = np.random.default_rng(N)
    x = np.zeros((N, 3))
    x[0] = rng.uniform(0, L, 3)
    for i in range(1, N):
        d = rng.standard_normal(3)
        x[i] = x[i - 1] + sep * d / np.linalg.norm(d)
    x32 = x.astype(np.float32)
    xd = x32.astype(np.float64)
    ctx = make_ctx(N, L, xi, grid, P, rcut, tol)
    ctx.pse_neighbors(dev(pos4(x32)))
    sets = nbr_sets_from_gpu(ctx)
    ref = nbo.neighbor_sets(x32, L, rcut)
    assert all(np.array_equal(a, b) for a, b in zip(sets, ref))
    if N == 3:
        assert all(len(s) == 0 for s in sets)
    F, S = synth.gaussian_inputs(N, 7)
    U, E = gpu_apply(ctx, F, S, 3)
    Uo, Eo = mob.mobility_apply(xd, L, A, ETA, xi, F, S, eps=1e-12)
    assert rel(np.hstack([U, E]), np.hstack([Uo, Eo])) < bar(tol)
    w1, w2 = synth.brownian_noise(N, grid, 9)
    UB, EB = torch.empty(N, 3, device='cuda'), torch.empty(N, 5, device='cuda')
    ctx.pse_brownian(1e-3, dev(w1.reshape(N, 8)), dev(w2), UB, EB)
    torch.cuda.synchronize()
    Ub, Eb = brn.brownian(xd, L, A, ETA, KT, xi, 1e-3, grid, w1, w2, eps=1e-12)
    assert rel(np.hstack([UB.cpu().numpy(), EB.cpu().numpy()]), np.hstack([Ub, Eb])) < bar(tol)
    ctx.close()


def test_calls_before_neighbors_fail_with_not_ready():
    import paper_1709_06946_b200 as pse
    N, L, xi, tol = 8, 16.0, 0.6, 1e-3
    _, _, _, rcut = pse.pse_suggest_params(N, L, A, tol, xi)
    ctx = make_ctx(N, L, xi, 32, 8, rcut, tol)
    F, S = synth.gaussian_inputs(N, 0)
    U, E = torch.empty(N, 3, device='cuda'), torch.empty(N, 5, device='cuda')
    with pytest.raises(pse.PSEError) as ei:
        ctx.pse_mobility_apply(dev(F), dev(S), U, E, 3)
    assert 'ENOTREADY' in str(ei.value) or ei.value.status == 5
    ctx.close()


def test_host_buffer_entry_points_match_device_ones():
    """pse_step_host / pse_mobility_apply_host (the end-to-end calls bench.py times: host buffers, copies inside the
    call, wave noise uploaded on a second stream) against pse_step / pse_mobility_apply on the same inputs, two
    consecutive steps so that the staging buffers are reused while the previous step may still be reading them."""
    import paper_1709_06946_b200 as pse
    N, tol, xi, dt = 2000, 1e-3, 0.5, 1e-3
    x, L = synth.rsa(N, 0.20, seed=31)
    x32 = x.astype(np.float32)
    st, grid, P, rcut = pse.pse_suggest_params(N, L, A, tol, xi)
    assert st == 0
    noises = [synth.brownian_noise(N, grid, 40 + i) for i in range(2)]
    ctx_d, ctx_h = make_ctx(N, L, xi, grid, P, rcut, tol), make_ctx(N, L, xi, grid, P, rcut, tol)
    pos_d = dev(pos4(x32))
    pos_h = torch.from_numpy(pos4(x32)).pin_memory()
    for w1, w2 in noises:
        ctx_d.pse_step(pos_d, dt, dev(w1.reshape(N, 8)), dev(w2))
        ctx_h.pse_step_host(pos_h, dt, torch.from_numpy(np.ascontiguousarray(w1.reshape(N, 8), dtype=np.float32)).pin_memory(),
                            torch.from_numpy(np.ascontiguousarray(w2, dtype=np.float32)).pin_memory())
    torch.cuda.synchronize()
    assert np.array_equal(pos_d.cpu().numpy(), pos_h.numpy())
    F, S = synth.gaussian_inputs(N, 3)
    ctx_d.pse_neighbors(pos_d)
    Ud, Ed = gpu_apply(ctx_d, F, S, 3)
    Uh, Eh = torch.empty(N, 3).pin_memory(), torch.empty(N, 5).pin_memory()
    ctx_h.pse_mobility_apply_host(pos_h, torch.from_numpy(F.astype(np.float32)).pin_memory(), torch.from_numpy(S.astype(np.float32)).pin_memory(), Uh, Eh)
    assert np.array_equal(Ud, Uh.numpy()) and np.array_equal(Ed, Eh.numpy())
    ctx_d.close(); ctx_h.close()


def test_bitwise_reproducible_across_contexts_and_repeats():
    """Stand-in for a race detector (compute-sanitizer is closed on this GPU pool): every kernel on the path has a fixed summation
    order (gather-form spread, ballot-ordered lists, 8-lane shuffle reductions), so two fresh contexts and repeated calls must
    agree BITWISE on the neighbour lists as sets, every masked product, the Brownian sample and three consecutive steps (checked
    path, then the fixed-count path replayed as CUDA graphs).  A shared-memory race or an atomics-ordered sum would break this."""
    import paper_1709_06946_b200 as pse
    N, tol, xi, dt = 20000, 1e-3, 0.55, 1e-4
    x, L = synth.rsa(N, 0.30, seed=61)
    x32 = x.astype(np.float32)
    st, grid, P, rcut = pse.pse_suggest_params(N, L, A, tol, xi)
    assert st == 0
    F, S = synth.gaussian_inputs(N, 6)
    w1, w2 = synth.brownian_noise(N, grid, 6)
    outs = []
    for rep in range(2):
        ctx = make_ctx(N, L, xi, grid, P, rcut, tol)
        pos = dev(pos4(x32))
        ctx.pse_neighbors(pos)
        o = {'sets': [s.tobytes() for s in nbr_sets_from_gpu(ctx)[:200]]}
        for name, (f, s_, u, e) in {'all': (1, 1, 1, 1), 'se': (0, 1, 0, 1), 'fe': (1, 0, 0, 1), 'fsu': (1, 1, 1, 0)}.items():
            U, E = torch.empty(N, 3, device='cuda'), torch.empty(N, 5, device='cuda')
            for _ in range(2):                      # repeated call on the same context
                ctx.pse_mobility_apply(dev(F) if f else None, dev(S) if s_ else None, U if u else None, E if e else None, 3)
                key = name + str(_)
                o[key] = (U.cpu().numpy().tobytes() if u else b'') + (E.cpu().numpy().tobytes() if e else b'')
            assert o[name + '0'] == o[name + '1']
        UB, EB = torch.empty(N, 3, device='cuda'), torch.empty(N, 5, device='cuda')
        ctx.pse_brownian(dt, dev(w1.reshape(N, 8)), dev(w2), UB, EB)
        o['brownian'] = UB.cpu().numpy().tobytes() + EB.cpu().numpy().tobytes()
        its = []
        for k in range(3):
            its.append(ctx.pse_step(pos, dt, dev(w1.reshape(N, 8)), dev(w2)))
        o['steps'] = pos.cpu().numpy().tobytes()
        o['its'] = its
        outs.append(o)
        ctx.close()
    for key in outs[0]:
        assert outs[0][key] == outs[1][key], key
