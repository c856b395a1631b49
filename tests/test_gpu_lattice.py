"""GPU parity on deformed lattices: pse_set_lattice + the existing calls against
oracle/lattice.py (direct Ewald sums with lattice vectors L A and k = (2 pi/L) A^-T n).  Bars as on the cube: neighbour sets bit-exact,
products and samples within max(2 tol, 1e-5) relative L2."""
import numpy as np
import pytest

import synth
from oracle import lattice as lat
from oracle import mobility as mob

pytestmark = pytest.mark.gpu
torch = pytest.importorskip('torch')

A, ETA, KT = 1.0, 1.0 / (6.0 * np.pi), 1.0
SHEAR, EXT = (1.0, 0.5, 1.0), (1.25, 0.0, 0.8)


def rel(a, b):
    return float(np.linalg.norm(np.asarray(a, float) - np.asarray(b, float)) / np.linalg.norm(np.asarray(b, float)))


def bar(tol):
    return max(2 * tol, 1e-5)


def dev(x):
    return torch.as_tensor(np.ascontiguousarray(x), dtype=torch.float32).cuda().contiguous()


def pos4(x):
    p = np.zeros((x.shape[0], 4), np.float32)
    p[:, :3] = x
    return p


def matrix(l3):
    return np.array([[l3[0], l3[1], 0.0], [0.0, l3[2], 0.0], [0.0, 0.0, 1.0]])


def deformed_suspension(N, phi, l3, seed, images=True):
    """A seeded hard-sphere suspension of the cube carried along by the deformation (x = A s: what Lees-Edwards / Kraynik-Reinelt
    boxes hold after straining), then every particle moved to a random periodic image (lattice vectors = columns of L A)."""
    s, L = synth.rsa(N, phi, seed=seed)
    Am = matrix(l3)
    x = s @ Am.T
    if images:
        n = np.random.default_rng(seed).integers(-1, 2, size=(N, 3))
        x = x + L * (n @ Am.T)
    return x.astype(np.float32), L


def make(N, L, xi, tol, l3, x32):
    import paper_1709_06946_b200 as pse
    st, g, p, rcut = pse.pse_suggest_params(N, L, A, tol, xi, lattice=l3)
    assert st == 0, 'rcut does not fit the deformed cell'
    ctx = pse.pse_create(N, L, A, ETA, KT, xi, g, p, rcut, tol)
    ctx.pse_set_lattice(*l3)
    ctx.pse_neighbors(dev(pos4(x32)))
    return ctx, rcut


def gpu_apply(ctx, F, S, which=3):
    N = ctx.N
    U, E = torch.empty(N, 3, device='cuda'), torch.empty(N, 5, device='cuda')
    ctx.pse_mobility_apply(dev(F), dev(S), U, E, which)
    torch.cuda.synchronize()
    return U.cpu().numpy(), E.cpu().numpy()


def nbr_sets(ctx):
    count, index = ctx.pse_get_neighbors()
    count, index = count.cpu().numpy(), index.cpu().numpy()
    off = np.concatenate([[0], np.cumsum(count)])
    return [np.sort(index[off[i]:off[i + 1]]) for i in range(len(count))]


@pytest.mark.parametrize('l3', [SHEAR, EXT, (1.0, -0.3, 1.0)])
def test_neighbour_sets_bit_exact_on_deformed_lattices(l3):
    N = 3000
    x32, L = deformed_suspension(N, 0.25, l3, seed=3)
    ctx, rcut = make(N, L, 0.6, 1e-3, l3, x32)
    got = nbr_sets(ctx)
    want = lat.neighbor_sets(x32, L, *l3, rcut)
    assert sum(len(w) for w in want) > 20 * N
    assert all(np.array_equal(g, w) for g, w in zip(got, want))


def test_identity_lattice_is_the_cube_bit_for_bit():
    import paper_1709_06946_b200 as pse
    N, xi, tol = 2000, 0.6, 1e-3
    x, L = synth.rsa(N, 0.2, seed=2)
    x32 = x.astype(np.float32)
    F, S = synth.gaussian_inputs(N, 1)
    st, g, p, rcut = pse.pse_suggest_params(N, L, A, tol, xi)
    assert pse.pse_suggest_params(N, L, A, tol, xi, lattice=(1.0, 0.0, 1.0)) == (st, g, p, rcut)
    outs = []
    for set_it in (False, True):
        ctx = pse.pse_create(N, L, A, ETA, KT, xi, g, p, rcut, tol)
        if set_it:
            ctx.pse_set_lattice(1.0, 0.7, 1.0)
            ctx.pse_set_lattice(1.0, 0.0, 1.0)
        ctx.pse_neighbors(dev(pos4(x32)))
        outs.append(gpu_apply(ctx, F, S))
    assert np.array_equal(outs[0][0], outs[1][0]) and np.array_equal(outs[0][1], outs[1][1])


@pytest.mark.parametrize('l3,tol', [(SHEAR, 1e-3), (SHEAR, 1e-4), (EXT, 1e-3)])
def test_product_on_deformed_lattice_against_direct_sums(l3, tol):
    """N = 300 all rows: total, and the real and wave halves separately (relative to the total)."""
    N, xi = 300, 0.55
    x32, L = deformed_suspension(N, 0.20, l3, seed=7)
    ctx, _ = make(N, L, xi, tol, l3, x32)
    F, S = synth.gaussian_inputs(N, 3)
    x = x32.astype(np.float64)
    halves = {part: lat.mobility_apply(x, L, matrix(l3), A, ETA, xi, F, S, eps=1e-10, part=part) for part in ('real', 'wave')}
    Uo, Eo = halves['real'][0] + halves['wave'][0], halves['real'][1] + halves['wave'][1]      # M = M_r + M_w (part='both' is this sum)
    U, E = gpu_apply(ctx, F, S)
    assert rel(U, Uo) < bar(tol) and rel(E, Eo) < bar(tol), (rel(U, Uo), rel(E, Eo))
    for which, part in ((1, 'real'), (2, 'wave')):
        Up, Ep = halves[part]
        Ug, Eg = gpu_apply(ctx, F, S, which)
        assert np.linalg.norm(Ug - Up) < bar(tol) * np.linalg.norm(Uo) and np.linalg.norm(Eg - Ep) < bar(tol) * np.linalg.norm(Eo), part
    # the cube's operator is a different one: the deformation is really in the numbers
    Uc, Ec = mob.mobility_apply(x, L, A, ETA, xi, F, S, eps=1e-8)
    assert rel(U, Uc) > 50 * bar(tol)


def test_product_sampled_rows_mid_size_sheared():
    N, xi, tol, l3 = 2000, 0.5, 1e-3, (1.0, 0.4, 1.0)
    x32, L = deformed_suspension(N, 0.25, l3, seed=11)
    ctx, _ = make(N, L, xi, tol, l3, x32)
    F, S = synth.gaussian_inputs(N, 4)
    rows = np.sort(np.random.default_rng(3).choice(N, 12, replace=False))
    Uo, Eo = lat.mobility_apply(x32.astype(np.float64), L, matrix(l3), A, ETA, xi, F, S, rows=rows, eps=1e-9)
    U, E = gpu_apply(ctx, F, S)
    assert rel(U[rows], Uo) < bar(tol) and rel(E[rows], Eo) < bar(tol), (rel(U[rows], Uo), rel(E[rows], Eo))


def test_a_shear_by_a_whole_lattice_vector_is_the_same_lattice_on_the_gpu():
    """gamma and gamma - 1 describe the same lattice: the same physical positions give the same product."""
    N, xi, tol = 800, 0.6, 1e-3
    x32, L = deformed_suspension(N, 0.2, (1.0, 0.3, 1.0), seed=5)
    F, S = synth.gaussian_inputs(N, 5)
    ctx_a, _ = make(N, L, xi, tol, (1.0, 0.3, 1.0), x32)
    ctx_b, _ = make(N, L, xi, tol, (1.0, -0.7, 1.0), x32)
    Ua, Ea = gpu_apply(ctx_a, F, S)
    Ub, Eb = gpu_apply(ctx_b, F, S)
    assert rel(Ub, Ua) < bar(tol) and rel(Eb, Ea) < bar(tol)


def test_brownian_sample_constrained_solve_and_overlap_forces_on_a_sheared_lattice():
    N, xi, tol, l3, dt = 150, 0.7, 1e-3, (1.0, 0.4, 1.0), 1e-3
    x32, L = deformed_suspension(N, 0.25, l3, seed=9)
    ctx, rcut = make(N, L, xi, tol, l3, x32)
    x, Am = x32.astype(np.float64), matrix(l3)
    w1, w2 = synth.brownian_noise(N, ctx.grid, 4)
    UB, EB = torch.empty(N, 3, device='cuda'), torch.empty(N, 5, device='cuda')
    ctx.pse_brownian(dt, dev(w1.reshape(N, 8)), dev(w2), UB, EB)
    Uo, Eo = lat.brownian(x, L, Am, A, ETA, KT, xi, dt, ctx.grid, w1, w2, eps=1e-10)
    assert rel(UB.cpu().numpy(), Uo) < bar(tol) and rel(EB.cpu().numpy(), Eo) < bar(tol), (rel(UB.cpu().numpy(), Uo), rel(EB.cpu().numpy(), Eo))
    # overlap forces: pairs closer than 2a from the oracle's image search
    ia, ib, rv = lat.real_pairs(x, L, Am, 2.0 * A)
    keep = ia != ib
    ia, rv = ia[keep], rv[keep]
    r = np.linalg.norm(rv, axis=1)
    Fo = np.zeros((N, 3))
    np.add.at(Fo, ia, (3 * np.pi * ETA * A * (2 * A - r) / dt / r)[:, None] * rv)
    assert np.abs(Fo).max() > 0
    Fp = torch.empty(N, 3, device='cuda')
    ctx.pse_hard_sphere_forces(dt, Fp)
    assert rel(Fp.cpu().numpy(), Fo) < 1e-4
    # constrained solve against the dense matrix of the deformed lattice
    from oracle import brownian as brn
    M = lat.dense(x, L, Am, A, ETA, xi, eps=1e-10)
    rng = np.random.default_rng(2)
    F, UBh, EBh = rng.standard_normal((N, 3)), rng.standard_normal((N, 3)), rng.standard_normal((N, 5))
    Us, Ss = brn.constrained_solve(M, N, UBh, EBh, F)
    U, S = torch.empty(N, 3, device='cuda'), torch.empty(N, 5, device='cuda')
    ctx.pse_constrained_solve(dev(F), dev(UBh), dev(EBh), U, S)
    assert rel(U.cpu().numpy(), Us) < 3 * bar(tol) and rel(S.cpu().numpy(), Ss) < 5 * bar(tol)
    # a step runs on the deformed lattice (positions stay unwrapped) and repeats bit for bit
    pos = dev(pos4(x32))
    p1, p2 = pos.clone(), pos.clone()
    ctx.pse_step(p1, dt, dev(w1.reshape(N, 8)), dev(w2))
    ctx.pse_step(p2, dt, dev(w1.reshape(N, 8)), dev(w2))
    assert torch.isfinite(p1).all() and torch.equal(p1, p2) and float((p1 - pos).abs().max()) > 0


def test_set_lattice_rejects_what_it_cannot_do():
    import paper_1709_06946_b200 as pse
    N = 64
    x, L = synth.rsa(N, 0.10, seed=1)
    st, g, p, rcut = pse.pse_suggest_params(N, L, A, 1e-3, 0.6)
    ctx = pse.pse_create(N, L, A, ETA, KT, 0.6, g, p, rcut, 1e-3)
    for bad in ((1.0, 0.0, 1.1), (-1.0, 0.0, -1.0), (2.0, 0.0, 0.5)):       # not volume preserving; negative; rcut no longer fits
        with pytest.raises(pse.PSEError) as e:
            ctx.pse_set_lattice(*bad)
        assert e.value.status == pse.PSE_EINVAL
    assert pse.pse_suggest_params(N, L, A, 1e-3, 0.6, lattice=(2.0, 0.0, 0.5))[0] == pse.PSE_EINVAL


def test_full_couplet_and_paper_window_on_a_sheared_lattice():
    """The torque / angular-velocity rows (pse_mobility_apply_full) and the paper's Gaussian window, both on a sheared cell."""
    import paper_1709_06946_b200 as pse
    from oracle import couplet as cpl
    N, xi, tol, l3 = 400, 0.55, 1e-3, (1.0, 0.4, 1.0)
    x32, L = deformed_suspension(N, 0.20, l3, seed=13)
    x, Am = x32.astype(np.float64), matrix(l3)
    F, S = synth.gaussian_inputs(N, 6)
    Lq = np.random.default_rng(6).standard_normal((N, 3))
    want = cpl.mobility_apply_full(x, L, A, ETA, xi, F, Lq, S, eps=1e-10, A=Am)
    for window in (pse.PSE_WINDOW_ES, pse.PSE_WINDOW_GAUSS):
        st, g, p, rcut = pse.pse_suggest_params(N, L, A, tol, xi, window, lattice=l3)
        assert st == 0
        ctx = pse.pse_create(N, L, A, ETA, KT, xi, g, p, rcut, tol, window=window)
        ctx.pse_set_lattice(*l3)
        ctx.pse_neighbors(dev(pos4(x32)))
        U, W, E = torch.empty(N, 3, device='cuda'), torch.empty(N, 3, device='cuda'), torch.empty(N, 5, device='cuda')
        ctx.pse_mobility_apply_full(dev(F), dev(Lq), dev(S), U, W, E)
        for got, w, name in zip((U, W, E), want, 'UWE'):
            assert rel(got.cpu().numpy(), w) < bar(tol), (window, name, rel(got.cpu().numpy(), w))


def test_config3_in_a_sheared_cell_against_the_lattice_reference():
    """`bench.py --shear 0.5`'s workload (N = 65 536, phi = 0.30, tol = 1e-3, xi = 0.575 -> grid 112, P = 4): U and E of the full
    product on 128 sampled particles against the fp64 lattice reference tier at its own xi = 0.45, tol 1e-7."""
    N, xi, tol, l3 = 65536, 0.575, 1e-3, SHEAR
    x32, L = deformed_suspension(N, 0.30, l3, seed=100, images=False)
    ctx, _ = make(N, L, xi, tol, l3, x32)
    assert (ctx.grid, ctx.P) == (112, 4)
    F, S = synth.gaussian_inputs(N, 1)
    rows = np.sort(np.random.default_rng(5).choice(N, 128, replace=False))
    Uo, Eo = lat.LatticeReference(L, matrix(l3), A, ETA, 0.45, tol=1e-7).apply(x32.astype(np.float64), F, S, rows)
    U, E = gpu_apply(ctx, F, S)
    for g, w, name in ((U[rows], Uo, 'U'), (E[rows], Eo, 'E')):
        worst = float(np.linalg.norm(g - w, axis=1).max() / np.sqrt((w * w).sum(axis=1).mean()))
        assert rel(g, w) < bar(tol) and worst < 10 * bar(tol), (name, rel(g, w), worst)


def test_sedimentation_velocity_error_on_a_sheared_grid_tracks_the_tolerance():
    """The experiment of the paper's Fig. 2: relative error of the sedimentation velocity of a random suspension in a
    cell sheared to gamma = 0.5, as a function of the requested tolerance, at several splitting parameters.  There, supports chosen
    with the orthorhombic bound miss the tolerance by an order of magnitude; here the window acts on lattice coordinates (reading
    R22), so the cube's P = 3, 4, 5 must meet the bar on the sheared grid as well.  Reference: direct sums of oracle.lattice."""
    N, l3 = 500, SHEAR
    F = np.tile(np.array([0.0, 0.0, -1.0]), (N, 1))
    S = np.zeros((N, 5))
    rows = []
    for cell in ((1.0, 0.0, 1.0), l3):                        # the same suspension in the cube and carried along by the shear
        x32, L = deformed_suspension(N, 0.15, cell, seed=21)
        Uo, _ = lat.mobility_apply(x32.astype(np.float64), L, matrix(cell), A, ETA, 0.6, F, S, eps=1e-10)
        for xi in (0.5, 0.65):
            for tol in (1e-2, 1e-3, 1e-4):
                ctx, _ = make(N, L, xi, tol, cell, x32)
                U, _ = gpu_apply(ctx, F, S)
                rows.append((cell[1], xi, tol, ctx.P, ctx.grid, rel(U, Uo)))
                ctx.close()
    print('\n'.join(f'gamma={r[0]} xi={r[1]} tol={r[2]:g} P={r[3]} grid={r[4]} err={r[5]:.2e}' for r in rows))
    cube, sheared = rows[:6], rows[6:]
    for (_, xi, tol, P, grid, err), (_, _, _, Pc, gridc, errc) in zip(sheared, cube):
        assert P == Pc == {1e-2: 3, 1e-3: 4, 1e-4: 5}[tol] and grid >= gridc and err < bar(tol), (xi, tol, err)
        assert err < 1.3 * errc + 0.2 * tol, (xi, tol, err, errc)          # the sheared grid is as accurate as the cube's
    assert all(sheared[i + 1][5] < sheared[i][5] for i in (0, 1, 3, 4))    # and the error falls with the tolerance at fixed xi


def test_lattice_edge_cases_pair_across_the_sheared_boundary_compression_and_repeats():
    """(1) Two spheres that are neighbours only through the sheared image (x1 = x0 + d + the lattice vector (gamma L, L, 0)): each is in
    the other's list and the product matches the direct sums; (2) a cell compressed along x (epsilon < 1); (3) bit-identical repeats."""
    import paper_1709_06946_b200 as pse
    L, xi, tol, g = 14.0, 0.7, 1e-3, 0.5
    x = np.array([[1.0, 0.3, 4.0], [1.0 + 1.5 + g * L, 0.3 + 1.2 + L, 4.5], [7.0, 7.0, 7.0]])
    x32 = x.astype(np.float32)
    ctx, rcut = make(3, L, xi, tol, (1.0, g, 1.0), x32)
    sets = nbr_sets(ctx)
    assert 1 in sets[0] and 0 in sets[1]
    F, S = synth.gaussian_inputs(3, 2)
    Uo, Eo = lat.mobility_apply(x32.astype(np.float64), L, lat.shear(g), A, ETA, xi, F, S, eps=1e-10)
    U, E = gpu_apply(ctx, F, S)
    assert rel(U, Uo) < bar(tol) and rel(E, Eo) < bar(tol)
    # the same pair in the cube would not interact through that image
    cube = lat.neighbor_sets(x32, L, 1.0, 0.0, 1.0, rcut)
    assert 1 not in cube[0]
    # (2), (3)
    l3 = (0.8, 0.0, 1.25)
    N = 300
    xs, Ls = deformed_suspension(N, 0.2, l3, seed=31)
    F, S = synth.gaussian_inputs(N, 3)
    outs = []
    for rep in range(2):
        ctx, _ = make(N, Ls, 0.6, 1e-3, l3, xs)
        outs.append(gpu_apply(ctx, F, S) + gpu_apply(ctx, F, S))
    assert all(np.array_equal(outs[0][0], o) for o in (outs[0][2], outs[1][0], outs[1][2]))
    Uo, Eo = lat.mobility_apply(xs.astype(np.float64), Ls, matrix(l3), A, ETA, 0.6, F, S, eps=1e-9)
    assert rel(outs[0][0], Uo) < bar(1e-3) and rel(outs[0][1], Eo) < bar(1e-3)


def test_strain_advanced_every_step_on_one_context_matches_fresh_contexts():
    """A flowing suspension ("the periodic lattice must deform"): pse_set_lattice before every pse_step on ONE context, whose
    captured step graphs stay alive because the kernels read A from device memory.  Each step must agree with a fresh context that is
    given that step's lattice (checked path, nothing captured), within the solver tolerance; a context left on the PREVIOUS strain
    must not (the check that this test can see a stale lattice at all)."""
    import paper_1709_06946_b200 as pse
    N, phi, xi, tol, dt = 4000, 0.2, 0.6, 1e-3, 1e-4
    s, L = synth.rsa(N, phi, seed=77)
    st, grid, P, rcut = pse.pse_suggest_params(N, L, A, tol, xi, lattice=SHEAR)
    assert st == 0
    strains = [0.10, 0.20, 0.30, 0.35, 0.40, 0.45, 0.50, 0.10]            # jumps large enough that a stale lattice shows; back down at the end

    def fresh_step(x32, gamma, w1, w2):
        c = pse.pse_create(N, L, A, ETA, KT, xi, grid, P, rcut, tol)
        c.pse_set_lattice(1.0, gamma, 1.0)
        p = dev(pos4(x32))
        c.pse_step(p, dt, dev(w1.reshape(N, 8)), dev(w2))
        out = p.cpu().numpy()[:, :3].copy()
        c.close()
        return out

    ctx = pse.pse_create(N, L, A, ETA, KT, xi, grid, P, rcut, tol)
    x32 = (s @ matrix((1.0, strains[0], 1.0)).T).astype(np.float32)
    worst, stale_seen = 0.0, 0.0
    for k, gamma in enumerate(strains):
        if k:                                                              # carry the suspension along: same lattice coordinates, new A
            sl = x32.astype(np.float64) @ np.linalg.inv(matrix((1.0, strains[k - 1], 1.0))).T
            x32 = (sl @ matrix((1.0, gamma, 1.0)).T).astype(np.float32)
        w1, w2 = synth.brownian_noise(N, grid, 100 + k)
        ctx.pse_set_lattice(1.0, gamma, 1.0)
        p = dev(pos4(x32))
        ctx.pse_step(p, dt, dev(w1.reshape(N, 8)), dev(w2))
        got = p.cpu().numpy()[:, :3]
        want = fresh_step(x32, gamma, w1, w2)
        e = rel(got - x32, want - x32)
        worst = max(worst, e)
        assert e < 5 * tol, (k, gamma, e)
        if k in (3, 7):
            stale = fresh_step(x32, strains[k - 1], w1, w2)
            stale_seen = max(stale_seen, rel(stale - x32, want - x32))
        x32 = got.astype(np.float32).copy()
    ctx.close()
    print('worst displacement difference', worst, 'a stale lattice would give', stale_seen)
    assert stale_seen > 20 * tol


def test_kraynik_reinelt_lattice_in_the_lab_frame():
    """Planar extension with Kraynik-Reinelt boundary conditions: in the lab frame the cell is the cube turned by the
    magic angle about z and then stretched, B = diag(e^eps, e^-eps, 1) Rz(theta), which is not triangular.  B = Q R with R upper
    triangular, positive diagonal, det 1: R is what pse_set_lattice takes and the library works in the frame x' = Q^T x.  The oracle
    sums over the lab-frame lattice L B n directly; U = Q U', E = Q E' Q^T.  All three entries of A differ from the cube's here.
    Run twice: with the basis as the flow leaves it (lattice vectors of length 1.32 and 0.97) and with the Gauss-reduced basis of the
    SAME lattice (0.97 and 1.04), which needs a grid that is a quarter smaller per side and must give the same answer."""
    import paper_1709_06946_b200 as pse
    from oracle import functions as fn
    N, xi, tol, eps_h = 500, 0.6, 1e-3, 0.4
    theta = np.arctan(0.5 * (np.sqrt(5.0) - 1.0))
    Rz = np.array([[np.cos(theta), -np.sin(theta), 0.0], [np.sin(theta), np.cos(theta), 0.0], [0.0, 0.0, 1.0]])
    B = np.diag([np.exp(eps_h), np.exp(-eps_h), 1.0]) @ Rz
    b1, b2 = B[:2, 0].copy(), B[:2, 1].copy()                  # Gauss reduction of the planar basis
    for _ in range(20):
        if b2 @ b2 < b1 @ b1:
            b1, b2 = b2, b1
        mu = np.rint(b1 @ b2 / (b1 @ b1))
        if mu == 0:
            break
        b2 = b2 - mu * b1
    Bred = np.eye(3)
    Bred[:2, 0], Bred[:2, 1] = b1, b2
    if np.linalg.det(Bred) < 0:
        Bred[:2, 1] = -b2
    assert abs(np.linalg.det(Bred) - 1) < 1e-12 and max(np.linalg.norm(Bred[:, :2], axis=0)) < 1.06 < 1.3 < np.linalg.norm(B[:, 0])
    s, L = synth.rsa(N, 0.2, seed=41)
    x_lab = s @ B.T                                            # the suspension carried along by the flow
    F, S = synth.gaussian_inputs(N, 4)
    Uo, Eo = lat.mobility_apply(x_lab, L, B, A, ETA, xi, F, S, eps=1e-10)
    grids = []
    for basis in (B, Bred):
        Q, R = np.linalg.qr(basis)
        sg = np.diag(np.sign(np.diag(R)))
        Q, R = Q @ sg, sg @ R
        assert np.allclose(Q @ R, basis) and abs(np.linalg.det(Q) - 1) < 1e-12 and abs(R[0, 0] * R[1, 1] - 1) < 1e-12 and abs(R[2, 2] - 1) < 1e-12
        l3 = (float(R[0, 0]), float(R[0, 1]), float(R[1, 1]))
        assert abs(l3[0] - 1) > 0.02 and abs(l3[1]) > 0.05
        # into the frame of the triangular lattice, through the library, and back
        x32 = (x_lab @ Q).astype(np.float32)
        Ff = F @ Q
        Sf = fn.to_coords(np.einsum('ji,njk,kl->nil', Q, fn.to_tensor(S), Q))
        ctx, rcut = make(N, L, xi, tol, l3, x32)
        grids.append(ctx.grid)
        sets = nbr_sets(ctx)
        want = lat.neighbor_sets(x32, L, *l3, rcut)
        assert all(np.array_equal(a_, b_) for a_, b_ in zip(sets, want))
        Uf, Ef = gpu_apply(ctx, Ff, Sf)
        U = Uf.astype(np.float64) @ Q.T
        E = fn.to_coords(np.einsum('ij,njk,lk->nil', Q, fn.to_tensor(Ef), Q))
        print('Kraynik-Reinelt lattice', l3, 'grid', ctx.grid, 'U', rel(U, Uo), 'E', rel(E, Eo))
        assert rel(U, Uo) < bar(tol) and rel(E, Eo) < bar(tol)
    assert grids[1] < grids[0]
