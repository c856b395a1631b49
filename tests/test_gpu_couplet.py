"""GPU parity of the full couplet: pse_mobility_apply_full / pse_constrained_solve_full through the C ABI
against oracle/couplet.py (direct Ewald sums, fp64) on the same seeded inputs.  Bar: relative L2 error max(2 tol, 1e-5) per output
block (U, Omega, E), as for the force / stresslet product (BASELINE.json north_star)."""
import numpy as np
import pytest

import synth
from oracle import couplet as cpl

pytestmark = pytest.mark.gpu
torch = pytest.importorskip('torch')

A, ETA, KT = 1.0, 1.0 / (6.0 * np.pi), 1.0


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


def inputs(N, seed):
    rng = np.random.default_rng(seed)
    F, S = synth.gaussian_inputs(N, seed)
    return F.astype(np.float64), rng.standard_normal((N, 3)), S.astype(np.float64)


def gpu_full(ctx, F, Lq, S, which=3):
    N = ctx.N
    U, W, E = torch.empty(N, 3, device='cuda'), torch.empty(N, 3, device='cuda'), torch.empty(N, 5, device='cuda')
    ctx.pse_mobility_apply_full(None if F is None else dev(F), None if Lq is None else dev(Lq), None if S is None else dev(S), U, W, E, which)
    torch.cuda.synchronize()
    return U.cpu().numpy(), W.cpu().numpy(), E.cpu().numpy()


def make(N, phi, xi, tol, seed, grid=None, P=None, squeeze=1.0):
    import paper_1709_06946_b200 as pse
    x, L = synth.rsa(N, phi, seed=seed)
    x, L = x * squeeze, L * squeeze
    x32 = x.astype(np.float32)
    st, g, p, rcut = pse.pse_suggest_params(N, L, A, tol, xi)
    assert st == 0
    ctx = pse.pse_create(N, L, A, ETA, KT, xi, grid or g, P or p, rcut, tol)
    ctx.pse_neighbors(dev(pos4(x32)))
    return ctx, x32.astype(np.float64), L


def test_full_couplet_config1_every_block_and_both_halves():
    """BASELINE.json configs[0] (N = 64, grid 32, P = 8, tol 1e-3) with a torque on every particle: all inputs together, every input
    block alone (a wrong sign in one coupling cannot hide in the total), and the real and wave halves separately."""
    xi, tol = 0.6, 1e-3
    ctx, x, L = make(64, 0.10, xi, tol, seed=1, grid=32, P=8)
    F, Lq, S = inputs(64, 0)
    want = cpl.mobility_apply_full(x, L, A, ETA, xi, F, Lq, S, eps=1e-10)
    got = gpu_full(ctx, F, Lq, S)
    for g, w, name in zip(got, want, 'UWE'):
        assert rel(g, w) < bar(tol), (name, rel(g, w))
    z3, z5 = np.zeros((64, 3)), np.zeros((64, 5))
    for Fi, Li, Si, name in ((F, None, None, 'F'), (None, Lq, None, 'L'), (None, None, S, 'S')):
        want = cpl.mobility_apply_full(x, L, A, ETA, xi, z3 if Fi is None else Fi, z3 if Li is None else Li, z5 if Si is None else Si, eps=1e-10)
        got = gpu_full(ctx, Fi, Li, Si)
        scale = max(np.linalg.norm(w) for w in want)
        for g, w, out in zip(got, want, 'UWE'):
            assert np.linalg.norm(g - w) < bar(tol) * scale, (name, out, np.linalg.norm(g - w) / scale)
    for which, part in ((1, 'real'), (2, 'wave')):
        want = cpl.mobility_apply_full(x, L, A, ETA, xi, F, Lq, S, eps=1e-10, part=part)
        got = gpu_full(ctx, F, Lq, S, which)
        tot = cpl.mobility_apply_full(x, L, A, ETA, xi, F, Lq, S, eps=1e-10)
        for g, w, t, out in zip(got, want, tot, 'UWE'):
            assert np.linalg.norm(g - w) < bar(tol) * np.linalg.norm(t), (part, out)
    # without a torque, U and E are those of the 8-component product
    U8, E8 = torch.empty(64, 3, device='cuda'), torch.empty(64, 5, device='cuda')
    ctx.pse_mobility_apply(dev(F), dev(S), U8, E8)
    U, W, E = gpu_full(ctx, F, None, S)
    assert rel(U, U8.cpu().numpy()) < 2e-6 and rel(E, E8.cpu().numpy()) < 2e-6


@pytest.mark.parametrize('tol', [1e-3, 1e-4])
def test_full_couplet_sampled_rows_with_overlaps(tol):
    """N = 1 500 at phi = 0.25, compressed 6 % (overlapping pairs: the regularised branch of every function), parameters from
    pse_suggest_params, 12 sampled particles against the direct sums."""
    N, xi = 1500, 0.55
    ctx, x, L = make(N, 0.25, xi, tol, seed=4, squeeze=0.94)
    F, Lq, S = inputs(N, 5)
    rows = np.sort(np.random.default_rng(2).choice(N, 12, replace=False))
    want = cpl.mobility_apply_full(x, L, A, ETA, xi, F, Lq, S, rows=rows, eps=1e-9)
    got = gpu_full(ctx, F, Lq, S)
    for g, w, name in zip(got, want, 'UWE'):
        assert rel(g[rows], w) < bar(tol), (name, rel(g[rows], w))
    # torque only: the couplings that exist only in the new rows
    z3, z5 = np.zeros((N, 3)), np.zeros((N, 5))
    want = cpl.mobility_apply_full(x, L, A, ETA, xi, z3, Lq, z5, rows=rows, eps=1e-9)
    got = gpu_full(ctx, None, Lq, None)
    for g, w, name in zip(got, want, 'UWE'):
        assert rel(g[rows], w) < 2 * bar(tol), (name, rel(g[rows], w))


def test_full_couplet_is_symmetric_on_the_gpu():
    """v . M w = w . M v for random 11N vectors (Eq. 31's matrix is symmetric): a transposed coupling fails this."""
    N, xi, tol = 600, 0.6, 1e-3
    ctx, x, L = make(N, 0.15, xi, tol, seed=8)
    v, w = inputs(N, 1), inputs(N, 2)
    Mv, Mw = gpu_full(ctx, *v), gpu_full(ctx, *w)
    dot = lambda a, b: float(sum((p.astype(np.float64) * q).sum() for p, q in zip(a, b)))
    vMw, wMv = dot((v[0], v[1], v[2]), Mw), dot((w[0], w[1], w[2]), Mv)
    assert abs(vMw - wMv) < 2 * tol * max(abs(vMw), abs(wMv), 1.0), (vMw, wMv)
    assert dot((v[0], v[1], v[2]), Mv) > 0


def test_constrained_solve_with_torques_against_dense_oracle():
    N, xi, tol = 48, 0.85, 1e-4
    ctx, x, L = make(N, 0.20, xi, tol, seed=3)
    M = cpl.dense_full(x, L, A, ETA, xi, eps=1e-10)
    rng = np.random.default_rng(9)
    F, Lq = rng.standard_normal((N, 3)), rng.standard_normal((N, 3))
    UB, EB = rng.standard_normal((N, 3)), rng.standard_normal((N, 5))
    Uo, Wo, So = cpl.constrained_solve_full(M, N, UB, np.zeros((N, 3)), EB, F, Lq)
    U, W, S = torch.empty(N, 3, device='cuda'), torch.empty(N, 3, device='cuda'), torch.empty(N, 5, device='cuda')
    it = ctx.pse_constrained_solve_full(dev(F), dev(Lq), dev(UB), dev(EB), U, W, S)
    assert 2 <= it <= 30
    assert rel(S.cpu().numpy(), So) < 5 * bar(tol) and rel(U.cpu().numpy(), Uo) < 3 * bar(tol) and rel(W.cpu().numpy(), Wo) < 3 * bar(tol), \
        (rel(S.cpu().numpy(), So), rel(U.cpu().numpy(), Uo), rel(W.cpu().numpy(), Wo))
    # no torque, no Omega asked for: the 8-component solve
    U2, S2 = torch.empty(N, 3, device='cuda'), torch.empty(N, 5, device='cuda')
    ctx.pse_constrained_solve_full(dev(F), None, dev(UB), dev(EB), U2, None, S2)
    U3, S3 = torch.empty(N, 3, device='cuda'), torch.empty(N, 5, device='cuda')
    ctx.pse_constrained_solve(dev(F), dev(UB), dev(EB), U3, S3)
    assert torch.equal(U2, U3) and torch.equal(S2, S3)


def test_full_couplet_at_config3_size_against_pse_reference():
    """bench.py's default workload (N = 65 536, phi = 0.30, tol = 1e-3, xi = 0.575, grid 100, P = 4) with torques: U, Omega and E on
    128 sampled particles against the fp64 reference tier (its own xi = 0.40, tol = 1e-7; pinned against the direct sums in
    tests/test_pse_reference.py), plus the worst sampled particle as in tests/test_gpu_reference.py."""
    from oracle import pse_reference as pr
    N, tol, xi = 65536, 1e-3, 0.575
    ctx, x, L = make(N, 0.30, xi, tol, seed=100)
    assert (ctx.grid, ctx.P) == (100, 4)
    F, Lq, S = inputs(N, 1)
    rows = np.sort(np.random.default_rng(5).choice(N, 128, replace=False))
    want = pr.PSEReference(L, A, ETA, 0.40, tol=1e-7).apply_full(x, F, Lq, S, rows=rows)
    got = gpu_full(ctx, F, Lq, S)
    for g, w, name in zip(got, want, 'UWE'):
        worst = float(np.linalg.norm(g[rows] - w, axis=1).max() / np.sqrt((w * w).sum(axis=1).mean()))
        assert rel(g[rows], w) < bar(tol) and worst < 10 * bar(tol), (name, rel(g[rows], w), worst)


@pytest.mark.parametrize('tol', [1e-3, 1e-4])
def test_brownian_sample_of_the_full_couplet_against_dense_oracle(tol):
    """pse_brownian_full at N = 300 (dense 3 300 x 3 300 principal root), U^B, Omega^B and E^B separately; the same wave noise through
    pse_brownian gives a U^B, E^B whose WAVE half is identical (same random fluid field)."""
    N, xi, dt = 300, 0.7, 1e-3
    ctx, x, L = make(N, 0.20, xi, tol, seed=6)
    _, w2 = synth.brownian_noise(N, ctx.grid, 7)
    w1 = np.random.default_rng(7).standard_normal((N, 11))
    UB, WB, EB = torch.empty(N, 3, device='cuda'), torch.empty(N, 3, device='cuda'), torch.empty(N, 5, device='cuda')
    it = ctx.pse_brownian_full(dt, dev(w1), dev(w2), UB, WB, EB)
    assert 3 <= it <= 40
    Uo, Wo, Eo = cpl.brownian_full(x, L, A, ETA, KT, xi, dt, ctx.grid, w1, w2, eps=1e-10)
    for g, w, name in zip((UB, WB, EB), (Uo, Wo, Eo), 'UWE'):
        assert rel(g.cpu().numpy(), w) < bar(tol), (name, rel(g.cpu().numpy(), w))
    # wave half alone (zero real-space noise): the 8-component call sees the same field
    U1, W1, E1 = torch.empty(N, 3, device='cuda'), torch.empty(N, 3, device='cuda'), torch.empty(N, 5, device='cuda')
    ctx.pse_brownian_full(dt, torch.zeros(N, 11, device='cuda'), dev(w2), U1, W1, E1)
    U2, E2 = torch.empty(N, 3, device='cuda'), torch.empty(N, 5, device='cuda')
    ctx.pse_brownian(dt, torch.zeros(N, 8, device='cuda'), dev(w2), U2, E2)
    assert torch.equal(U1, U2) and torch.equal(E1, E2)
    Uw, Ww, Ew = cpl.wave_sqrt_apply_full(x, L, A, ETA, xi, ctx.grid, w2)
    assert rel(W1.cpu().numpy(), np.sqrt(2 * KT / dt) * Ww) < bar(tol)


def test_step_with_external_torques_against_dense_oracle():
    """pse_step_full at N = 48, tol 1e-4: displacement and angular velocities against oracle.couplet.step_full (dense matrices), with
    overlapping pairs (F^P != 0) and a torque on every sphere; without torques the displacement is pse_step's."""
    N, xi, tol, dt = 48, 0.85, 1e-4, 1e-3
    ctx, x, L = make(N, 0.20, xi, tol, seed=3, squeeze=0.93)
    w1, w2 = synth.brownian_noise(N, ctx.grid, 2)
    Lq = 20.0 * np.random.default_rng(5).standard_normal((N, 3))
    xo, Uo, Wo, So = cpl.step_full(x, L, A, ETA, KT, xi, dt, ctx.grid, w1, w2, Lq, eps=1e-10)
    pos = dev(pos4(x.astype(np.float32)))
    W = torch.empty(N, 3, device='cuda')
    gi, li = ctx.pse_step_full(pos, dt, dev(Lq), dev(w1.reshape(N, 8)), dev(w2), W)
    assert 2 <= gi <= 30 and 2 <= li <= 40
    d = pos[:, :3].cpu().numpy().astype(np.float64) - x
    d -= L * np.round(d / L)                                        # the library wraps into [0, L)
    assert rel(d, xo - x) < 3 * bar(tol) and rel(W.cpu().numpy(), Wo) < 3 * bar(tol), (rel(d, xo - x), rel(W.cpu().numpy(), Wo))
    # the torques really moved the spheres, and without them the step is pse_step's
    p0, p1 = dev(pos4(x.astype(np.float32))), dev(pos4(x.astype(np.float32)))
    ctx.pse_step_full(p0, dt, None, dev(w1.reshape(N, 8)), dev(w2))
    ctx.pse_step(p1, dt, dev(w1.reshape(N, 8)), dev(w2))
    d0 = (p0 - dev(pos4(x.astype(np.float32))))[:, :3].cpu().numpy()
    d1 = (p1 - dev(pos4(x.astype(np.float32))))[:, :3].cpu().numpy()
    d0 -= L * np.round(d0 / L); d1 -= L * np.round(d1 / L)
    assert rel(d0, d1) < 3 * bar(tol) and rel(d, d0) > 10 * bar(tol)


def test_edge_cases_single_sphere_odd_grid_and_bitwise_repeats():
    """(1) One sphere: the GPU reproduces the exact periodic rotational self-mobility Omega = L/(8 pi eta a^3) (1 - (4 pi/3)(a/L)^3)
    (pin C1 of the oracle) within the bar; (2) an odd grid (planes padded to 16-byte starts, no TMA) with an odd support;
    (3) two contexts and repeated calls agree bit for bit (every kernel of the full-couplet path has a fixed summation order)."""
    import paper_1709_06946_b200 as pse
    # (1)
    L, xi, tol = 12.0, 0.7, 1e-4
    st, g, p, rcut = pse.pse_suggest_params(1, L, A, tol, xi)
    ctx = pse.pse_create(1, L, A, ETA, KT, xi, g, p, rcut, tol)
    ctx.pse_neighbors(dev(pos4(np.array([[0.3, 11.9, 5.5]], np.float32))))
    Lq = np.array([[0.2, -1.0, 0.5]])
    U, W, E = gpu_full(ctx, None, Lq, None)
    want = Lq / (8 * np.pi * ETA * A**3) * (1.0 - 4 * np.pi / 3 * (A / L)**3)
    assert rel(W, want) < bar(tol) and np.abs(U).max() < bar(tol) * np.abs(want).max() and np.abs(E).max() < bar(tol) * np.abs(want).max()
    # (2)
    N, xi, tol = 120, 0.6, 1e-3
    x, L = synth.rsa(N, 0.15, seed=17)
    x32 = x.astype(np.float32)
    st, g, p, rcut = pse.pse_suggest_params(N, L, A, tol, xi)
    outs = []
    for rep in range(2):
        ctx = pse.pse_create(N, L, A, ETA, KT, xi, 27, 5, rcut, tol)          # 27^3: odd, not a multiple of 4
        ctx.pse_neighbors(dev(pos4(x32)))
        F, Lq, S = inputs(N, 9)
        a_ = gpu_full(ctx, F, Lq, S)
        b_ = gpu_full(ctx, F, Lq, S)
        w1 = np.random.default_rng(3).standard_normal((N, 11))
        _, w2 = synth.brownian_noise(N, 27, 3)
        UB, WB, EB = torch.empty(N, 3, device='cuda'), torch.empty(N, 3, device='cuda'), torch.empty(N, 5, device='cuda')
        ctx.pse_brownian_full(1e-3, dev(w1), dev(w2), UB, WB, EB)
        assert all(np.array_equal(u, v) for u, v in zip(a_, b_))
        outs.append(a_ + (UB.cpu().numpy(), WB.cpu().numpy(), EB.cpu().numpy()))
    assert all(np.array_equal(u, v) for u, v in zip(*outs))
    want = cpl.mobility_apply_full(x32.astype(np.float64), L, A, ETA, xi, F, Lq, S, eps=1e-9)
    for g_, w_, name in zip(outs[0][:3], want, 'UWE'):
        assert rel(g_, w_) < bar(tol), (name, rel(g_, w_))


def test_translational_rotational_brownian_covariance():
    """<[U^B; Omega^B][U^B; Omega^B]^T> = (2 kT/dt) M_{script-U script-F} (Eq. 71 for the 11-component sample): two spheres
    at r = 2.5a, 8 000 draws of pse_brownian_full with fresh device noise, against the 12 x 12 block of the oracle's dense matrix
    (which contains the translation-rotation coupling of the pair)."""
    import paper_1709_06946_b200 as pse
    N, L, xi, tol, dt, ndraw = 2, 16.0, 0.5, 1e-3, 1e-2, 8000
    x = np.array([[4.0, 4.0, 4.0], [6.0, 5.5, 4.0]])
    st, g, p, rcut = pse.pse_suggest_params(N, L, A, tol, xi)
    ctx = pse.pse_create(N, L, A, ETA, KT, xi, g, p, rcut, tol)
    ctx.pse_neighbors(dev(pos4(x.astype(np.float32))))
    gen = torch.Generator(device='cuda')
    gen.manual_seed(7)
    w1 = torch.empty(N, 11, device='cuda')
    w2 = torch.empty(3, g, g, g // 2 + 1, 2, device='cuda')
    UB, WB, EB = torch.empty(N, 3, device='cuda'), torch.empty(N, 3, device='cuda'), torch.empty(N, 5, device='cuda')
    acc = torch.zeros(12, 12, device='cuda', dtype=torch.float64)
    for _ in range(ndraw):
        w1.normal_(generator=gen)
        w2.normal_(generator=gen)
        ctx.pse_brownian_full(dt, w1, w2, UB, WB, EB)
        v = torch.cat([UB, WB], dim=1).reshape(-1).double()
        acc += torch.outer(v, v)
    C = (acc / ndraw).cpu().numpy() * dt / (2 * KT)
    M = cpl.dense_full(x, L, A, ETA, xi, eps=1e-10)
    keep = np.array([11 * i + c for i in range(N) for c in range(6)])
    Mo = M[np.ix_(keep, keep)]
    err = np.linalg.norm(C - Mo) / np.linalg.norm(Mo)
    tr_block = np.abs(Mo[:3, 9:12]).max()                            # U_1 <- L_2: the rotlet coupling, must be resolved
    print(f'brownian_full covariance: rel Frobenius error {err:.3f}, max |C - M| {np.abs(C - Mo).max():.4f}, rotlet block {tr_block:.4f}')
    assert err < 0.05
    assert np.abs(C[:3, 9:12] - Mo[:3, 9:12]).max() < 0.5 * tr_block + 4 * np.sqrt(Mo[0, 0] * Mo[9, 9] / ndraw)
