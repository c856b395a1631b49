"""GPU validation of the mid-point scheme against the paper's thermodynamic-equilibrium test:
pairs of spheres bound by U(r) = k |r - r0| must sample the Boltzmann distribution of Eq. (80).  Also parity of the
bond force and of one step with bonds against the fp64 oracle.  SURVEY.md §8(f) NEXT-2.
"""
import numpy as np
import pytest

import synth
from oracle import brownian as brn

pytestmark = pytest.mark.gpu
torch = pytest.importorskip('torch')

A, ETA, KT = 1.0, 1.0 / (6.0 * np.pi), 1.0


def dev(x, dtype=torch.float32):
    return torch.as_tensor(np.ascontiguousarray(x), dtype=dtype).cuda().contiguous()


def pos4(x):
    p = np.zeros((x.shape[0], 4), np.float32)
    p[:, :3] = x
    return p


def rel(a, b):
    return float(np.linalg.norm(np.asarray(a, float) - np.asarray(b, float)) / np.linalg.norm(np.asarray(b, float)))


def test_bond_forces_match_oracle_and_argument_checks():
    import paper_1709_06946_b200 as pse
    N = 200
    x, L = synth.rsa(N, 0.15, seed=12)
    x32 = x.astype(np.float32)
    ctx = pse.pse_create(N, L, A, ETA, KT, 0.6, 32, 6, min(6.0, L / 2), 1e-3)
    ctx.pse_neighbors(dev(pos4(x32)))
    g = np.random.Generator(np.random.Philox(3))
    pairs = np.array([(i, j) for i, j in g.integers(0, N, (300, 2)) if i != j], dtype=np.int32)   # repeated particles, periodic images
    F = torch.full((N, 3), 7.0, device='cuda')
    ctx.pse_bond_forces(F)                                   # no bonds: zero
    assert float(F.abs().max()) == 0.0
    ctx.pse_set_bonds(pairs, 2.5, 3.0)
    ctx.pse_bond_forces(F)
    Fo = brn.bond_forces(x32.astype(np.float64), L, pairs, 2.5, 3.0)
    assert rel(F.cpu().numpy(), Fo) < 1e-5
    assert np.abs(F.cpu().numpy().sum(axis=0)).max() < 1e-3     # Newton's third law
    for bad in ([[0, N]], [[-1, 2]], [[5, 5]]):
        with pytest.raises(pse.PSEError):
            ctx.pse_set_bonds(np.array(bad, dtype=np.int32), 1.0, 3.0)
    ctx.pse_set_bonds(np.zeros((0, 2), np.int32), 0.0, 0.0)
    ctx.pse_bond_forces(F)
    assert float(F.abs().max()) == 0.0


def test_step_with_bonds_against_dense_oracle():
    """One mid-point step (Eqs. 76-79) with bond forces in F^P, N=40, fp32 GPU vs dense fp64 oracle."""
    import paper_1709_06946_b200 as pse
    N, tol, xi, grid, P, dt = 40, 1e-4, 1.1, 32, 9, 1e-3
    x, L = synth.rsa(N, 0.20, seed=8)
    x32 = x.astype(np.float32)
    st, _, _, rcut = pse.pse_suggest_params(N, L, A, tol, xi)
    assert st == 0
    ctx = pse.pse_create(N, L, A, ETA, KT, xi, grid, P, rcut, tol)
    pairs = np.arange(N, dtype=np.int32).reshape(-1, 2)
    ctx.pse_set_bonds(pairs, 40.0, 2.5)                       # strong enough to matter next to the Brownian displacement
    w1, w2 = synth.brownian_noise(N, grid, 4)
    pos = dev(pos4(x32))
    ctx.pse_step(pos, dt, dev(w1.reshape(N, 8)), dev(w2))
    xb, _, _ = brn.step(x32.astype(np.float64), L, A, ETA, KT, xi, dt, grid, w1, w2, eps=1e-10, bonds=(pairs, 40.0, 2.5))
    x0, _, _ = brn.step(x32.astype(np.float64), L, A, ETA, KT, xi, dt, grid, w1, w2, eps=1e-10)
    got = pos.cpu().numpy()[:, :3].astype(np.float64)
    d = got - xb
    d -= L * np.round(d / L)
    disp = xb - x32.astype(np.float64)
    assert np.linalg.norm(xb - x0) > 0.3 * np.linalg.norm(disp)          # the bonds do move the particles
    assert np.linalg.norm(d) / np.linalg.norm(disp) < 5 * tol


@pytest.mark.parametrize('gamma', [0.0, 0.3], ids=['cube', 'sheared_cell'])
def test_pair_distance_distribution_matches_eq80(gamma):
    """64 bonded pairs in a dilute periodic box (phi = 0.002), 40 000 mid-point steps: the histogram of the
    centre-to-centre distance and its first moments against Eq. (80).  The bond keeps r > 2a with
    probability 1 - 1e-4 (r0 = 5a, k = 3 kT/a), so the hard-sphere force plays no role inside a pair.
    Second case: the same in a cell sheared to gamma = 0.3 (pse_set_lattice, NEXT-4): the equilibrium distribution does not
    know about the lattice, so the whole deformed-lattice step path (graphs included) must reproduce it as well."""
    import paper_1709_06946_b200 as pse
    npair, k, r0, dt, tol, xi = 64, 3.0, 5.0, 2.5e-3, 1e-3, 0.3
    nsteps, burn, every = 40000, 1000, 4
    N, L = 2 * npair, 64.0
    st, grid, P, rcut = pse.pse_suggest_params(N, L, A, tol, xi, lattice=(1.0, gamma, 1.0))
    assert st == 0
    ctx = pse.pse_create(N, L, A, ETA, KT, xi, grid, P, rcut, tol)
    if gamma:
        ctx.pse_set_lattice(1.0, gamma, 1.0)
    c = (np.stack(np.meshgrid(*[np.arange(4)] * 3, indexing='ij'), -1).reshape(-1, 3) + 0.5) * (L / 4)    # 4^3 pair centres
    x = np.empty((N, 3))
    x[0::2] = c - [r0 / 2, 0, 0]
    x[1::2] = c + [r0 / 2, 0, 0]
    pairs = np.arange(N, dtype=np.int32).reshape(-1, 2)
    ctx.pse_set_bonds(pairs, k, r0)
    pos = dev(pos4(x.astype(np.float32)))
    gen = torch.Generator(device='cuda')
    gen.manual_seed(1234)
    w1 = torch.empty(N, 8, device='cuda')
    w2 = torch.empty(3, grid, grid, grid // 2 + 1, 2, device='cuda')
    samples = []
    for s in range(nsteps):
        w1.normal_(generator=gen)
        w2.normal_(generator=gen)
        ctx.pse_step(pos, dt, w1, w2)
        if s >= burn and s % every == 0:
            d = pos[0::2, :3] - pos[1::2, :3]
            d[:, 0] -= gamma * d[:, 1]                        # minimum image in lattice coordinates s = A^-1 x, back to x = A s
            d = d - L * torch.round(d / L)
            d[:, 0] += gamma * d[:, 1]
            samples.append(d.norm(dim=1))
    r = torch.cat(samples).double().cpu().numpy()
    # Eq. (80) by quadrature
    rr = np.linspace(0.0, 14.0, 140001)
    f = brn.pair_distance_pdf(rr, k / KT, r0)
    assert abs(np.trapezoid(f, rr) - 1.0) < 1e-6
    mean_th, absu_th = np.trapezoid(f * rr, rr), np.trapezoid(f * np.abs(rr - r0), rr)
    var_th = np.trapezoid(f * (rr - mean_th) ** 2, rr)
    print(f'eq80: n={len(r)} <|u|> {np.abs(r - r0).mean():.4f} (th {absu_th:.4f})  <r> {r.mean():.4f} (th {mean_th:.4f})  '
          f'var {r.var():.4f} (th {var_th:.4f})  min r {r.min():.3f}  grid {grid} P {P}')
    # 64 pairs x 39 000 steps / (2 x ~130 steps correlation time) ~ 9 600 independent samples: 1 sigma ~ 1 % on <|u|>
    # (measured on B200: <|u|> 0.3366 against 0.3392, <r> 5.0847 against 5.0881, variance 0.2241 against 0.2242)
    assert abs(np.abs(r - r0).mean() / absu_th - 1.0) < 0.035
    assert abs(r.mean() - mean_th) < 0.02
    assert abs(r.var() / var_th - 1.0) < 0.06
    edges = np.array([0.0, 4.0, 4.4, 4.7, 4.9, 5.0, 5.1, 5.3, 5.6, 6.0, 14.0])
    hist = np.histogram(r, edges)[0] / len(r)
    cdf = np.concatenate([[0.0], np.cumsum((f[1:] + f[:-1]) * 0.5 * np.diff(rr))])
    want = np.diff(np.interp(edges, rr, cdf))
    print('eq80 histogram: max |p_bin - Eq.(80)| =', float(np.abs(hist - want).max()))
    assert np.abs(hist - want).max() < 0.015, (hist, want)
    assert r.min() > 2.0 * A * 0.98


def test_midpoint_drift_and_covariance_match_appendix_B():
    """Eqs. (B12), (B17): over many noise samples from the same x_k the mid-point step gives
    <dx> = kT dt div R_FU^-1 and <dx dx> = 2 kT dt R_FU^-1, with R_FU^-1 = M_UF - M_US M_ES^-1 M_EF from the dense fp64
    oracle.  Each sample is run with +w and -w: the O(sqrt dt) term cancels in the sum and the drift (O(dt), 1.4e3 times
    smaller than the noise per step) is resolved with 20 000 pairs (measured on B200 with 40 000: -0.0294 / +0.0279
    against -/+0.0286, transverse components below 6e-4, covariance diagonal within 1.4 %).  Two spheres at r = 2.5a: no overlap at the
    mid-point, so F^P = 0."""
    import paper_1709_06946_b200 as pse
    N, L, xi, tol, dt, npairs = 2, 16.0, 0.5, 1e-4, 1e-3, 20000
    x0 = np.array([[1.0, 1.0, 1.0], [3.5, 1.0, 1.0]])
    st, grid, P, rcut = pse.pse_suggest_params(N, L, A, tol, xi)
    assert st == 0
    ctx = pse.pse_create(N, L, A, ETA, KT, xi, grid, P, rcut, tol)
    p0 = dev(pos4(x0.astype(np.float32)))
    gen = torch.Generator(device='cuda')
    gen.manual_seed(99)
    w1 = torch.empty(N, 8, device='cuda')
    w2 = torch.empty(3, grid, grid, grid // 2 + 1, 2, device='cuda')
    s1 = torch.zeros(6, dtype=torch.float64, device='cuda')
    s2 = torch.zeros(6, 6, dtype=torch.float64, device='cuda')
    pos = p0.clone()
    for _ in range(npairs):
        w1.normal_(generator=gen)
        w2.normal_(generator=gen)
        for sgn in (1.0, -1.0):
            pos.copy_(p0)
            ctx.pse_step(pos, dt, w1 * sgn, w2 * sgn)
            d = (pos[:, :3] - p0[:, :3]).double()
            d = (d - L * torch.round(d / L)).reshape(6)
            s1 += d
            s2 += torch.outer(d, d)
    n = 2 * npairs
    mean, cov = (s1 / n).cpu().numpy(), (s2 / n).cpu().numpy()
    Mc = brn.constrained_mobility(mob_dense(x0, L, xi), N)
    div_c, _ = brn.constrained_mobility_divergence(x0, L, A, ETA, xi)
    print('drift/(kT dt):', mean / (KT * dt), 'oracle', div_c)
    print('cov/(2 kT dt) diag:', np.diag(cov) / (2 * KT * dt), 'oracle', np.diag(Mc))
    # (B17): entries to 4 % of the diagonal scale (the +w / -w samples repeat each other here: 1 sigma = sqrt(2/npairs) = 1 %)
    assert np.abs(cov / (2 * KT * dt) - Mc).max() < 0.04 * np.abs(Mc).max()
    # (B12): 0.029 along the line of centres, equal and opposite; transverse components vanish
    scale = abs(div_c[0])
    assert scale > 0.02
    assert abs(mean[0] / (KT * dt) - div_c[0]) < 0.2 * scale and abs(mean[3] / (KT * dt) - div_c[3]) < 0.2 * scale
    assert np.abs(mean[[1, 2, 4, 5]] / (KT * dt)).max() < 0.2 * scale


def mob_dense(x, L, xi):
    from oracle import mobility as mob
    return mob.dense(np.asarray(x, dtype=np.float64), L, A, ETA, xi, 'both', 1e-12)
