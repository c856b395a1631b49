#!/usr/bin/env python
"""bench.py — constrained Brownian-dynamics steps/s (and grand-mobility products/s) of libpse on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload config3|config4|config2|tiny] [--impl ours|reference]

One "step" is one pass of the whole hot path: pse_step = neighbour build, Brownian sample
(Lanczos + wave-space square root), mid-point move, neighbour build, hard-sphere forces, GMRES stresslet solve
(~10 full products), final move.  Inputs are seeded synthetic hard-sphere suspensions (synth/, recipe in DESIGN.md).
Prints ONE JSON line on rank 0.  Multi-GPU (torchrun): independent replicas, no data-path collective.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

A, ETA, KT = 1.0, 1.0 / (6.0 * np.pi), 1.0

WORKLOADS = {
    # name: N, phi, tol, xi, dt, relax sweeps          (BASELINE.json configs; xi is the free tuning knob)
    'tiny': dict(N=4096, phi=0.20, tol=1e-3, xi=0.5, dt=1e-3, relax=0),
    'config2': dict(N=4096, phi=0.20, tol=1e-4, xi=0.5, dt=1e-3, relax=0),
    'config3': dict(N=65536, phi=0.30, tol=1e-3, xi=0.575, dt=1e-4, relax=2),   # largest xi that keeps the 100^3 grid
    'config4': dict(N=1048576, phi=0.10, tol=1e-3, xi=0.34, dt=1e-4, relax=0),
    # fractal aggregates (d_f ~ 1.8, 32-sphere clusters); tol and xi are swept with --tol / --xi
    'config5': dict(N=262144, phi=0.05, tol=1e-3, xi=0.28, dt=1e-4, relax=0, fractal=True),
}


def peaks():
    try:
        with open(os.path.join(ROOT, 'MEASURED_PEAKS.json')) as f:
            return float(json.load(f)['hbm_gbs']), 'measured (MEASURED_PEAKS.json hbm_gbs)'
    except Exception:
        return 6650.0, 'fallback (B200_PROFILING.md)'


class ClockSampler:
    """nvidia-smi clocks and throttle reasons sampled DURING the timed region."""
    Q = ('clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,'
         'clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap')

    def __init__(self, index=0):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(['nvidia-smi', f'--id={self.index}', f'--query-gpu={self.Q}', '--format=csv,noheader,nounits',
                                          '-lms', '100'], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(',')])

    def stop(self):
        if not self.proc:
            return {'sm_mhz': None, 'sm_max_mhz': None, 'reasons': ['nvidia-smi unavailable']}
        time.sleep(0.15)
        self.proc.terminate()
        self.th.join(timeout=2)
        sm = [float(r[0]) for r in self.rows if r and r[0].replace('.', '').isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) > 1 and r[1].replace('.', '').isdigit()]
        names = ['hw_slowdown', 'hw_thermal_slowdown', 'sw_thermal_slowdown', 'sw_power_cap']
        reasons = [n for i, n in enumerate(names) if any(len(r) > 2 + i and r[2 + i].lower().startswith('active') for r in self.rows)]
        return {'sm_mhz': float(np.median(sm)) if sm else None, 'sm_max_mhz': max(mx) if mx else None, 'reasons': reasons,
                'samples': len(sm)}


# dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed ncu --set full captures (profiles/r2_traffic.md), default
# workloads only; other workloads report null.
# fp32 operations per pair evaluation of real_pairs_kernel (ncu: fadd + fmul + 2 ffma predicated-on thread instructions / pairs,
# profiles/r1_ncu_kernels.md; the kernel is unchanged since): 162 for the full 8 x 8 product (Lanczos iterations), 129 for S -> E
# (GMRES iterations); a step runs seven of each plus two mixed products, so their mean is used
FLOP_PER_PAIR = 0.5 * (162.0 + 129.0)
N_SM, FP32_LANES_PER_SM = 148, 128                # B200: 4 sub-partitions x 32 fp32 lanes per SM (blackwell guide), FMA = 2 flop
NCU_TRAFFIC = {'config3': {'real': 17375488, 'spread': 6934784, 'interp': 25789440, 'scale': 12053760, 'neighbors': 1096704},
               'config4': {'real': 372716288, 'spread': 264503808, 'interp': 327649280, 'scale': 271386112, 'neighbors': 251827968}}


def max_over_ranks(ms, device=None):
    """Replica aggregation: the job's time is the slowest rank's; no data-path collective."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(ms)
    t = torch.tensor([float(ms)], dtype=torch.float64, device=device if device is not None else 'cpu')
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def replica_throughput(steps, world, ms_max):
    """Whole-job steps/s of `world` independent replicas that each ran `steps` steps in at most ms_max ms."""
    return world * steps * 1e3 / ms_max


def make_suspension(wl, seed):
    import synth
    if wl.get('fractal'):
        return synth.fractal_aggregates(wl['N'], wl['phi'], seed=seed)
    x, L = synth.rsa(wl['N'], wl['phi'], seed=seed)
    if wl['relax']:
        x = synth.relax_overlaps(x, L, sweeps=wl['relax'], seed=seed)
    return x, L


def choose_params(wl, L, need_gpu_lib=True):
    """grid, P, r_cut of the run from pse_suggest_params (host-only entry point of libpse.so: parameter arithmetic, no kernels)."""
    import paper_1709_06946_b200 as pse
    st, grid, P, rcut = pse.pse_suggest_params(wl['N'], L, A, wl['tol'], wl['xi'], lattice=(1.0, wl.get('shear', 0.0), 1.0))
    if st != 0:
        raise RuntimeError(f'no valid PSE parameters for {wl}')
    return grid, P, rcut


def planes_per_launch(g):
    """Mean number of grids (planes) each wave-space kernel touches per launch inside one pse_step with g GMRES
    iterations (the products carry only the components they need): M_EF F (3 in, 5 out), g x M_ES v
    (5 in, 5 out), the final [F;S] -> U product (8 in, 3 out) and the Brownian half pass (3 noise planes in, 8 out)."""
    fwd = (3 + 5 * g + 8) / (g + 2)
    inv = (5 + 5 * g + 3 + 8) / (g + 3)
    scale = ((3 + 5) + 10 * g + (8 + 3) + (3 + 8)) / (g + 3)
    return {'spread': fwd, 'fft_fwd': fwd, 'scale': scale, 'fft_inv': inv, 'interp': inv}


def algorithmic_bytes(N, M, nb_mean, g=None):
    """Per-launch algorithmic bytes of each phase: fp32, G = M^3 grid points.
    g = None: a full product (8 grids in, 8 out); else the launch mix of a step with g GMRES iterations."""
    G, Gh = float(M) ** 3, float(M) * M * (M // 2 + 1)
    pl = planes_per_launch(g) if g is not None else {'spread': 8, 'fft_fwd': 8, 'scale': 16, 'fft_inv': 8, 'interp': 8}
    return {
        'neighbors': 16 * N + 8 * N + 2 * 4 * N * nb_mean,      # positions, sort keys/permutation, list written (count + fill pass reads excluded)
        'real': 16 * N + 32 * N + 32 * N + 4 * N * nb_mean,     # compulsory DRAM: pos, in, out, neighbour indices
        'spread': 16 * N + pl['spread'] * (4 * N + 4 * G),      # particles read, each grid written once
        'fft_fwd': pl['fft_fwd'] * (4 * G + 8 * Gh),            # one-pass lower bound: real grid in, half spectrum out
        'scale': pl['scale'] * 8 * Gh,                          # one complex per half-spectrum mode per plane read or written
        'fft_inv': pl['fft_inv'] * (8 * Gh + 4 * G),
        'interp': 16 * N + pl['interp'] * (4 * G + 4 * N),      # each grid read once, particles read/written
    }


def run_ours(args, wl, rank, world):
    import torch
    import paper_1709_06946_b200 as pse
    dev = torch.device('cuda', int(os.environ.get('LOCAL_RANK', 0)))
    torch.cuda.set_device(dev)
    N, dt = wl['N'], wl['dt']
    x, L = make_suspension(wl, seed=100 + rank)
    grid, P, rcut = choose_params(wl, L)
    ctx = pse.pse_create(N, L, A, ETA, KT, wl['xi'], grid, P, rcut, wl['tol'])
    if wl.get('shear'):                              # Lees-Edwards cell of strain gamma (Eq. 56): the suspension is carried along, x = A s
        ctx.pse_set_lattice(1.0, wl['shear'], 1.0)
        x = x.copy()
        x[:, 0] += wl['shear'] * x[:, 1]
    pos = torch.zeros(N, 4, device=dev)
    pos[:, :3] = torch.from_numpy(x.astype(np.float32)).to(dev)
    gen = torch.Generator(device=dev); gen.manual_seed(1234 + rank)
    K, W = args.steps, args.warmup
    nshape = (3, grid, grid, grid // 2 + 1, 2)

    def noise():
        return (torch.randn(N, 8, device=dev, generator=gen), torch.randn(nshape, device=dev, generator=gen))

    flush = torch.empty(256 * 1024 * 1024 // 4, device=dev)
    iters = []

    def timed_steps(n, profiled=False):
        """n steps, each bracketed by its own CUDA events on the library's stream, L2 flushed in between."""
        total = 0.0
        for _ in range(n):
            nr, nw = noise()
            flush.fill_(1.0)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            gi, li = ctx.pse_step(pos, dt, nr, nw)
            e1.record()
            torch.cuda.synchronize()
            total += e0.elapsed_time(e1)
            iters.append((gi, li))
        return total

    timed_steps(W)
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
    torch.cuda.synchronize()
    sampler = ClockSampler(dev.index or 0)
    sampler.start()
    l0 = ctx.pse_kernel_launches()
    iters.clear()
    ms = timed_steps(K)
    launches = ctx.pse_kernel_launches() - l0
    clocks = sampler.stop()
    torch.cuda.synchronize()
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
        ms = max_over_ranks(ms, dev)
    gm = float(np.mean([i[0] for i in iters])); lz = float(np.mean([i[1] for i in iters]))
    out = dict(ms=ms, launches=launches, clocks=clocks, gmres=gm, lanczos=lz, grid=grid, P=P, rcut=rcut, L=L)
    if rank != 0:
        return out
    # ---- per-phase times (profiled pass, same steps, CUDA events inside the library) ----
    ctx.pse_set_profiling(True)
    ctx.pse_get_timings()
    kp = max(1, min(K, 5))
    timed_steps(kp)
    phases = ctx.pse_get_timings()
    ctx.pse_set_profiling(False)
    ctx.pse_neighbors(pos)
    count, _ = ctx.pse_get_neighbors()
    nb_mean = float(count.float().mean().item())
    out.update(phases=phases, nb_mean=nb_mean, profiled_steps=kp)
    # ---- product throughput (device resident) ----
    F, S = torch.randn(N, 3, device=dev, generator=gen), torch.randn(N, 5, device=dev, generator=gen)
    U, E = torch.empty(N, 3, device=dev), torch.empty(N, 5, device=dev)
    for _ in range(3):
        ctx.pse_mobility_apply(F, S, U, E)
    mv = 0.0
    nmv = 20
    for _ in range(nmv):
        flush.fill_(1.0)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); ctx.pse_mobility_apply(F, S, U, E); e1.record()
        torch.cuda.synchronize()
        mv += e0.elapsed_time(e1)
    out['matvec_ms'] = mv / nmv
    # the same with torques and angular velocities (Eq. 31's full couplet, 11 components)
    Lq, W = torch.randn(N, 3, device=dev, generator=gen), torch.empty(N, 3, device=dev)
    for _ in range(3):
        ctx.pse_mobility_apply_full(F, Lq, S, U, W, E)
    mv = 0.0
    for _ in range(nmv):
        flush.fill_(1.0)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); ctx.pse_mobility_apply_full(F, Lq, S, U, W, E); e1.record()
        torch.cuda.synchronize()
        mv += e0.elapsed_time(e1)
    out['matvec_full_ms'] = mv / nmv
    # ---- end to end through the C ABI with host buffers ----
    hpos = pos.cpu().pin_memory()
    hnr = torch.randn(N, 8).pin_memory(); hnw = torch.randn(nshape).pin_memory()
    ke = max(1, min(K, 10))
    for _ in range(2):
        ctx.pse_step_host(hpos, dt, hnr, hnw)
    e2e = 0.0
    for _ in range(ke):
        hnr.normal_(); hnw.normal_()
        flush.fill_(1.0)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        ctx.pse_step_host(hpos, dt, hnr, hnw)          # synchronises internally after the D2H copy
        e2e += (time.perf_counter() - t0) * 1e3
    out.update(e2e_ms=e2e / ke, h2d=int(hpos.numel() * 4 + hnr.numel() * 4 + hnw.numel() * 4), d2h=int(hpos.numel() * 4), e2e_steps=ke)
    if wl.get('shear'):
        # a flowing suspension: the strain changes before every step (here it recedes from the value the grid was sized for, the
        # particles carried along), which must not cost the captured step graphs (the kernels read the lattice from device memory)
        g, dg, fl = float(wl['shear']), 1e-4, 0.0
        for k in range(3 + ke):
            nr, nw = noise()
            pos[:, 0] -= dg * pos[:, 1]
            g -= dg
            flush.fill_(1.0)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); ctx.pse_set_lattice(1.0, g, 1.0); ctx.pse_step(pos, dt, nr, nw); e1.record()
            torch.cuda.synchronize()
            if k >= 3:
                fl += e0.elapsed_time(e1)
        out['flow_ms'] = fl / ke
    return out


def direct_oracle_sample(wl, nsteps):
    """The direct O(N^2) oracle, as it stands, on a bounded sample of the workload: one dense mid-point step (Eqs. 76-79) of
    N_s spheres at the workload's volume fraction and tolerance.  Returns (seconds per oracle step, N_s, cores, text)."""
    import synth
    from oracle import brownian as brn
    Ns = 128
    x, L = synth.rsa(Ns, wl['phi'], seed=7)
    s = np.sqrt(-np.log(wl['tol']))
    xi = max(wl['xi'], 1.02 * s / (0.5 * L - 2 * A))                 # keep rcut = s/xi + 2a <= L/2 in the small box
    Mg = 16
    while Mg < 2 * xi * s * L / np.pi:
        Mg += 2
    eps = min(1e-10, wl['tol'] * 1e-4)
    times = []
    for k in range(nsteps):
        w1, w2 = synth.brownian_noise(Ns, Mg, seed=k)
        t0 = time.perf_counter()
        xn, _, _ = brn.step(x, L, A, ETA, KT, xi, wl['dt'], Mg, w1, w2, eps=eps)
        times.append(time.perf_counter() - t0)
        x = xn % L
    text = (f'oracle.brownian.step (dense fp64 direct Ewald, eps={eps:g}) on N_s={Ns} spheres at phi={wl["phi"]}, xi={xi:.3f}, '
            f'{nsteps} step(s); steps/s scaled to the workload by N_s/N (linear, generous: the oracle is O(N^2) and worse)')
    return float(np.mean(times)), Ns, host_threads(), text


def host_threads():
    try:
        from threadpoolctl import threadpool_info
        return max([p.get('num_threads', 1) for p in threadpool_info()] + [os.cpu_count() or 1])
    except Exception:
        return os.cpu_count() or 1


class ReferenceStepper:
    """The fp64 CPU PSE reference (oracle/pse_reference.py: linked-cell pair sum, Gaussian NUFFT of Eq. 42 with scipy's FFT,
    textbook Lanczos and GMRES), as it stands, on the workload itself: same particles, xi, grid and r_cut as the GPU run, the
    paper's Gaussian window at the support its own bound gives for the tolerance, Krylov tolerances = the Ewald tolerance.
    If one step would take too long the particle number is reduced at fixed phi, tol, xi (PSE is O(N))."""

    def __init__(self, wl, budget_s=25.0):
        import synth
        from oracle import pse_reference as pr
        self.pr, self.wl, self.synth = pr, wl, synth
        self.N = wl['N']
        self.x, self.L = make_suspension(wl, seed=100)
        self.grid, _, self.rcut = choose_params(wl, self.L, need_gpu_lib=False)
        self.P = pr.gaussian_support(wl['tol'])
        self.k = 0
        self.budget_s = budget_s
        self.cores = max(pr.threads(), os.cpu_count() or 1)

    def shrink(self, factor):
        """Sub-sample: N/factor particles at the same volume fraction (fresh RSA placement), same tol, xi."""
        wl = dict(self.wl, N=max(4096, int(self.N // factor)), relax=0, fractal=False)
        self.N = wl['N']
        self.x, self.L = make_suspension(wl, seed=100)
        self.grid, _, self.rcut = choose_params(wl, self.L, need_gpu_lib=False)

    def step(self):
        wl = self.wl
        w1, w2 = self.synth.brownian_noise(self.N, self.grid, seed=1000 + self.k)
        self.k += 1
        t0 = time.perf_counter()
        xn, _, _, its = self.pr.step(self.x, self.L, A, ETA, KT, wl['xi'], wl['dt'], self.grid, w1, w2, tol=wl['tol'], krylov_tol=wl['tol'],
                                     params=dict(M=self.grid, P=self.P, rcut=self.rcut))
        dt_s = time.perf_counter() - t0
        self.x = xn % self.L
        return dt_s, its

    def describe(self, nsteps):
        scaled = '' if self.N == self.wl['N'] else f'; N_s={self.N} of N={self.wl["N"]} at the same phi, steps/s scaled by N_s/N (PSE is O(N))'
        return (f'oracle.pse_reference.step (fp64 PSE: linked-cell pair sum + Gaussian NUFFT P={self.P} on the {self.grid}^3 grid, scipy FFT, '
                f'fp64 Lanczos/GMRES to tol) on the workload itself: N={self.N}, xi={self.wl["xi"]}, r_cut={self.rcut:.3f}, {nsteps} full step(s)' + scaled)


def describe(name, wl):
    kind = 'spheres in 32-sphere fractal aggregates' if wl.get('fractal') else 'hard spheres'
    return (f'{name}: N={wl["N"]} {kind}, phi={wl["phi"]}, Ewald tol={wl["tol"]}, xi={wl["xi"]}, dt={wl["dt"]}, kT=1, RSA placement'
            + (f' + {wl["relax"]} relax sweeps (BASELINE.json: 1000; equilibration does not change the kernels\' work)' if wl['relax'] else ''))


def assemble(name, wl, r, K, world, overridden):
    """Measured numbers of one workload -> the keys of the JSON line that depend on it."""
    ms_step = r['ms'] / K
    value = replica_throughput(K, world, r['ms'])                     # replicas: all ranks' steps / max-over-ranks time
    peak, peak_src = peaks()
    ab = algorithmic_bytes(wl['N'], r['grid'], r['nb_mean'], r['gmres'])
    phases = {}
    for ph, (ms, n) in r['phases'].items():
        if n == 0:
            continue
        avg = ms / n
        e = {'ms_per_step': ms / r['profiled_steps'], 'launches_per_step': n / r['profiled_steps'], 'avg_ms': avg}
        if ph in ab:
            e['alg_GBps'] = ab[ph] / (avg * 1e-3) / 1e9
            e['frac_of_hbm_peak'] = e['alg_GBps'] / peak
        if ph == 'real':                         # the pair kernel is not a streaming kernel: also report pair evaluations per second
            e['pairs_per_sec'] = wl['N'] * r['nb_mean'] / (avg * 1e-3)
        phases[ph] = e
    dom = max((p for p in phases if p in ab), key=lambda p: phases[p]['ms_per_step'])
    fft_share = (phases.get('fft_fwd', {}).get('ms_per_step', 0) + phases.get('fft_inv', {}).get('ms_per_step', 0)) / \
        max(sum(p['ms_per_step'] for p in phases.values()), 1e-9)
    out = {'value': value, 'ms_per_step': ms_step}
    out['config'] = {'workload': describe(name, wl), 'N': wl['N'], 'phi': wl['phi'], 'tol': wl['tol'], 'xi': wl['xi'], 'dt': wl['dt'],
                     'grid': r['grid'], 'rcut': round(r['rcut'], 4), 'L': round(r['L'], 4)}
    if wl.get('shear'):
        out['config']['lattice'] = f"simple shear, strain {wl['shear']} (Eq. 56): lattice vectors = columns of L [[1, {wl['shear']}, 0], [0, 1, 0], [0, 0, 1]]"
    out['run'] = {'window': 'exponential of semicircle', 'P': r['P'], 'mean_neighbors': round(r['nb_mean'], 2), 'gmres_iters': r['gmres'],
                  'lanczos_iters': r['lanczos'], 'parallelism': f'replicas x{world}' if world > 1 else 'single GPU',
                  'l2': 'flushed (256 MiB write) between timed steps; each step bracketed by its own CUDA events'}
    out['matvecs_per_sec'] = 1e3 / r['matvec_ms']
    out['matvecs_full_couplet_per_sec'] = 1e3 / r['matvec_full_ms']      # [U;Omega;E] = M [F;L;S], 11 components
    out['ptps'] = value * wl['N']
    if 'flow_ms' in r:
        out['strain_advanced_every_step_steps_per_sec'] = 1e3 / r['flow_ms']      # pse_set_lattice before every pse_step
    out['clocks'] = r['clocks']
    out['gpu_launches'] = int(r['launches'])
    out['e2e'] = {'value': 1e3 / r['e2e_ms'], 'unit': 'steps/s', 'h2d_bytes_per_step': r['h2d'], 'd2h_bytes_per_step': r['d2h'],
                  'api': 'pse_step_host (pinned host buffers, copies inside the timed call)', 'steps': r['e2e_steps']}
    traffic = None if overridden else NCU_TRAFFIC.get(name, {}).get(dom)
    out['roofline'] = {'bound': 'hbm', 'kernel': dom, 'achieved': phases[dom]['alg_GBps'], 'peak': peak, 'unit': 'GB/s',
                       'frac': phases[dom]['alg_GBps'] / peak, 'traffic': traffic, 'peak_source': peak_src,
                       'note': 'algorithmic bytes per launch / mean launch duration from CUDA events inside the library over '
                               f'{r["profiled_steps"]} profiled steps; ' + (
                                   'at this size the grids are L2-resident (see DESIGN.md §5)' if 64 * r['grid']**3 < 100e6 else
                                   'the 8 real + 8 spectral grids exceed the L2 (see DESIGN.md §5)')}
    if dom == 'real':
        # the pair kernel moves few bytes per flop (its gathers are served by L1/L2): the binding roofline is fp32 issue, not HBM
        hbm_view = {k: out['roofline'][k] for k in ('achieved', 'peak', 'unit', 'frac')}
        clock_ghz = (r['clocks'].get('sm_mhz') or r['clocks'].get('sm_max_mhz') or 1965.0) / 1e3
        peak_tf = N_SM * FP32_LANES_PER_SM * 2 * clock_ghz / 1e3
        tf = phases['real']['pairs_per_sec'] * FLOP_PER_PAIR / 1e12
        out['roofline'].update({'bound': 'alu', 'achieved': tf, 'peak': peak_tf, 'unit': 'TFLOP/s', 'frac': tf / peak_tf, 'hbm_view': hbm_view,
                                'peak_source': f'{N_SM} SMs x {FP32_LANES_PER_SM} fp32 lanes x 2 flop x {clock_ghz:.3f} GHz (median SM clock under load in this run)',
                                'note': f'pair evaluations/s x {FLOP_PER_PAIR:.1f} fp32 operations per pair (ncu count, profiles/); the kernel is bound by the L1 request '
                                        'rate of its gathers and by instruction issue, its DRAM traffic (traffic, bytes per launch) is the neighbour list; '
                                        'hbm_view = algorithmic bytes / launch time against the measured HBM peak'})
    out['phases'] = phases
    out['cufft_share_of_step'] = fft_share
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument('--gpus', type=int, default=1)
    ap.add_argument('--steps', type=int, default=20)
    ap.add_argument('--warmup', type=int, default=3)
    ap.add_argument('--workload', default='config3', choices=sorted(WORKLOADS))
    ap.add_argument('--impl', default='ours', choices=['ours', 'reference'])
    ap.add_argument('--no-cpu-baseline', action='store_true')
    ap.add_argument('--no-config4', action='store_true', help='skip the 1M-particle block that the default run adds')
    ap.add_argument('--xi', type=float, default=None, help='override the splitting parameter (tuning knob, PAPER.md:154)')
    ap.add_argument('--tol', type=float, default=None, help='override the Ewald tolerance of the workload')
    ap.add_argument('--particles', type=int, default=None, help='override N of the workload (size sweep; phi, tol and xi are kept)')
    ap.add_argument('--shear', type=float, default=None, help='run the workload in a sheared periodic cell of this strain (Eq. 56, PAPER.md:318); '
                                                               'implies --no-cpu-baseline (the reference tier is cubic)')
    args = ap.parse_args()
    wl = dict(WORKLOADS[args.workload])
    overridden = bool(args.xi or args.tol or args.particles or args.shear)
    if args.shear:
        if args.impl == 'reference':
            raise SystemExit('bench.py: --shear has no reference arm (oracle/pse_reference.py is cubic)')
        wl['shear'] = args.shear
        args.no_cpu_baseline = True
    if args.xi:
        wl['xi'] = args.xi
    if args.tol:
        wl['tol'] = args.tol
    if args.particles:
        wl['N'] = args.particles
    rank, world = int(os.environ.get('RANK', 0)), int(os.environ.get('WORLD_SIZE', 1))
    base = {'metric': 'constrained_bd_steps_per_sec', 'unit': 'steps/s', 'n_gpus': args.gpus, 'steps': args.steps, 'warmup': args.warmup,
            'higher_is_better': True, 'scaling': 'weak', 'vs_baseline': None, 'dtype': 'f32', 'data': 'synthetic'}

    if args.impl == 'reference':
        # the oracle's fast tier on the SAME workload (config identical to our arm's), on the host cores; rank 0 only
        if rank != 0:
            return
        rs = ReferenceStepper(wl)
        sec0, _ = rs.step()                                          # first warm-up step doubles as the cost probe
        total = sec0 * (args.steps + args.warmup)
        if total > 240.0:                                            # keep the whole run within a few minutes
            rs.shrink(total / 240.0)
            rs.step()
        for _ in range(max(0, args.warmup - 1)):
            rs.step()
        times, its = [], None
        for _ in range(args.steps):
            t, its = rs.step()
            times.append(t)
        val = (1.0 / float(np.mean(times))) * rs.N / wl['N']
        grid, _, rcut = choose_params(wl, make_suspension(wl, seed=100)[1]) if rs.N != wl['N'] else (rs.grid, None, rs.rcut)
        L = synth_box(wl)
        config = {'workload': describe(args.workload, wl), 'N': wl['N'], 'phi': wl['phi'], 'tol': wl['tol'], 'xi': wl['xi'], 'dt': wl['dt'],
                  'grid': grid, 'rcut': round(rcut, 4), 'L': round(L, 4)}
        text = rs.describe(args.steps)
        line = dict(base, impl='reference', value=val, ms_per_step=1e3 / val, config=config,
                    run={'window': 'Gaussian (PAPER.md:263)', 'P': rs.P, 'lanczos_gmres_iters_last_step': list(its), 'N_timed': rs.N},
                    cpu_baseline={'value': val, 'unit': 'steps/s', 'cores': rs.cores, 'kind': 'oracle', 'tier': 'pse_reference', 'sample': text},
                    e2e={'value': val, 'unit': 'steps/s', 'h2d_bytes_per_step': 0, 'd2h_bytes_per_step': 0})
        line['dtype'] = 'f64'
        print(json.dumps(line))
        return

    if world > 1:
        import torch
        import torch.distributed as dist
        torch.cuda.set_device(int(os.environ.get('LOCAL_RANK', 0)))
        dist.init_process_group('nccl')
    r = run_ours(args, wl, rank, world)
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
        dist.destroy_process_group()
    if rank != 0:
        return
    line = dict(base, **assemble(args.workload, wl, r, args.steps, world, overridden))
    if args.workload == 'config3' and not overridden and world == 1 and not args.no_config4:
        # the large-N point the metric is quoted on (BASELINE.json configs[3]), measured in the same invocation
        wl4 = dict(WORKLOADS['config4'])
        a4 = argparse.Namespace(**dict(vars(args), steps=max(2, min(args.steps, 10)), warmup=3))
        r4 = run_ours(a4, wl4, rank, world)
        blk = assemble('config4', wl4, r4, a4.steps, world, False)
        blk.update(steps=a4.steps, warmup=a4.warmup)
        blk['hbm_fraction_per_kernel'] = {k: round(v['frac_of_hbm_peak'], 4) for k, v in blk['phases'].items() if 'frac_of_hbm_peak' in v}
        line['config4'] = blk
        # the headline workload once more in a sheared periodic cell (NEXT-4; Eq. 56 at strain 0.5, the largest a Lees-Edwards cell reaches)
        wls = dict(wl, shear=0.5)
        rsh = run_ours(a4, wls, rank, world)
        line['sheared_cell'] = {'strain': 0.5, 'value': replica_throughput(a4.steps, world, rsh['ms']), 'unit': 'steps/s', 'ms_per_step': rsh['ms'] / a4.steps,
                                'grid': rsh['grid'], 'P': rsh['P'], 'matvecs_per_sec': 1e3 / rsh['matvec_ms'], 'e2e_steps_per_sec': 1e3 / rsh['e2e_ms'],
                                'strain_advanced_every_step_steps_per_sec': 1e3 / rsh['flow_ms'],
                                'steps': a4.steps, 'warmup': a4.warmup}
    if not args.no_cpu_baseline and world == 1:          # the CPU baseline is reported at N = 1 only
        rs = ReferenceStepper(wl)
        sec, its = rs.step()
        if sec > 40.0:
            rs.shrink(sec / 20.0)
            sec, its = rs.step()
        line['cpu_baseline'] = {'value': (1.0 / sec) * rs.N / wl['N'], 'unit': 'steps/s', 'cores': rs.cores, 'kind': 'oracle', 'tier': 'pse_reference',
                                'sample': rs.describe(1), 'seconds_per_step': sec, 'lanczos_gmres_iters': list(its)}
        sec, Ns, cores, text = direct_oracle_sample(wl, 1)
        line['cpu_baseline_direct'] = {'value': (1.0 / sec) * Ns / wl['N'], 'unit': 'steps/s', 'cores': cores, 'kind': 'oracle', 'tier': 'direct O(N^2) sums',
                                       'sample': text, 'seconds_per_sample_step': sec}
    print(json.dumps(line))


def synth_box(wl):
    import synth
    return synth.box_length(wl['N'], wl['phi'])


if __name__ == '__main__':
    main()
