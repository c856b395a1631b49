"""CPU-only checks of the boundary: the C-ABI library loads, exports every symbol include/pse.h declares, its
host-side logic (parameter chooser, argument validation, no-GPU behaviour) works, and the multi-rank (replica)
aggregation of bench.py runs under gloo with world_size 2."""
import ctypes
import os
import re
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope='module')
def pse():
    sys.path.insert(0, ROOT)
    import __graft_entry__ as ge
    ge.build()
    import paper_1709_06946_b200 as pse
    return pse


def test_library_exports_every_declared_symbol(pse):
    hdr = open(os.path.join(ROOT, 'include', 'pse.h')).read()
    declared = set(re.findall(r'\b(pse_[a-z_]+)\s*\(', hdr))
    assert {'pse_create', 'pse_neighbors', 'pse_mobility_apply', 'pse_brownian', 'pse_step'} <= declared
    lib = ctypes.CDLL(pse.LIB_PATH)
    for name in declared:
        assert hasattr(lib, name), name
    assert declared == set(pse.EXPORTS)


def test_suggest_params_rules(pse):
    st, grid, P, rcut = pse.pse_suggest_params(64, 13.892, 1.0, 1e-3, 0.6)
    assert st == 0 and P == 4                       # exponential-of-semicircle window: P = ceil(-log10 tol) + 1
    assert abs(rcut - (np.sqrt(-np.log(1e-3)) / 0.6 + 1.0)) < 1e-12 and rcut <= 13.892 / 2
    n = grid
    for p in (2, 3, 5, 7):
        while n % p == 0:
            n //= p
    assert n == 1 and grid >= 1.07 * 2 * 0.6 * np.sqrt(-np.log(1e-3)) * 13.892 / np.pi
    # above 64 the cheapest measured cuFFT size is taken (profiles/r1_cufft_sizes.md): 90 -> 90, 320 -> 343, 97 -> 100
    assert pse.pse_suggest_params(65536, 97.084, 1.0, 1e-3, 0.5)[1] == 90
    assert pse.pse_suggest_params(65536, 97.084, 1.0, 1e-3, 0.55)[1] == 100
    assert pse.pse_suggest_params(65536, 97.084, 1.0, 1e-3, 0.575)[1] == 100        # bench.py's config3
    assert pse.pse_suggest_params(65536, 97.084, 1.0, 1e-3, 0.58)[1] == 108
    for tol, want in [(1e-2, 3), (1e-3, 4), (1e-4, 5)]:
        assert pse.pse_suggest_params(4096, 44.1, 1.0, tol, 0.5)[2] == want
    assert pse.pse_suggest_params(64, 13.892, 1.0, 1e-3, 0.3)[0] == pse.PSE_EINVAL      # rcut > L/2
    assert pse.pse_suggest_params(0, 13.892, 1.0, 1e-3, 0.6)[0] == pse.PSE_EINVAL


def test_suggest_params_on_deformed_lattices(pse):
    """pse_suggest_params_lattice (host only): the grid grows by the largest column norm of A, P stays, and the cutoff must fit the
    deformed cell in lattice coordinates (reading R22)."""
    base = pse.pse_suggest_params(4096, 44.1, 1.0, 1e-3, 0.5)
    assert pse.pse_suggest_params(4096, 44.1, 1.0, 1e-3, 0.5, lattice=(1.0, 0.0, 1.0)) == base
    st, grid, P, rcut = pse.pse_suggest_params(4096, 44.1, 1.0, 1e-3, 0.5, lattice=(1.0, 0.5, 1.0))
    assert st == 0 and P == base[2] and rcut == base[3]
    need = 1.07 * 2 * 0.5 * np.sqrt(-np.log(1e-3)) * 44.1 / np.pi
    assert grid >= need * np.sqrt(1.25) > base[1] * 0.999 and grid > base[1]
    st, grid2, _, _ = pse.pse_suggest_params(4096, 44.1, 1.0, 1e-3, 0.5, lattice=(1.25, 0.0, 0.8))
    assert st == 0 and grid2 >= need * 1.25
    assert pse.pse_suggest_params(4096, 44.1, 1.0, 1e-3, 0.5, lattice=(1.0, 0.0, 1.2))[0] == pse.PSE_EINVAL      # det A != 1
    assert pse.pse_suggest_params(64, 13.892, 1.0, 1e-3, 0.6, lattice=(1.0, 1.0, 1.0))[0] == pse.PSE_EINVAL      # 5.38 * sqrt2 > L/2


def test_create_validates_arguments_and_fails_loudly_without_gpu(pse):
    import torch
    eta = 1 / (6 * np.pi)
    bad = [dict(rcut=8.0), dict(rcut=1.5), dict(P=40), dict(grid=4), dict(N=0)]
    base = dict(N=64, L=13.892, a=1.0, eta=eta, kT=1.0, xi=0.6, grid=32, P=8, rcut=5.3, tol=1e-3)
    for b in bad:
        with pytest.raises(pse.PSEError) as e:
            pse.pse_create(**dict(base, **b))
        assert e.value.status == pse.PSE_EINVAL
    if not torch.cuda.is_available():
        with pytest.raises(pse.PSEError) as e:
            pse.pse_create(**base)
        assert e.value.status == pse.PSE_ECUDA and 'no CPU fallback' in str(e.value)


def _rank_main(rank, world, port, q):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR='127.0.0.1', MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group('gloo', rank=rank, world_size=world)
    sys.path.insert(0, ROOT)
    import bench
    ms = bench.max_over_ranks(10.0 + 5.0 * rank)
    dist.barrier()
    q.put((rank, ms, bench.replica_throughput(4, world, ms)))
    dist.destroy_process_group()


def test_replica_aggregation_gloo_world2():
    import torch.multiprocessing as mp
    ctx = mp.get_context('spawn')
    q = ctx.Queue()
    procs = [ctx.Process(target=_rank_main, args=(r, 2, 29571, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, val in res:
        assert ms == 15.0 and abs(val - 2 * 4 * 1e3 / 15.0) < 1e-9


def test_bench_algorithmic_bytes_formula():
    sys.path.insert(0, ROOT)
    import bench
    ab = bench.algorithmic_bytes(1000, 10, 20.0)
    assert ab['spread'] == 48 * 1000 + 32 * 1000 and ab['scale'] == 2 * 64 * 10 * 10 * 6
    pl = bench.planes_per_launch(7)
    assert abs(pl['spread'] - 46 / 9) < 1e-12 and abs(pl['interp'] - 51 / 10) < 1e-12 and abs(pl['scale'] - 100 / 10) < 1e-12
    assert ab['real'] == 80 * 1000 + 4 * 1000 * 20.0
