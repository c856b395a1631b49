"""pse_hard_sphere_forces_noalloc (include/pse.h): the Heyes-Melrose overlap force with its linked-cell scratch in a static
__device__ array, for callers that cannot call cudaMalloc.  Checked against the existing path (pse_neighbors +
pse_hard_sphere_forces) and the oracle on calls in a row that share the scratch.  Collected last on purpose."""
import ctypes

import numpy as np
import pytest

import synth

A, ETA, DT = 1.0, 1.0 / (6.0 * np.pi), 1e-3
BAR = 1e-4                     # the bar of test_gpu_parity.test_hard_sphere_forces_match_oracle


def rel(a, b):
    a, b = np.asarray(a, dtype=np.float64), np.asarray(b, dtype=np.float64)
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def test_rejects_sizes_beyond_the_static_scratch_before_touching_the_gpu():
    import paper_1709_06946_b200 as pse
    lib = ctypes.CDLL(pse.LIB_PATH)
    lib.pse_hard_sphere_forces_noalloc.argtypes = [ctypes.c_int] + [ctypes.c_double] * 4 + [ctypes.c_void_p] * 3 + [ctypes.c_char_p, ctypes.c_size_t]
    msg = ctypes.create_string_buffer(256)
    dummy = ctypes.c_void_p(256)                             # never dereferenced: the argument checks come first
    st = lib.pse_hard_sphere_forces_noalloc(pse.PSE_NOALLOC_MAX_N + 1, 500.0, A, ETA, DT, dummy, dummy, None, msg, len(msg))
    assert st == pse.PSE_EOVERFLOW and b'PSE_NOALLOC_MAX_N = 1048576' in msg.value
    st = lib.pse_hard_sphere_forces_noalloc(100, 3.9, A, ETA, DT, dummy, dummy, None, msg, len(msg))
    assert st == pse.PSE_EINVAL and b'minimum image' in msg.value
    st = lib.pse_hard_sphere_forces_noalloc(0, 10.0, A, ETA, DT, dummy, dummy, None, None, 0)
    assert st == pse.PSE_EINVAL


def _cases():
    """(positions fp32 [N][3], L, what): three boxes whose cell grids differ, so that each call finds the other's leftovers."""
    out = []
    x, L = synth.rsa(20000, 0.30, seed=11)                   # 31 cells per side of edge just over 2a; compressed 5 %: many overlaps
    out.append(((x * 0.95).astype(np.float32), L * 0.95, 'dense'))
    x, L = synth.rsa(40, 0.25, seed=5)                       # 3 cells per side, FEWER particles than the call before,
    x, L = x * 0.9, L * 0.9                                  # positions unwrapped by whole boxes
    shift = np.random.default_rng(0).integers(-2, 3, size=x.shape)
    out.append(((x + shift * L).astype(np.float32), L, 'tiny'))
    x, L = synth.rsa(20000, 0.01, seed=3)                    # L = 203: the 64-cells-per-side cap (cells of 3.2 a); overlaps made
    u = np.random.default_rng(1).standard_normal((1000, 3))  # by moving 1000 particles next to their index neighbour
    x[1:2000:2] = (x[0:2000:2] + 1.7 * u / np.linalg.norm(u, axis=1, keepdims=True)) % L
    out.append((x.astype(np.float32), L, 'dilute'))
    return out


def _existing_path(pse, torch, pos, L):
    """pse_neighbors + pse_hard_sphere_forces on a context (which allocates); xi and grid do not enter this force."""
    N = pos.shape[0]
    xi = 0.5 * max(1.0, 28.0 / L)
    st, grid, P, rcut = pse.pse_suggest_params(N, L, A, 1e-3, xi)
    assert st == 0
    ctx = pse.pse_create(N, L, A, ETA, 1.0, xi, grid, P, rcut, 1e-3)
    ctx.pse_neighbors(pos)
    F = torch.empty(N, 3, device='cuda')
    ctx.pse_hard_sphere_forces(DT, F)
    out = F.cpu().numpy()
    ctx.close()
    return out


@pytest.mark.gpu
def test_no_alloc_entry_point_equals_the_existing_path_on_calls_in_a_row():
    import torch
    import paper_1709_06946_b200 as pse
    from oracle import pse_reference as pr
    cases, dev, want = _cases(), [], []
    for x32, L, what in cases:
        pos = torch.zeros(x32.shape[0], 4, device='cuda')
        pos[:, :3] = torch.from_numpy(x32).cuda()
        dev.append((pos, torch.full((x32.shape[0], 3), float('nan'), device='cuda')))
        want.append(_existing_path(pse, torch, pos, L))
        assert (np.abs(want[-1]).max(axis=1) > 0).sum() >= 10, what
        if what != 'tiny':                                   # the existing path itself, where the input needs no fp32 wrap
            assert rel(want[-1], pr.heyes_melrose(x32.astype(np.float64), L, A, ETA, DT)) < BAR, what

    # first call on this device in this process: looks up the address of the static array
    pse.pse_hard_sphere_forces_noalloc(cases[0][1], A, ETA, DT, dev[0][0], torch.empty_like(dev[0][1]))
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for (pos, F), (_, L, _) in zip(dev, cases):              # calls in a row on one stream, sharing the static scratch
        pse.pse_hard_sphere_forces_noalloc(L, A, ETA, DT, pos, F)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0              # the device's free memory did not move: nothing was allocated
    for (_, F), w, (_, _, what) in zip(dev, want, cases):
        g = F.cpu().numpy()
        assert np.isfinite(g).all(), what
        assert rel(g, w) < BAR, (what, rel(g, w))
        assert rel(g, w) < 1e-6, (what, rel(g, w))           # same per-pair terms; only the fp32 summation order differs
        assert np.array_equal(g != 0, w != 0), what          # the same particles overlap
        one = (np.abs(w).max(axis=1) > 0)
        assert one.sum() > 0

    # repeats agree bit for bit (fixed summation order), whatever the scratch held before
    (pos, F1), L = dev[0], cases[0][1]
    F1 = F1.clone()
    F2 = torch.empty_like(F1)
    pse.pse_hard_sphere_forces_noalloc(cases[1][1], A, ETA, DT, dev[1][0], dev[1][1])
    pse.pse_hard_sphere_forces_noalloc(L, A, ETA, DT, pos, F2)
    assert torch.equal(F1, F2)
    # a side stream
    s = torch.cuda.Stream()
    F3 = torch.empty_like(F1)
    torch.cuda.synchronize()
    with torch.cuda.stream(s):
        pse.pse_hard_sphere_forces_noalloc(L, A, ETA, DT, pos, F3, stream=s)
    s.synchronize()
    assert torch.equal(F1, F3)
    # beyond the maximum: a clear error, nothing launched
    n = pse.PSE_NOALLOC_MAX_N + 1
    with pytest.raises(pse.PSEError) as e:
        pse.pse_hard_sphere_forces_noalloc(500.0, A, ETA, DT, torch.zeros(n, 4, device='cuda'), torch.empty(n, 3, device='cuda'))
    assert e.value.status == pse.PSE_EOVERFLOW and 'exceeds the static scratch' in str(e.value)
