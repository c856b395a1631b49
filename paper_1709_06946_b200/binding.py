"""ctypes binding of libpse.so — argument marshalling only; every step of the path runs in the CUDA library.

Function names mirror include/pse.h.  Tensors are torch CUDA tensors (torch is used for device memory and
streams only).  There is no CPU fallback: if libpse.so is missing or no CUDA device is present the calls raise.
"""
import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, 'libpse.so')

PSE_OK, PSE_EINVAL, PSE_ENOMEM, PSE_ECUDA, PSE_ECUFFT, PSE_ENOTREADY, PSE_ENOCONV, PSE_EOVERFLOW = range(8)
PSE_REAL, PSE_WAVE, PSE_BOTH = 1, 2, 3
PSE_WINDOW_GAUSS, PSE_WINDOW_ES = 0, 1
PSE_NOALLOC_MAX_N = 1 << 20
PHASES = ('neighbors', 'real', 'spread', 'fft_fwd', 'scale', 'fft_inv', 'interp', 'vector', 'pack')
_STATUS = {0: 'PSE_OK', 1: 'PSE_EINVAL', 2: 'PSE_ENOMEM', 3: 'PSE_ECUDA', 4: 'PSE_ECUFFT', 5: 'PSE_ENOTREADY',
           6: 'PSE_ENOCONV', 7: 'PSE_EOVERFLOW'}

EXPORTS = ('pse_suggest_params', 'pse_suggest_params_window', 'pse_suggest_params_lattice', 'pse_set_lattice', 'pse_create', 'pse_create_window', 'pse_destroy', 'pse_neighbors', 'pse_mobility_apply', 'pse_brownian',
           'pse_constrained_solve', 'pse_mobility_apply_full', 'pse_constrained_solve_full', 'pse_brownian_full', 'pse_step_full', 'pse_hard_sphere_forces', 'pse_hard_sphere_forces_noalloc', 'pse_set_bonds', 'pse_bond_forces', 'pse_step', 'pse_mobility_apply_host', 'pse_step_host', 'pse_get_neighbors', 'pse_set_profiling',
           'pse_get_timings', 'pse_kernel_launches', 'pse_get_table', 'pse_last_error', 'pse_version')


class PSEError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f'{_STATUS.get(status, status)}: {msg}')
        self.status = status


def load_library():
    if not os.path.exists(LIB_PATH):
        raise ImportError(f'{LIB_PATH} not found: build it with `python paper_1709_06946_b200/build.py` '
                          '(there is no CPU fallback)')
    lib = C.CDLL(LIB_PATH)
    vp, dbl, i32 = C.c_void_p, C.c_double, C.c_int
    lib.pse_suggest_params.argtypes = [i32, dbl, dbl, dbl, dbl, C.POINTER(i32), C.POINTER(i32), C.POINTER(dbl)]
    lib.pse_create.argtypes = [C.POINTER(vp), i32, dbl, dbl, dbl, dbl, dbl, i32, i32, dbl, dbl, vp]
    lib.pse_suggest_params_window.argtypes = [i32, dbl, dbl, dbl, dbl, i32, C.POINTER(i32), C.POINTER(i32), C.POINTER(dbl)]
    lib.pse_create_window.argtypes = [C.POINTER(vp), i32, dbl, dbl, dbl, dbl, dbl, i32, i32, dbl, dbl, i32, vp]
    lib.pse_suggest_params_lattice.argtypes = [i32, dbl, dbl, dbl, dbl, i32, dbl, dbl, dbl, C.POINTER(i32), C.POINTER(i32), C.POINTER(dbl)]
    lib.pse_set_lattice.argtypes = [vp, dbl, dbl, dbl]
    lib.pse_destroy.argtypes = [vp]
    lib.pse_neighbors.argtypes = [vp, vp]
    lib.pse_mobility_apply.argtypes = [vp, vp, vp, vp, vp, i32]
    lib.pse_brownian.argtypes = [vp, dbl, vp, vp, vp, vp, C.POINTER(i32)]
    lib.pse_constrained_solve.argtypes = [vp, vp, vp, vp, vp, vp, C.POINTER(i32)]
    lib.pse_hard_sphere_forces.argtypes = [vp, dbl, vp]
    lib.pse_mobility_apply_full.argtypes = [vp, vp, vp, vp, vp, vp, vp, i32]
    lib.pse_step_full.argtypes = [vp, vp, dbl, vp, vp, vp, vp, C.POINTER(i32), C.POINTER(i32)]
    lib.pse_brownian_full.argtypes = [vp, dbl, vp, vp, vp, vp, vp, C.POINTER(i32)]
    lib.pse_constrained_solve_full.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, C.POINTER(i32)]
    lib.pse_hard_sphere_forces_noalloc.argtypes = [i32, dbl, dbl, dbl, dbl, vp, vp, vp, C.c_char_p, C.c_size_t]
    lib.pse_set_bonds.argtypes = [vp, vp, i32, dbl, dbl]
    lib.pse_bond_forces.argtypes = [vp, vp]
    lib.pse_step.argtypes = [vp, vp, dbl, vp, vp, C.POINTER(i32), C.POINTER(i32)]
    lib.pse_mobility_apply_host.argtypes = [vp, vp, vp, vp, vp, vp]
    lib.pse_step_host.argtypes = [vp, vp, dbl, vp, vp, C.POINTER(i32), C.POINTER(i32)]
    lib.pse_get_neighbors.argtypes = [vp, vp, vp, C.c_size_t, C.POINTER(C.c_size_t)]
    lib.pse_set_profiling.argtypes = [vp, i32]
    lib.pse_get_timings.argtypes = [vp, C.POINTER(C.c_float), C.POINTER(i32), i32]
    lib.pse_kernel_launches.argtypes = [vp]
    lib.pse_kernel_launches.restype = C.c_longlong
    lib.pse_get_table.argtypes = [vp, vp, i32, C.POINTER(i32), C.POINTER(dbl)]
    lib.pse_last_error.argtypes = [vp]
    lib.pse_last_error.restype = C.c_char_p
    lib.pse_version.restype = C.c_char_p
    return lib


_lib = load_library()


def _ptr(t, shape=None, dtype=torch.float32):
    if t is None:
        return None
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.is_contiguous()):
        raise TypeError('expected a contiguous CUDA tensor')
    if t.dtype != dtype:
        raise TypeError(f'expected dtype {dtype}, got {t.dtype}')
    if shape is not None and tuple(t.shape) != tuple(shape):
        raise ValueError(f'expected shape {tuple(shape)}, got {tuple(t.shape)}')
    return C.c_void_p(t.data_ptr())


def _hptr(t, shape):
    if not (isinstance(t, torch.Tensor) and not t.is_cuda and t.is_contiguous() and t.dtype == torch.float32):
        raise TypeError('expected a contiguous float32 CPU tensor')
    if tuple(t.shape) != tuple(shape):
        raise ValueError(f'expected shape {tuple(shape)}, got {tuple(t.shape)}')
    return C.c_void_p(t.data_ptr())


def pse_version():
    return _lib.pse_version().decode()


def pse_suggest_params(N, L, a, tol, xi, window=PSE_WINDOW_ES, lattice=(1.0, 0.0, 1.0)):
    """-> (status, grid, P, rcut); see include/pse.h (pse_suggest_params_window / _lattice).  lattice = (a11, a12, a22)."""
    g, p, rc = C.c_int(), C.c_int(), C.c_double()
    st = _lib.pse_suggest_params_lattice(N, L, a, tol, xi, window, lattice[0], lattice[1], lattice[2], C.byref(g), C.byref(p), C.byref(rc))
    return st, g.value, p.value, rc.value


def pse_hard_sphere_forces_noalloc(L, a, eta, dt, pos, F, stream=None):
    """Heyes-Melrose overlap forces without a context and without any allocation (static device scratch; see include/pse.h).
    pos [N][4], F [N][3] CUDA float32 tensors on the current device; N <= PSE_NOALLOC_MAX_N."""
    N = int(pos.shape[0]) if isinstance(pos, torch.Tensor) and pos.dim() == 2 else -1
    msg = C.create_string_buffer(256)
    sp = C.c_void_p(stream.cuda_stream) if stream is not None else None
    st = _lib.pse_hard_sphere_forces_noalloc(N, L, a, eta, dt, _ptr(pos, (N, 4)), _ptr(F, (N, 3)), sp, msg, len(msg))
    if st != PSE_OK:
        raise PSEError(st, msg.value.decode())


class Context:
    """Owns a pse_ctx*.  Methods are one-to-one with the C calls of the same name."""

    def __init__(self, N, L, a, eta, kT, xi, grid, P, rcut, tol, stream=None, window=PSE_WINDOW_ES):
        self.N, self.L, self.grid, self.P = int(N), float(L), int(grid), int(P)
        self._h = C.c_void_p()
        # the library enqueues on this stream (NULL = legacy default stream, which torch's default stream is ordered with);
        # inputs produced on another torch stream must be ordered before the calls by the caller
        sp = C.c_void_p(stream.cuda_stream) if stream is not None else None
        st = _lib.pse_create_window(C.byref(self._h), N, L, a, eta, kT, xi, grid, P, rcut, tol, window, sp)
        if st != PSE_OK:
            msg = _lib.pse_last_error(self._h).decode() if self._h else 'allocation failed'
            if self._h:
                _lib.pse_destroy(self._h)
                self._h = C.c_void_p()
            raise PSEError(st, msg)

    def _check(self, st, allow=()):
        if st != PSE_OK and st not in allow:
            raise PSEError(st, _lib.pse_last_error(self._h).decode())
        return st

    def close(self):
        if getattr(self, '_h', None):
            _lib.pse_destroy(self._h)
            self._h = C.c_void_p()

    __del__ = close

    def pse_set_lattice(self, a11, a12, a22):
        """Deformed lattice A = [[a11, a12, 0], [0, a22, 0], [0, 0, 1]] (simple shear: (1, gamma, 1); extension: (eps, 0, 1/eps))."""
        self._check(_lib.pse_set_lattice(self._h, float(a11), float(a12), float(a22)))

    def pse_neighbors(self, pos):
        self._check(_lib.pse_neighbors(self._h, _ptr(pos, (self.N, 4))))

    def pse_mobility_apply(self, F, S, U, E, which=PSE_BOTH):
        N = self.N
        self._check(_lib.pse_mobility_apply(self._h, _ptr(F, (N, 3)), _ptr(S, (N, 5)), _ptr(U, (N, 3)), _ptr(E, (N, 5)), which))

    def pse_brownian(self, dt, noise_real, noise_wave, UB, EB, allow_noconv=False):
        N, M = self.N, self.grid
        it = C.c_int()
        self._check(_lib.pse_brownian(self._h, dt, _ptr(noise_real, (N, 8)), _ptr(noise_wave, (3, M, M, M // 2 + 1, 2)),
                                      _ptr(UB, (N, 3)), _ptr(EB, (N, 5)), C.byref(it)), (PSE_ENOCONV,) if allow_noconv else ())
        return it.value

    def pse_constrained_solve(self, F, UB, EB, U, S):
        N = self.N
        it = C.c_int()
        self._check(_lib.pse_constrained_solve(self._h, _ptr(F, (N, 3)), _ptr(UB, (N, 3)), _ptr(EB, (N, 5)),
                                               _ptr(U, (N, 3)), _ptr(S, (N, 5)), C.byref(it)))
        return it.value

    def pse_mobility_apply_full(self, F, Lq, S, U, W, E, which=PSE_BOTH):
        """[U; Omega; E] = M [F; L; S] (torque Lq [N][3] in, angular velocity W [N][3] out); any tensor may be None."""
        N = self.N
        self._check(_lib.pse_mobility_apply_full(self._h, _ptr(F, (N, 3)), _ptr(Lq, (N, 3)), _ptr(S, (N, 5)),
                                                 _ptr(U, (N, 3)), _ptr(W, (N, 3)), _ptr(E, (N, 5)), which))

    def pse_step_full(self, pos, dt, Lq, noise_real, noise_wave, W=None):
        """pse_step with external torques Lq [N][3] (or None); angular velocities to W [N][3] (or None).  -> (gmres, lanczos) iterations."""
        N, M = self.N, self.grid
        gi, li = C.c_int(), C.c_int()
        self._check(_lib.pse_step_full(self._h, _ptr(pos, (N, 4)), dt, _ptr(Lq, (N, 3)), _ptr(noise_real, (N, 8)),
                                       _ptr(noise_wave, (3, M, M, M // 2 + 1, 2)), _ptr(W, (N, 3)), C.byref(gi), C.byref(li)))
        return gi.value, li.value

    def pse_brownian_full(self, dt, noise_real, noise_wave, UB, WB, EB):
        """11-component Brownian slip: noise_real [N][11] (Ux..Uz, Ox..Oz, e1..e5), outputs UB, WB (Omega^B), EB."""
        N, M = self.N, self.grid
        it = C.c_int()
        self._check(_lib.pse_brownian_full(self._h, dt, _ptr(noise_real, (N, 11)), _ptr(noise_wave, (3, M, M, M // 2 + 1, 2)),
                                           _ptr(UB, (N, 3)), _ptr(WB, (N, 3)), _ptr(EB, (N, 5)), C.byref(it)))
        return it.value

    def pse_constrained_solve_full(self, F, Lq, UB, EB, U, W, S):
        N = self.N
        it = C.c_int()
        self._check(_lib.pse_constrained_solve_full(self._h, _ptr(F, (N, 3)), _ptr(Lq, (N, 3)), _ptr(UB, (N, 3)), _ptr(EB, (N, 5)),
                                                    _ptr(U, (N, 3)), _ptr(W, (N, 3)), _ptr(S, (N, 5)), C.byref(it)))
        return it.value

    def pse_hard_sphere_forces(self, dt, F):
        self._check(_lib.pse_hard_sphere_forces(self._h, dt, _ptr(F, (self.N, 3))))

    def pse_set_bonds(self, pairs, k, r0):
        """pairs: host int32 array-like (n, 2)."""
        import numpy as np
        p = np.ascontiguousarray(np.asarray(pairs, dtype=np.int32).reshape(-1, 2))
        self._check(_lib.pse_set_bonds(self._h, p.ctypes.data_as(C.c_void_p) if len(p) else None, len(p), float(k), float(r0)))

    def pse_bond_forces(self, F):
        self._check(_lib.pse_bond_forces(self._h, _ptr(F, (self.N, 3))))

    def pse_step(self, pos, dt, noise_real, noise_wave):
        N, M = self.N, self.grid
        gi, li = C.c_int(), C.c_int()
        self._check(_lib.pse_step(self._h, _ptr(pos, (N, 4)), dt, _ptr(noise_real, (N, 8)),
                                  _ptr(noise_wave, (3, M, M, M // 2 + 1, 2)), C.byref(gi), C.byref(li)))
        return gi.value, li.value

    def pse_mobility_apply_host(self, pos, F, S, U, E):
        """Host (CPU, ideally pinned) float32 tensors; copies are inside the call."""
        N = self.N
        self._check(_lib.pse_mobility_apply_host(self._h, _hptr(pos, (N, 4)), _hptr(F, (N, 3)), _hptr(S, (N, 5)),
                                                 _hptr(U, (N, 3)), _hptr(E, (N, 5))))

    def pse_step_host(self, pos, dt, noise_real, noise_wave):
        N, M = self.N, self.grid
        gi, li = C.c_int(), C.c_int()
        self._check(_lib.pse_step_host(self._h, _hptr(pos, (N, 4)), dt, _hptr(noise_real, (N, 8)),
                                       _hptr(noise_wave, (3, M, M, M // 2 + 1, 2)), C.byref(gi), C.byref(li)))
        return gi.value, li.value

    def pse_get_neighbors(self):
        """-> (count [N] int32 tensor, index [total] int32 tensor) in original particle numbering."""
        total = C.c_size_t()
        count = torch.empty(self.N, dtype=torch.int32, device='cuda')
        self._check(_lib.pse_get_neighbors(self._h, _ptr(count, dtype=torch.int32), None, 0, C.byref(total)))
        index = torch.empty(max(total.value, 1), dtype=torch.int32, device='cuda')
        self._check(_lib.pse_get_neighbors(self._h, _ptr(count, dtype=torch.int32), _ptr(index, dtype=torch.int32), index.numel(), C.byref(total)))
        return count, index[:total.value]

    def pse_set_profiling(self, on):
        self._check(_lib.pse_set_profiling(self._h, int(bool(on))))

    def pse_get_timings(self):
        n = len(PHASES)
        ms, cnt = (C.c_float * n)(), (C.c_int * n)()
        self._check(_lib.pse_get_timings(self._h, ms, cnt, n))
        return {PHASES[i]: (float(ms[i]), int(cnt[i])) for i in range(n)}

    def pse_kernel_launches(self):
        return int(_lib.pse_kernel_launches(self._h))

    def pse_get_table(self):
        import numpy as np
        n, dr = C.c_int(), C.c_double()
        self._check(_lib.pse_get_table(self._h, None, 0, C.byref(n), C.byref(dr)))
        tab = np.empty((n.value, 8), dtype=np.float32)
        self._check(_lib.pse_get_table(self._h, tab.ctypes.data_as(C.c_void_p), n.value, C.byref(n), C.byref(dr)))
        return tab, dr.value


def pse_create(N, L, a, eta, kT, xi, grid, P, rcut, tol, stream=None, window=PSE_WINDOW_ES):
    return Context(N, L, a, eta, kT, xi, grid, P, rcut, tol, stream, window)
