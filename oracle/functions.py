"""Scalar building blocks of the oracle (fp64, numpy/scipy).  Test infrastructure only.

Notation follows PAPER.md / SURVEY.md §8:  s0(x) = sin x / x  and  s1(x) = 3 (sin x - x cos x)/x^3 are the
U/F and D/C shape factors; H(k, xi) = (1 + k^2/4xi^2) exp(-k^2/4xi^2) is Hasimoto's
splitting function (Eq. 28).
"""
import numpy as np
from scipy.special import spherical_jn

SQ2 = np.sqrt(2.0)
SQ6 = np.sqrt(6.0)


def basis():
    """Orthonormal basis e^1..e^5 of symmetric traceless 3x3 tensors (e^p : e^q = delta_pq).

    (xx-yy)/sqrt2, (2zz-xx-yy)/sqrt6, (xy+yx)/sqrt2, (xz+zx)/sqrt2, (yz+zy)/sqrt2  — DESIGN.md reading R9
    (the paper only says the stresslet has 5 independent components).
    """
    e = np.zeros((5, 3, 3))
    e[0, 0, 0], e[0, 1, 1] = 1 / SQ2, -1 / SQ2
    e[1, 0, 0], e[1, 1, 1], e[1, 2, 2] = -1 / SQ6, -1 / SQ6, 2 / SQ6
    e[2, 0, 1] = e[2, 1, 0] = 1 / SQ2
    e[3, 0, 2] = e[3, 2, 0] = 1 / SQ2
    e[4, 1, 2] = e[4, 2, 1] = 1 / SQ2
    return e


def to_tensor(s5):
    """5 coordinates (..., 5) -> symmetric traceless tensors (..., 3, 3)."""
    return np.einsum('...q,qij->...ij', np.asarray(s5, dtype=np.float64), basis())


def to_coords(T):
    """Symmetric traceless tensors (..., 3, 3) -> 5 coordinates (..., 5):  s^q = e^q : T."""
    return np.einsum('...ij,qij->...q', np.asarray(T, dtype=np.float64), basis())


def s0(x):
    """sin x / x."""
    return spherical_jn(0, x)


def s1(x):
    """3 (sin x - x cos x) / x^3 = 3 j1(x)/x; -> 1 as x -> 0."""
    x = np.asarray(x, dtype=np.float64)
    out = np.ones_like(x)
    nz = np.abs(x) > 1e-8
    out[nz] = 3.0 * spherical_jn(1, x[nz]) / x[nz]
    return out


def hasimoto_H(k, xi):
    """Eq. (28)."""
    q = k * k / (4.0 * xi * xi)
    return (1.0 + q) * np.exp(-q)


def _jl_over_x(l, x):
    """j_l(x)/x with the x -> 0 limit (1/3 for l=1, 0 for l>=2)."""
    x = np.asarray(x, dtype=np.float64)
    out = np.full_like(x, 1.0 / 3.0 if l == 1 else 0.0)
    nz = np.abs(x) > 1e-12
    out[nz] = spherical_jn(l, x[nz]) / x[nz]
    return out


NAMES = ('F1', 'F2', 'G1', 'G2', 'Z0', 'Z2', 'Z4')


def free_space(r, a):
    """Free-space (H == 1) scalar functions, in units of 1/(6 pi eta a).  SURVEY.md §8(c) O2.

    For r > 2a these are the Rotne-Prager / Faxen forms (1 + a^2/3 lap) J etc.; for r <= 2a the overlap
    forms (F1, F2: Rotne-Prager-Yamakawa).  rho = r/a; G carries 1/a and Z carries 1/a^2.
    """
    rho = np.asarray(r, dtype=np.float64) / a
    far = rho > 2.0
    rf = np.where(far, rho, 3.0)         # dummy 3.0 keeps the unused branch finite
    out = {}
    out['F1'] = np.where(far, 3 / (4 * rf) + 1 / (2 * rf**3), 1 - 9 * rho / 32)
    out['F2'] = np.where(far, 3 / (2 * rf) - 1 / rf**3, 1 - 3 * rho / 16)
    out['G1'] = np.where(far, 3 * (5 * rf**2 + 8) / (20 * rf**4), 3 * rho * (64 - 25 * rho) / 320) / a
    out['G2'] = np.where(far, -3 * (5 * rf**2 - 8) / (20 * rf**4), 3 * rho * (5 * rho - 16) / 320) / a
    out['Z0'] = np.where(far, 0.0, 9 * (rho - 2)**2 * (rho + 4) / 32) / a**2
    out['Z2'] = np.where(far, 9 / (2 * rf**3), -9 * rho * (rho**2 - 6) / 64) / a**2
    out['Z4'] = np.where(far, 9 * (5 * rf**2 - 14) / (4 * rf**5), 9 * rho * (rho**2 + 8) / 512) / a**2
    return out


def wave_integrals(r, xi, a, order=16, decay=50.0):
    """Gaussian-damped wave integrals W_X(r; xi): the inverse Fourier transforms of
    the summands of Eqs. (21)-(24) over all of k-space, angular part done with
    <exp(ik.r) khat...khat> -> spherical Bessel j_l(kr).  Panelled Gauss-Legendre on [0, 2 xi sqrt(decay)].

    W_F1 = (3a/pi) int dk H s0^2 [j0(kr) - j1(kr)/kr]        W_F2 = (3a/pi) int dk H s0^2 2 j1(kr)/kr
    W_G1 = (3a/pi) int dk k H s0 s1 [j1(kr) - j2(kr)/kr]     W_G2 = -(3a/pi) int dk k H s0 s1 j2(kr)/kr
    W_Zl = (3a/pi) int dk k^2 H s1^2 j_l(kr),  l = 0, 2, 4
    """
    r = np.atleast_1d(np.asarray(r, dtype=np.float64))
    kmax = 2.0 * xi * np.sqrt(decay)
    rmax = float(r.max()) if r.size else 0.0
    npanel = int(np.ceil(kmax * (rmax + 2 * a) / np.pi)) + 8
    xg, wg = np.polynomial.legendre.leggauss(order)
    edges = np.linspace(0.0, kmax, npanel + 1)
    half = 0.5 * (edges[1:] - edges[:-1])
    mid = 0.5 * (edges[1:] + edges[:-1])
    k = (mid[:, None] + half[:, None] * xg[None, :]).ravel()
    w = (half[:, None] * wg[None, :]).ravel()
    Hk = hasimoto_H(k, xi)
    c00 = w * Hk * s0(k * a)**2
    c01 = w * Hk * k * s0(k * a) * s1(k * a)
    c11 = w * Hk * k * k * s1(k * a)**2
    pref = 3.0 * a / np.pi
    out = {n: np.empty_like(r) for n in NAMES}
    chunk = max(1, 4_000_000 // k.size)
    for lo in range(0, r.size, chunk):
        x = r[lo:lo + chunk, None] * k[None, :]
        sl = slice(lo, lo + chunk)
        j0, j1, j2, j4 = (spherical_jn(l, x) for l in (0, 1, 2, 4))
        j1x, j2x = _jl_over_x(1, x), _jl_over_x(2, x)
        out['F1'][sl] = pref * ((j0 - j1x) @ c00)
        out['F2'][sl] = pref * ((2 * j1x) @ c00)
        out['G1'][sl] = pref * ((j1 - j2x) @ c01)
        out['G2'][sl] = -pref * (j2x @ c01)
        out['Z0'][sl] = pref * (j0 @ c11)
        out['Z2'][sl] = pref * (j2 @ c11)
        out['Z4'][sl] = pref * (j4 @ c11)
    return out


def real_space_functions(r, xi, a):
    """R_X(r) = Free_X(r) - W_X(r; xi): the scalar functions of M^(r), Eqs. (25)-(27),
    in the parametrisation of SURVEY.md §8(c) O2 (Appendix A of the paper is garbled)."""
    fr, wv = free_space(r, a), wave_integrals(r, xi, a)
    return {n: np.atleast_1d(fr[n]) - wv[n] for n in NAMES}


def rank4_combinations(R):
    """A, B, C, D of SURVEY.md §8(c) O2 from R_Z0, R_Z2, R_Z4 (Bessel recurrences)."""
    j1x = (R['Z0'] + R['Z2']) / 3.0
    j3x = (R['Z2'] + R['Z4']) / 7.0
    j2xx = (j1x + j3x) / 5.0
    return j1x - 2.0 * j2xx, 2.0 * j3x - R['Z2'] / 2.0, j3x, -R['Z4']
