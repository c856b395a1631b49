"""Closed forms exactly as PRINTED in Appendix A of the paper (cited line by line) — used only as pins for the
oracle's quadrature-based real-space functions.  Restated from /root/reference/PAPER.md; never used by the
product path.  Only the items the survey found sound are here (F1, F2, G2, self term A4); G1 case 2, K1, K2 are
garbled in the extraction (SURVEY.md §8(c) errata) and are not transcribed.
"""
import numpy as np
from scipy.special import erfc

SP = np.sqrt(np.pi)


def _combine(c, r, a, xi):
    """Eq. (A2) / (A6)."""
    return (c[0] + c[1] * np.exp(-r**2 * xi**2) + c[2] * np.exp(-(r - 2 * a)**2 * xi**2)
            + c[3] * np.exp(-(r + 2 * a)**2 * xi**2) + c[4] * erfc(r * xi)
            + c[5] * erfc((r - 2 * a) * xi) + c[6] * erfc((r + 2 * a) * xi))


def F1(r, a, xi):
    """PAPER.md:617 (case 1, r > 2a) and PAPER.md:628 (case 2, r <= 2a)."""
    c = [0.0 if r > 2 * a else -(r - 2 * a)**2 * (4 * a**2 + 4 * a * r + 9 * r**2) / (32 * a * r**3),
         (18 * r**2 * xi**2 + 3) / (64 * SP * a * r**2 * xi**3),
         (2 * xi**2 * (2 * a - r) * (4 * a**2 + 4 * a * r + 9 * r**2) - 2 * a - 3 * r) / (128 * SP * a * r**3 * xi**3),
         (-2 * xi**2 * (2 * a + r) * (4 * a**2 - 4 * a * r + 9 * r**2) + 2 * a - 3 * r) / (128 * SP * a * r**3 * xi**3),
         (3 - 36 * r**4 * xi**4) / (128 * a * r**3 * xi**4),
         (4 * xi**4 * (r - 2 * a)**2 * (4 * a**2 + 4 * a * r + 9 * r**2) - 3) / (256 * a * r**3 * xi**4),
         (4 * xi**4 * (2 * a + r)**2 * (4 * a**2 - 4 * a * r + 9 * r**2) - 3) / (256 * a * r**3 * xi**4)]
    return _combine(c, r, a, xi)


def F2(r, a, xi):
    """PAPER.md:621 (case 1) and PAPER.md:632 (case 2)."""
    c = [0.0 if r > 2 * a else (2 * a - r)**3 * (2 * a + 3 * r) / (16 * a * r**3),
         (6 * r**2 * xi**2 - 3) / (32 * SP * a * r**2 * xi**3),
         (-2 * xi**2 * (r - 2 * a)**2 * (2 * a + 3 * r) + 2 * a + 3 * r) / (64 * SP * a * r**3 * xi**3),
         (2 * xi**2 * (2 * a + r)**2 * (2 * a - 3 * r) - 2 * a + 3 * r) / (64 * SP * a * r**3 * xi**3),
         -3 * (4 * r**4 * xi**4 + 1) / (64 * a * r**3 * xi**4),
         (3 - 4 * xi**4 * (2 * a - r)**3 * (2 * a + 3 * r)) / (128 * a * r**3 * xi**4),
         (3 - 4 * xi**4 * (2 * a - 3 * r) * (2 * a + r)**3) / (128 * a * r**3 * xi**4)]
    return _combine(c, r, a, xi)


def G2(r, a, xi):
    """PAPER.md:674 (case 1) and PAPER.md:680 (case 2).  Equals 2 x the coefficient that Eq. (22) implies for
    the tensor form (A5) at a = 1 (SURVEY.md errata): pinned as  G2_printed = 2 R_G2."""
    p5 = 16 * a**3 + 24 * a**2 * r + 14 * a * r**2 + 5 * r**3
    m5 = 16 * a**3 - 24 * a**2 * r + 14 * a * r**2 - 5 * r**3
    c = [0.0 if r > 2 * a else -3 * (128 * a**6 - 80 * a**4 * r**2 + 16 * a * r**5 - 5 * r**6) / (160 * a**4 * r**4),
         (-6 * r**4 * xi**4 + 3 * r**2 * xi**2 - 9) / (64 * SP * a**4 * r**3 * xi**5),
         (6 * xi**4 * (r - 2 * a)**2 * p5 - 3 * xi**2 * p5 + 18 * a + 45 * r) / (640 * SP * a**4 * r**4 * xi**5),
         (-6 * xi**4 * (2 * a + r)**2 * m5 + 3 * xi**2 * m5 - 18 * a + 45 * r) / (640 * SP * a**4 * r**4 * xi**5),
         (12 * r**6 * xi**6 + 9 * r**2 * xi**2 - 9) / (128 * a**4 * r**4 * xi**6),
         (12 * xi**6 * (128 * a**6 - 80 * a**4 * r**2 + 16 * a * r**5 - 5 * r**6) - 45 * r**2 * xi**2 + 45) / (1280 * a**4 * r**4 * xi**6),
         (12 * xi**6 * (128 * a**6 - 80 * a**4 * r**2 - 16 * a * r**5 - 5 * r**6) - 45 * r**2 * xi**2 + 45) / (1280 * a**4 * r**4 * xi**6)]
    return _combine(c, r, a, xi)


def self_UF(a, xi):
    """Eq. (A4)."""
    return (1 - np.exp(-4 * a**2 * xi**2) + 4 * SP * a * xi * erfc(2 * a * xi)) / (4 * SP * xi * a)


# Hasimoto's periodic self-mobility of a point force on a simple cubic lattice, with the finite-size Faxen term:
# 6 pi eta a mu = 1 - 2.8372974795 a/L + (4 pi/3)(a/L)^3 (Hasimoto 1959, ref. 18 of the paper).
HASIMOTO_C = 2.8372974795
