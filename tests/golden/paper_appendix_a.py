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


def G1_case1(r, a, xi):
    """First scalar function of M_UC for r > 2a.  g3 is printed there with the numerator ending "+ 18a - 45r^4";
    the r <= 2a print of the same coefficient ends "+ 18 a - 45 r", which is the dimensionally consistent one
    and is used here.  Equals -2 x the coefficient that Eq. (22) implies for the tensor form (A5) at a = 1 (SURVEY.md errata):
    pinned as  G1_printed = -2 R_G1  for r > 2a.  The r <= 2a case is garbled and not transcribed."""
    assert r > 2 * a
    c = [0.0,
         (-30 * r**4 * xi**4 + 15 * r**2 * xi**2 + 9) / (64 * SP * a**4 * r**3 * xi**5),
         (3 * xi**2 * (2 * a - r) * (8 * a**2 + 16 * a * r + 25 * r**2)
          - 6 * xi**4 * (2 * a - r) * (32 * a**4 + 32 * a**3 * r + 44 * a**2 * r**2 + 36 * a * r**3 + 25 * r**4)
          - 9 * (2 * a + 5 * r)) / (640 * SP * a**4 * r**4 * xi**5),
         (-3 * xi**2 * (2 * a + r) * (8 * a**2 - 16 * a * r + 25 * r**2)
          + 6 * xi**4 * (2 * a + r) * (32 * a**4 - 32 * a**3 * r + 44 * a**2 * r**2 - 36 * a * r**3 + 25 * r**4)
          + 18 * a - 45 * r) / (640 * SP * a**4 * r**4 * xi**5),
         (60 * r**6 * xi**6 + 9 * r**2 * xi**2 + 9) / (128 * a**4 * r**4 * xi**6),
         -3 * (512 * a**6 * xi**6 + 5 * r**2 * xi**2 * (64 * a**4 * xi**4 + 3) - 256 * a * r**5 * xi**6 + 100 * r**6 * xi**6 + 15)
         / (1280 * a**4 * r**4 * xi**6),
         -3 * (512 * a**6 * xi**6 + 5 * r**2 * xi**2 * (64 * a**4 * xi**4 + 3) + 256 * a * r**5 * xi**6 + 100 * r**6 * xi**6 + 15)
         / (1280 * a**4 * r**4 * xi**6)]
    return _combine(c, r, a, xi)


def K3(r, a, xi):
    """Third scalar function of M_DC, PAPER.md:723 (case 1, r > 2a) and PAPER.md:737 (case 2, r <= 2a); the two cases differ in
    k0 only.  Equals (R_Z2 + R_Z4)/7 (the combination C of SURVEY.md 8(c) O2) at a = 1."""
    k0 = 0.0 if r > 2 * a else 9 * (4 * a**2 - r**2)**3 * (4 * a**2 + r**2) / (512 * a**6 * r**5)
    k56 = 9 * (16 * xi**8 * (r**2 - 4 * a**2)**3 * (4 * a**2 + r**2) + 24 * r**2 * xi**4 * (12 * a**2 + r**2)
               - 48 * xi**2 * (10 * a**2 + r**2) + 45) / (16384 * a**6 * r**5 * xi**8)
    c = [k0,
         9 * (32 * a**2 * xi**2 * (-2 * r**4 * xi**4 + r**2 * xi**2 + 15) + 8 * r**6 * xi**6 - 4 * r**4 * xi**4 + 18 * r**2 * xi**2 - 45)
         / (4096 * SP * a**6 * r**4 * xi**7),
         9 * (-8 * xi**6 * (r - 2 * a)**2 * (2 * a + r)**3 * (4 * a**2 + r**2) + 4 * xi**4 * (2 * a + r)**3 * (4 * a**2 + r**2)
              - 6 * xi**2 * (2 * a + r)**2 * (2 * a + 3 * r) + 45 * (r - 2 * a)) / (8192 * SP * a**6 * r**5 * xi**7),
         9 * (-8 * xi**6 * (r - 2 * a)**3 * (2 * a + r)**2 * (4 * a**2 + r**2) + 4 * xi**4 * (r - 2 * a)**3 * (4 * a**2 + r**2)
              + 6 * xi**2 * (r - 2 * a)**2 * (2 * a - 3 * r) + 45 * (2 * a + r)) / (8192 * SP * a**6 * r**5 * xi**7),
         9 * (8 * xi**2 * (4 * a**2 * (4 * r**6 * xi**6 - 9 * r**2 * xi**2 + 15) - 2 * r**8 * xi**6 - 3 * r**4 * xi**2 + 6 * r**2) - 45)
         / (8192 * a**6 * r**5 * xi**8),
         k56, k56]
    return _combine(c, r, a, xi)


def self_DC_bracket(a, xi):
    """The bracket of Eq. (A12), PAPER.md:744 (= K1(r -> 0)); carries a stray 1/a (SURVEY.md errata), invisible at a = 1.
    On a symmetric traceless S the tensor (dd + dd - 4dd) acts as -3, so  R_Z0(0)/5 = -3 x bracket  at a = 1."""
    return (-3 * (6 * a**2 * xi**2 + 1) / (80 * SP * a**6 * xi**3) + 3 * (10 * a**2 * xi**2 + 1) / (80 * SP * a**6 * xi**3) * np.exp(-4 * a**2 * xi**2)
            - 3 / (10 * a**3) * erfc(2 * a * xi))
