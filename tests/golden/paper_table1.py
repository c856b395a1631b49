"""Numbers exactly as PRINTED in the paper's section on deformed FFT grids (restated from /root/reference/PAPER.md; used only as pins
for oracle/lattice.py, never by the product path).

TABLE I: "Maximum eigenvalue of A^T A for different values of gamma for both simple shear and planar extensional
lattice deformations.  The Gaussian kernel support size for an error bound of 1e-3 is also reported."
The row gamma = 0.5 prints lambda_ext = 2.25 without its epsilon (the extraction lost it; 2.25 = 1.5^2 by Eq. 59) and without P_ext.
"""

# (gamma, lambda_max^shear, P_shear)
SHEAR_ROWS = ((0.0, 1.00, 5), (0.1, 1.11, 6), (0.5, 1.64, 7), (1.0, 2.62, 8))
# (epsilon, lambda_max^ext, P_ext or None)
EXTENSION_ROWS = ((1.0, 1.00, 5), (1.1, 1.21, 6), (1.5, 2.25, None), (2.0, 4.00, 10))

# "if simulation parameters were chosen to satisfy a tolerance of 1e-3 with gamma = 0.5 (epsilon = 0.5) using the bounds
# for orthorhombic lattice ..., the actual expected error would be (1e-3)^(1/lambda_max^shear) = 0.015 for simple shear and ... = 0.046
# for planar extension"  (the second uses lambda = 2.25, the value printed in the gamma = 0.5 row)
EXPECTED_ERROR_SHEAR_G05 = 0.015
EXPECTED_ERROR_EXT = 0.046
