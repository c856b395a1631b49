"""Seeded synthetic inputs shared by the oracle tests, the GPU parity tests and bench.py.

Holds none of the method's arithmetic: only particle placement (random sequential addition, fractal
aggregates) and Philox Gaussian vectors.  Stands in for the paper's "random suspensions of hard spheres"
(PAPER.md:559, 569); recipe in DESIGN.md.
"""
from .suspensions import box_length, rsa, relax_overlaps, fractal_aggregates  # noqa: F401
from .noise import gaussian_inputs, brownian_noise  # noqa: F401
