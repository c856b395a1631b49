"""CPU fp64 oracle for the PSE grand-mobility path of arxiv 1709.06946 (Fiore & Swan).

TEST INFRASTRUCTURE ONLY.  Nothing under ``paper_1709_06946_b200/`` (the CUDA product path) imports,
links or calls this package, and this package imports nothing from the product path.  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may use it.

It is a plain, slow, obviously-correct statement of what the path computes:

* ``functions``  – shape factors, Hasimoto splitting function, the seven real-space scalar functions
                   (free-space closed form minus a Gaussian-damped 1-D wave integral; SURVEY.md §8(c) O2,
                   replacing the garbled Appendix A of PAPER.md:589-744).
* ``mobility``   – direct O(N^2) Ewald sums of Eqs. (21)-(27): dense 8N x 8N assembly,
                   and row-sampled application for larger N.
* ``brownian``   – Eq. (71)/(74)/(76) sample: principal square root of the dense
                   real-space matrix plus the direct non-uniform sum of the wave-space factor over the
                   grid's wave vectors; the mid-point step Eqs. (76)-(79); the bond force of
                   the equilibrium test potential U = k|r - r0| and Eq. (80); the constrained
                   mobility R_FU^-1 of Eq. (B15) and its divergence, the drift of Eq. (B12).
* ``neighbors``  – brute-force fp32 neighbour sets.
* ``pse_reference`` (+ ``pse_ref.c``, ``krylov``) – second tier: the paper's own fast scheme in fp64 (linked-cell pair sum,
                   Gaussian NUFFT of Eq. 42 with scipy's FFT, textbook Lanczos / GMRES), pinned against the direct sums at
                   N <= 4 096; the parity reference at N >= 65 536 and bench.py's second timed CPU baseline.

* ``couplet``    – the full couplet of Eq. (31): torque in, angular velocity out, 11N x 11N matrix, constrained
                   solve and mid-point step with torques, 11-component Brownian sample (reading R21).  Pins C1-C10
                   (tests/test_oracle_couplet.py): exact periodic rotational self-mobility, textbook pair forms incl. overlap,
                   xi-independence per block, SPD, covariance identity of the wave factor, reduction to the 8-component step.
* ``lattice``    – deformed periodic cells (reading R22): Eqs. (55)-(59), direct sums with lattice vectors L A,
                   fp32 neighbour sets, Brownian sample, and ``LatticeReference``, the NUFFT tier in lattice coordinates.
                   Pins L1-L8 (tests/test_oracle_lattice.py): Table I as printed (tests/golden/paper_table1.py), identity
                   lattice, lattice equivalence gamma -> gamma +- 1, a rectangular box written out by hand, xi-independence, SPD,
                   covariance identity of the sheared wave factor, the reference tier against the direct sums.

Pins (tests/test_oracle_*.py, ``-m "not gpu"``): Hasimoto periodic self-mobility, xi-independence of
M_r + M_w, symmetry and positive-definiteness of M, M_r, M_w, textbook RPY / RPY-overlap free-space
limits, printed closed forms F1, F2 of Appendix A, exact covariance identity
A_w A_w^T = M_w(grid modes), Schur-complement constraint solve, bond force = -grad U, Eq. (80) normalised
Boltzmann density, a short two-sphere run against Eq. (80), div M_UF = 0, printed K3 / G1 (r > 2a) / (A12)
(PAPER.md:670, 723, 737, 744), the mid-point step written out by hand from the dense matrices, the Brownian amplitude
against its dense factors, and the Heyes-Melrose force (not in the paper; reading R12) by the property that defines it:
a free-draining pair ends at contact after one dt.  The PSE reference is pinned in tests/test_pse_reference.py.

Parity unpinned: none of the functions on the timed path; the RSA / aggregate generators live in synth/ (no method
arithmetic) and are checked only for "no overlaps".
"""
