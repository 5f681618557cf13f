"""CPU ORACLE for the DGFS collision operator of arXiv 1903.04670 -- TEST INFRASTRUCTURE ONLY.

Plain, slow, numpy fp64.  Follows the paper step by step (PAPER.md Algo 1 P:166-212,
Algo 2 P:219-244, Eq. 1-23) in the paper's order and notation; library primitives used as
steps: numpy.fft (FFT), numpy.polynomial.legendre.leggauss (Gauss-Legendre nodes),
scipy.special.roots_jacobi / j0 (VSS angular integral).  No blocking, fusion or reordering.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It shares no code with the CUDA path (paper_1903_04670_b200/) and
neither imports the other.

Pins (tests/test_oracle_*.py, `-m "not gpu"`): brute-force wrapped Galerkin sum (Eq. 11+13),
exact-kernel Galerkin sum (Eq. 12), closed-form Krook-Wu solution and printed Table 1 errors
(P:263-327), Table 2 Knudsen numbers, table closed forms, shift/permutation/
bilinearity invariants, shift identity of Eq. 8, conservation and Maxwellian-null trends.
Parity-unpinned functions: none for the collision path.  dg.py (readings DG-1..3, the paper
gives no formulas) is PARITY-UNPINNED against the paper and pinned only by textbook properties
(tests/test_oracle_dg.py) -- see its header.
"""
