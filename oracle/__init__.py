"""oracle/ -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

A plain, slow, direct-summation CPU implementation of what the hot path of
arXiv:2402.01282 computes (scale-discretised directional wavelet transforms on
the sphere and the ball), written from the paper's definitions and the
readings listed in DESIGN.md.  It is independent of the CUDA path: it imports
nothing from paper_2402_01282_b200/, shares no code, header, table or constant
with it, and no expected value here ever comes from the GPU.

Only tests/, __graft_entry__.smoke() and bench.py's `cpu_baseline` /
`--impl reference` legs may import, build or call anything in this package.

Parity status: every function is pinned by tests/test_oracle_*.py
(closed forms, mpmath factorial sums, orthogonality, admissibility, brute-force
Eq. 16 sums, least squares, Gauss-Laguerre moments).  Nothing is "parity
unpinned".
"""
