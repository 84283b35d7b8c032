"""CPU oracle for MB-SCB transient slab S_N transport with OCI and SI.

TEST INFRASTRUCTURE, NOT THE PRODUCT.  The arithmetic lives in
`mbscb_oracle.c` (plain C, fp64, written from the paper); this file is only a
ctypes loader.  Only tests/, `__graft_entry__.smoke()` and bench.py's
cpu_baseline / `--impl reference` legs may import it.  It shares no code with
`paper_2305_13555_b200/` and neither imports the other.
"""
from .mbscb import Oracle, gauss_legendre, A4, cell_matrix, lu_factor, lu_solve, threads_available  # noqa: F401
