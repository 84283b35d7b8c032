"""bench.py's tuned CPU leg (numpy + BLAS restatement of the interface-reduced iteration, reported next to the plain
oracle so that the GPU/CPU ratio is not inflated by the oracle's deliberate slowness) must compute the method: same
iteration counts and fluxes as the oracle on small versions of the shared-block configs."""
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from oracle import Oracle  # noqa: E402
from workloads import make_problem  # noqa: E402


@pytest.mark.parametrize("cfg,cells", [(1, 20), (2, 50), (3, 60), (4, 12)])
def test_cpu_blas_leg_matches_the_oracle(cfg, cells):
    import bench
    p = make_problem(cfg, cells=cells)
    c, o = bench.CpuBlasReduced(p), Oracle.from_problem(p)
    for k in range(3):
        o.set_source(p.source(k))
        assert c.step(p.source(k), p.tol, p.max_iters) == o.oci_step(p.tol, p.max_iters)[1]
        ref = o.angular_flux().reshape(cells, -1)
        assert np.max(np.abs(c.Psi - ref)) < 1e-12 * np.max(np.abs(ref))
        assert np.max(np.abs(c.phi - o.scalar_flux())) < 1e-12 * np.max(np.abs(ref))
