"""Seeded random problems (cells 1 ... 4000, S2 ... S64, all boundary kinds, shared and per-cell blocks) through the default
paths of oci_step and si_step against the oracle: whatever kernel family, one-launch step or scan variant oci_setup picks
for a shape must give the oracle's iterates (1e-12 at a fixed iteration count) and its iteration counts (converged)."""
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from workloads.configs import Problem  # noqa: E402

VAC, INC, REF = 0, 1, 2


def _rel(a, b):
    return np.max(np.abs(a - b)) / max(np.max(np.abs(b)), 1e-300)


def _random_problem(rng):
    N = int(rng.choice([2, 4, 6, 8, 12, 16, 32, 64]))
    J = int(rng.choice([1, 2, 3, 7, 15, 16, 17, 33, 64, 65, 100, 129, 255, 300, 513, 1000, 1500, 2049, 4000]))
    if J * N > 70000:
        J = max(1, 70000 // N)
    hetero = rng.random() < 0.25

    def bc():
        k = int(rng.choice([VAC, INC, REF]))
        return (k, float(rng.uniform(0.1, 2.0)) if k == INC else 0.0)

    if hetero:
        dx, st = rng.uniform(0.1, 1.0, J), rng.uniform(0.2, 4.0, J)
        ss = st * rng.uniform(0.1, 0.95, J)
    else:
        dx, st = np.full(J, rng.uniform(0.1, 1.0)), np.full(J, rng.uniform(0.5, 3.0))
        ss = st * rng.uniform(0.1, 0.95)
    q = rng.uniform(0, 1, (J, 4))
    return Problem(0, "fuzz", N, J, dx, st, ss, float(rng.uniform(0.5, 3.0)), float(rng.uniform(0.05, 1.0)), 2, bc(), bc(),
                   rng.uniform(0, 1, (J, N, 2)), _source=lambda step: q), q


@pytest.mark.gpu
@pytest.mark.parametrize("seed", [11, 12, 13])
def test_random_shapes_against_the_oracle(seed):
    import paper_2305_13555_b200 as P
    from oracle import Oracle, threads_available
    rng = np.random.default_rng(seed)
    for case in range(30):
        p, q = _random_problem(rng)
        for scheme in ("oci", "si"):
            for tol, max_iters in ((-1.0, 3), (1e-10, 100_000)):
                g, o = P.OCI.from_problem(p), Oracle.from_problem(p, threads=threads_available())
                what = dict(seed=seed, case=case, N=p.n_angles, J=p.cells, bc=(p.bc_left, p.bc_right), scheme=scheme, tol=tol, info=g.get_info())
                for k in range(2):
                    g.set_source(q)
                    o.set_source(q)
                    a = (g.oci_step if scheme == "oci" else g.si_step)(tol, max_iters)
                    b = (o.oci_step if scheme == "oci" else o.si_step)(tol, max_iters)
                    assert a[0] == b[0] and abs(a[1] - b[1]) <= (0 if tol < 0 else 1), (what, a, b)
                lim = 1e-12 if tol < 0 else 1e-8
                assert _rel(g.get_angular_flux(), o.angular_flux()) < lim, what
                assert _rel(g.get_scalar_flux(), o.scalar_flux()) < lim, what
                g.close()
