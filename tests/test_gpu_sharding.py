"""Row f4 on one GPU: W shards of one slab held in one process and stepped together (the launches of the shards are
interleaved on one stream, so every pull is ordered behind all pushes: the single-device emulation the profiling guide
asks for) must reproduce the UNSHARDED run of the same library bit for bit - the per-cell arithmetic does not depend
on which shard a cell lives in and the stopping rule is a maximum, which is exact - with the same iteration counts;
and that unsharded run is held to the oracle by tests/test_gpu_parity.py (one case is checked against it here too)."""
import numpy as np
import pytest

from workloads import make_problem

pytestmark = pytest.mark.gpu
VAC, INC, REF = 0, 1, 2


def _run_unsharded(p, steps, tol, max_iters):
    import paper_2305_13555_b200 as P
    # the three-pass kernels the shards run (a small unsharded slab would otherwise take the one-launch step, whose sums
    # run in another order)
    g = P.OCI.from_problem(p, iteration=P.ITERATION_REDUCED, small_step=0)
    its = []
    for k in range(steps):
        g.set_source(p.source(k))
        its.append(g.oci_step(tol, max_iters)[:2])
    out = (its, g.get_angular_flux(), g.get_scalar_flux(), g.get_info()["reduced_kernel"])
    g.close()
    return out


def _run_sharded(p, world, steps, tol, max_iters):
    from paper_2305_13555_b200.sharding import ShardedOCI
    s = ShardedOCI.local(p, world)
    its = []
    for k in range(steps):
        s.set_source(k)
        its.append(s.step(tol, max_iters)[:2])
    out = (its, s.get_angular_flux(), s.get_scalar_flux())
    s.close()
    return out


def _custom(J, N, bcL, bcR, seed, hetero):
    from workloads.configs import Problem
    rng = np.random.default_rng(seed)
    if hetero:
        dx, st = rng.uniform(0.1, 1.0, J), rng.uniform(0.2, 4.0, J)
        ss = st * rng.uniform(0.1, 0.95, J)
    else:
        dx, st, ss = np.full(J, 0.37), np.full(J, 1.7), np.full(J, 1.1)
    q = rng.uniform(0, 1, (J, 4))
    return Problem(0, "custom", N, J, dx, st, ss, 1.3, 0.13, 3, bcL, bcR, rng.uniform(0, 1, (J, N, 2)), _source=lambda step: q)


@pytest.mark.parametrize("world", [2, 3])
@pytest.mark.parametrize("J,N,bcL,bcR,hetero", [
    (40, 4, (INC, 1.0), (VAC, 0.0), False),       # GEMV kernels, shared block
    (301, 16, (REF, 0.0), (VAC, 0.0), False),     # resident kernels (config-2 block size), mirror at one end
    (500, 32, (REF, 0.0), (REF, 0.0), False),     # resident kernels (config-3 block size), mirrors at both ends
    (200, 64, (VAC, 0.0), (INC, 0.5), False),     # operator-in-registers kernels
    (150, 48, (INC, 0.3), (REF, 0.0), False),     # K-tiled kernels
    (90, 16, (VAC, 0.0), (VAC, 0.0), True),       # per-cell blocks (GEMV, config-5 style)
])
def test_sharded_equals_unsharded_bit_for_bit(J, N, bcL, bcR, hetero, world):
    p = _custom(J, N, bcL, bcR, seed=J + N, hetero=hetero)
    for tol, mx in ((-1.0, 5), (1e-10, 10_000)):
        a = _run_unsharded(p, 3, tol, mx)
        b = _run_sharded(p, world, 3, tol, mx)
        assert a[0] == b[0], (a[0], b[0])                         # status and iteration count of every step
        assert np.array_equal(a[1], b[1]) and np.array_equal(a[2], b[2])


def test_sharded_config3_against_the_oracle_and_restart():
    import paper_2305_13555_b200 as P
    from oracle import Oracle
    from paper_2305_13555_b200.sharding import ShardedOCI
    p = make_problem(3, cells=1000)
    o = Oracle.from_problem(p, threads=8)
    s = ShardedOCI.local(p, 4)
    for k in range(2):
        s.set_source(k)
        o.set_source(p.source(k))
        a, b = s.step(p.tol, p.max_iters), o.oci_step(p.tol, p.max_iters)
        assert a[:2] == b[:2]
    den = np.max(np.abs(o.angular_flux()))
    assert np.max(np.abs(s.get_angular_flux() - o.angular_flux())) / den < 1e-9
    s.set_flux_from_problem()                                   # restart: the ghost rows are exchanged again
    o.set_flux(p.psi0)
    assert s.step(-1.0, 3)[:2] == (1, 3) == o.oci_step(-1.0, 3)[:2]
    assert np.max(np.abs(s.get_angular_flux() - o.angular_flux())) / den < 1e-12
    # si_step and the FULL form are refused on a shard; a HALO face without an attachment cannot step
    with pytest.raises(P.OCIError) as e:
        s.shards[0].si_step()
    assert e.value.code == -1
    s.close()
    g = P.OCI(np.ones(4), np.ones(4), np.full(4, 0.5), 1.0, 0.1, 4, (P.BC_HALO, 0.0), (P.BC_VACUUM, 0.0))
    g.setup()
    g.set_flux(np.zeros((4, 4, 2)))
    with pytest.raises(P.OCIError) as e:
        g.oci_step()
    assert e.value.code == -2
    g.close()
