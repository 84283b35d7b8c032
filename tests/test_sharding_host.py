"""Row f4, host side (no GPU): the partition of a slab into contiguous cell ranges, the per-shard problem (cut faces
become OCI_BC_HALO, everything else is a slice), the mailbox size the C ABI reports, the call-order / argument errors of
oci_shard_attach that need no device - and the same partition logic across two real processes (gloo, world_size 2)."""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import pytest

import paper_2305_13555_b200 as P
from paper_2305_13555_b200.sharding import partition, shard_problem
from workloads import make_problem

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.parametrize("cells,world", [(1, 1), (7, 1), (7, 2), (8, 3), (100, 7), (131072, 8), (64, 64)])
def test_partition_is_contiguous_balanced_and_complete(cells, world):
    parts = partition(cells, world)
    assert len(parts) == world and parts[0][0] == 0 and parts[-1][1] == cells
    sizes = [b - a for a, b in parts]
    assert all(parts[i][1] == parts[i + 1][0] for i in range(world - 1))
    assert max(sizes) - min(sizes) <= 1 and min(sizes) >= 1 and sizes == sorted(sizes, reverse=True)
    with pytest.raises(ValueError):
        partition(world - 1, world)


@pytest.mark.parametrize("cfg,cells,world", [(1, 20, 2), (3, 50, 3), (5, 33, 4), (4, 10, 1)])
def test_shard_problem_slices_and_marks_the_cuts(cfg, cells, world):
    p = make_problem(cfg, cells=cells)
    shards = [shard_problem(p, r, world) for r in range(world)]
    for name in ("dx", "sigma_t", "sigma_s", "psi0"):
        assert np.array_equal(np.concatenate([getattr(s, name) for s in shards]), getattr(p, name))
    for r, s in enumerate(shards):
        assert s.bc_left == (p.bc_left if r == 0 else (P.BC_HALO, 0.0))
        assert s.bc_right == (p.bc_right if r == world - 1 else (P.BC_HALO, 0.0))
        assert s.n_angles == p.n_angles and s.dt == p.dt and s.v == p.v and s.unknowns == s.cells * 4 * p.n_angles
    for step in (0, 1):
        full = p.source(step)
        parts = [s.source(step) for s in shards]
        if full is None:
            assert all(q is None for q in parts)
        else:
            assert np.array_equal(np.concatenate(parts), full)
    assert p.cells == cells and p.bc_left[0] != P.BC_HALO                    # the original is untouched


def test_mailbox_size_and_host_side_errors():
    # halo [2][2][N] + norms [2][W][2] + flags [W], 8 bytes each
    assert P.shard_mailbox_bytes(32, 4) == 8 * (4 * 32 + 4 * 4 + 4)
    assert P.shard_mailbox_bytes(32, 65) == 0 and P.shard_mailbox_bytes(1, 2) == 0
    g = P.OCI(np.ones(4), np.ones(4), np.full(4, 0.5), 1.0, 0.1, 4, (P.BC_VACUUM, 0.0), (P.BC_HALO, 0.0))   # HALO is a valid kind
    with pytest.raises(P.OCIError) as e:
        g.shard_attach(0, 2, [16, 32])
    assert e.value.code == -2                                                # before oci_setup
    with pytest.raises(P.OCIError) as e:
        g.oci_step()
    assert e.value.code == -2
    g.close()


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_two_gloo_ranks_build_consistent_shards():
    """world_size 2 on CPU: each rank derives its shard from the same global problem; the ranks exchange what they
    hold at the cut (edge dx and the cut's BC kinds) and their cell ranges, and rank 0 checks the slab is tiled."""
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr", "127.0.0.1",
           "--master-port", str(_free_port()), os.path.join(ROOT, "tests", "_shard_worker.py")]
    r = subprocess.run(cmd, cwd=ROOT, env=dict(os.environ, OMP_NUM_THREADS="1", CUDA_VISIBLE_DEVICES=""), capture_output=True,
                       text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [json.loads(ln) for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = lines[0]
    assert d["ranges"] == [[0, 19], [19, 37]] and d["cells_total"] == 37
    assert d["cut_bcs"] == [[P.BC_VACUUM, P.BC_HALO], [P.BC_HALO, P.BC_VACUUM]]
    assert d["edge_match"] is True and d["mailbox_bytes"] == P.shard_mailbox_bytes(64, 2)
