"""Row f4 plumbing: one slab sharded over several GPUs by contiguous cell ranges (include/oci.h
"oci_shard_*").  Host logic only: the partition, the per-shard problem (cut faces become OCI_BC_HALO), the mailboxes
every rank can address, and a small driver object.  The exchange itself (edge half rows and the two norms, stored
straight into the peers' mailboxes by stream-ordered kernels) lives in csrc/shard_exchange.cu.

Two ways to hold the shards:
  * `ShardedOCI.local(p, world)`: all shards in THIS process on one device and stream (the single-GPU emulation the
    tests use: the launches of the shards are interleaved so that every pull is ordered behind all pushes);
  * `ShardedOCI.distributed(p)`: one shard per process / GPU under torch.distributed (NCCL for the rendezvous only);
    the mailboxes are one symmetric-memory allocation, so every rank holds peer-mapped addresses of all of them.
"""
from __future__ import annotations

import copy

import numpy as np

from . import binding as B


def partition(cells: int, world: int):
    """Contiguous, balanced cell ranges [(start, stop)] * world; the first `cells % world` shards get one more cell."""
    if world < 1 or cells < world:
        raise ValueError("need at least one cell per shard")
    base, extra = divmod(cells, world)
    out, start = [], 0
    for r in range(world):
        stop = start + base + (1 if r < extra else 0)
        out.append((start, stop))
        start = stop
    return out


def shard_problem(p, rank: int, world: int):
    """The sub-problem of shard `rank`: its cells' materials and initial condition, the slab's own boundary
    conditions at the slab's ends and OCI_BC_HALO at the cuts.  `p` is a workloads.Problem (or anything with the same
    fields); the returned object is a shallow copy with sliced arrays and a sliced source."""
    start, stop = partition(p.cells, world)[rank]
    q = copy.copy(p)
    q.cells = stop - start
    q.dx, q.sigma_t, q.sigma_s = (np.ascontiguousarray(a[start:stop]) for a in (p.dx, p.sigma_t, p.sigma_s))
    q.psi0 = np.ascontiguousarray(p.psi0[start:stop])
    q.bc_left = p.bc_left if rank == 0 else (B.BC_HALO, 0.0)
    q.bc_right = p.bc_right if rank == world - 1 else (B.BC_HALO, 0.0)
    src = p._source

    def sliced(step, _src=src, _a=start, _b=stop):
        full = None if _src is None else _src(step)
        return None if full is None else np.ascontiguousarray(full[_a:_b])

    q._source = sliced
    q.cell_range = (start, stop)
    return q


class ShardedOCI:
    """The shards of one slab held by this process, stepped together."""

    def __init__(self, shards, ranks, world, keep):
        self.shards, self.ranks, self.world, self._keep = shards, ranks, world, keep

    @classmethod
    def local(cls, p, world, device="cuda:0", iteration=None, reduced_kernel=None):
        import torch
        dev = torch.device(device)
        nbytes = B.shard_mailbox_bytes(p.n_angles, world)
        boxes = [torch.zeros(nbytes, dtype=torch.uint8, device=dev) for _ in range(world)]
        shards = []
        for r in range(world):
            sp = shard_problem(p, r, world)
            g = B.OCI.from_problem(sp, device=device, set_flux=False, iteration=iteration, reduced_kernel=reduced_kernel)
            g.shard_attach(r, world, [b.data_ptr() for b in boxes])
            g.set_flux(sp.psi0)
            g.problem = sp
            shards.append(g)
        return cls(shards, list(range(world)), world, boxes)

    @classmethod
    def distributed(cls, p, device=None, group=None):
        """One shard per rank of the torch.distributed group (backend NCCL).  The mailboxes are rows of one
        symmetric-memory tensor: `rendezvous` hands every rank the peer-mapped address of every row."""
        import torch
        import torch.distributed as dist
        import torch.distributed._symmetric_memory as symm
        rank, world = dist.get_rank(group), dist.get_world_size(group)
        dev = torch.device(device if device is not None else f"cuda:{torch.cuda.current_device()}")
        nbytes = (B.shard_mailbox_bytes(p.n_angles, world) + 255) // 256 * 256
        box = symm.empty(nbytes, dtype=torch.uint8, device=dev)
        hdl = symm.rendezvous(box, group=group if group is not None else dist.group.WORLD)
        ptrs = [int(hdl.buffer_ptrs[r]) for r in range(world)]
        sp = shard_problem(p, rank, world)
        g = B.OCI.from_problem(sp, device=str(dev), set_flux=False)
        g.shard_attach(rank, world, ptrs)
        torch.cuda.synchronize(dev)
        dist.barrier(group)                        # every rank's mailbox is zeroed before anybody pushes
        g.set_flux(sp.psi0)
        g.problem = sp
        return cls([g], [rank], world, (box, hdl))

    def set_flux_from_problem(self):
        for g in self.shards:
            g.set_flux(g.problem.psi0)

    def set_source(self, step):
        for g in self.shards:
            g.set_source(g.problem.source(step))

    def step(self, tol=1e-10, max_iters=10_000):
        return B.shard_step(self.shards, tol, max_iters)

    def get_scalar_flux(self):
        return np.concatenate([g.get_scalar_flux() for g in self.shards], axis=0)

    def get_angular_flux(self):
        return np.concatenate([g.get_angular_flux() for g in self.shards], axis=0)

    def close(self):
        for g in self.shards:
            g.close()
        self.shards = []
