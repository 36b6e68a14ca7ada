"""The multi-process executor: one process per GPU, virtual device -> rank.

The paper's unit of work is one sender and all of its receivers ("broadcast based resharding"), and unit
tasks are independent.  So the whole task shards over ranks with NO collective: every rank builds the
same plan with rs_plan_opts.src_owner / rank, which leaves in its execute table only the unit tasks whose chosen sender
it holds; it runs them with ONE launch of the same kernels, whose destination pointers are local shards or shards of
other ranks mapped through CUDA IPC -- the slice crosses NVLink as the kernel's own stores ("the sender's GPU issues the
writes").  torch.distributed is plumbing here: it carries the IPC handles and the barrier, nothing of the data path.

This module holds no method arithmetic: which rank runs which unit task is decided inside the library.  There is no
fallback: without peer access between two GPUs the import fails loudly.
"""
import torch
import torch.distributed as dist

from . import reshard as rs


def round_robin_owner(n_devices, world):
    """virtual device r lives on rank r mod world: the mapping bench.py and the tests use"""
    return [r % world for r in range(n_devices)]


class ShardedReshard:
    """plan = reshard_plan_ex(..., src_owner, rank); bind() exchanges the IPC handles of the destination shards;
    execute() is this rank's single launch; wait() makes every rank's stores visible to every rank."""

    def __init__(self, shape, elem_bytes, src_mesh, src_spec, dst_mesh, dst_spec, src_owner, dst_owner, flags=0, opts=None, group=None):
        self.group = group
        self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)
        self.src_owner, self.dst_owner = list(src_owner), list(dst_owner)
        self.plan = rs.Plan(shape, elem_bytes, src_mesh, src_spec, dst_mesh, dst_spec, flags,
                            dict(opts or {}, src_owner=self.src_owner, rank=self.rank))
        assert len(self.src_owner) == self.plan.info.n_src and len(self.dst_owner) == self.plan.info.n_dst
        # destination shards this rank's unit tasks write (a query of the plan, not arithmetic of ours)
        self.writes = sorted({q for s in self.plan.slices() if self.src_owner[s["sender"]] == self.rank for q in s["receivers"]})
        self.src_ptrs = self.dst_ptrs = None

    def bind(self, src_local, dst_local):
        """src_local: {source device r: device tensor} for every r this rank holds; dst_local likewise for the
        destination shards it holds.  Collective: every rank must call it."""
        assert sorted(src_local) == [r for r, o in enumerate(self.src_owner) if o == self.rank]
        assert sorted(dst_local) == [q for q, o in enumerate(self.dst_owner) if o == self.rank]
        mine = {q: rs.ipc_export(t.data_ptr()) for q, t in dst_local.items()}
        everyone = [None] * self.world
        dist.all_gather_object(everyone, mine, group=self.group)
        self.src_ptrs = [src_local[r].data_ptr() if r in src_local else 0 for r in range(self.plan.info.n_src)]
        self.dst_ptrs = []
        for q in range(self.plan.info.n_dst):
            if q in dst_local:
                self.dst_ptrs.append(dst_local[q].data_ptr())
            elif q in self.writes:
                self.dst_ptrs.append(rs.ipc_import(everyone[self.dst_owner[q]][q]))   # peer memory: NVLink stores
            else:
                self.dst_ptrs.append(0)
        self._keep = (src_local, dst_local)
        dist.barrier(group=self.group)

    def execute(self, stream=0):
        self.plan.execute(self.src_ptrs, self.dst_ptrs, stream)

    def wait(self):
        """after this every destination shard of every rank is complete"""
        torch.cuda.synchronize()
        dist.barrier(group=self.group)

    def my_bytes(self):
        o = self.plan.op_info(rs.RS_OP_EXECUTE)
        return o.read_bytes + o.write_bytes

    def close(self):
        dist.barrier(group=self.group)                      # nobody is still writing into a peer
        rs.ipc_release_all()
        dist.barrier(group=self.group)                      # nobody frees memory a peer still maps
        self.plan.close()
