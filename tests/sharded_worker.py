"""One rank of the multi-process executor test (tests/test_sharded.py starts two of these on cuda:0 -- CUDA IPC works
between processes on the same GPU, so the peer-store path is checked bit for bit under the 1-GPU gpurun; only the
NVLink number stays unmeasured).  argv: workload names.  Exit code 0 = every shard this rank holds equals the oracle."""
import sys

import numpy as np
import torch
import torch.distributed as dist

from oracle import data_oracle as do
from paper_2211_05322_b200 import inputs, sharded
from paper_2211_05322_b200 import reshard as rs


def main(names):
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    torch.cuda.set_device(0)
    dev = torch.device("cuda:0")
    for name in names:
        w = inputs.get_workload(name)
        e = inputs.elem_bytes(w.dtype)
        D = inputs.global_tensor(w)
        src = do.shards_from_global(D, w.src_mesh, w.src_spec)
        so, dow = sharded.round_robin_owner(len(src), world), sharded.round_robin_owner(do.num_devices(w.dst_mesh), world)
        x = sharded.ShardedReshard(w.shape, e, w.src_mesh, w.src_spec, w.dst_mesh, w.dst_spec, so, dow)
        src_local = {r: torch.from_numpy(src[r]).to(dev) for r in range(len(src)) if so[r] == rank}
        dst_local = {q: torch.full((x.plan.info.dst_shard_bytes,), 0x5A, dtype=torch.uint8, device=dev) for q in range(len(dow)) if dow[q] == rank}
        x.bind(src_local, dst_local)
        n0 = rs.launch_count()
        x.execute(torch.cuda.current_stream().cuda_stream)
        assert rs.launch_count() == n0 + (1 if x.plan.op_info(rs.RS_OP_EXECUTE).n_tiles else 0)   # one launch per rank that holds a chosen sender
        x.wait()
        # every rank moved its share only, and the shares add up to the whole task
        shares = [None] * world
        dist.all_gather_object(shares, x.my_bytes())
        assert sum(shares) == x.plan.info.unique_read_bytes + x.plan.info.write_bytes, shares
        peers = [None] * world
        dist.all_gather_object(peers, sum(1 for q in x.writes if x.dst_owner[q] != rank))
        assert sum(peers) > 0 or world == 1, "no peer store in this test"
        for q, t in dst_local.items():
            want = do.reshard_device(w.shape, e, w.src_mesh, w.src_spec, w.dst_mesh, w.dst_spec, src, q, D.dtype, n_threads=do.max_threads())
            assert np.array_equal(t.cpu().numpy(), want.view(np.uint8).reshape(-1)), "%s: rank %d, destination shard %d differs from the oracle" % (name, rank, q)
        for call in (lambda: x.plan.pack(x.src_ptrs, 1), lambda: x.plan.host_workspace_bytes() >= 0 or (_ for _ in ()).throw(rs.ReshardError(1, "refused"))):
            try:
                call()
                raise SystemExit("a sharded plan must refuse pack / execute_host")
            except rs.ReshardError:
                pass
        x.close()
        del src_local, dst_local
        torch.cuda.empty_cache()
    dist.destroy_process_group()
    print("rank %d ok: %s" % (rank, ", ".join(names)))


if __name__ == "__main__":
    main(sys.argv[1:])
