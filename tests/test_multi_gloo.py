"""N > 1 path on CPU: world_size-2 gloo run of the bench's barrier + max-over-ranks timing, and of the
host planner on both ranks (replicas build identical plans)."""
import os
import socket

import torch
import torch.multiprocessing as mp

from paper_2211_05322_b200 import multi


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    import torch.distributed as dist
    from paper_2211_05322_b200 import reshard as rs
    multi.init("gloo")
    assert multi.world() == world
    multi.barrier()
    ms = multi.max_over_ranks(10.0 + 5.0 * rank)          # rank 1 is the slow replica
    p = rs.Plan((8, 16, 32), 2, (2, 4), "S0,R,S1", (2, 4), "S0,S1,R", rs.RS_HOST_ONLY)
    sig = torch.tensor([p.info.n_slices, p.info.max_sender_bytes, p.op_info(0).n_tiles], dtype=torch.int64)
    gathered = [torch.zeros_like(sig) for _ in range(world)]
    dist.all_gather(gathered, sig)
    same = all(torch.equal(g, sig) for g in gathered)
    multi.barrier()
    out.put((rank, ms, multi.job_gbs(3e9, ms, world), same))
    dist.destroy_process_group()


def test_two_rank_timing_and_identical_plans():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, gbs, same in res:
        assert ms == 15.0                                   # max over ranks, on every rank
        assert abs(gbs - 2 * 3e9 / 15e-3 / 1e9) < 1e-9      # all ranks' bytes / slowest time
        assert same


def test_single_process_is_identity():
    assert multi.world() == 1
    assert multi.max_over_ranks(7.5) == 7.5
    assert multi.job_gbs(1e9, 1.0, 1) == 1000.0
