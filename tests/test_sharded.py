"""The multi-process executor (first half): rs_plan_opts.src_owner / rank.

CPU (gloo, world_size 2, host-only plans): the ranks' execute tables partition the unit tasks, and replaying them
into one set of destination buffers gives the oracle's result with every byte written exactly once.
GPU: two processes on cuda:0 exchange CUDA IPC handles and store into each other's shards (tests/sharded_worker.py)."""
import os
import socket
import subprocess
import sys

import numpy as np
import pytest
import torch.multiprocessing as mp

import table_interp as ti
from oracle import data_oracle as do
from paper_2211_05322_b200 import reshard as rs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

CASES = [
    ((8, 8, 8), (2, 4), "S0,R,R", (2, 4), "R,R,R"),                  # full broadcast: 2 slices, 8 receivers each
    ((8, 16, 12), (2, 4), "S0,S1,R", (4, 2), "S1,R,S0"),             # config 4 in small
    ((4, 8, 4, 4), (1, 4), "S1,R,R,R", (2, 2), "R,S0,R,R"),          # config 3'' in small: multicast to 2
    ((7, 9), (2, 4), "S1,S0", (4, 2), "S0,S1"),                      # uneven (R5)
    ((8, 8, 8), (2, 4), "R,R,R", (2, 4), "S0,S1,R"),                 # 8 candidate senders per slice: Eq. 4 spreads them
]


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _bytes(a):
    return np.ascontiguousarray(a).view(np.uint8).reshape(-1)


def _worker(rank, world, port, out):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    import torch.distributed as dist
    dist.init_process_group("gloo")
    results = []
    for shape, sm, ss, dm, ds in CASES:
        n_src, n_dst = do.num_devices(sm), do.num_devices(dm)
        owner = [r % world for r in range(n_src)]
        p = rs.Plan(shape, 2, sm, ss, dm, ds, rs.RS_HOST_ONLY, dict(src_owner=owner, rank=rank))
        full = rs.Plan(shape, 2, sm, ss, dm, ds, rs.RS_HOST_ONLY)
        D = (np.arange(int(np.prod(shape)), dtype=np.int64) * 2654435761 % 251 + 1).astype(np.int16).reshape(shape)
        src = do.shards_from_global(D, sm, ss)
        want = do.reshard(shape, sm, ss, dm, ds, src)
        dst = [np.zeros(want[0].nbytes, np.uint8) for _ in range(n_dst)]
        cnt = [np.zeros(want[0].nbytes, np.int32) for _ in range(n_dst)]
        # this rank's launch reads only shards it holds: the others are not even passed
        mine = [_bytes(s) if owner[r] == rank else np.zeros(0, np.uint8) for r, s in enumerate(src)]
        ti.replay(p, rs.RS_OP_EXECUTE, mine, dst, cnt)
        tasks, _d, _s = ti.tables(p, rs.RS_OP_EXECUTE)
        o = p.op_info(rs.RS_OP_EXECUTE)
        mine_senders = sorted(s["sender"] for s in p.slices() if owner[s["sender"]] == rank)
        assert sorted(int(t["src_buf"]) for t in tasks) == mine_senders            # exactly this rank's unit tasks
        assert p.slices() == full.slices()                                            # same plan on every rank
        assert p.op_info(rs.RS_OP_PACK).n_tiles == 0 and p.op_info(rs.RS_OP_EXECUTE_SLABS).n_tiles == 0
        parts = [None] * world
        dist.all_gather_object(parts, (dst, cnt, o.read_bytes, o.write_bytes))
        if rank == 0:
            total = [sum(pt[1][q] for pt in parts) for q in range(n_dst)]
            merged = [sum(pt[0][q].astype(np.int32) for pt in parts).astype(np.uint8) for q in range(n_dst)]   # disjoint writes: sum = union
            local = do.local_shape(shape, dm, ds)
            for q in range(n_dst):
                lo, hi = do.device_box(shape, dm, ds, q)
                once = np.zeros(local + (2,), np.int32)
                once[tuple(slice(0, h - l) for l, h in zip(lo, hi))] = 1
                assert np.array_equal(total[q], once.reshape(-1)), "ranks together do not write every byte exactly once"
                assert np.array_equal(merged[q], _bytes(want[q])), "union of the ranks' launches differs from the oracle"
            assert sum(pt[2] for pt in parts) == full.info.unique_read_bytes and sum(pt[3] for pt in parts) == full.info.write_bytes
        results.append(len(tasks))
    dist.barrier()
    out.put((rank, results))
    dist.destroy_process_group()


def test_two_ranks_partition_the_unit_tasks():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = dict(q.get(timeout=180) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert sum(1 for i in range(len(CASES)) if res[0][i] and res[1][i]) >= 3
    for i, (shape, sm, ss, dm, ds) in enumerate(CASES):
        n = rs.Plan(shape, 2, sm, ss, dm, ds, rs.RS_HOST_ONLY).info.n_slices
        assert res[0][i] + res[1][i] == n                     # a partition (a rank may hold no chosen sender at all)


def test_owner_arguments():
    with pytest.raises(rs.ReshardError):
        rs.Plan((8, 8), 2, (2, 2), "S0,R", (2, 2), "R,S0", rs.RS_HOST_ONLY, dict(src_owner=[0, 0, 1, 1], rank=-1))
    with pytest.raises(rs.ReshardError):
        rs.Plan((8, 8), 2, (2, 2), "S0,R", (2, 2), "R,S0", rs.RS_HOST_ONLY | rs.RS_WITH_STRATEGIES, dict(src_owner=[0, 0, 1, 1], rank=0))
    p = rs.Plan((8, 8), 2, (2, 2), "S0,R", (2, 2), "R,S0", rs.RS_HOST_ONLY, dict(src_owner=[0, 0, 1, 1], rank=5))   # holds nothing
    assert p.op_info(rs.RS_OP_EXECUTE).n_tiles == 0 and p.info.n_slices == 4
    with pytest.raises(rs.ReshardError):
        rs.Plan.group([p], rs.RS_HOST_ONLY)


@pytest.mark.gpu
def test_two_processes_on_one_gpu_store_into_each_others_shards():
    """c3'' (every slice multicast to 2 receivers), a full-broadcast sweep point (1 + 8) and config 2: bit-exact against
    the oracle on every rank, one launch per rank, peer stores through CUDA IPC"""
    port = _free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE="2", LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port),
                   PYTHONPATH=os.pathsep.join([ROOT, os.path.join(ROOT, "tests")]))
        procs.append(subprocess.Popen([sys.executable, os.path.join(ROOT, "tests", "sharded_worker.py"), "c3ii", "sweep_P5_m8_16MiB", "c2", "c1i"],
                                      env=env, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True, cwd=ROOT))
    outs = [p.communicate(timeout=600)[0] for p in procs]
    for rank, (p, out) in enumerate(zip(procs, outs)):
        assert p.returncode == 0 and "rank %d ok" % rank in out, "\n".join("---- rank %d ----\n%s" % (r, o[-2500:]) for r, o in enumerate(outs))
