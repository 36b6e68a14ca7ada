"""reshard_execute_static: the entry point that allocates nothing (include/reshard.h).  Collected LAST (the name):
the suite runs with pytest -x, so a failure here hides no other test.

The plan is built with RS_HOST_ONLY (no CUDA call, no device block); the kernels read their tables from the library's
file-scope static device array.  Checked against the existing path (reshard_execute on an ordinary plan), tolerance 0
like every parity test here (a pure copy), on calls in a row that SHARE the array: different layouts, so that the second
call must not see the first call's tables, and the first layout once more."""
import numpy as np
import pytest
import torch

from oracle import data_oracle as do
from paper_2211_05322_b200 import reshard as rs

import gpu_util as gu

pytestmark = pytest.mark.gpu

CASES = [
    # (shape, dtype, src mesh, src spec, dst mesh, dst spec, path flag)
    ((8, 320, 64, 64), np.int16, (1, 4), "S1,R,R,R", (2, 2), "R,S0,R,R", rs.RS_PATH_AUTO),    # config 3'': multicast to 2, TMA ring
    ((64, 96, 160), np.int16, (2, 4), "S0,R,S1", (2, 4), "S0,S1,R", rs.RS_PATH_AUTO),        # 32 unit tasks, register path, segments
    ((50, 70, 97), np.uint8, (2, 4), "S0,S1,R", (3, 2), "S1,R,S0", rs.RS_PATH_AUTO),         # uneven, nothing aligned: shifted kernels
    ((16, 1024, 1024), np.int16, (2, 4), "S0,R,S1", (2, 4), "S0,S1,R", rs.RS_PATH_TMAP),     # tensor-map copies (maps encoded per call)
    ((8, 8, 8), np.float32, (2, 4), "S0,R,R", (2, 4), "R,R,R", rs.RS_PATH_BULK),             # 1 + 8 broadcast, tiny
]


def _device_inputs(shape, dtype, sm, ss, seed):
    e = np.dtype(dtype).itemsize
    D = np.frombuffer(np.random.default_rng(seed).bytes(int(np.prod(shape)) * e), dtype=dtype).reshape(shape)
    return [gu.to_dev(x) for x in do.shards_from_global(D, sm, ss)]


def _run(plan, call, src_d, fill):
    dst = [torch.full((plan.info.dst_shard_bytes,), fill, dtype=torch.uint8, device=gu.dev()) for _ in range(plan.info.n_dst)]
    call(gu.ptrs(src_d), gu.ptrs(dst), gu.stream())
    return dst


def test_execute_static_equals_execute_on_calls_in_a_row():
    launches = rs.launch_count()
    order = [0, 1, 2, 3, 4, 0, 1]                                  # back to back, no synchronisation in between: stream order
    got, want = [], []
    for n, i in enumerate(order):
        shape, dtype, sm, ss, dm, ds, flag = CASES[i]
        e = np.dtype(dtype).itemsize
        src_d = _device_inputs(shape, dtype, sm, ss, seed=100 + n)
        host_only = rs.Plan(shape, e, sm, ss, dm, ds, flag | rs.RS_HOST_ONLY)          # no CUDA call, no device allocation
        ordinary = rs.Plan(shape, e, sm, ss, dm, ds, flag)
        with pytest.raises(rs.ReshardError):                                            # the existing path refuses a host-only plan
            host_only.execute(gu.ptrs(src_d), gu.ptrs(src_d), gu.stream())
        got.append(_run(host_only, host_only.execute_static, src_d, 0xA5))
        want.append(_run(ordinary, ordinary.execute, src_d, 0xA5))
        assert host_only.op_info(rs.RS_OP_EXECUTE).path == ordinary.op_info(rs.RS_OP_EXECUTE).path
    torch.cuda.synchronize()
    assert rs.launch_count() - launches == 2 * len(order)                               # one kernel launch per call, both ways
    for n, (g, w) in enumerate(zip(got, want)):
        for q, (a, b) in enumerate(zip(g, w)):
            assert torch.equal(a, b), "call %d (case %d), device %d: reshard_execute_static differs from reshard_execute" % (n, order[n], q)


def test_execute_static_on_an_ordinary_plan_and_against_the_oracle():
    """the entry point also takes a plan that has a device block (it does not use it); result = the oracle's"""
    shape, dtype, sm, ss, dm, ds, flag = CASES[1]
    e = np.dtype(dtype).itemsize
    for rep in range(2):                                                                # two calls in a row on one plan
        D = np.frombuffer(np.random.default_rng(7 + rep).bytes(int(np.prod(shape)) * e), dtype=dtype).reshape(shape)
        src = do.shards_from_global(D, sm, ss)
        want = do.reshard(shape, sm, ss, dm, ds, src, fill=0x5A)
        p = rs.Plan(shape, e, sm, ss, dm, ds, flag)
        dst = _run(p, p.execute_static, [gu.to_dev(x) for x in src], 0x5A)
        torch.cuda.synchronize()
        for q, w in enumerate(want):
            assert dst[q].cpu().numpy().tobytes() == w.tobytes(), "rep %d device %d" % (rep, q)


def test_execute_static_rejects_plans_beyond_the_array():
    """4096 unit tasks need 4096 x (224 + 16 + 16) bytes > RS_STATIC_TABLE_BYTES = 256 KiB: a clear error, nothing launched"""
    p = rs.Plan((64, 64, 64), 2, (8, 8), "S01,R,R", (8, 8), "R,S01,R", rs.RS_HOST_ONLY)
    assert p.info.n_slices == 4096
    src = [torch.zeros(p.info.src_shard_bytes, dtype=torch.uint8, device=gu.dev()) for _ in range(p.info.n_src)]
    dst = [torch.zeros(p.info.dst_shard_bytes, dtype=torch.uint8, device=gu.dev()) for _ in range(p.info.n_dst)]
    launches = rs.launch_count()
    with pytest.raises(rs.ReshardError) as ei:
        p.execute_static(gu.ptrs(src), gu.ptrs(dst), gu.stream())
    assert ei.value.code == rs.RS_EUNSUPPORTED and "262144" in str(ei.value) and "reshard_execute" in str(ei.value)
    assert rs.launch_count() == launches
