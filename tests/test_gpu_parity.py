"""-m gpu parity tests: the CUDA path, called through the C ABI, against the CPU oracle.
Bar: bit-exact (pure copy, tolerance 0) -- BASELINE.json north_star."""
import numpy as np
import pytest
import torch

import gpu_util as gu
from oracle import data_oracle as do
from oracle import plan_oracle as po
from paper_2211_05322_b200 import inputs
from paper_2211_05322_b200 import reshard as rs

pytestmark = pytest.mark.gpu

PATHS = [rs.RS_PATH_AUTO, rs.RS_PATH_LSU, rs.RS_PATH_BULK, rs.RS_PATH_BULK_SHIFT, rs.RS_PATH_TMAP]

SMALL = [
    ((8, 16), (1, 2), "S0,R", (1, 2), "R,S0"),                      # config 1 literal
    ((8, 16), (1, 2), "S1,R", (1, 2), "R,S1"),                      # config 1 intent
    ((4, 8, 16), (2, 4), "S0,R,S1", (2, 4), "S0,S1,R"),
    ((4, 8, 4, 4), (1, 4), "S0,R,R,R", (2, 2), "R,S0,S1,R"),
    ((4, 8, 4, 4), (1, 4), "S1,R,R,R", (2, 2), "R,S0,R,R"),
    ((8, 16, 12), (2, 4), "S0,S1,R", (4, 2), "S1,R,S0"),
    ((8, 8, 4), (2, 4), "R,S01,R", (2, 4), "S01,R,R"),
    ((6, 6, 2), (2, 3), "RRR", (3, 2), "RRR"),
    ((12, 6), (2, 3), "S0,S1", (3, 2), "S0,S1"),
    ((8, 8, 8), (2, 4), "R,R,S0", (2, 4), "S0,R,R"),
    ((8, 8, 8), (2, 4), "S0,R,R", (2, 4), "R,R,R"),
    ((8, 8, 8), (2, 4), "R,R,R", (2, 4), "S0,S1,R"),
    ((4, 6, 5, 3), (2, 2), "S0,S1,R,R", (2, 2), "S1,R,R,R"),        # odd extents: 2-byte vectors at most
    ((16, 7), (4,), "S0,R", (2,), "R,R"),
    ((1,), (1,), "R", (1,), "R"),                                    # degenerate: one element
    ((8, 6, 2, 16), (2, 2), "S0,R,R,S1", (2, 2), "R,S0,R,S1"),       # GENERIC tiles
    ((6, 4, 2, 3, 8), (2,), "R,R,R,R,S0", (2,), "S0,R,R,R,R"),
    ((64, 96, 160), (2, 4), "S0,R,S1", (2, 4), "S0,S1,R"),           # several tiles + ragged tail (160*e/4)
    ((48, 1000), (2, 2), "S0,S1", (2, 2), "S1,S0"),
    ((3, 5, 7), (1,), "R,R,R", (1,), "R,R,R"),                       # 1 device -> 1 device: memcpy
    # uneven partitions (R5): padded buffers, short and empty shards
    ((10,), (3,), "S0", (4,), "S0"),
    ((7, 9), (2, 4), "S1,S0", (4, 2), "S0,S1"),
    ((7, 5, 3), (2, 3), "S1,R,S0", (3, 2), "R,S0,S1"),
    ((2, 6), (4,), "S0,R", (2,), "S0,R"),
    ((90, 100, 40), (2, 4), "S0,R,R", (3, 4), "S0,R,R"),             # Table 2 case 6 in small
    ((50, 70, 96), (2, 4), "S0,S1,R", (3, 2), "S1,R,S0"),            # uneven on three dims, several tiles
]


@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("dtype", [np.uint8, np.int16, np.float32, np.int64, np.dtype("V16")])
@pytest.mark.parametrize("case", SMALL, ids=[str(i) for i in range(len(SMALL))])
def test_execute_bit_exact_small(case, dtype, path):
    shape, sm, ss, dm, ds = case
    _p, got, want = gu.run_small(shape, dtype, sm, ss, dm, ds, flags=path)
    for q, (g, w) in enumerate(zip(got, want)):
        assert g.tobytes() == w.tobytes(), "device %d differs" % q


@pytest.mark.parametrize("alg", [rs.RS_SCHED_NAIVE, rs.RS_SCHED_LOAD_BALANCE, rs.RS_SCHED_DFS, rs.RS_SCHED_GREEDY, rs.RS_SCHED_ENSEMBLE])
@pytest.mark.parametrize("case", [SMALL[i] for i in (3, 4, 6, 7, 9, 10, 11, 17)])
def test_scheduled_plans_move_the_same_bytes(case, alg):
    """S3.2 changes senders and table order, never the result (R10)"""
    shape, sm, ss, dm, ds = case
    for dph in (1, 2):
        p, got, want = gu.run_small(shape, np.int16, sm, ss, dm, ds, opts=dict(
            schedule=alg, src_devices_per_host=dph, dst_devices_per_host=dph, seed=3, node_budget=5000))
        assert p.schedule()["info"].makespan >= p.schedule()["info"].busiest_host_bytes
        for g, w in zip(got, want):
            assert g.tobytes() == w.tobytes()


@pytest.mark.parametrize("off", [(2, 0), (0, 2), (4, 8), (1, 3), (16, 16)])
@pytest.mark.parametrize("path", PATHS)
def test_under_aligned_shard_pointers(off, path):
    """plan allows 16-byte vectors; the caller's pointers do not: narrower accesses, same bytes"""
    _p, got, want = gu.run_small((64, 96, 160), np.int16, (2, 4), "S0,R,S1", (2, 4), "S0,S1,R", flags=path,
                                 src_offset=off[0], dst_offset=off[1])
    for g, w in zip(got, want):
        assert g.tobytes() == w.tobytes()


LONG_UNALIGNED = [
    ((5, 9, 4099), (2,), "S0,R,R", (2, 2), "R,S0,R"),                  # 20 KiB runs cut into chunks, k = 2, uneven on two dims
    ((4, 40, 2203), (2,), "R,R,S0", (2, 2), "S0,R,R"),                 # 1102-byte rows, several per tile, k = 2
    ((3, 6, 9001), (1,), "R,R,R", (2, 4), "R,S0,R"),                   # 9001-byte rows, k = 4, whole rows adjacent in the receivers
    ((2, 11, 6146), (2, 2), "S0,R,S1", (2, 2), "S1,S0,R"),             # 3073-byte rows, 1 : 1 (u4 in small)
]


@pytest.mark.parametrize("mode", [1, 2])
@pytest.mark.parametrize("dtype", [np.uint8, np.int16])
@pytest.mark.parametrize("case", LONG_UNALIGNED, ids=[str(i) for i in range(len(LONG_UNALIGNED))])
def test_unaligned_long_rows_register_and_bulk_stores(case, dtype, mode):
    """rs_copy_bulk_shift on rows of 1-20 KiB that are not 16-byte aligned: stores from registers (rs_tuning.shift_mode 1) and
    bodies realigned in the ring + cp.async.bulk stores (2); receivers congruent modulo 16 (one bulk store per row and
    receiver) and not (falls back to registers); pointers moved by odd byte counts; ring shapes from 1 to 8 warps"""
    shape, sm, ss, dm, ds = case
    e = np.dtype(dtype).itemsize
    for so, dofs in [(0, 0), (e, 3 * e), (lambda r: (5 * r * e) % 16, lambda q: (7 * q * e + e) % 16), (16, lambda q: 16 if q % 2 else 0)]:
        for warps, stages in [(0, 0), (1, 2), (8, 2), (3, 5)]:
            tuning = dict(shift_mode=mode, shift_warps=warps, shift_stages=stages)
            p, got, want = gu.run_small(shape, dtype, sm, ss, dm, ds, flags=rs.RS_PATH_BULK_SHIFT, src_offset=so, dst_offset=dofs,
                                        opts=dict(tuning=tuning))
            assert p.op_info(rs.RS_OP_EXECUTE).path == rs.RS_PATH_BULK_SHIFT
            for q, (g, w) in enumerate(zip(got, want)):
                assert g.tobytes() == w.tobytes(), (case, dtype, mode, warps, stages, q)


@pytest.mark.parametrize("narrow", [1, -1])
@pytest.mark.parametrize("dtype", [np.uint8, np.int16, np.float32, np.int64])
def test_register_path_at_the_layouts_own_vector_width(dtype, narrow):
    """layouts that are not 16-byte aligned on the register path: vectors of 8 / 4 / 2 / 1 bytes (rs_tuning.lsu_narrow = 1) and the
    16-byte shift kernel (-1) -- FAST, SPLIT and GENERIC tiles, multicast, odd pointer offsets"""
    e = np.dtype(dtype).itemsize
    for i in (2, 9, 10, 13, 14, 16, 21, 24, 25):
        shape, sm, ss, dm, ds = SMALL[i]
        for so, dofs in [(0, 0), (e, 3 * e)]:
            _p, got, want = gu.run_small(shape[:-1] + (shape[-1] + 1,), dtype, sm, ss, dm, ds, flags=rs.RS_PATH_LSU, src_offset=so, dst_offset=dofs,
                                         opts=dict(tuning=dict(lsu_narrow=narrow)))
            for q, (g, w) in enumerate(zip(got, want)):
                assert g.tobytes() == w.tobytes(), (i, dtype, narrow, so, q)


@pytest.mark.parametrize("path", [rs.RS_PATH_LSU, rs.RS_PATH_BULK, rs.RS_PATH_BULK_SHIFT])
@pytest.mark.parametrize("tile", [128, 1024, 4096])
def test_tile_sizes_and_ring_depths(tile, path):
    """rs_plan_opts.tuning: other tile sizes, ring depths and warp counts, same bytes"""
    for stages, look, warps in [(2, 1, 1), (3, 2, 4), (8, 4, 2), (6, 5, 8)]:
        tuning = dict(lsu_tile_bytes=tile, bulk_tile_bytes=tile, shift_tile_bytes=tile, bulk_stages=stages, bulk_lookahead=look,
                      bulk_warps=warps, shift_stages=stages, shift_lookahead=look, shift_warps=warps)
        for case in (SMALL[2], SMALL[15], SMALL[17], SMALL[18]):
            shape, sm, ss, dm, ds = case
            p, got, want = gu.run_small(shape, np.int32, sm, ss, dm, ds, flags=path, opts=dict(tuning=tuning))
            assert p.op_info(rs.RS_OP_EXECUTE).tile_bytes <= max(tile, 128)
            for g, w in zip(got, want):
                assert g.tobytes() == w.tobytes()
        if path == rs.RS_PATH_LSU:
            break


@pytest.mark.parametrize("name", ["c1", "c1i", "c3", "c3i", "c3ii", "c2"])
@pytest.mark.parametrize("path", PATHS)
def test_baseline_configs_against_full_oracle(name, path):
    """configs 1-3 of BASELINE.json (and the prose-intent variants, R21): every element vs the oracle"""
    w = inputs.get_workload(name)
    e = inputs.elem_bytes(w.dtype)
    D = inputs.global_tensor(w)
    src = do.shards_from_global(D, w.src_mesh, w.src_spec)
    p = rs.Plan(w.shape, e, w.src_mesh, w.src_spec, w.dst_mesh, w.dst_spec, path)
    src_d = [gu.to_dev(s) for s in src]
    dst_d = [torch.full((p.info.dst_shard_bytes,), 0x5A, dtype=torch.uint8, device=gu.dev()) for _ in range(p.info.n_dst)]
    p.execute(gu.ptrs(src_d), gu.ptrs(dst_d), gu.stream())
    torch.cuda.synchronize()
    n_thr = do.max_threads()
    for q in range(p.info.n_dst):
        want = do.reshard_device(w.shape, e, w.src_mesh, w.src_spec, w.dst_mesh, w.dst_spec, src, q, D.dtype, n_threads=n_thr)
        assert dst_d[q].cpu().numpy().tobytes() == want.tobytes(), "%s: device %d differs" % (name, q)


def _check_full_size(w, path=rs.RS_PATH_AUTO, n_samples=4096):
    """full-size check in the bench's launch configuration: (1) every element of every dst shard equals
    basic slicing of D with the ORACLE's box (on device), (2) sampled elements equal what the oracle's
    per-element source map says, (3) values are a function of the global index, so (1) needs no source."""
    e = inputs.elem_bytes(w.dtype)
    D, src = gu.workload_on_device(w)
    p = rs.Plan(w.shape, e, w.src_mesh, w.src_spec, w.dst_mesh, w.dst_spec, path)
    dst = [torch.empty(p.local_shape(rs.RS_DST), dtype=D.dtype, device=gu.dev()) for _ in range(p.info.n_dst)]
    for t in dst:
        t.view(torch.uint8).fill_(0x5A)
    p.execute(gu.ptrs(src), gu.ptrs(dst), gu.stream())
    torch.cuda.synchronize()
    idx = gu.oracle_slices(w.shape, w.dst_mesh, w.dst_spec)
    local = do.local_shape(w.shape, w.dst_mesh, w.dst_spec)
    assert tuple(local) == tuple(p.local_shape(rs.RS_DST))
    for q in range(p.info.n_dst):                             # padding (R5) must still hold the 0x5A fill
        assert torch.equal(dst[q].view(torch.uint8), gu.padded(D, idx[q], local, 0x5A).view(torch.uint8)), "%s dev %d" % (w.name, q)
    rng = np.random.default_rng(7)
    n_local = int(np.prod(p.local_shape(rs.RS_DST)))
    flat_src = [s.reshape(-1) for s in src]
    for q in range(p.info.n_dst):
        js = rng.integers(0, n_local, size=n_samples // p.info.n_dst + 1)
        js[0], js[-1] = 0, n_local - 1
        srcs = [do.element_source(w.shape, w.src_mesh, w.src_spec, w.dst_mesh, w.dst_spec, q, int(j)) for j in js]
        keep = [i for i, s in enumerate(srcs) if s[0] >= 0]   # (q, j) in the padding has no source
        if not keep:
            continue
        js, srcs = js[keep], [srcs[i] for i in keep]
        got = dst[q].reshape(-1)[torch.from_numpy(js).to(gu.dev())].cpu()
        want = torch.stack([flat_src[d][l] for d, l, _g in srcs]).cpu()
        assert torch.equal(got.view(torch.uint8), want.view(torch.uint8))
        gl = D.reshape(-1)[torch.tensor([g for _d, _l, g in srcs], device=gu.dev())].cpu()
        assert torch.equal(got.view(torch.uint8), gl.view(torch.uint8))
    return p


@pytest.mark.parametrize("path", PATHS)
def test_config4_full_size(path):
    _check_full_size(inputs.get_workload("c4"), path)


@pytest.mark.parametrize("name", ["c2", "t2_9", "sweep_P1_m8_1024MiB", "sweep_P2_m8_256MiB", "sweep_P4_m4_64MiB", "c3ii"])
def test_tensor_map_path_full_size(name):
    """RS_PATH_TMAP on the short-run layouts it is meant for: full tiles move by cp.async.bulk.tensor (one load, one store
    per receiver), ragged tiles by per-row bulk copies, in one launch; execute, pack and unpack"""
    import table_interp as ti
    w = inputs.get_workload(name)
    p = _check_full_size(w, rs.RS_PATH_TMAP, n_samples=512)
    assert p.op_info(rs.RS_OP_EXECUTE).path == rs.RS_PATH_TMAP
    tasks, _d, _s = ti.tables(p, rs.RS_OP_EXECUTE)
    if name in ("c2", "t2_9", "sweep_P1_m8_1024MiB", "sweep_P4_m4_64MiB"):   # runs of 512 B .. 2 KiB; the others (4 KiB, 1.25 MiB
        assert tasks["tmap_ok"].all(), "no task of %s takes the tensor-map copies" % name   # runs) keep the per-row copies
    e = inputs.elem_bytes(w.dtype)
    D, src = gu.workload_on_device(w)
    arena = torch.empty(p.info.arena_bytes, dtype=torch.uint8, device=gu.dev())
    dst = [torch.zeros(p.local_shape(rs.RS_DST), dtype=D.dtype, device=gu.dev()) for _ in range(p.info.n_dst)]
    p.pack(gu.ptrs(src), arena.data_ptr(), gu.stream())
    p.unpack(arena.data_ptr(), gu.ptrs(dst), gu.stream())
    torch.cuda.synchronize()
    idx = gu.oracle_slices(w.shape, w.dst_mesh, w.dst_spec)
    for q in range(p.info.n_dst):
        assert torch.equal(dst[q], D[idx[q]])


@pytest.mark.parametrize("path", [rs.RS_PATH_AUTO, rs.RS_PATH_LSU])
@pytest.mark.parametrize("name", ["u4", "u4b", "u1", "a4", "x:1024x1024x1040:u8:2x4:RRS01:2x4:S01RR"])   # the last: 130-byte rows at 1-byte alignment
def test_unaligned_uneven_full_size(name, path):
    """1-1.5 GiB with nothing aligned (a4: 16-byte aligned and nothing more): TMA loads + shifted stores (AUTO; bulk stores of
    realigned rows for u4 / u4b, register stores for u1's 2 KiB rows, the plain TMA ring for a4) and the register path (LSU)"""
    if name == "a4":
        p = _check_full_size(inputs.get_workload(name), path)
        assert p.op_info(rs.RS_OP_EXECUTE).path == (rs.RS_PATH_BULK if path == rs.RS_PATH_AUTO else rs.RS_PATH_LSU)
        return
    p = _check_full_size(inputs.get_workload(name), path)
    assert p.op_info(rs.RS_OP_EXECUTE).path == (rs.RS_PATH_BULK_SHIFT if path == rs.RS_PATH_AUTO else rs.RS_PATH_LSU)


@pytest.mark.parametrize("path", [rs.RS_PATH_AUTO, rs.RS_PATH_LSU])
@pytest.mark.parametrize("name", ["r128", "r128m", "fm_hw", "fm_hwm"])
def test_short_rows_full_size(name, path):
    """the paper's microbenchmark tensor with 128-byte runs (last dim sharded 8 ways), 1 : 1 and 1 + 4: tensor-map boxes of 64 rows
    (AUTO) and the register path; a feature map resharded from a split of H to a split of W (64-byte rows in spans of 32: one FAST tile
    per span, slices that share source rows walked together), 1 : 1 (AUTO: registers) and 1 + 2 (AUTO: tensor maps)"""
    p = _check_full_size(inputs.get_workload(name), path)
    auto = rs.RS_PATH_LSU if name == "fm_hw" else rs.RS_PATH_TMAP
    assert p.op_info(rs.RS_OP_EXECUTE).path == (auto if path == rs.RS_PATH_AUTO else rs.RS_PATH_LSU)


@pytest.mark.parametrize("pair", sorted(inputs.SWEEP_PAIRS))
@pytest.mark.parametrize("meshes", ["m8", "m4"])
def test_sweep_1gib_full_size(pair, meshes):
    _check_full_size(inputs.sweep_workload(pair, meshes, 1 << 30))


@pytest.mark.parametrize("pair", sorted(inputs.SWEEP_PAIRS))
@pytest.mark.parametrize("meshes", ["m8", "m4"])
def test_sweep_4gib_maximum_size(pair, meshes):
    """2^31 elements: byte offsets beyond 2^32 (all 12 pair x mesh combinations of BASELINE config 5)"""
    _check_full_size(inputs.sweep_workload(pair, meshes, 4 << 30), n_samples=1024)
    torch.cuda.empty_cache()


@pytest.mark.parametrize("mib", [1, 4, 16, 64, 256])
@pytest.mark.parametrize("meshes", ["m8", "m4"])
@pytest.mark.parametrize("pair", sorted(inputs.SWEEP_PAIRS))
def test_sweep_small_sizes(pair, meshes, mib):
    """every point of BASELINE config 5 below 1 GiB: AUTO changes kernel and launch shape inside this range"""
    _check_full_size(inputs.sweep_workload(pair, meshes, mib << 20), n_samples=512)


@pytest.mark.parametrize("name", ["c4", "sweep_P5_m8_1024MiB"])
def test_full_size_every_byte_against_the_oracles_own_output(name):
    """the headline config (and one 1 GiB multicast point) against reshard_oracle ITSELF: the oracle computes
    every destination shard from host source shards, the GPU shards are copied back and compared byte
    for byte; execute and pack -> unpack"""
    w = inputs.get_workload(name)
    e = inputs.elem_bytes(w.dtype)
    D = inputs.global_tensor(w)
    src = do.shards_from_global(D, w.src_mesh, w.src_spec)
    del D
    p = rs.Plan(w.shape, e, w.src_mesh, w.src_spec, w.dst_mesh, w.dst_spec)
    src_d = [torch.from_numpy(s).to(gu.dev()) for s in src]
    dst_d = [torch.full((p.info.dst_shard_bytes,), 0x5A, dtype=torch.uint8, device=gu.dev()) for _ in range(p.info.n_dst)]
    dst2_d = [torch.full((p.info.dst_shard_bytes,), 0xA5, dtype=torch.uint8, device=gu.dev()) for _ in range(p.info.n_dst)]
    arena = torch.empty(p.info.arena_bytes, dtype=torch.uint8, device=gu.dev())
    p.execute(gu.ptrs(src_d), gu.ptrs(dst_d), gu.stream())
    p.pack(gu.ptrs(src_d), arena.data_ptr(), gu.stream())
    p.unpack(arena.data_ptr(), gu.ptrs(dst2_d), gu.stream())
    torch.cuda.synchronize()
    n_thr = do.max_threads()
    want = np.empty(do.local_shape(w.shape, w.dst_mesh, w.dst_spec), dtype=src[0].dtype)
    for q in range(p.info.n_dst):
        do.reshard_device(w.shape, e, w.src_mesh, w.src_spec, w.dst_mesh, w.dst_spec, src, q, src[0].dtype, n_threads=n_thr, out=want)
        wb = want.view(np.uint8).reshape(-1)
        assert np.array_equal(dst_d[q].cpu().numpy(), wb), "%s: execute, device %d differs from the oracle" % (name, q)
        assert np.array_equal(dst2_d[q].cpu().numpy(), wb), "%s: pack -> unpack, device %d differs from the oracle" % (name, q)


def test_pack_arena_contents_full_size_c4():
    """config 4: every message of the arena equals the concatenation, in slice-id order, of the sender's boxes
    (plan oracle's message table and tile boxes; the slicing itself is torch basic slicing on the device)"""
    w = inputs.get_workload("c4")
    e = inputs.elem_bytes(w.dtype)
    _D, src = gu.workload_on_device(w)
    del _D
    p = rs.Plan(w.shape, e, w.src_mesh, w.src_spec, w.dst_mesh, w.dst_spec)
    arena = torch.full((p.info.arena_bytes,), 0x77, dtype=torch.uint8, device=gu.dev())
    p.pack(gu.ptrs(src), arena.data_ptr(), gu.stream())
    torch.cuda.synchronize()
    tasks = po.unit_tasks(w.shape, w.src_mesh, w.src_spec, w.dst_mesh, w.dst_spec)
    senders = [s["sender"] for s in p.slices()]
    table = po.message_table(tasks, senders)
    msgs = p.messages()
    assert len(msgs) == len(table)
    used = torch.zeros(p.info.arena_bytes, dtype=torch.bool, device=gu.dev())
    for m, (s, r, ids, n_elems) in zip(msgs, table):
        assert (m["sender"], m["receiver"], m["slice_ids"], m["bytes"]) == (s, r, ids, n_elems * e)
        lo, _hi = po.tile_box(w.shape, w.src_mesh, w.src_spec, s)
        parts = [src[s][tuple(slice(a - l, b - l) for a, b, l in zip(tasks[i]["lo"], tasks[i]["hi"], lo))].reshape(-1) for i in ids]
        payload = torch.cat(parts).view(torch.uint8)
        assert torch.equal(arena[m["offset"]:m["offset"] + m["bytes"]], payload), "message (%d, %d)" % (s, r)
        used[m["offset"]:m["offset"] + m["bytes"]] = True
    assert bool((arena[~used] == 0x77).all())                           # padding between messages untouched


@pytest.mark.parametrize("case", [1, 2, 3, 4, 5, 6, 7, 8, 9])
def test_table2_cases_full_size(case):
    """the paper's microbenchmark layouts on (1024,1024,512) at 2 B/elt"""
    _check_full_size(inputs.table2_workload(case), n_samples=512)


def test_a_to_b_to_a_is_identity_on_every_replica():
    for name in ("c3ii", "c2", "t2_3"):
        w = inputs.get_workload(name)
        e = inputs.elem_bytes(w.dtype)
        _D, src = gu.workload_on_device(w)
        fwd = rs.Plan(w.shape, e, w.src_mesh, w.src_spec, w.dst_mesh, w.dst_spec)
        bwd = rs.Plan(w.shape, e, w.dst_mesh, w.dst_spec, w.src_mesh, w.src_spec)
        mid = [torch.empty(fwd.info.dst_shard_bytes, dtype=torch.uint8, device=gu.dev()) for _ in range(fwd.info.n_dst)]
        back = [torch.zeros_like(s) for s in src]
        fwd.execute(gu.ptrs(src), gu.ptrs(mid), gu.stream())
        bwd.execute(gu.ptrs(mid), gu.ptrs(back), gu.stream())
        torch.cuda.synchronize()
        for a, b in zip(src, back):
            assert torch.equal(a, b)


@pytest.mark.parametrize("lb", [rs.RS_LB_GREEDY, rs.RS_LB_NAIVE])
@pytest.mark.parametrize("path", [rs.RS_PATH_LSU, rs.RS_PATH_BULK])
def test_executed_sender_is_the_planned_sender(lb, path):
    """R12: replicas carry their device id; what lands tells which replica the kernel read"""
    for shape, sm, ss, dm, ds in [((8, 8, 64), (2, 4), "R,R,S0", (2, 4), "S0,R,R"), ((8, 8, 64), (2, 4), "R,R,R", (2, 4), "S0,S1,R"),
                                  ((16, 8, 64), (2, 3), "RRR", (3, 2), "RRR"), ((24, 64), (2, 3), "S0,R", (3, 2), "S0,R")]:
        p = rs.Plan(shape, 4, sm, ss, dm, ds, lb | path)
        src = [torch.full(p.local_shape(rs.RS_SRC), r, dtype=torch.int32, device=gu.dev()) for r in range(p.info.n_src)]
        dst = [torch.full(p.local_shape(rs.RS_DST), -1, dtype=torch.int32, device=gu.dev()) for _ in range(p.info.n_dst)]
        p.execute(gu.ptrs(src), gu.ptrs(dst), gu.stream())
        torch.cuda.synchronize()
        for s in p.slices():
            for q in s["receivers"]:
                lo, _hi = do.device_box(shape, dm, ds, q)
                box = tuple(slice(a - l, b - l) for a, b, l in zip(s["lo"], s["hi"], lo))
                assert (dst[q][box] == s["sender"]).all()
        assert all((d >= 0).all() for d in dst)


@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("case", [SMALL[i] for i in (2, 4, 5, 8, 10, 12, 15, 17)])
def test_pack_unpack_equals_execute_equals_oracle(case, path):
    shape, sm, ss, dm, ds = case
    D = np.frombuffer(np.random.default_rng(3).bytes(int(np.prod(shape)) * 2), dtype=np.int16).reshape(shape)
    src = do.shards_from_global(D, sm, ss)
    want = do.reshard(shape, sm, ss, dm, ds, src)
    p = rs.Plan(shape, 2, sm, ss, dm, ds, path)
    src_d = [gu.to_dev(s) for s in src]
    arena = torch.full((p.info.arena_bytes,), 0x77, dtype=torch.uint8, device=gu.dev())
    dst_d = [torch.full((p.info.dst_shard_bytes,), 0x5A, dtype=torch.uint8, device=gu.dev()) for _ in want]
    p.pack(gu.ptrs(src_d), arena.data_ptr(), gu.stream())
    p.unpack(arena.data_ptr(), gu.ptrs(dst_d), gu.stream())
    torch.cuda.synchronize()
    for q, wq in enumerate(want):
        assert dst_d[q].cpu().numpy().tobytes() == wq.tobytes()
    # message contents: concatenation of the sender's boxes in slice-id order (plan oracle, numpy slicing)
    tasks = po.unit_tasks(shape, sm, ss, dm, ds)
    ref = po.pack_messages(shape, sm, ss, tasks, [s["sender"] for s in p.slices()], src)
    host = arena.cpu().numpy()
    used = np.zeros(host.size, bool)
    for m, (s, r, payload) in zip(p.messages(), ref):
        assert (m["sender"], m["receiver"]) == (s, r)
        assert host[m["offset"]:m["offset"] + m["bytes"]].tobytes() == payload.tobytes()
        used[m["offset"]:m["offset"] + m["bytes"]] = True
    assert (host[~used] == 0x77).all()                               # padding between messages untouched


def test_pack_unpack_full_size_c4_and_multicast():
    for name in ("c4", "sweep_P5_m8_1024MiB"):
        w = inputs.get_workload(name)
        e = inputs.elem_bytes(w.dtype)
        D, src = gu.workload_on_device(w)
        p = rs.Plan(w.shape, e, w.src_mesh, w.src_spec, w.dst_mesh, w.dst_spec)
        arena = torch.empty(p.info.arena_bytes, dtype=torch.uint8, device=gu.dev())
        dst = [torch.empty(p.local_shape(rs.RS_DST), dtype=D.dtype, device=gu.dev()) for _ in range(p.info.n_dst)]
        p.pack(gu.ptrs(src), arena.data_ptr(), gu.stream())
        p.unpack(arena.data_ptr(), gu.ptrs(dst), gu.stream())
        torch.cuda.synchronize()
        idx = gu.oracle_slices(w.shape, w.dst_mesh, w.dst_spec)
        for q in range(p.info.n_dst):
            assert torch.equal(dst[q], D[idx[q]])
        del arena, dst, src, D
        torch.cuda.empty_cache()


def test_execute_host_buffers_and_side_stream():
    w = inputs.get_workload("c3ii")
    e = inputs.elem_bytes(w.dtype)
    D = inputs.global_tensor(w)
    src = do.shards_from_global(D, w.src_mesh, w.src_spec)
    want = do.reshard(w.shape, w.src_mesh, w.src_spec, w.dst_mesh, w.dst_spec, src, n_threads=do.max_threads())
    p = rs.Plan(w.shape, e, w.src_mesh, w.src_spec, w.dst_mesh, w.dst_spec)
    src_h = [torch.from_numpy(s.copy()).pin_memory() for s in src]
    dst_h = [torch.empty(p.local_shape(rs.RS_DST), dtype=torch.int16).pin_memory() for _ in want]
    ws = torch.empty(p.host_workspace_bytes(), dtype=torch.uint8, device=gu.dev())
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        up, down = p.execute_host(gu.ptrs(src_h), gu.ptrs(dst_h), ws.data_ptr(), side.cuda_stream)
    side.synchronize()
    assert up == p.info.tensor_bytes and down == p.info.write_bytes
    for g, wq in zip(dst_h, want):
        assert g.numpy().tobytes() == wq.tobytes()


def test_one_launch_per_call_and_loud_failure():
    p = rs.Plan((8, 8, 64), 2, (2, 4), "S0,R,S1", (2, 4), "S0,S1,R")
    src = [torch.zeros(p.info.src_shard_bytes, dtype=torch.uint8, device=gu.dev()) for _ in range(8)]
    dst = [torch.zeros(p.info.dst_shard_bytes, dtype=torch.uint8, device=gu.dev()) for _ in range(8)]
    n0 = rs.launch_count()
    p.execute(gu.ptrs(src), gu.ptrs(dst), gu.stream())
    assert rs.launch_count() == n0 + 1                                # single-launch kernel (north_star item 2)
    with pytest.raises(rs.ReshardError):
        p.execute(gu.ptrs(src), [0] * 8, gu.stream())                 # null destination: refused, not skipped
    torch.cuda.synchronize()


@pytest.mark.parametrize("case", [
    ((6, 1024, 2048), (2, 2), "S0,R,S1", (3,), "S0,R,R"),            # 3 slabs, l_0 = 6, 2-way x 3-way cuts on dim 0
    ((64, 512, 1024), (2, 4), "R,R,S0", (2, 4), "S0,R,R"),           # replicas: only the chosen senders are uploaded
    ((48, 256, 1024), (2, 4), "S0,R,R", (2, 4), "R,R,R"),            # full broadcast: every slab lands on 8 devices
    ((5, 1024, 2048), (2,), "R,S0,R", (4,), "R,R,S0"),               # l_0 = 5 not divisible by the slab count
    ((40, 300, 1000), (2, 2), "S0,S1,R", (2, 2), "S1,S0,R"),         # 8-byte-aligned runs only: LSU path per slab
])
def test_execute_host_pipeline_cases(case):
    shape, sm, ss, dm, ds = case
    D = np.frombuffer(np.random.default_rng(11).bytes(int(np.prod(shape)) * 2), dtype=np.int16).reshape(shape)
    src = do.shards_from_global(D, sm, ss)
    want = do.reshard(shape, sm, ss, dm, ds, src, n_threads=do.max_threads())
    p = rs.Plan(shape, 2, sm, ss, dm, ds)
    used = {s["sender"] for s in p.slices()}
    src_h = [torch.from_numpy(s.copy()).pin_memory() if r in used else None for r, s in enumerate(src)]
    dst_h = [torch.full(p.local_shape(rs.RS_DST), 0x5A5A, dtype=torch.int16).pin_memory() for _ in want]
    ws = torch.empty(p.host_workspace_bytes(), dtype=torch.uint8, device=gu.dev())
    for _ in range(2):                                               # twice: the plan-owned streams/events are reused
        up, down = p.execute_host([t.data_ptr() if t is not None else 0 for t in src_h], gu.ptrs(dst_h),
                                  ws.data_ptr(), gu.stream())
        torch.cuda.current_stream().synchronize()                    # the caller's stream alone must be enough
        assert up == p.info.tensor_bytes and down == p.info.write_bytes
        for q, (g, wq) in enumerate(zip(dst_h, want)):
            assert g.numpy().tobytes() == wq.tobytes(), "device %d" % q
            g.fill_(0x5A5A)


@pytest.mark.parametrize("strategy", [rs.RS_STRATEGY_BROADCAST, rs.RS_STRATEGY_SENDRECV, rs.RS_STRATEGY_ALLGATHER,
                                      rs.RS_STRATEGY_ALLGATHER_LOCAL])
@pytest.mark.parametrize("path", [rs.RS_PATH_AUTO, rs.RS_PATH_LSU])
@pytest.mark.parametrize("case", [SMALL[i] for i in (0, 3, 4, 7, 9, 10, 13, 17, 20, 23, 24)])
def test_strategies_reach_the_oracle_result(case, path, strategy):
    """send/recv, all-gather and broadcast are routes to the SAME destination layout"""
    shape, sm, ss, dm, ds = case
    rng = np.random.default_rng(11)
    D = rng.integers(-2 ** 15, 2 ** 15, size=shape).astype(np.int16)
    src = do.shards_from_global(D, sm, ss)
    want = do.reshard(shape, sm, ss, dm, ds, src, fill=0xA5)
    p = rs.Plan(shape, 2, sm, ss, dm, ds, path | rs.RS_WITH_STRATEGIES, dict(dst_devices_per_host=2))
    src_d = [gu.to_dev(s) for s in src]
    dst_d = [torch.full((w.nbytes,), 0xA5, dtype=torch.uint8, device=gu.dev()) for w in want]
    n0 = rs.launch_count()
    p.execute_strategy(strategy, gu.ptrs(src_d), gu.ptrs(dst_d), gu.stream())
    torch.cuda.synchronize()
    gather = {rs.RS_STRATEGY_ALLGATHER: rs.RS_OP_AG_GATHER, rs.RS_STRATEGY_ALLGATHER_LOCAL: rs.RS_OP_AGL_GATHER}.get(strategy)
    assert rs.launch_count() - n0 == (2 if gather is not None and p.op_info(gather).n_tiles else 1)
    for q, w in enumerate(want):
        assert dst_d[q].cpu().numpy().tobytes() == w.tobytes(), "device %d differs" % q


def test_strategies_full_size_multicast_and_refusal():
    w = inputs.sweep_workload("P5", "m8", 256 << 20)               # 1 read + 8 writes at 256 MiB
    e = inputs.elem_bytes(w.dtype)
    D, src = gu.workload_on_device(w)
    p = rs.Plan(w.shape, e, w.src_mesh, w.src_spec, w.dst_mesh, w.dst_spec, rs.RS_WITH_STRATEGIES, dict(dst_devices_per_host=4))
    idx = gu.oracle_slices(w.shape, w.dst_mesh, w.dst_spec)
    for strategy in (rs.RS_STRATEGY_SENDRECV, rs.RS_STRATEGY_ALLGATHER, rs.RS_STRATEGY_ALLGATHER_LOCAL):
        dst = [torch.zeros(p.local_shape(rs.RS_DST), dtype=D.dtype, device=gu.dev()) for _ in range(p.info.n_dst)]
        p.execute_strategy(strategy, gu.ptrs(src), gu.ptrs(dst), gu.stream())
        torch.cuda.synchronize()
        for q in range(p.info.n_dst):
            assert torch.equal(dst[q], D[idx[q]])
    plain = rs.Plan(w.shape, e, w.src_mesh, w.src_spec, w.dst_mesh, w.dst_spec)
    with pytest.raises(rs.ReshardError):
        plain.execute_strategy(rs.RS_STRATEGY_SENDRECV, gu.ptrs(src), gu.ptrs(dst), gu.stream())


def test_cuda_graph_capture_and_replay():
    """execute / pack / unpack only enqueue kernels: a whole step can be captured once and replayed
    (small, launch-bound reshards are the case for it)"""
    w = inputs.get_workload("c3ii")
    e = inputs.elem_bytes(w.dtype)
    D, src = gu.workload_on_device(w)
    p = rs.Plan(w.shape, e, w.src_mesh, w.src_spec, w.dst_mesh, w.dst_spec)
    dst = [torch.zeros(p.local_shape(rs.RS_DST), dtype=D.dtype, device=gu.dev()) for _ in range(p.info.n_dst)]
    dst2 = [torch.zeros_like(t) for t in dst]
    arena = torch.zeros(p.info.arena_bytes, dtype=torch.uint8, device=gu.dev())
    g = torch.cuda.CUDAGraph()
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.graph(g, stream=side):
        s = torch.cuda.current_stream().cuda_stream
        p.execute(gu.ptrs(src), gu.ptrs(dst), s)
        p.pack(gu.ptrs(src), arena.data_ptr(), s)
        p.unpack(arena.data_ptr(), gu.ptrs(dst2), s)
    torch.cuda.synchronize()
    assert all(int(t.abs().sum()) == 0 for t in dst)                   # capture does not execute
    idx = gu.oracle_slices(w.shape, w.dst_mesh, w.dst_spec)
    for _ in range(3):
        for t in dst + dst2:
            t.zero_()
        g.replay()
        torch.cuda.synchronize()
        for q in range(p.info.n_dst):
            assert torch.equal(dst[q], D[idx[q]]) and torch.equal(dst2[q], D[idx[q]])


def test_one_plan_many_host_threads_and_streams():
    """include/reshard.h 'Threading': a plan is immutable; threads may execute it concurrently on their own streams"""
    import threading
    w = inputs.get_workload("c2")
    e = inputs.elem_bytes(w.dtype)
    D, src = gu.workload_on_device(w)
    p = rs.Plan(w.shape, e, w.src_mesh, w.src_spec, w.dst_mesh, w.dst_spec)
    idx = gu.oracle_slices(w.shape, w.dst_mesh, w.dst_spec)
    outs, errs = {}, []

    def work(tid):
        try:
            torch.cuda.set_device(0)
            st = torch.cuda.Stream()
            dst = [torch.zeros(p.local_shape(rs.RS_DST), dtype=D.dtype, device=gu.dev()) for _ in range(p.info.n_dst)]
            st.wait_stream(torch.cuda.default_stream())
            for _ in range(5):
                p.execute(gu.ptrs(src), gu.ptrs(dst), st.cuda_stream)
            st.synchronize()
            outs[tid] = dst
        except Exception as ex:                                        # noqa: BLE001
            errs.append(ex)

    torch.cuda.synchronize()
    ts = [threading.Thread(target=work, args=(i,)) for i in range(4)]
    [t.start() for t in ts]
    [t.join() for t in ts]
    assert not errs and len(outs) == 4
    for dst in outs.values():
        for q in range(p.info.n_dst):
            assert torch.equal(dst[q], D[idx[q]])


@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("case", [
    ((2, 3, 2, 2, 4, 2, 2, 6), (2, 2, 2, 2), "S0,R,S1,R,S2,R,R,S3", (2, 2, 2, 2), "R,S3,R,S2,R,S1,S0,R"),
    ((128, 4), (128,), "S0,R", (2, 4, 4, 4), "R,S0123"),
    ((256, 64), (1,), "R,R", (128,), "R,R"),
])
def test_maximum_ranks_and_device_counts(case, path):
    """RS_MAX_NDIM = 8 tensor dims, RS_MAX_MESH_NDIM = 4 mesh dims, RS_MAX_DEVICES = 128 devices per mesh"""
    shape, sm, ss, dm, ds = case
    _p, got, want = gu.run_small(shape, np.int16, sm, ss, dm, ds, flags=path)
    for g, w in zip(got, want):
        assert g.tobytes() == w.tobytes()


@pytest.mark.parametrize("tuning", [dict(pace_permille=5), dict(pace_permille=850), dict(pace_permille=-1), dict(no_pdl=1),
                                    dict(pace_permille=300, no_pdl=1, bulk_warps=4, bulk_tile_bytes=2048), dict(task_order=1),
                                    dict(tiles_per_worker=1), dict(small_op_bytes_mib=-1), dict(lsu_ctas_per_sm=1)])
def test_rate_matching_and_launch_switches_change_no_byte(tuning):
    """rs_plan_opts.tuning: pacing (down to a crawl), programmatic dependent launch off, task order, other shapes -- same bytes;
    back-to-back dependent launches (B reads what A wrote) stay ordered with PDL on and off"""
    for path in (rs.RS_PATH_AUTO, rs.RS_PATH_BULK, rs.RS_PATH_TMAP):
        for case in (SMALL[9], SMALL[10], SMALL[17], SMALL[18]):          # 1 + 4, 1 + 8 multicast, several tiles per warp
            shape, sm, ss, dm, ds = case
            p, got, want = gu.run_small(shape, np.int32, sm, ss, dm, ds, flags=path, opts=dict(tuning=tuning))
            for g, w in zip(got, want):
                assert g.tobytes() == w.tobytes()
    w = inputs.get_workload("sweep_P5_m8_16MiB")                            # 1 + 8 at 144 MiB moved: paced by default
    e = inputs.elem_bytes(w.dtype)
    D, src = gu.workload_on_device(w)
    fwd = rs.Plan(w.shape, e, w.src_mesh, w.src_spec, w.dst_mesh, w.dst_spec, 0, dict(tuning=tuning))
    bwd = rs.Plan(w.shape, e, w.dst_mesh, w.dst_spec, w.src_mesh, w.src_spec, 0, dict(tuning=tuning))
    if not tuning.get("pace_permille"):
        assert fwd.op_info(rs.RS_OP_EXECUTE).pace_permille == 825
    mid = [torch.zeros(fwd.info.dst_shard_bytes, dtype=torch.uint8, device=gu.dev()) for _ in range(fwd.info.n_dst)]
    back = [torch.zeros_like(s) for s in src]
    for _ in range(3):                                                      # a chain of dependent launches, no host sync in between
        fwd.execute(gu.ptrs(src), gu.ptrs(mid), gu.stream())
        bwd.execute(gu.ptrs(mid), gu.ptrs(back), gu.stream())
    torch.cuda.synchronize()
    for a, b in zip(src, back):
        assert torch.equal(a, b)


@pytest.mark.parametrize("cap", [1, 7, 64])
def test_max_ctas_caps_the_grid_not_the_result(cap):
    """rs_plan_opts.max_ctas: fewer CTAs (SMs left to other streams), same bytes"""
    for case in (SMALL[2], SMALL[10], SMALL[17], SMALL[25]):
        shape, sm, ss, dm, ds = case
        for path in (rs.RS_PATH_AUTO, rs.RS_PATH_LSU, rs.RS_PATH_BULK_SHIFT):
            p, got, want = gu.run_small(shape, np.int16, sm, ss, dm, ds, flags=path, opts=dict(max_ctas=cap))
            assert p.op_info(rs.RS_OP_EXECUTE).grid <= cap
            for g, w in zip(got, want):
                assert g.tobytes() == w.tobytes()
    w = inputs.get_workload("c4")
    p = rs.Plan(w.shape, 2, w.src_mesh, w.src_spec, w.dst_mesh, w.dst_spec, 0, dict(max_ctas=cap))
    assert p.op_info(rs.RS_OP_EXECUTE).grid == cap


@pytest.mark.parametrize("case", [
    ((70, 300, 1001), (2, 2), "S0,S1,R", (3, 2), "S1,S0,R"),          # uneven on dims 0 and 1, odd runs: shifted kernels per slab
    ((45, 260, 1024), (2, 4), "S0,R,R", (3, 4), "S0,R,R"),            # Table 2 case 6 in small: short last shard on dim 0
    ((9, 64, 4096), (4,), "S0,R,R", (2, 3), "S1,S0,R"),               # 9 rows over 4 and over 3 devices
])
def test_execute_host_uneven_layouts(case):
    """host buffers are padded too (R5, R11); only the valid boxes are specified after reshard_execute_host"""
    shape, sm, ss, dm, ds = case
    D = np.frombuffer(np.random.default_rng(5).bytes(int(np.prod(shape)) * 2), dtype=np.int16).reshape(shape)
    src = do.shards_from_global(D, sm, ss, pad=0x11)
    want = do.reshard(shape, sm, ss, dm, ds, src, n_threads=do.max_threads())
    for opts in (None, dict(schedule=rs.RS_SCHED_ENSEMBLE, src_devices_per_host=2, dst_devices_per_host=2)):
        p = rs.Plan(shape, 2, sm, ss, dm, ds, 0, opts)
        src_h = [torch.from_numpy(s.copy()).pin_memory() for s in src]
        dst_h = [torch.zeros(p.local_shape(rs.RS_DST), dtype=torch.int16).pin_memory() for _ in want]
        ws = torch.empty(p.host_workspace_bytes(), dtype=torch.uint8, device=gu.dev())
        p.execute_host(gu.ptrs(src_h), gu.ptrs(dst_h), ws.data_ptr(), gu.stream())
        torch.cuda.current_stream().synchronize()
        for q, (g, wq) in enumerate(zip(dst_h, want)):
            lo, hi = do.device_box(shape, dm, ds, q)
            valid = tuple(slice(0, h - l) for l, h in zip(lo, hi))
            assert np.array_equal(g.numpy()[valid], wq[valid]), "device %d" % q


def _random_layout(rng):
    ndim = int(rng.integers(1, 5))
    meshes = [(1, 2), (2, 2), (2, 4), (4, 2), (2, 3), (3, 2), (1, 4), (4,), (3,), (2, 2, 2)]

    def side():
        mesh = meshes[int(rng.integers(len(meshes)))]
        axes = list(rng.permutation(len(mesh)))
        spec = []
        for _ in range(ndim):
            take = int(rng.integers(0, 3)) if axes else 0
            mine = [axes.pop() for _ in range(min(take, len(axes)))]
            spec.append("S" + "".join(str(a) for a in mine) if mine else "R")
        return mesh, ",".join(spec)
    sm, ss = side()
    dm, ds = side()
    inner = int(rng.choice([1, 3, 8, 17, 64, 100, 257, 1000]))
    shape = tuple(int(rng.choice([1, 2, 5, 7, 12, 16, 33])) for _ in range(ndim - 1)) + (inner,)
    return shape, sm, ss, dm, ds


@pytest.mark.parametrize("seed", range(20))
def test_random_layouts_alignments_and_paths(seed):
    """fuzz: 12 seeded layouts per seed (even and uneven, 1..4 dims, runs of 1..1000 elements), every element size,
    shard pointers at random byte offsets, every executor, with and without a schedule -- bit-exact, guard bands intact"""
    rng = np.random.default_rng(2211_05322 + seed)
    dtypes = [np.uint8, np.int16, np.float32, np.int64, np.dtype("V16")]
    members = []                                                   # the same layouts once more, as ONE group launch
    for _ in range(12):
        shape, sm, ss, dm, ds = _random_layout(rng)
        dtype = dtypes[int(rng.integers(len(dtypes)))]
        members.append((shape, dtype, sm, ss, dm, ds))
        path = PATHS[int(rng.integers(len(PATHS)))]
        so, dofs = (int(rng.integers(0, 16)), int(rng.integers(0, 16))) if rng.integers(2) else (0, 0)
        opts = dict(schedule=int(rng.integers(1, 6)), src_devices_per_host=int(rng.integers(1, 3)), node_budget=2000) if rng.integers(3) == 0 else None
        _p, got, want = gu.run_small(shape, dtype, sm, ss, dm, ds, flags=path, seed=seed, src_offset=so, dst_offset=dofs, opts=opts)
        for q, (g, w) in enumerate(zip(got, want)):
            assert g.tobytes() == w.tobytes(), (shape, sm, ss, dm, ds, dtype, path, so, dofs, opts, q)
        if rng.integers(3) == 0:                                   # another route to the same layout, and pack -> unpack
            strategy = int(rng.integers(1, 4))
            e = np.dtype(dtype).itemsize
            p = rs.Plan(shape, e, sm, ss, dm, ds, path | rs.RS_WITH_STRATEGIES, dict(dst_devices_per_host=int(rng.integers(1, 4))))
            D = np.frombuffer(np.random.default_rng(seed).bytes(int(np.prod(shape)) * e), dtype=dtype).reshape(shape)
            src_d = [gu.to_dev(x) for x in do.shards_from_global(D, sm, ss)]
            for route in ("strategy", "pack"):
                dst_d = [torch.full((w.nbytes,), 0xA5, dtype=torch.uint8, device=gu.dev()) for w in want]
                if route == "strategy":
                    p.execute_strategy(strategy, gu.ptrs(src_d), gu.ptrs(dst_d), gu.stream())
                else:
                    arena = torch.zeros(max(1, p.info.arena_bytes), dtype=torch.uint8, device=gu.dev())
                    p.pack(gu.ptrs(src_d), arena.data_ptr(), gu.stream())
                    p.unpack(arena.data_ptr(), gu.ptrs(dst_d), gu.stream())
                torch.cuda.synchronize()
                for q, w in enumerate(want):
                    assert dst_d[q].cpu().numpy().tobytes() == w.tobytes(), (shape, sm, ss, dm, ds, dtype, path, route, strategy, q)
    plans, src_d, wants = [], [], []
    for shape, dtype, sm, ss, dm, ds in members:
        e = np.dtype(dtype).itemsize
        if len(src_d) + do.num_devices(sm) > 128 or len(wants) + do.num_devices(dm) > 128:
            break
        D = np.frombuffer(np.random.default_rng(seed + len(plans)).bytes(int(np.prod(shape)) * e), dtype=dtype).reshape(shape)
        src = do.shards_from_global(D, sm, ss)
        wants += do.reshard(shape, sm, ss, dm, ds, src, fill=0xA5)
        src_d += [gu.to_dev(x) for x in src]
        plans.append(rs.Plan(shape, e, sm, ss, dm, ds))
    g = rs.Plan.group(plans, PATHS[seed % len(PATHS)])
    dst_d = [torch.full((w.nbytes,), 0xA5, dtype=torch.uint8, device=gu.dev()) for w in wants]
    g.execute(gu.ptrs(src_d), gu.ptrs(dst_d), gu.stream())
    torch.cuda.synchronize()
    for q, w in enumerate(wants):
        assert dst_d[q].cpu().numpy().tobytes() == w.tobytes(), ("group", seed, q)


@pytest.mark.parametrize("nodes,gpus", [(1, 3), (4, 2)])
def test_fig5_single_sender_full_size(nodes, gpus):
    """one sender, a replicated receiver mesh, 1 GiB: every receiver ends with the whole tensor"""
    _check_full_size(inputs.fig5_workload(nodes, gpus), n_samples=256)


@pytest.mark.parametrize("path", [rs.RS_PATH_AUTO, rs.RS_PATH_LSU, rs.RS_PATH_BULK_SHIFT])
def test_plan_group_runs_every_member_in_one_launch(path):
    """reshard_plan_group (many resharding tasks per stage boundary): one launch, every member bit-exact"""
    members = [SMALL[i] for i in (2, 4, 9, 10, 17, 21, 25)]
    plans, src_d, want = [], [], []
    rng = np.random.default_rng(3)
    for shape, sm, ss, dm, ds in members:
        D = rng.integers(-2 ** 15, 2 ** 15, size=shape).astype(np.int16)
        src = do.shards_from_global(D, sm, ss)
        want += do.reshard(shape, sm, ss, dm, ds, src, fill=0xA5)
        src_d += [gu.to_dev(s) for s in src]
        plans.append(rs.Plan(shape, 2, sm, ss, dm, ds, path))
    g = rs.Plan.group(plans, path)
    for p in plans:
        p.close()                                                  # the group owns its own tables
    dst_d = [torch.full((w.nbytes,), 0xA5, dtype=torch.uint8, device=gu.dev()) for w in want]
    n0 = rs.launch_count()
    g.execute(gu.ptrs(src_d), gu.ptrs(dst_d), gu.stream())
    torch.cuda.synchronize()
    assert rs.launch_count() == n0 + 1
    for q, w in enumerate(want):
        assert dst_d[q].cpu().numpy().tobytes() == w.tobytes(), "group buffer %d" % q


def test_unet_boundary_group_full_size():
    """four feature maps of a U-shaped network on one stage boundary, one launch"""
    ws = [inputs.unet_workload(l) for l in range(4)]
    plans, src, dst, expect = [], [], [], []
    for w in ws:
        D, s = gu.workload_on_device(w)
        p = rs.Plan(w.shape, 2, w.src_mesh, w.src_spec, w.dst_mesh, w.dst_spec)
        plans.append(p)
        src += s
        dst += [torch.zeros(p.local_shape(rs.RS_DST), dtype=D.dtype, device=gu.dev()) for _ in range(p.info.n_dst)]
        expect += [D[idx] for idx in gu.oracle_slices(w.shape, w.dst_mesh, w.dst_spec)]
    g = rs.Plan.group(plans)
    n0 = rs.launch_count()
    g.execute(gu.ptrs(src), gu.ptrs(dst), gu.stream())
    torch.cuda.synchronize()
    assert rs.launch_count() == n0 + 1
    for got, want in zip(dst, expect):
        assert torch.equal(got, want)


def _random_mid_size_task(rng):
    """a seeded task of 48-320 MiB: 2-4 dims, meshes of 2-32 devices, even and uneven extents, inner dims from 16 elements to thousands"""
    ndim = int(rng.integers(2, 5))
    meshes = [(2, 4), (4, 2), (1, 4), (2, 2), (8,), (2,), (4, 4), (4, 8), (2, 3), (1, 1)]

    def side():
        mesh = meshes[int(rng.integers(len(meshes)))]
        axes = list(rng.permutation(len(mesh)))
        spec = []
        for _ in range(ndim):
            take = int(rng.integers(0, 3)) if axes else 0
            mine = [axes.pop() for _ in range(min(take, len(axes)))]
            spec.append("S" + "".join(str(a) for a in mine) if mine else "R")
        return mesh, "".join(spec)
    sm, ss = side()
    dm, ds = side()
    dtype = ["u8", "bf16", "fp32", "i64"][int(rng.integers(4))]
    e = inputs.elem_bytes(dtype)
    inner = int(rng.choice([16, 32, 64, 100, 256, 257, 512, 1000, 2050, 4096, 12288]))
    mids = [int(rng.choice([4, 7, 16, 32, 33, 64, 128, 320])) for _ in range(ndim - 2)]
    target = int(rng.integers(48, 321)) << 20
    outer = max(1, target // (e * inner * int(np.prod(mids or [1]))))
    shape = (outer,) + tuple(mids) + (inner,)
    name = "x:%s:%s:%s:%s:%s:%s" % ("x".join(map(str, shape)), dtype, "x".join(map(str, sm)), ss, "x".join(map(str, dm)), ds)
    return name


@pytest.mark.parametrize("seed", range(96))
def test_random_mid_size_tasks_under_auto(seed):
    """48-320 MiB tasks under AUTO, where the launch rules switch kernels and shapes (tensor maps for short rows, span tiles, source- and
    destination-order segments, paced shapes, both store paths of the shifted kernel): execute and pack -> unpack, every destination byte
    against basic slicing of D with the ORACLE's boxes, padding untouched"""
    rng = np.random.default_rng(5322_2211 + seed)
    w = inputs.get_workload(_random_mid_size_task(rng))
    e = inputs.elem_bytes(w.dtype)
    D, src = gu.workload_on_device(w)
    if D.numel() * e * (1 + do.num_devices(w.dst_mesh)) > (40 << 30):
        pytest.skip("destination side larger than the box")
    p = rs.Plan(w.shape, e, w.src_mesh, w.src_spec, w.dst_mesh, w.dst_spec)
    idx = gu.oracle_slices(w.shape, w.dst_mesh, w.dst_spec)
    local = do.local_shape(w.shape, w.dst_mesh, w.dst_spec)
    want = [gu.padded(D, idx[q], local, 0x5A).view(torch.uint8) for q in range(p.info.n_dst)]
    for route in ("execute", "pack"):
        dst = [torch.empty(tuple(local), dtype=D.dtype, device=gu.dev()) for _ in range(p.info.n_dst)]
        for t in dst:
            t.view(torch.uint8).fill_(0x5A)
        if route == "execute":
            p.execute(gu.ptrs(src), gu.ptrs(dst), gu.stream())
        else:
            arena = torch.empty(max(1, p.info.arena_bytes), dtype=torch.uint8, device=gu.dev())
            p.pack(gu.ptrs(src), arena.data_ptr(), gu.stream())
            p.unpack(arena.data_ptr(), gu.ptrs(dst), gu.stream())
        torch.cuda.synchronize()
        for q in range(p.info.n_dst):
            assert torch.equal(dst[q].view(torch.uint8), want[q]), (w.name, route, q, p.op_info(rs.RS_OP_EXECUTE).path)
