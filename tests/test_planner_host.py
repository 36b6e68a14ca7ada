"""Host logic of libreshard.so on the CPU box (no compute calls, RS_HOST_ONLY plans):
exported symbols, planner (a1..a4) against the plan oracle and the paper's facts, and the flat
task/tile tables (a5) replayed by the TEST-ONLY interpreter tests/table_interp.py against the
C data oracle."""
import os
import re
import subprocess

import numpy as np
import pytest
from hypothesis import given, settings, strategies as st

import golden_io
import table_interp as ti
from oracle import data_oracle as do
from oracle import plan_oracle as po
from paper_2211_05322_b200 import inputs
from paper_2211_05322_b200 import reshard as rs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HOST = rs.RS_HOST_ONLY

LAYOUTS = [
    ((8, 16), (1, 2), "S0,R", (1, 2), "R,S0"),
    ((8, 16), (1, 2), "S1,R", (1, 2), "R,S1"),
    ((4, 8, 16), (2, 4), "S0,R,S1", (2, 4), "S0,S1,R"),
    ((4, 8, 4, 4), (1, 4), "S0,R,R,R", (2, 2), "R,S0,S1,R"),
    ((4, 8, 4, 4), (1, 4), "S1,R,R,R", (2, 2), "R,S0,R,R"),
    ((8, 16, 12), (2, 4), "S0,S1,R", (4, 2), "S1,R,S0"),
    ((8, 8, 4), (2, 4), "R,S01,R", (2, 4), "S01,R,R"),
    ((6, 6, 2), (2, 3), "RRR", (3, 2), "RRR"),
    ((12, 6), (2, 3), "S0,S1", (3, 2), "S0,S1"),
    ((12, 6), (2, 3), "S0,R", (3, 2), "S0,R"),
    ((8, 8, 8), (2, 4), "R,R,S0", (2, 4), "S0,R,R"),
    ((8, 8, 8), (2, 4), "S0,R,R", (2, 4), "R,R,R"),
    ((8, 8, 8), (2, 4), "R,R,R", (2, 4), "S0,S1,R"),
    ((8, 4), (2, 2), "S0,S1", (4,), "S0,R"),
    ((4, 6, 5, 3), (2, 2), "S0,S1,R,R", (2, 2), "S1,R,R,R"),      # odd inner extents: narrow vectors
    ((16, 7), (4,), "S0,R", (2,), "R,R"),
    # uneven partitions (R5): padded shard buffers, short / empty last shards, unequal slices
    ((10,), (3,), "S0", (4,), "S0"),
    ((5, 4), (2, 2), "S0,R", (2, 2), "R,S1"),
    ((7, 9), (2, 4), "S1,S0", (4, 2), "S0,S1"),
    ((7, 5, 3), (2, 3), "S1,R,S0", (3, 2), "R,S0,S1"),
    ((2, 6), (4,), "S0,R", (2,), "S0,R"),
    ((9, 10, 4), (2, 4), "S0,R,R", (3, 4), "S0,R,R"),               # Table 2 case 6 in small
    ((11, 6), (2, 4), "S01,R", (2, 3), "R,S10"),
]


def _plan(shape, e, sm, ss, dm, ds, flags=0, opts=None):
    return rs.Plan(shape, e, sm, ss, dm, ds, flags | HOST, opts)


# ---------------------------------------------------------------- the boundary

def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "reshard.h")).read()
    declared = sorted(set(re.findall(r"RS_API[^;(]*?\b(reshard_\w+)\s*\(", hdr)))
    assert declared == sorted(rs.SYMBOLS)
    out = subprocess.run(["nm", "-D", "--defined-only", rs.LIB_PATH], capture_output=True, text=True, check=True).stdout
    exported = sorted(l.split()[-1] for l in out.splitlines() if " T " in l)
    assert exported == declared                       # nothing else leaks out of the library
    for name in declared:
        assert hasattr(rs._lib(), name)
    assert "sm_100a" in rs.version()


def test_only_sm_100a_code_in_library():
    out = subprocess.run(["cuobjdump", "-lelf", rs.LIB_PATH], capture_output=True, text=True)
    if out.returncode != 0:
        pytest.skip("cuobjdump unavailable")
    archs = set(re.findall(r"sm_\d+a?", out.stdout))
    assert archs == {"sm_100a"}


def test_error_codes():
    def code(*a, **k):
        with pytest.raises(rs.ReshardError) as ei:
            _plan(*a, **k)
        return ei.value.code
    assert code((8, 8), 2, (2, 2), "S0,S0", (2, 2), "R,R") == rs.RS_ESPEC          # axis used twice (R3)
    assert code((8, 8), 2, (2, 2), "S2,R", (2, 2), "R,R") == rs.RS_ESPEC           # axis out of range
    assert code((8, 8), 2, (2, 2), "S0", (2, 2), "R,R") == rs.RS_ESPEC             # too few entries
    assert code((8, 8), 2, (2, 2), "S0,R,R", (2, 2), "R,R") == rs.RS_ESPEC         # too many
    assert code((8, 8), 2, (2, 2), "S,R", (2, 2), "R,R") == rs.RS_ESPEC            # S without axis
    assert code((8, 8), 2, (2, 2), "X,R", (2, 2), "R,R") == rs.RS_ESPEC
    assert code((6, 8), 2, (2, 4), "S1,R", (2, 2), "R,R", rs.RS_EVEN_ONLY) == rs.RS_EDIVIS     # 6 % 4, strict mode (R5)
    assert code((1024, 1024, 512), 2, (2, 4), "S0RR", (3, 4), "S0RR", rs.RS_EVEN_ONLY) == rs.RS_EDIVIS   # Table 2 case 6
    assert _plan((6, 8), 2, (2, 4), "S1,R", (2, 2), "R,R").local_shape(rs.RS_SRC) == (2, 8)    # default: padded last shard
    assert code((8, 8), 3, (2, 2), "R,R", (2, 2), "R,R") == rs.RS_EINVAL           # elem_bytes
    assert code((8, 0), 2, (2, 2), "R,R", (2, 2), "R,R") == rs.RS_EINVAL
    assert code((8, 8), 2, (0, 2), "R,R", (2, 2), "R,R") == rs.RS_EINVAL
    assert code((8, 8), 2, (16, 16), "R,R", (2, 2), "R,R") == rs.RS_EUNSUPPORTED   # > RS_MAX_DEVICES
    p = _plan((8, 8), 2, (2, 2), "R,R", (2, 2), "R,R")
    with pytest.raises(rs.ReshardError) as ei:                                      # host-only plan refuses to run
        p.execute([1] * 4, [1] * 4)
    assert ei.value.code == rs.RS_EINVAL


def test_spec_spellings():
    a = _plan((8, 8, 8), 2, (2, 4), "S01,R,R", (2, 4), "R,S0,S1").slices()
    for text in ("(S01, R, R)", "S^{01}RR", "s01 r r", "[S_01,R,R]"):
        assert _plan((8, 8, 8), 2, (2, 4), text, (2, 4), "RS0S1").slices() == a


# ---------------------------------------------------------------- a1..a3 against the paper and the plan oracle

def test_fig2_worked_example():
    """PAPER.md:62, 86, 90."""
    g = golden_io.load("fig2_example.txt")
    shape = tuple(g["matrix_shape"])
    a0, b0 = g["mesh_a_devices"][0], g["mesh_b_devices"][0]
    D = np.array(g["matrix_values"]).reshape(shape)
    p1 = _plan(shape, 4, g["mesh_a"], g["spec1"], g["mesh_b"], g["spec2"])
    s = p1.slices()
    assert len(s) == g["task1_num_unit_tasks"][0]
    box = tuple(slice(l, h) for l, h in zip(s[0]["lo"], s[0]["hi"]))
    assert D[box].reshape(-1).tolist() == g["task1_first_slice_elements"]
    assert [r + b0 for r in s[0]["receivers"]] == g["task1_first_receivers"]
    for local in (0, 1):                                   # devices 4, 5 hold elements 0..7
        lo, hi = p1.device_box(rs.RS_DST, local)
        assert D[lo[0]:hi[0], lo[1]:hi[1]].reshape(-1).tolist() == g["spec2_device4_elements"]
    p2 = _plan(shape, 4, g["mesh_b"], g["spec2"], g["mesh_a"], g["spec3"])
    s = p2.slices()
    assert len(s) == g["task2_num_unit_tasks"][0]
    box = tuple(slice(l, h) for l, h in zip(s[0]["lo"], s[0]["hi"]))
    assert D[box].reshape(-1).tolist() == g["task2_first_slice_elements"]
    assert [r + a0 for r in s[0]["receivers"]] == g["task2_first_receivers"]
    assert [x + b0 for x in s[0]["senders"]] == [4, 5]


def test_table2_facts():
    """PAPER.md:282 (case 4: 64 unit tasks), 320 (case 8: one broadcast; case 2 naive: first node)."""
    g = golden_io.load("table2_facts.txt")
    shape = tuple(g["tensor_shape"])

    def plan(case, flags=0):
        ss, ds, sm, dm = inputs.TABLE2[case]
        return _plan(shape, 2, sm, ss, dm, ds, flags)
    assert plan(4).info.n_slices == g["case4_num_unit_tasks"][0]
    p8 = plan(8)
    assert p8.info.n_slices == g["case8_num_unit_tasks"][0]
    assert len(p8.slice(0)["senders"]) == 6 and len(p8.slice(0)["receivers"]) == 6
    naive = plan(2, rs.RS_LB_NAIVE)
    assert {s["sender"] // 4 for s in naive.slices()} == {g["case2_naive_sender_node"][0]}
    assert naive.info.max_sender_bytes == naive.info.tensor_bytes            # everything from one device
    greedy = plan(2)
    assert greedy.info.max_sender_bytes == greedy.info.tensor_bytes // 2
    for case in (1, 2, 3, 4, 5, 7, 8, 9):
        p = plan(case)
        assert sum(p.sender_bytes()) == p.info.tensor_bytes                  # lower bound


@pytest.mark.parametrize("shape,sm,ss,dm,ds", LAYOUTS)
def test_slices_match_plan_oracle(shape, sm, ss, dm, ds):
    p = _plan(shape, 2, sm, ss, dm, ds)
    tasks = po.unit_tasks(shape, sm, ss, dm, ds)
    got = p.slices()
    assert len(got) == len(tasks) == p.info.n_slices
    for g, t in zip(got, tasks):
        assert g["lo"] == t["lo"] and g["hi"] == t["hi"]
        assert g["senders"] == t["senders"] and g["receivers"] == t["receivers"]
        assert g["sender"] in t["senders"]                                   # Eq. 2
    for side, mesh, spec in ((rs.RS_SRC, sm, ss), (rs.RS_DST, dm, ds)):
        assert p.local_shape(side) == do.local_shape(shape, mesh, spec)
        for r in range(po.n_devices(mesh)):
            assert p.device_box(side, r) == po.tile_box(shape, mesh, spec, r)
    assert p.info.write_bytes == sum(t["size"] * len(t["receivers"]) for t in tasks) * 2
    assert p.info.unique_read_bytes == int(np.prod(shape)) * 2


# ---------------------------------------------------------------- a4: sender choice

@pytest.mark.parametrize("shape,sm,ss,dm,ds", LAYOUTS)
def test_sender_choice_objective(shape, sm, ss, dm, ds):
    tasks = po.unit_tasks(shape, sm, ss, dm, ds)
    n_src = po.n_devices(sm)
    greedy = _plan(shape, 2, sm, ss, dm, ds)
    naive = _plan(shape, 2, sm, ss, dm, ds, rs.RS_LB_NAIVE)
    assert [s["sender"] for s in naive.slices()] == po.naive_senders(tasks)
    assert naive.info.max_sender_bytes == po.max_load(tasks, po.naive_senders(tasks), n_src, 2)
    loads = po.sender_loads(tasks, [s["sender"] for s in greedy.slices()], n_src, 2)
    assert loads == greedy.sender_bytes() and max(loads) == greedy.info.max_sender_bytes
    assert greedy.info.max_sender_bytes <= po.max_load(tasks, po.greedy_senders(tasks, 2), n_src, 2)
    assert greedy.info.max_sender_bytes <= naive.info.max_sender_bytes
    try:
        opt = po.bruteforce_optimum(tasks, n_src, 2)
    except ValueError:
        return
    assert greedy.info.max_sender_bytes == opt            # BASELINE: equals the brute-force optimum


def test_unequal_slices_need_the_exact_finish():
    """2-way x 3-way cuts give slices of 3 sizes; LPT alone can miss the optimum (R9)."""
    shape, sm, ss, dm, ds = (12, 12), (2, 3), "S0,R", (3, 2), "S0,S1"
    for shape, sm, ss, dm, ds in [((12, 12), (2, 3), "S0,R", (3, 2), "S0,S1"), ((12, 6), (2, 3), "S0,R", (3, 2), "S0,R"),
                                  ((24, 12), (4, 3), "R,R", (3, 4), "S0,S1")]:
        tasks = po.unit_tasks(shape, sm, ss, dm, ds)
        p = _plan(shape, 1, sm, ss, dm, ds)
        try:
            assert p.info.max_sender_bytes == po.bruteforce_optimum(tasks, po.n_devices(sm), 1)
        except ValueError:
            assert p.info.max_sender_bytes <= po.max_load(tasks, po.greedy_senders(tasks, 1), po.n_devices(sm), 1)


# ---------------------------------------------------------------- a5: tables replayed against the data oracle

def _bytes(a):
    return np.ascontiguousarray(a).view(np.uint8).reshape(-1)


def _valid_bytes(shape, mesh, spec, e):
    """per device: 1 for every byte of the padded shard buffer that holds an element of D (oracle boxes)"""
    out = []
    local = do.local_shape(shape, mesh, spec)
    for r in range(do.num_devices(mesh)):
        lo, hi = do.device_box(shape, mesh, spec, r)
        m = np.zeros(local + (e,), np.int32)
        m[tuple(slice(0, h - l) for l, h in zip(lo, hi))] = 1
        out.append(m.reshape(-1))
    return out


def _check_tables(shape, dtype, sm, ss, dm, ds, flags=0, tuning=None, opts=None):
    e = np.dtype(dtype).itemsize
    once = _valid_bytes(shape, dm, ds, e)
    if tuning:
        opts = dict(opts or {}, tuning=tuning)
    p = _plan(shape, e, sm, ss, dm, ds, flags, opts)
    for op in (rs.RS_OP_EXECUTE, rs.RS_OP_PACK, rs.RS_OP_UNPACK, rs.RS_OP_EXECUTE_SLABS):
        mine, theirs = ti.tiles(p, op), ti.lib_tiles(p, op)       # the decode restated here vs the routine the kernels run
        assert mine.tobytes() == theirs.tobytes(), "tile decode of op %d differs" % op
    D = (np.arange(int(np.prod(shape)), dtype=np.int64) * 2654435761 % 251 + 1).astype(dtype).reshape(shape)
    src = do.shards_from_global(D, sm, ss)
    want = do.reshard(shape, sm, ss, dm, ds, src)
    n_dst = len(want)
    # execute
    dst = [np.zeros(want[0].nbytes, np.uint8) for _ in range(n_dst)]
    cnt = [np.zeros(want[0].nbytes, np.int32) for _ in range(n_dst)]
    ti.replay(p, rs.RS_OP_EXECUTE, [_bytes(s) for s in src], dst, cnt)
    for q in range(n_dst):
        assert np.array_equal(dst[q], _bytes(want[q])), "execute tables differ from the oracle on device %d" % q
        assert np.array_equal(cnt[q], once[q]), "execute tables do not write every byte exactly once (padding: never)"
    # the slab-cut execute table that reshard_execute_host pipelines over: same result, same exactly-once
    dst3 = [np.zeros(want[0].nbytes, np.uint8) for _ in range(n_dst)]
    cnt3 = [np.zeros(want[0].nbytes, np.int32) for _ in range(n_dst)]
    ti.replay(p, rs.RS_OP_EXECUTE_SLABS, [_bytes(s) for s in src], dst3, cnt3)
    for q in range(n_dst):
        assert np.array_equal(dst3[q], _bytes(want[q])) and np.array_equal(cnt3[q], once[q])
    # pack -> message contents as the plan oracle states them -> unpack
    arena = [np.zeros(p.info.arena_bytes, np.uint8)]
    acnt = [np.zeros(p.info.arena_bytes, np.int32)]
    ti.replay(p, rs.RS_OP_PACK, [_bytes(s) for s in src], arena, acnt)
    tasks = po.unit_tasks(shape, sm, ss, dm, ds)
    senders = [s["sender"] for s in p.slices()]
    msgs = p.messages()
    ref = po.pack_messages(shape, sm, ss, tasks, senders, src)
    assert [(m["sender"], m["receiver"]) for m in msgs] == [(s, r) for s, r, _ in ref]
    covered = np.zeros(p.info.arena_bytes, bool)
    for m, (s, r, payload) in zip(msgs, ref):
        assert m["bytes"] == payload.nbytes and m["offset"] % 256 == 0
        assert np.array_equal(arena[0][m["offset"]:m["offset"] + m["bytes"]], _bytes(payload))
        covered[m["offset"]:m["offset"] + m["bytes"]] = True
    assert sum(m["bytes"] for m in msgs) == p.info.write_bytes
    assert np.array_equal(acnt[0] == 1, covered) and (acnt[0][~covered] == 0).all()
    dst2 = [np.zeros(want[0].nbytes, np.uint8) for _ in range(n_dst)]
    cnt2 = [np.zeros(want[0].nbytes, np.int32) for _ in range(n_dst)]
    ti.replay(p, rs.RS_OP_UNPACK, arena, dst2, cnt2)
    for q in range(n_dst):
        assert np.array_equal(dst2[q], _bytes(want[q]))
        assert np.array_equal(cnt2[q], once[q])
    return p


@pytest.mark.parametrize("shape,sm,ss,dm,ds", LAYOUTS)
@pytest.mark.parametrize("dtype", [np.uint8, np.int16, np.int64])
def test_tables_replay_equals_oracle(shape, sm, ss, dm, ds, dtype):
    _check_tables(shape, dtype, sm, ss, dm, ds)


@pytest.mark.parametrize("tile", [128, 256, 1024])
@pytest.mark.parametrize("path", [rs.RS_PATH_LSU, rs.RS_PATH_BULK])
def test_tables_with_tiny_tiles_cover_every_tile_kind(tile, path):
    """small tile sizes force column-split rows, FAST row groups and GENERIC tiles at test sizes"""
    tuning = {"lsu_tile_bytes": tile, "bulk_tile_bytes": tile}
    kinds = set()
    for shape, sm, ss, dm, ds in [((4, 6, 64), (2, 2), "S0,S1,R", (2, 2), "S1,S0,R"),      # long runs -> column split
                                  ((8, 16, 16), (2, 4), "S0,R,S1", (2, 4), "S0,S1,R"),     # short runs, wide ext0
                                  ((8, 6, 2, 16), (2, 2), "S0,R,R,S1", (2, 2), "R,S0,R,S1"),  # ext0 = 2 -> GENERIC
                                  ((6, 4, 2, 3, 8), (2,), "R,R,R,R,S0", (2,), "S0,R,R,R,R")]:
        p = _check_tables(shape, np.int32, sm, ss, dm, ds, flags=path, tuning=tuning)
        tiles = ti.tiles(p, rs.RS_OP_EXECUTE)
        for t in tiles:
            kinds.add("split" if t["n_rows"] == 1 and t["flags"] & 1 else "fast" if t["flags"] & 1 else "generic")
        assert p.op_info(rs.RS_OP_EXECUTE).tile_bytes <= max(tile, 128)
        assert all(int(t["n_rows"]) * int(t["col_bytes"]) <= max(tile, 128) for t in tiles)
    assert kinds == {"split", "fast", "generic"}


def test_alignment_class_and_path_choice():
    p = _plan((16, 1024, 4096), 2, (2, 4), "S0,R,S1", (2, 4), "S0,S1,R")
    oi = p.op_info(rs.RS_OP_EXECUTE)
    assert oi.vec_bytes == 16 and oi.path == rs.RS_PATH_TMAP and oi.min_run_bytes == 2048     # config 2: 2 KiB rows, 256 MiB moved
    assert oi.read_bytes == p.info.tensor_bytes and oi.write_bytes == p.info.tensor_bytes
    p = _plan((4, 6, 5, 3), 2, (2, 2), "S0,S1,R,R", (2, 2), "S1,R,R,R")          # runs of 15 elements = 30 B
    oi = p.op_info(rs.RS_OP_EXECUTE)
    assert oi.vec_bytes == 2 and oi.path == rs.RS_PATH_LSU
    p = _plan((4, 6, 5, 3), 2, (2, 2), "S0,S1,R,R", (2, 2), "S1,R,R,R", rs.RS_PATH_BULK)
    assert p.op_info(rs.RS_OP_EXECUTE).path == rs.RS_PATH_BULK_SHIFT              # TMA stores need 16-byte everything
    p = _plan((32, 2048, 12290), 2, (2, 4), "S0,S1,R", (4, 2), "S1,R,S0")           # long runs of 6145 B: 2-byte class
    oi = p.op_info(rs.RS_OP_EXECUTE)
    assert oi.vec_bytes == 2 and oi.path == rs.RS_PATH_BULK_SHIFT and oi.smem_bytes <= 227 * 1024
    p = _plan((16, 1024, 4096), 2, (2, 4), "S0,R,S1", (2, 4), "S0,S1,R", rs.RS_PATH_BULK_SHIFT)
    assert p.op_info(rs.RS_OP_EXECUTE).path == rs.RS_PATH_BULK_SHIFT              # forceable on aligned layouts too
    p = _plan((8, 16), 4, (1, 2), "S1,R", (1, 2), "R,S1")                         # c1i: 32-byte runs
    assert p.op_info(rs.RS_OP_EXECUTE).path == rs.RS_PATH_LSU
    assert _plan((8, 16), 4, (1, 2), "S1,R", (1, 2), "R,S1", rs.RS_PATH_BULK).op_info(0).path == rs.RS_PATH_BULK


@pytest.mark.parametrize("name", ["c2", "c3", "c3i", "c3ii", "c4", "t2_4", "sweep_P5_m8_1024MiB", "sweep_P2_m8_4096MiB"])
def test_full_size_tables_cover_every_byte_once(name):
    """at BASELINE sizes: interval arithmetic over the tile table instead of replaying bytes"""
    w = inputs.get_workload(name)
    p = _plan(w.shape, inputs.elem_bytes(w.dtype), w.src_mesh, w.src_spec, w.dst_mesh, w.dst_spec)
    for op in (rs.RS_OP_EXECUTE, rs.RS_OP_PACK, rs.RS_OP_UNPACK):
        tasks, dsts, _segs = ti.tables(p, op)
        tiles = ti.tiles(p, op)
        assert tiles.tobytes() == ti.lib_tiles(p, op).tobytes()
        oi = p.op_info(op)
        assert oi.n_tiles == len(tiles) and oi.table_bytes == 224 * oi.n_tasks + 16 * oi.n_dsts + 16 * oi.n_segs
        T = tasks[tiles["task"]]
        nbytes = tiles["n_rows"].astype(np.int64) * tiles["col_bytes"].astype(np.int64)
        assert int(nbytes.sum()) == oi.read_bytes
        assert int((nbytes * T["k"]).sum()) == oi.write_bytes
        assert int(nbytes.max()) <= oi.tile_bytes
        assert (tiles["col_bytes"] % 16 == 0).all() and oi.vec_bytes == 16
        # the largest byte any FAST tile touches stays inside its buffers
        fast = (tiles["flags"] & 1) == 1
        assert fast.all()
        last_s = T["src_off"] + tiles["a"].astype(np.int64) + (tiles["n_rows"].astype(np.int64) - 1) * T["sstride"][:, 0] + tiles["col_bytes"]
        src_cap = p.info.src_shard_bytes if op != rs.RS_OP_UNPACK else p.info.arena_bytes
        assert int(last_s.max()) <= src_cap
        dst_cap = p.info.dst_shard_bytes if op != rs.RS_OP_PACK else p.info.arena_bytes
        for j in range(int(T["k"].max())):
            has = T["k"] > j
            D = dsts[(T["dst_first"] + j)[has]]
            last_d = D["off"] + tiles["b"].astype(np.int64)[has] + (tiles["n_rows"].astype(np.int64)[has] - 1) * T["dstride"][:, 0][has] + tiles["col_bytes"][has]
            assert int(last_d.max()) <= dst_cap


_SPECS2 = ["R", "S0", "S1", "S01", "S10"]


@st.composite
def _layouts(draw):
    ndim = draw(st.integers(1, 4))

    def side():
        mesh = draw(st.sampled_from([(1, 2), (2, 2), (2, 4), (4, 2), (2, 3), (3, 2), (1, 4), (4,), (3,)]))
        while True:
            spec = [draw(st.sampled_from(_SPECS2)) for _ in range(ndim)]
            axes = "".join(s[1:] for s in spec)
            if len(set(axes)) == len(axes) and all(int(a) < len(mesh) for a in axes):
                return mesh, ",".join(spec)
    sm, ss = side()
    dm, ds = side()
    shape = tuple(draw(st.sampled_from([12, 24, 7, 10, 1])) for _ in range(ndim))     # even and uneven (R5) splits
    if ndim >= 3:
        shape = tuple(min(s, 12) for s in shape)
    return shape, sm, ss, dm, ds, draw(st.sampled_from([np.uint8, np.int16, np.int32])), draw(st.sampled_from([128, 512, 16384]))


@settings(max_examples=60, deadline=None)
@given(_layouts())
def test_random_layouts_tables_equal_oracle(layout):
    shape, sm, ss, dm, ds, dtype, tile = layout
    even = all(l % k == 0 for mesh, spec in ((sm, ss), (dm, ds))
               for l, k in zip(shape, po.degrees(shape, mesh, po.parse_spec(spec, len(shape), len(mesh)))))
    if not even:
        with pytest.raises(rs.ReshardError) as ei:
            _plan(shape, 1, sm, ss, dm, ds, rs.RS_EVEN_ONLY)
        assert ei.value.code == rs.RS_EDIVIS
    _check_tables(shape, dtype, sm, ss, dm, ds, tuning={"lsu_tile_bytes": tile, "bulk_tile_bytes": tile})


def test_slab_table_cuts_dim0_when_large():
    """>= 8 MiB per slab, at most 16 slabs, never more than l_0"""
    p = _plan((32, 2048, 12288), 2, (2, 4), "S0,S1,R", (4, 2), "S1,R,S0")
    assert p.op_info(rs.RS_OP_EXECUTE_SLABS).n_tasks == 16 * 32 // 2      # 16 slabs x the 16 slices each slab meets
    p = _plan((6, 1024, 2048), 2, (2, 2), "S0,R,S1", (3,), "S0,R,R")       # 24 MiB -> 3 slabs over l_0 = 6
    tiles = ti.tiles(p, rs.RS_OP_EXECUTE_SLABS)
    assert p.op_info(rs.RS_OP_EXECUTE_SLABS).read_bytes == p.info.tensor_bytes
    assert int((tiles["n_rows"].astype(np.int64) * tiles["col_bytes"]).sum()) == p.info.tensor_bytes
    p = _plan((8, 16), 4, (1, 2), "S1,R", (1, 2), "R,S1")                  # tiny: one slab == the execute table
    assert p.op_info(rs.RS_OP_EXECUTE_SLABS).n_tasks == p.op_info(rs.RS_OP_EXECUTE).n_tasks


# ---------------------------------------------------------------- alternative strategies

@pytest.mark.parametrize("shape,sm,ss,dm,ds", LAYOUTS)
def test_strategy_tables_replay_equals_oracle(shape, sm, ss, dm, ds):
    """send/recv and scatter + all-gather reach the oracle's result; their byte counts are 2k per slice byte"""
    dtype, e = np.int16, 2
    p = _plan(shape, e, sm, ss, dm, ds, rs.RS_WITH_STRATEGIES)
    D = (np.arange(int(np.prod(shape)), dtype=np.int64) * 2654435761 % 251 + 1).astype(dtype).reshape(shape)
    src = do.shards_from_global(D, sm, ss)
    want = do.reshard(shape, sm, ss, dm, ds, src)
    once = _valid_bytes(shape, dm, ds, e)
    n_dst, r_B = len(want), p.info.write_bytes // p.info.tensor_bytes
    # send/recv: one launch, every destination byte written once, the source read r_B times
    dst = [np.zeros(want[0].nbytes, np.uint8) for _ in range(n_dst)]
    cnt = [np.zeros(want[0].nbytes, np.int32) for _ in range(n_dst)]
    ti.replay(p, rs.RS_OP_SENDRECV, [_bytes(s) for s in src], dst, cnt)
    for q in range(n_dst):
        assert np.array_equal(dst[q], _bytes(want[q])) and np.array_equal(cnt[q], once[q])
    oi = p.op_info(rs.RS_OP_SENDRECV)
    assert oi.read_bytes == oi.write_bytes == p.info.tensor_bytes * r_B and oi.n_tasks == sum(len(s["receivers"]) for s in p.slices())
    # all-gather: phase 1 writes every part once somewhere, phase 2 (reading destination shards) completes every shard
    dst = [np.zeros(want[0].nbytes, np.uint8) for _ in range(n_dst)]
    cnt = [np.zeros(want[0].nbytes, np.int32) for _ in range(n_dst)]
    ti.replay(p, rs.RS_OP_AG_SCATTER, [_bytes(s) for s in src], dst, cnt)
    assert sum(int(c.sum()) for c in cnt) == p.info.tensor_bytes            # one copy of D in total after the scatter
    ti.replay(p, rs.RS_OP_AG_GATHER, dst, dst, cnt)
    for q in range(n_dst):
        assert np.array_equal(dst[q], _bytes(want[q])) and np.array_equal(cnt[q], once[q])
    a, g = p.op_info(rs.RS_OP_AG_SCATTER), p.op_info(rs.RS_OP_AG_GATHER)
    assert a.read_bytes == a.write_bytes == p.info.tensor_bytes
    assert g.read_bytes == g.write_bytes == p.info.tensor_bytes * (r_B - 1)
    # local all-gather: per receiver host; with one device per host it degenerates to send/recv bytes
    for dph in (1, 2, 4):
        pl = _plan(shape, e, sm, ss, dm, ds, rs.RS_WITH_STRATEGIES, dict(dst_devices_per_host=dph))
        dst = [np.zeros(want[0].nbytes, np.uint8) for _ in range(n_dst)]
        cnt = [np.zeros(want[0].nbytes, np.int32) for _ in range(n_dst)]
        ti.replay(pl, rs.RS_OP_AGL_SCATTER, [_bytes(s) for s in src], dst, cnt)
        hosts_per_slice = [len({r // dph for r in sl["receivers"]}) for sl in pl.slices()]
        slice_bytes = [int(np.prod([h - l for l, h in zip(sl["lo"], sl["hi"])])) * e for sl in pl.slices()]
        assert sum(int(c.sum()) for c in cnt) == sum(h * b for h, b in zip(hosts_per_slice, slice_bytes))   # one copy per HOST
        assert pl.op_info(rs.RS_OP_AGL_SCATTER).read_bytes == sum(h * b for h, b in zip(hosts_per_slice, slice_bytes))
        ti.replay(pl, rs.RS_OP_AGL_GATHER, dst, dst, cnt)
        for q in range(n_dst):
            assert np.array_equal(dst[q], _bytes(want[q])) and np.array_equal(cnt[q], once[q])
        ls, lg = pl.op_info(rs.RS_OP_AGL_SCATTER), pl.op_info(rs.RS_OP_AGL_GATHER)
        assert ls.write_bytes + lg.write_bytes == pl.info.write_bytes
    # without the flag the tables are not built
    assert _plan(shape, e, sm, ss, dm, ds).op_info(rs.RS_OP_SENDRECV).n_tasks == 0


MAXIMA = [
    ((2, 3, 2, 2, 4, 2, 2, 6), (2, 2, 2, 2), "S0,R,S1,R,S2,R,R,S3", (2, 2, 2, 2), "R,S3,R,S2,R,S1,S0,R"),   # RS_MAX_NDIM, RS_MAX_MESH_NDIM
    ((128, 4), (128,), "S0,R", (2, 4, 4, 4), "R,S0123"),                                                    # RS_MAX_DEVICES on both sides
    ((256, 2), (1,), "R,R", (128,), "R,R"),                                                                  # one slice, 128 receivers
]


@pytest.mark.parametrize("shape,sm,ss,dm,ds", MAXIMA)
def test_maximum_ranks_and_device_counts(shape, sm, ss, dm, ds):
    _check_tables(shape, np.int16, sm, ss, dm, ds)
    with pytest.raises(rs.ReshardError) as ei:
        _plan(shape + (2,) * (9 - len(shape)), 2, sm, ss + ",R" * (9 - len(shape)), dm, ds + ",R" * (9 - len(shape)))
    assert ei.value.code == rs.RS_EINVAL                      # more than RS_MAX_NDIM dims


def test_launch_shapes_follow_the_measured_rules():
    """what AUTO picks for the benchmark workloads (148-SM part)"""
    def shape_of(name, op=rs.RS_OP_EXECUTE, **opts):
        w = inputs.get_workload(name)
        p = _plan(w.shape, inputs.elem_bytes(w.dtype), w.src_mesh, w.src_spec, w.dst_mesh, w.dst_spec, 0, opts or None)
        o = p.op_info(op)
        return o.path, o.grid, o.block, o.pace_permille
    assert shape_of("c4") == (rs.RS_PATH_BULK, 132, 128, 860)                     # large 1 : 1 operations: 4 warps x 12 KiB on 132 SMs, paced
    assert shape_of("sweep_P1_m8_1024MiB") == (rs.RS_PATH_BULK, 132, 128, 860)    # ... rows of 2 KiB (holds under power-limited clocks)
    assert shape_of("sweep_P2_m8_1024MiB", rs.RS_OP_UNPACK) == (rs.RS_PATH_BULK, 132, 128, 860)   # ... 4 KiB rows (2 unpaced warps: 6.6 TB/s idle, 4.5 hot)
    assert shape_of("x:256x2048x1024:bf16:2x4:S0RS1:2x4:S0S1R") == (rs.RS_PATH_BULK, 132, 256, 860)   # ... rows of 512 bytes: 8 warps x 6 KiB
    assert shape_of("x:64x2048x4096:bf16:4x8:S0S1R:8x4:S1RS0") == (rs.RS_PATH_BULK, 132, 128, 860)    # ... rows of 1 KiB
    assert shape_of("sweep_P3_m8_256MiB") == (rs.RS_PATH_BULK, 132, 128, 860)     # ... from 384 MiB moved on
    assert shape_of("sweep_P3_m8_128MiB") == (rs.RS_PATH_BULK, 148, 64, 880)      # below: 2 warps on every SM, paced when the runs are >= 1 MiB and 128 MiB move
    assert shape_of("sweep_P3_m8_32MiB") == (rs.RS_PATH_BULK, 148, 64, 0)
    assert shape_of("c2", rs.RS_OP_PACK) == (rs.RS_PATH_BULK, 148, 64, 0)         # 128 + 128 MiB, under the WIDE_11 size: 2 unpaced warps on every SM
    assert shape_of("sweep_P5_m8_1024MiB") == (rs.RS_PATH_BULK, 148, 64, 825)     # 1 read + 8 writes: every SM, rate matched
    assert shape_of("sweep_P5_m8_1024MiB", rs.RS_OP_UNPACK) == (rs.RS_PATH_BULK, 132, 128, 860)   # its unpack is a 1 : 1 copy of 512 MiB runs
    assert shape_of("fig5_1x1") == (rs.RS_PATH_BULK, 132, 128, 860)               # one sender, one receiver, one 1 GiB run
    assert shape_of("t2_4") == (rs.RS_PATH_BULK, 132, 128, 860)                   # 128 KiB runs, 1 : 1
    assert shape_of("sweep_P5_m8_16MiB") == (rs.RS_PATH_BULK, 148, 128, 825)      # write-heavy, 144 MiB moved: paced, 4 warps
    assert shape_of("t2_9") == (rs.RS_PATH_BULK, 148, 256, 820)                   # 512-byte runs, 1 + 4: 8 warps; rows adjacent in the receivers
    assert shape_of("u4") == (rs.RS_PATH_BULK_SHIFT, 148, 256, 850)               # nothing aligned, 6 KiB rows: 8 warps, bulk stores, paced
    assert shape_of("u1") == (rs.RS_PATH_BULK_SHIFT, 148, 256, 850)               # nothing aligned, 2 KiB rows: 8 warps, register stores, paced
    assert shape_of("x:64x2046x4100:bf16:2x4:S0RS1:2x4:S0RR") == (rs.RS_PATH_BULK_SHIFT, 148, 256, 800)   # ... to 4 receivers: a lower target
    assert shape_of("x:107101x257:i64:1x2:RS1:2x1:S0R")[::3] == (rs.RS_PATH_BULK_SHIFT, 0)                # ... rows of 1 KiB: issue-bound, unpaced
    assert shape_of("c2") == (rs.RS_PATH_TMAP, 148, 128, 860)                     # 256 MiB moved in 2 KiB rows: tensor-map copies, 4 warps, paced
    assert shape_of("sweep_P1_m8_1024MiB")[0] == shape_of("sweep_P2_m8_64MiB")[0] == rs.RS_PATH_BULK   # too large / rows of 4 KiB
    assert shape_of("c3") == (rs.RS_PATH_BULK, 148, 64, 0)                        # 20 + 20 MiB: the TMA ring from 32 MiB moved on
    assert shape_of("sweep_P1_m8_16MiB")[:2] == (rs.RS_PATH_LSU, 4 * 148)         # small operations: register path, 4 CTAs per SM
    assert shape_of("sweep_P1_m8_1MiB")[0] == rs.RS_PATH_LSU
    assert shape_of("r128") == (rs.RS_PATH_TMAP, 132, 128, 860)                   # 128-byte rows at 1 + 1 GiB: boxes of 64 rows, paced, 132 of 148 SMs like every large 1 : 1 operation
    assert shape_of("r128m") == (rs.RS_PATH_TMAP, 148, 128, 775)                  # ... 1 + 4 GiB
    assert shape_of("r128", rs.RS_OP_PACK)[0] == rs.RS_PATH_BULK                  # its pack copies whole 64 KiB runs
    p = _plan((262144, 4, 64), 2, (2,), "R,R,S0", (2,), "R,S0,R", 0)              # 64-byte rows, but only 2 per span: no box fits
    assert p.op_info(rs.RS_OP_EXECUTE).path == rs.RS_PATH_LSU                     # ... so AUTO falls back to the register path
    assert shape_of("c4", max_ctas=48) == (rs.RS_PATH_BULK, 48, 128, 0)           # capped: more warps per CTA
    assert shape_of("sweep_P5_m8_1024MiB", tuning=dict(pace_permille=-1))[3] == 0  # rate matching can be switched off


def test_plan_group_merges_execute_tables():
    """reshard_plan_group: the members' execute tables in one table, buffer ids shifted; replay equals every member's oracle result"""
    members = [((4, 8, 16), np.int16, (2, 4), "S0,R,S1", (2, 4), "S0,S1,R"),
               ((8, 8, 8), np.int16, (2, 4), "S0,R,R", (2, 4), "R,R,R"),
               ((7, 9), np.int16, (2, 4), "S1,S0", (4, 2), "S0,S1"),
               ((16, 7), np.int16, (4,), "S0,R", (2,), "R,R")]
    plans, srcs, wants = [], [], []
    for shape, dt, sm, ss, dm, ds in members:
        plans.append(_plan(shape, 2, sm, ss, dm, ds))
        D = (np.arange(int(np.prod(shape)), dtype=np.int64) * 2654435761 % 251 + len(plans)).astype(dt).reshape(shape)
        src = do.shards_from_global(D, sm, ss)
        srcs += [_bytes(x) for x in src]
        wants += [_bytes(w) for w in do.reshard(shape, sm, ss, dm, ds, src)]
    g = rs.Plan.group(plans, HOST)
    assert g.info.n_src == len(srcs) == 28 and g.info.n_dst == len(wants) == 26
    assert g.info.unique_read_bytes == sum(p.info.tensor_bytes for p in plans)
    assert g.info.write_bytes == sum(p.info.write_bytes for p in plans)
    assert g.op_info(rs.RS_OP_EXECUTE).n_tasks == sum(p.info.n_slices for p in plans)
    dst = [np.zeros(w.size, np.uint8) for w in wants]
    ti.replay(g, rs.RS_OP_EXECUTE, srcs, dst)
    for q, w in enumerate(wants):
        assert np.array_equal(dst[q], w), "group buffer %d" % q
    for call in (lambda: g.pack([1] * 28, 1), lambda: g.local_shape(rs.RS_SRC), lambda: g.schedule(), lambda: rs.Plan.group([g], HOST)):
        with pytest.raises(rs.ReshardError):
            call()
    big = [_plan((256, 2), 4, (1,), "R,R", (128,), "R,R")] * 2          # 256 destination shards: too many for one launch
    with pytest.raises(rs.ReshardError) as ei:
        rs.Plan.group(big, HOST)
    assert ei.value.code == rs.RS_EUNSUPPORTED


def test_plan_is_o_slices_not_o_bytes():
    """PAPER.md:482-492 (App. B.2): the plan is the slice list, nothing finer.  Table bytes and plan time do not
    grow with the tensor: tiles are decoded on the device (csrc/tables.h), never stored."""
    import time
    sizes = {}
    for mib in (1, 64, 1024, 4096):
        w = inputs.sweep_workload("P1", "m8", mib << 20)
        p = _plan(w.shape, 2, w.src_mesh, w.src_spec, w.dst_mesh, w.dst_spec)
        sizes[mib] = [p.op_info(op).table_bytes for op in (rs.RS_OP_EXECUTE, rs.RS_OP_PACK, rs.RS_OP_UNPACK)]
        assert p.op_info(rs.RS_OP_EXECUTE).n_tiles >= (mib << 20) // 16384
    assert sizes[1024] == sizes[4096] and max(max(v) for v in sizes.values()) <= 32 * (224 + 16 + 16)   # 32 unit tasks: a task, a destination
    # and at most one segment each (slices that share rows form one segment, so a small tensor with short runs may have fewer)
    for name in ("c1", "c2", "c3", "c3i", "c3ii", "c4", "sweep_P5_m8_4096MiB", "sweep_P1_m8_4096MiB", "t2_4"):
        w = inputs.get_workload(name)
        e = inputs.elem_bytes(w.dtype)
        _plan(w.shape, e, w.src_mesh, w.src_spec, w.dst_mesh, w.dst_spec)                    # warm
        t0 = time.perf_counter()
        p = _plan(w.shape, e, w.src_mesh, w.src_spec, w.dst_mesh, w.dst_spec)
        dt = time.perf_counter() - t0
        for op in (rs.RS_OP_EXECUTE, rs.RS_OP_PACK, rs.RS_OP_UNPACK):
            assert p.op_info(op).table_bytes < 64 << 10, (name, op)
        assert dt < 0.02, "%s: host plan took %.1f ms" % (name, dt * 1e3)                      # round 1: 18-225 ms


def test_destination_order_segments():
    """slices that share destination rows (config 2: four slices fill a quarter of every row of a receiver's
    shard) form one segment walked round-robin = in destination address order; rs_tuning.task_order and a
    schedule (tables in order of S_i) switch it off"""
    w = inputs.get_workload("c2")
    p = _plan(w.shape, 2, w.src_mesh, w.src_spec, w.dst_mesh, w.dst_spec)
    tasks, dsts, segs = ti.tables(p, rs.RS_OP_EXECUTE)
    assert len(tasks) == 32 and len(segs) == 8 and (segs["n_members"] == 4).all()
    tiles = ti.tiles(p, rs.RS_OP_EXECUTE)
    T = tasks[tiles["task"]]
    key = dsts[T["dst_first"]]["buf"].astype(np.int64) * (1 << 40) + dsts[T["dst_first"]]["off"] + tiles["b"].astype(np.int64)
    assert (np.diff(key) > 0).all()                                   # ascending (buffer, address)
    for opts in (dict(tuning=dict(task_order=1)), dict(schedule=rs.RS_SCHED_LOAD_BALANCE)):
        q = _plan(w.shape, 2, w.src_mesh, w.src_spec, w.dst_mesh, w.dst_spec, 0, opts)
        _t, _d, segs = ti.tables(q, rs.RS_OP_EXECUTE)
        assert len(segs) == 32 and (segs["n_members"] == 1).all()
        assert (np.diff(ti.tiles(q, rs.RS_OP_EXECUTE)["task"].astype(np.int64)) >= 0).all()   # task by task
    _t, _d, segs = ti.tables(p, rs.RS_OP_PACK)                        # pack writes dense messages: nothing to interleave
    assert (segs["n_members"] == 1).all()
