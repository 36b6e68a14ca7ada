"""TEST-ONLY interpreter of the library's flat task tables (reshard_op_tables).

A plan stores tasks and segments, never tiles (csrc/tables.h): the kernels DECODE tile t where they
need it.  This module restates that decode in numpy, from the layout comments of tables.h alone, and
replays the resulting tile list on numpy byte buffers exactly as the kernels are specified to, so
the host planner's tables can be checked against the oracle on the CPU box.  The library's own
decode (reshard_op_tiles: the routine the kernels run, compiled for the host) is compared with
this one tile by tile.  Not a product path; nothing under paper_2211_05322_b200/ imports it.
"""
import numpy as np

TASK = np.dtype([("src_off", "<i8"), ("run_bytes", "<i8"), ("src_buf", "<i4"), ("k", "<i4"), ("dst_first", "<i4"), ("nd", "<i4"),
                 ("kind", "<u4"), ("chunk_bytes", "<u4"), ("n_chunks", "<u4"), ("rows_per_tile", "<u4"),
                 ("tiles_per_span", "<u4"), ("n_tiles", "<u4"), ("n_rows", "<u4"), ("tmap_ok", "<u4"),
                 ("ext", "<u4", 8), ("sstride", "<i8", 8), ("dstride", "<i8", 8)])
DST = np.dtype([("off", "<i8"), ("buf", "<i4"), ("pad", "<i4")])
SEG = np.dtype([("tile_begin", "<u4"), ("first_task", "<u4"), ("n_members", "<u4"), ("tiles_each", "<u4")])
TILE = np.dtype([("task", "<u4"), ("n_rows", "<u4"), ("col_bytes", "<u4"), ("flags", "<u4"), ("a", "<u8"), ("b", "<u8")])
assert TASK.itemsize == 224 and DST.itemsize == 16 and SEG.itemsize == 16 and TILE.itemsize == 32
FAST = 1
SPLIT, FASTK, GENERIC = 0, 1, 2


def tables(plan, op):
    t, d, g = plan.op_tables(op)
    return np.frombuffer(t, TASK), np.frombuffer(d, DST), np.frombuffer(g, SEG)


def lib_tiles(plan, op):
    """the tile list as the library decodes it (reshard_op_tiles)"""
    return np.frombuffer(plan.op_tiles(op), TILE)


def _row_offsets(T, first, row):
    """byte offsets (source, destination) of linear rows `row` (int64 array) over row dims first..nd-1"""
    so = np.zeros(row.shape, np.int64)
    do = np.zeros(row.shape, np.int64)
    row = row.copy()
    for i in range(first, int(T["nd"])):
        e = int(T["ext"][i])
        c = row % e
        row //= e
        so += c * int(T["sstride"][i])
        do += c * int(T["dstride"][i])
    return so, do, row


def task_tiles(T, task_id):
    """all tiles of one task, in its own order u = 0 .. n_tiles-1 (tables.h: SPLIT / FAST / GENERIC)"""
    n = int(T["n_tiles"])
    u = np.arange(n, dtype=np.int64)
    out = np.zeros(n, TILE)
    out["task"] = task_id
    B = int(T["run_bytes"])
    kind = int(T["kind"])
    if kind == SPLIT:
        nc, chunk = int(T["n_chunks"]), int(T["chunk_bytes"])
        row, cc = u // nc, u % nc
        so, do, rest = _row_offsets(T, 0, row)
        assert (rest == 0).all()
        c0 = cc * chunk
        out["n_rows"] = 1
        out["col_bytes"] = np.minimum(chunk, B - c0)
        out["flags"] = FAST
        out["a"] = so + c0
        out["b"] = do + c0
    elif kind == FASTK:
        tps, rpt, ext0 = int(T["tiles_per_span"]), int(T["rows_per_tile"]), int(T["ext"][0])
        span, g = u // tps, u % tps
        so, do, rest = _row_offsets(T, 1, span)
        assert (rest == 0).all()
        r0 = g * rpt
        out["n_rows"] = np.minimum(rpt, ext0 - r0)
        out["col_bytes"] = B
        out["flags"] = FAST
        out["a"] = so + r0 * int(T["sstride"][0])
        out["b"] = do + r0 * int(T["dstride"][0])
    else:
        assert kind == GENERIC
        rpt, R = int(T["rows_per_tile"]), int(T["n_rows"])
        r0 = u * rpt
        out["n_rows"] = np.minimum(rpt, R - r0)
        out["col_bytes"] = B
        out["flags"] = 0
        out["a"] = r0
        out["b"] = 0
    return out


def tiles(plan, op):
    """the operation's tile list in walk order, decoded HERE: inside a segment of G members tile v is tile v // G
    of member v % G"""
    tasks, _d, segs = tables(plan, op)
    n_tiles = plan.op_info(op).n_tiles
    out = np.zeros(n_tiles, TILE)
    seen = np.zeros(n_tiles, bool)
    for s in segs:
        G, each, begin = int(s["n_members"]), int(s["tiles_each"]), int(s["tile_begin"])
        for m in range(G):
            t = int(s["first_task"]) + m
            assert int(tasks[t]["n_tiles"]) == each
            idx = begin + np.arange(each) * G + m
            assert not seen[idx].any()
            out[idx] = task_tiles(tasks[t], t)
            seen[idx] = True
    assert seen.all(), "segments do not cover the tile range"
    return out


def replay(plan, op, src_bufs, dst_bufs, count=None, tile_list=None):
    """src_bufs / dst_bufs: lists of 1-D uint8 arrays.  count (optional): list of int32 arrays of the
    same sizes as dst_bufs, incremented for every byte written (exactly-once check)."""
    tasks, dsts, _segs = tables(plan, op)
    if tile_list is None:
        tile_list = tiles(plan, op)
    for tile in tile_list:
        T = tasks[tile["task"]]
        cb = int(tile["col_bytes"])
        for r in range(int(tile["n_rows"])):
            if tile["flags"] & FAST:
                so = int(tile["a"]) + r * int(T["sstride"][0])
                do = int(tile["b"]) + r * int(T["dstride"][0])
            else:
                lin = int(tile["a"]) + r
                so = do = int(tile["b"])
                for i in range(int(T["nd"])):
                    e = int(T["ext"][i])
                    c, lin = lin % e, lin // e
                    so += c * int(T["sstride"][i])
                    do += c * int(T["dstride"][i])
                assert lin == 0
            s0 = int(T["src_off"]) + so
            row = src_bufs[int(T["src_buf"])][s0:s0 + cb]
            assert row.size == cb, "source read out of bounds"
            for j in range(int(T["k"])):
                D = dsts[int(T["dst_first"]) + j]
                d0 = int(D["off"]) + do
                out = dst_bufs[int(D["buf"])]
                assert d0 >= 0 and d0 + cb <= out.size, "destination write out of bounds"
                out[d0:d0 + cb] = row
                if count is not None:
                    count[int(D["buf"])][d0:d0 + cb] += 1
