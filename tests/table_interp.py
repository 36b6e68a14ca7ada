"""TEST-ONLY interpreter of the library's flat task/tile tables (reshard_op_tables).

It replays a tile table on numpy byte buffers exactly as the kernels are specified to
(csrc/tables.h), so the host planner's tables can be checked against the oracle on the CPU box.
It is not a product path and nothing under paper_2211_05322_b200/ imports it.
"""
import numpy as np

TASK = np.dtype([("src_off", "<i8"), ("src_buf", "<i4"), ("k", "<i4"), ("dst_first", "<i4"), ("nd", "<i4"),
                 ("run_bytes", "<i8"), ("ext", "<u4", 8), ("sstride", "<i8", 8), ("dstride", "<i8", 8)])
DST = np.dtype([("off", "<i8"), ("buf", "<i4"), ("pad", "<i4")])
TILE = np.dtype([("task", "<u4"), ("n_rows", "<u4"), ("col_bytes", "<u4"), ("flags", "<u4"), ("a", "<u8"), ("b", "<u8")])
assert TASK.itemsize == 192 and DST.itemsize == 16 and TILE.itemsize == 32
FAST = 1


def tables(plan, op):
    t, d, l = plan.op_tables(op)
    return np.frombuffer(t, TASK), np.frombuffer(d, DST), np.frombuffer(l, TILE)


def replay(plan, op, src_bufs, dst_bufs, count=None):
    """src_bufs / dst_bufs: lists of 1-D uint8 arrays.  count (optional): list of int32 arrays of the
    same sizes as dst_bufs, incremented for every byte written (exactly-once check)."""
    tasks, dsts, tiles = tables(plan, op)
    for tile in tiles:
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
