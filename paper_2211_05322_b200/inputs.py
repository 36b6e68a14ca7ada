"""Seeded synthetic inputs and the workload table (shared by tests, bench.py and smoke()).

This module holds NONE of the method's arithmetic: no tile boxes, no slices, no plans.  It
only (a) names the workloads of BASELINE.json / SURVEY.md S8(d) as (shape, dtype, meshes,
specs) tuples and (b) produces the values of the global tensor D as a pure function of the
global linear index g, so every destination element is checkable on its own:

    kind "index": value(g) = g                       (config 1: fp32, "values = global linear index")
    kind "bits" : value(g) = low 8*e bits of mix64(seed + g)   ("seeded uniform bit patterns")

Payloads are opaque bytes to the method (R22): 16-bit floats are carried as int16 bit
patterns so comparisons are NaN-safe.  The paper's microbenchmark tensor has a stated shape
and unstated contents; the GPT shapes follow its [B,S,H] family,
the U-Transformer shape is BASELINE.json's stand-in.  Nothing here comes from a dataset.
"""
from collections import namedtuple

import numpy as np

SEED_BASE = 221105322000

Workload = namedtuple("Workload", "name shape dtype src_mesh src_spec dst_mesh dst_spec kind seed")

_M64 = (1 << 64) - 1


def mix64_np(x):
    """splitmix64 finaliser on a uint64 numpy array (wrapping arithmetic)."""
    x = x.astype(np.uint64, copy=True)
    with np.errstate(over="ignore"):
        x ^= x >> np.uint64(30)
        x *= np.uint64(0xBF58476D1CE4E5B9)
        x ^= x >> np.uint64(27)
        x *= np.uint64(0x94D049BB133111EB)
        x ^= x >> np.uint64(31)
    return x


def _container(dtype):
    """numpy container dtype for an element type name."""
    return {"fp32": np.float32, "bf16": np.int16, "fp16": np.int16, "u8": np.uint8,
            "i32": np.int32, "i64": np.int64}[dtype]


def elem_bytes(dtype):
    return np.dtype(_container(dtype)).itemsize


def global_tensor(w, chunk=1 << 24):
    """D as a numpy array of w.shape in the container dtype (host)."""
    n = int(np.prod(w.shape))
    ct = np.dtype(_container(w.dtype))
    out = np.empty(n, dtype=ct)
    for a in range(0, n, chunk):
        b = min(n, a + chunk)
        g = np.arange(a, b, dtype=np.uint64)
        if w.kind == "index":
            out[a:b] = g.astype(ct)
        else:
            bits = mix64_np(g + np.uint64(w.seed % (1 << 64)))
            out[a:b] = (bits & np.uint64((1 << (8 * ct.itemsize)) - 1)).astype(
                np.dtype("u%d" % ct.itemsize)).view(ct)
    return out.reshape(w.shape)


def global_tensor_torch(w, device, chunk=1 << 26):
    """same values as global_tensor(), generated on `device` with torch integer ops
    (int64 wraps like uint64; logical shifts are emulated with masks)."""
    import torch
    n = int(np.prod(w.shape))
    tdt = {"fp32": torch.float32, "bf16": torch.int16, "fp16": torch.int16, "u8": torch.uint8,
           "i32": torch.int32, "i64": torch.int64}[w.dtype]
    out = torch.empty(n, dtype=tdt, device=device)

    def i64(v):  # python int (uint64 value) -> wrapped int64
        v &= _M64
        return v - (1 << 64) if v >= (1 << 63) else v

    def lsr(x, s):
        return (x >> s) & ((1 << (64 - s)) - 1)

    nb = 8 * out.element_size()
    for a in range(0, n, chunk):
        b = min(n, a + chunk)
        g = torch.arange(a, b, dtype=torch.int64, device=device)
        if w.kind == "index":
            out[a:b] = g.to(tdt)
            continue
        x = g + i64(w.seed)
        x = x ^ lsr(x, 30)
        x = x * i64(0xBF58476D1CE4E5B9)
        x = x ^ lsr(x, 27)
        x = x * i64(0x94D049BB133111EB)
        x = x ^ lsr(x, 31)
        if nb == 64:
            out[a:b] = x
        else:
            lo = x & ((1 << nb) - 1)
            if tdt != torch.uint8:
                lo = torch.where(lo >= (1 << (nb - 1)), lo - (1 << nb), lo)   # to signed container
            out[a:b] = lo.to(tdt)
    return out.reshape(w.shape)


# ------------------------------------------------------------------ BASELINE.json configs

def _w(name, shape, dtype, sm, ss, dm, ds, kind="bits", cid=0):
    return Workload(name, tuple(shape), dtype, tuple(sm), ss, tuple(dm), ds, kind, SEED_BASE + cid)


# Spec strings and mesh shapes are taken literally (R21); the primed variants are
# the prose-intent readings of BASELINE.json configs 1 and 3.
CONFIGS = {
    "c1":   _w("c1", (8, 16), "fp32", (1, 2), "S0,R", (1, 2), "R,S0", "index", 1),
    "c1i":  _w("c1i", (8, 16), "fp32", (1, 2), "S1,R", (1, 2), "R,S1", "index", 1),
    "c2":   _w("c2", (16, 1024, 4096), "bf16", (2, 4), "S0,R,S1", (2, 4), "S0,S1,R", "bits", 2),
    "c3":   _w("c3", (8, 320, 64, 64), "fp16", (1, 4), "S0,R,R,R", (2, 2), "R,S0,S1,R", "bits", 3),
    "c3i":  _w("c3i", (8, 320, 64, 64), "fp16", (1, 4), "S1,R,R,R", (2, 2), "R,S0,S1,R", "bits", 3),
    "c3ii": _w("c3ii", (8, 320, 64, 64), "fp16", (1, 4), "S1,R,R,R", (2, 2), "R,S0,R,R", "bits", 3),
    "c4":   _w("c4", (32, 2048, 12288), "bf16", (2, 4), "S0,S1,R", (4, 2), "S1,R,S0", "bits", 4),
    # config 4's layout pair on extents that divide nothing: uneven partitions on all three dims and runs of
    # 6145 B at 2-byte alignment (the "tiling, padding" case of PAPER.md:259 at GPT-activation size)
    "u4":   _w("u4", (30, 2047, 12290), "bf16", (2, 4), "S0,S1,R", (4, 2), "S1,R,S0", "bits", 6),
    "u4b":  _w("u4b", (30, 2047, 24579), "u8", (2, 4), "S0,S1,R", (4, 2), "S1,R,S0", "bits", 7),
    # sweep pair P1 at 1 GiB on extents that divide nothing: 2050-byte destination rows at 2-byte alignment
    "u1":   _w("u1", (64, 2046, 4100), "bf16", (2, 4), "S0,R,S1", (2, 4), "S0,S1,R", "bits", 9),
    # the paper's microbenchmark tensor with its LAST dim sharded 8 ways on one side: 128-byte runs (register path at full size)
    "r128": _w("r128", (1024, 1024, 512), "bf16", (2, 4), "R,R,S01", (2, 4), "S01,R,R", "bits", 10),
    "r128m": _w("r128m", (1024, 1024, 512), "bf16", (2, 4), "R,R,S01", (2, 4), "S0,R,R", "bits", 11),
    # a feature map resharded from a split of H to a split of W: 64-byte rows, 32 of them per span (tiles cannot cross a span)
    "fm_hw": _w("fm_hw", (64, 640, 64, 64), "fp16", (2, 2), "S0,R,S1,R", (2, 2), "S0,R,R,S1", "bits", 12),
    "fm_hwm": _w("fm_hwm", (64, 640, 64, 64), "fp16", (1, 2), "R,R,S1,R", (2, 2), "R,R,R,S1", "bits", 13),
    # the same pair with rows that are 16-byte aligned and nothing more (6160-byte runs): the least the TMA path accepts
    "a4":   _w("a4", (32, 2048, 12320), "bf16", (2, 4), "S0,S1,R", (4, 2), "S1,R,S0", "bits", 8),
}

# config 5: six layout pairs (BASELINE.json configs[4]) on two mesh pairs.
SWEEP_PAIRS = {
    "P1": ("S0,R,S1", "S0,S1,R"),
    "P2": ("R,R,S0", "S0,R,R"),
    "P3": ("S0,S1,R", "S1,S0,R"),
    "P4": ("R,S0,S1", "R,S1,S0"),
    "P5": ("S0,R,R", "R,R,R"),
    "P6": ("R,R,R", "S0,S1,R"),
}
SWEEP_MESHES = {"m8": ((2, 4), (2, 4)), "m4": ((1, 4), (2, 2))}
SWEEP_BYTES = [(1 << 20) * 4 ** j for j in range(7)]          # 1 MiB ... 4 GiB


def sweep_shape(nbytes):
    """[B, S, 4096] bf16 with B, S multiples of 8."""
    rows = nbytes // (4096 * 2)                 # B*S
    if nbytes >= (128 << 20):
        S = 2048
    else:
        S = max(16, rows // 8)
    B = rows // S
    assert B * S * 4096 * 2 == nbytes and B % 8 == 0 and S % 8 == 0, (nbytes, B, S)
    return (B, S, 4096)


def sweep_workload(pair, meshes, nbytes):
    (sm, dm), (ss, ds) = SWEEP_MESHES[meshes], SWEEP_PAIRS[pair]
    name = "sweep_%s_%s_%dMiB" % (pair, meshes, nbytes >> 20)
    return _w(name, sweep_shape(nbytes), "bf16", sm, ss, dm, ds, "bits", 5)


# Table 2 of the paper, tensor (1024,1024,512) at 2 B/elt.
# Case 6 needs an uneven partition ((2,4)->(3,4), padded in the paper) and is listed for the
# uneven-partition extension only.
TABLE2 = {
    1: ("S0RR", "S0RR", (2, 4), (2, 4)),
    2: ("RRR", "S0RR", (2, 4), (2, 4)),
    3: ("RS0R", "S0RR", (2, 4), (2, 4)),
    4: ("RS01R", "S01RR", (2, 4), (2, 4)),
    5: ("S1RR", "S0RR", (2, 4), (2, 4)),
    6: ("S0RR", "S0RR", (2, 4), (3, 4)),
    7: ("S1RR", "RRR", (1, 4), (2, 4)),
    8: ("RRR", "RRR", (2, 3), (3, 2)),
    9: ("RS0R", "RRS0", (2, 4), (2, 4)),
}


def table2_workload(case, shape=(1024, 1024, 512)):
    ss, ds, sm, dm = TABLE2[case]
    return _w("table2_case%d" % case, shape, "bf16", sm, ss, dm, ds, "bits", 20 + case)


def fig5_workload(nodes, gpus_per_node, shape=(1024, 1024, 512)):
    """PAPER.md:255 (S5.1.1): one sender GPU, a receiver mesh of `nodes` x `gpus_per_node` GPUs, both fully
    replicated, "the message size keeps 1GB" (2 B/element here)."""
    return _w("fig5_%dx%d" % (nodes, gpus_per_node), shape, "bf16", (1,), "RRR", (nodes, gpus_per_node), "RRR", "bits", 40 + 8 * nodes + gpus_per_node)


FIG5 = [(1, 1), (1, 2), (1, 3), (1, 4), (2, 2), (3, 2), (4, 2)]     # group 1: one node, 1-4 GPUs; group 2: 2 GPUs per node, 1-4 nodes


# The skip connections of a U-shaped network put several feature maps of different resolution on one stage
# boundary.  The paper gives no shapes; these four follow config 3's [8, 320, 64, 64] down a
# 2x-per-level U (channels x2, resolution /2), same layout pair as c3ii.  Synthetic stand-ins.
UNET_LEVELS = [(320, 64), (640, 32), (1280, 16), (1280, 8)]


def unet_workload(level):
    c, hw = UNET_LEVELS[level]
    return _w("unet_l%d" % level, (8, c, hw, hw), "fp16", (1, 4), "S1,R,R,R", (2, 2), "R,S0,R,R", "bits", 60 + level)


def get_workload(name):
    """'c1'..'c4', 'c1i', 'c3i', 'c3ii', 'u4', 't2_<case>', 'sweep_<pair>_<m8|m4>_<MiB>', 'fig5_<nodes>x<gpus>', or any task as
    'x:<shape>:<dtype>:<src mesh>:<src spec>:<dst mesh>:<dst spec>'."""
    if name.startswith("x:"):
        # any task spelled out: x:<shape>:<dtype>:<src mesh>:<src spec>:<dst mesh>:<dst spec>, e.g. x:64x2048x4096:bf16:4x8:S0S1R:8x4:S1RS0 (specs without commas, so that names can be listed)
        _x, shape, dtype, sm, ss, dm, ds = name.split(":")
        dims = lambda s: tuple(int(v) for v in s.split("x"))
        return _w(name, dims(shape), dtype, dims(sm), ss, dims(dm), ds, "bits", 99)
    if name.startswith("unet_l"):
        return unet_workload(int(name[6:]))
    if name.startswith("fig5_"):
        a, b = name[5:].split("x")
        return fig5_workload(int(a), int(b))
    if name in CONFIGS:
        return CONFIGS[name]
    if name.startswith("t2_"):
        return table2_workload(int(name[3:]))
    if name.startswith("sweep_"):
        _s, pair, meshes, mib = name.split("_")
        return sweep_workload(pair, meshes, int(mib.replace("MiB", "")) << 20)
    raise KeyError(name)
