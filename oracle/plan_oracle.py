"""Plan-side oracle: unit-task decomposition and sender choice, step by step from the paper.

TEST INFRASTRUCTURE, NOT THE PRODUCT.  Pure Python (small inputs only), written from
PAPER.md alone; shares no code with paper_2211_05322_b200/ and neither imports the other.

What it follows (PAPER.md:<line>, section):
  tile boxes        PAPER.md:78-86   S2.2 device mesh / sharding spec / data slice
  unit tasks        PAPER.md:482-492 App. B.2: Cut(d) -> I_d -> slices = I_0 x ... x I_{n-1};
                                     senders N_i = source devices owning the slice,
                                     receivers M_i = destination devices requiring it
  naive senders     PAPER.md:163     lowest-indexed device
  greedy senders    PAPER.md:167-171 Eq. 4: sort tasks by descending T_i, give each to the
                                     currently lightest candidate sender
  optimum of Eq. 4  PAPER.md:169     brute force over all sender assignments (tiny inputs)

Readings: R1 row-major device ids; R2 S^{01}: first listed axis most significant;
R3 a mesh axis shards at most one tensor dim; R5 uneven partitions: every shard has the padded
extent c = ceil(l/k), shard p holds [min(pc, l), min((p+1)c, l)); R6 one unit task per
B.2 slice; R7 T_i = slice bytes (independent of #receivers); R8 balance per (virtual) device;
R9 ties: tasks by (bytes desc, slice id asc), senders by (load, device id).
Slice id = row-major rank in I_0 x ... x I_{n-1} (dim 0 slowest): a convention of this build,
stated in include/reshard.h too.

Pins: tests/test_plan_oracle_pins.py (Fig. 2 unit tasks, Table 2 case 4 = 64 tasks, case 8 = 1,
case 2 naive vs greedy, lower bound sum = size(D), exact cover by painting).
"""
import itertools
import re

import numpy as np


class SpecError(ValueError):
    pass


class DivisError(ValueError):
    pass


def parse_spec(spec, ndim, mesh_ndim):
    """'S0,R,S1' / 'S01RR' / 'RRR' -> tuple of axis tuples, () for R.  PAPER.md:84."""
    entries = re.findall(r"[Rr]|[Ss][\^{_ ]*\d*\}?", re.sub(r"[,\s()\[\]]", "", spec))
    if "".join(entries) != re.sub(r"[,\s()\[\]]", "", spec):
        raise SpecError("unparsable spec %r" % spec)
    out, used = [], set()
    for e in entries:
        if e in "Rr":
            out.append(())
            continue
        axes = tuple(int(ch) for ch in re.sub(r"\D", "", e))
        if not axes:
            raise SpecError("S without mesh axis in %r" % spec)
        for a in axes:
            if a >= mesh_ndim:
                raise SpecError("mesh axis %d out of range in %r" % (a, spec))
            if a in used:
                raise SpecError("mesh axis %d used twice in %r" % (a, spec))  # R3
            used.add(a)
        out.append(axes)
    if len(out) != ndim:
        raise SpecError("spec %r has %d entries for %d dims" % (spec, len(out), ndim))
    return tuple(out)


def n_devices(mesh):
    n = 1
    for m in mesh:
        n *= m
    return n


def device_coords(mesh, r):
    """row-major: (2,2) mesh is [[0,1],[2,3]]."""
    return tuple(int(x) for x in np.unravel_index(r, tuple(mesh)))


def degrees(shape, mesh, axes_per_dim, even_only=False):
    ks = []
    for l, axes in zip(shape, axes_per_dim):
        k = 1
        for a in axes:
            k *= mesh[a]
        if even_only and l % k:
            raise DivisError("dim of length %d not divisible by degree %d" % (l, k))
        ks.append(k)
    return ks


def ceil_div(a, b):
    return -(-a // b)


def tile_box(shape, mesh, spec, r):
    """[lo, hi) per tensor dim of the piece of D held by device r."""
    axes_per_dim = parse_spec(spec, len(shape), len(mesh))
    ks = degrees(shape, mesh, axes_per_dim)
    c = device_coords(mesh, r)
    lo, hi = [], []
    for l, k, axes in zip(shape, ks, axes_per_dim):
        p = 0
        for a in axes:               # R2: first listed axis most significant
            p = p * mesh[a] + c[a]
        ext = ceil_div(l, k)                                # R5: padded extent, clipped box
        lo.append(min(p * ext, l))
        hi.append(min((p + 1) * ext, l))
    return tuple(lo), tuple(hi)


def cutpoints(shape, src_mesh, src_spec, dst_mesh, dst_spec):
    """Cut(d) = {0, l_d} U {j l_d/k_A} U {j l_d/k_B}; with uneven partitions the
    shard boundaries are j*ceil(l_d/k), clipped to l_d (R5)."""
    ka = degrees(shape, src_mesh, parse_spec(src_spec, len(shape), len(src_mesh)))
    kb = degrees(shape, dst_mesh, parse_spec(dst_spec, len(shape), len(dst_mesh)))
    cuts = []
    for l, a, b in zip(shape, ka, kb):
        s = {0, l}
        s.update(min(j * ceil_div(l, a), l) for j in range(1, a))
        s.update(min(j * ceil_div(l, b), l) for j in range(1, b))
        cuts.append(sorted(s))
    return cuts


def unit_tasks(shape, src_mesh, src_spec, dst_mesh, dst_spec):
    """App. B.2: list of unit tasks in slice-id order.
    Each task: dict(lo, hi, size (elements), senders N_i, receivers M_i)."""
    cuts = cutpoints(shape, src_mesh, src_spec, dst_mesh, dst_spec)
    intervals = [list(zip(c[:-1], c[1:])) for c in cuts]          # I_d
    src_boxes = [tile_box(shape, src_mesh, src_spec, r) for r in range(n_devices(src_mesh))]
    dst_boxes = [tile_box(shape, dst_mesh, dst_spec, r) for r in range(n_devices(dst_mesh))]

    def inside(lo, hi, box):
        return all(bl <= l and h <= bh for l, h, bl, bh in zip(lo, hi, box[0], box[1]))

    tasks = []
    for combo in itertools.product(*intervals):                   # I_0 x I_1 x ... (row-major)
        lo = tuple(iv[0] for iv in combo)
        hi = tuple(iv[1] for iv in combo)
        size = 1
        for l, h in zip(lo, hi):
            size *= h - l
        senders = [r for r, b in enumerate(src_boxes) if inside(lo, hi, b)]
        receivers = [r for r, b in enumerate(dst_boxes) if inside(lo, hi, b)]
        tasks.append(dict(lo=lo, hi=hi, size=size, senders=senders, receivers=receivers))
    return tasks


def naive_senders(tasks):
    """the first (lowest-indexed) device."""
    return [min(t["senders"]) for t in tasks]


def greedy_senders(tasks, elem_bytes=1):
    """sort by descending T_i, assign to the currently lightest candidate."""
    load = {}
    order = sorted(range(len(tasks)), key=lambda i: (-tasks[i]["size"], i))       # R9
    chosen = [None] * len(tasks)
    for i in order:
        s = min(tasks[i]["senders"], key=lambda d: (load.get(d, 0), d))
        chosen[i] = s
        load[s] = load.get(s, 0) + tasks[i]["size"] * elem_bytes
    return chosen


def sender_loads(tasks, senders, n_src, elem_bytes=1):
    load = [0] * n_src
    for t, s in zip(tasks, senders):
        assert s in t["senders"], "Eq. 2 violated: sender does not hold the slice"
        load[s] += t["size"] * elem_bytes
    return load


def max_load(tasks, senders, n_src, elem_bytes=1):
    """objective of Eq. 4."""
    return max(sender_loads(tasks, senders, n_src, elem_bytes))


def bruteforce_optimum(tasks, n_src, elem_bytes=1, limit=2_000_000):
    """min over ALL sender assignments of max per-sender bytes (Eq. 4), by enumeration."""
    total = 1
    for t in tasks:
        total *= len(t["senders"])
        if total > limit:
            raise ValueError("too many assignments to enumerate")
    best = None
    for choice in itertools.product(*[t["senders"] for t in tasks]):
        m = max_load(tasks, choice, n_src, elem_bytes)
        if best is None or m < best:
            best = m
    return best


def paint_cover(shape, dst_mesh, dst_spec, tasks):
    """count, for every (dst device, local element), how many (task, receiver) pairs write it."""
    counts = []
    for q in range(n_devices(dst_mesh)):
        lo, hi = tile_box(shape, dst_mesh, dst_spec, q)
        cnt = np.zeros([h - l for l, h in zip(lo, hi)], dtype=np.int32)
        for t in tasks:
            if q in t["receivers"]:
                sl = tuple(slice(a - l, b - l) for a, b, l in zip(t["lo"], t["hi"], lo))
                cnt[sl] += 1
        counts.append(cnt)
    return counts


def message_table(tasks, senders):
    """wire model of this build (north_star item 3): message (s, r) is the concatenation, in
    ascending slice id, of every slice with sender s and r in M_i, each dense row-major.
    Messages are ordered by (s, r).  Returns list of (s, r, [slice ids], elements)."""
    groups = {}
    for i, (t, s) in enumerate(zip(tasks, senders)):
        for r in t["receivers"]:
            groups.setdefault((s, r), []).append(i)
    return [(s, r, ids, sum(tasks[i]["size"] for i in ids)) for (s, r), ids in sorted(groups.items())]


def pack_messages(shape, src_mesh, src_spec, tasks, senders, src_shards):
    """bytes of every message, built with numpy basic slicing of the SENDER's shard."""
    out = []
    for s, r, ids, _n in message_table(tasks, senders):
        lo, _hi = tile_box(shape, src_mesh, src_spec, s)
        parts = []
        for i in ids:
            t = tasks[i]
            sl = tuple(slice(a - l, b - l) for a, b, l in zip(t["lo"], t["hi"], lo))
            parts.append(np.ascontiguousarray(src_shards[s][sl]).reshape(-1))
        out.append((s, r, np.concatenate(parts)))
    return out
