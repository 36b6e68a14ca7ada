"""Pins of the plan-side oracle (oracle/plan_oracle.py): the paper's worked example, the
facts it states about Table 2, closed forms and brute-force invariants."""
import numpy as np
import pytest
from hypothesis import given, settings, strategies as st

import golden_io
from oracle import plan_oracle as po
from paper_2211_05322_b200 import inputs


def _elements(t, shape):
    D = np.arange(np.prod(shape)).reshape(shape)
    return D[tuple(slice(l, h) for l, h in zip(t["lo"], t["hi"]))].reshape(-1).tolist()


def test_fig2_unit_tasks():
    """PAPER.md:90 and App. B.1."""
    g = golden_io.load("fig2_example.txt")
    shape = tuple(g["matrix_shape"])
    a0, b0 = g["mesh_a_devices"][0], g["mesh_b_devices"][0]
    t1 = po.unit_tasks(shape, g["mesh_a"], g["spec1"], g["mesh_b"], g["spec2"])
    assert len(t1) == g["task1_num_unit_tasks"][0]
    assert _elements(t1[0], shape) == g["task1_first_slice_elements"]
    assert [r + b0 for r in t1[0]["receivers"]] == g["task1_first_receivers"]
    assert [s + a0 for s in t1[0]["senders"]] == [0]                 # "each device holds a unique slice"
    assert all(len(t["receivers"]) == 2 and len(t["senders"]) == 1 for t in t1)
    t2 = po.unit_tasks(shape, g["mesh_b"], g["spec2"], g["mesh_a"], g["spec3"])
    assert len(t2) == g["task2_num_unit_tasks"][0]
    assert _elements(t2[0], shape) == g["task2_first_slice_elements"]
    assert [r + a0 for r in t2[0]["receivers"]] == g["task2_first_receivers"]
    assert [s + b0 for s in t2[0]["senders"]] == [4, 5]              # PAPER.md:86 replicas of the top slice


def test_fig2_spec2_boxes():
    g = golden_io.load("fig2_example.txt")
    for local in (0, 1):                                              # devices 4 and 5: elements 0..7
        assert po.tile_box((4, 4), g["mesh_b"], g["spec2"], local) == ((0, 0), (2, 4))
    for local in (2, 3):
        assert po.tile_box((4, 4), g["mesh_b"], g["spec2"], local) == ((2, 0), (4, 4))


# (shape, mesh, spec, device, lo, hi) -- worked out by hand from PAPER.md:82-84
HAND_BOXES = [
    ((4, 8, 6), (2, 4), "S0,S1,R", 6, (2, 4, 0), (4, 6, 6)),
    ((4, 8, 6), (2, 4), "S1,R,S0", 6, (2, 0, 3), (3, 8, 6)),
    ((4, 8, 6), (2, 4), "R,S01,R", 6, (0, 6, 0), (4, 7, 6)),
    ((4, 8, 6), (2, 4), "R,S10,R", 6, (0, 5, 0), (4, 6, 6)),
    ((4, 8, 8), (4, 2), "S1,R,S0", 5, (2, 0, 4), (4, 8, 6)),
    ((8, 16), (1, 2), "S0,R", 1, (0, 0), (8, 16)),
    ((8, 16), (1, 2), "R,S1", 1, (0, 8), (8, 16)),
    ((6, 4), (3,), "S0,R", 2, (4, 0), (6, 4)),
    ((2, 4, 6, 8), (2, 2), "R,S0,S1,R", 3, (0, 2, 3, 0), (2, 4, 6, 8)),
]


@pytest.mark.parametrize("shape,mesh,spec,dev,lo,hi", HAND_BOXES)
def test_tile_box_hand_written(shape, mesh, spec, dev, lo, hi):
    assert po.tile_box(shape, mesh, spec, dev) == (lo, hi)


def test_table2_facts():
    g = golden_io.load("table2_facts.txt")
    shape = tuple(g["tensor_shape"])

    def tasks(case):
        ss, ds, sm, dm = inputs.TABLE2[case]
        return po.unit_tasks(shape, sm, ss, dm, ds), sm

    t4, _ = tasks(4)
    assert len(t4) == g["case4_num_unit_tasks"][0]
    t8, _ = tasks(8)
    assert len(t8) == g["case8_num_unit_tasks"][0]
    assert len(t8[0]["senders"]) == 6 and len(t8[0]["receivers"]) == 6
    # case 2 under Naive: everything from the first node (devices 0..3 of the (2,4) mesh)
    t2, sm = tasks(2)
    naive = po.naive_senders(t2)
    assert all(s // sm[1] == g["case2_naive_sender_node"][0] for s in naive)
    assert len(set(naive)) == 1
    greedy = po.greedy_senders(t2)
    assert len(set(greedy)) == len(t2)                               # load balance spreads them
    assert po.max_load(t2, greedy, 8) * 2 == po.max_load(t2, naive, 8)


# slices / candidate senders / receivers per slice, derived by hand from Table 2
TABLE2_HAND = {1: (2, 4, 4), 2: (2, 8, 4), 3: (4, 4, 4), 4: (64, 1, 1), 5: (4, 2, 4),
               7: (4, 1, 8), 8: (1, 6, 6), 9: (4, 4, 4)}


@pytest.mark.parametrize("case", sorted(TABLE2_HAND))
def test_table2_decomposition_counts(case):
    ss, ds, sm, dm = inputs.TABLE2[case]
    shape = (16, 16, 8)                                               # same structure, tiny
    tasks = po.unit_tasks(shape, sm, ss, dm, ds)
    n, ns, nr = TABLE2_HAND[case]
    assert len(tasks) == n
    assert all(len(t["senders"]) == ns and len(t["receivers"]) == nr for t in tasks)
    assert sum(t["size"] for t in tasks) == np.prod(shape)            # lower bound


def test_table2_case6_uneven_partition():
    """(2,4) -> (3,4), dim 0 = 1024 over 3 shards, "pad it in case 6" (R5)."""
    g = golden_io.load("table2_facts.txt")
    ss, ds, sm, dm = inputs.TABLE2[6]
    shape = tuple(g["tensor_shape"])
    c = g["case6_padded_extent"][0]
    assert po.ceil_div(shape[0], 3) == c and 3 * c == g["case6_padded_dim0"][0]
    boxes = sorted({(po.tile_box(shape, dm, ds, r)[0][0], po.tile_box(shape, dm, ds, r)[1][0]) for r in range(12)})
    assert [x for b in boxes for x in b] == g["case6_dst_dim0_boxes"]
    assert po.cutpoints(shape, sm, ss, dm, ds)[0] == g["case6_dim0_cutpoints"]
    tasks = po.unit_tasks(shape, sm, ss, dm, ds)
    assert len(tasks) == g["case6_num_unit_tasks"][0]
    assert sum(t["size"] for t in tasks) == np.prod(shape)            # PAPER.md:90, padding is never sent
    assert [len(t["senders"]) for t in tasks] == [4] * 4 and [len(t["receivers"]) for t in tasks] == [4] * 4
    with pytest.raises(po.DivisError):                                # the strict "evenly sharded" reading
        po.degrees(shape, dm, po.parse_spec(ds, 3, 2), even_only=True)


@pytest.mark.parametrize("shape,sm,ss,dm,ds", [((10,), (3,), "S0", (4,), "S0"), ((7, 9), (2, 4), "S1,S0", (4, 2), "S0,S1"),
                                               ((2, 6), (4,), "S0,R", (2,), "S0,R"), ((11, 6), (2, 4), "S01,R", (2, 3), "R,S10")])
def test_uneven_unit_tasks_cover_exactly_once(shape, sm, ss, dm, ds):
    tasks = po.unit_tasks(shape, sm, ss, dm, ds)
    assert sum(t["size"] for t in tasks) == np.prod(shape) and all(t["size"] > 0 for t in tasks)
    assert all(t["senders"] and t["receivers"] for t in tasks)
    for cnt in po.paint_cover(shape, dm, ds, tasks):
        assert (cnt == 1).all()
    # the brute-force optimum of Eq. 4 is reachable although slice sizes differ
    n_src = po.n_devices(sm)
    assert po.max_load(tasks, po.greedy_senders(tasks), n_src) >= po.bruteforce_optimum(tasks, n_src)


def test_cutpoints_follow_b2():
    """PAPER.md:488-492 on a 2-way x 3-way dim."""
    cuts = po.cutpoints((12, 6), (2, 3), "S0,S1", (3, 2), "S0,S1")
    assert cuts == [[0, 4, 6, 8, 12], [0, 2, 3, 4, 6]]
    tasks = po.unit_tasks((12, 6), (2, 3), "S0,S1", (3, 2), "S0,S1")
    assert len(tasks) == 4 * 4                                         # prod (#Cut(d) - 1)
    assert tasks[0]["lo"] == (0, 0) and tasks[0]["hi"] == (4, 2)
    assert tasks[1]["lo"] == (0, 2) and tasks[1]["hi"] == (4, 3)       # slice id is row-major
    assert sorted({t["size"] for t in tasks}) == [2, 4, 8]             # unequal slices


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
]


@pytest.mark.parametrize("shape,sm,ss,dm,ds", LAYOUTS)
def test_exact_cover_and_containment(shape, sm, ss, dm, ds):
    tasks = po.unit_tasks(shape, sm, ss, dm, ds)
    cuts = po.cutpoints(shape, sm, ss, dm, ds)
    assert len(tasks) == int(np.prod([len(c) - 1 for c in cuts]))
    assert sum(t["size"] for t in tasks) == int(np.prod(shape))
    for cnt in po.paint_cover(shape, dm, ds, tasks):
        assert (cnt == 1).all()
    # every slice lies in exactly one source tile (its replica group) and N_i is that whole group
    src_boxes = [po.tile_box(shape, sm, ss, r) for r in range(po.n_devices(sm))]
    for t in tasks:
        assert t["senders"] and t["receivers"]
        boxes = {src_boxes[s] for s in t["senders"]}
        assert len(boxes) == 1
        assert sorted(t["senders"]) == [r for r, b in enumerate(src_boxes) if b in boxes]


@pytest.mark.parametrize("shape,sm,ss,dm,ds", LAYOUTS)
def test_greedy_vs_naive_vs_bruteforce(shape, sm, ss, dm, ds):
    tasks = po.unit_tasks(shape, sm, ss, dm, ds)
    n_src = po.n_devices(sm)
    naive = po.max_load(tasks, po.naive_senders(tasks), n_src)
    greedy = po.max_load(tasks, po.greedy_senders(tasks), n_src)
    assert greedy <= naive
    try:
        opt = po.bruteforce_optimum(tasks, n_src)
    except ValueError:
        return
    assert opt <= greedy
    sizes = {t["size"] for t in tasks}
    if len(sizes) == 1:
        # closed form for equal slices: max over replica groups of ceil(n_G / r_G) * size
        groups = {}
        for t in tasks:
            groups.setdefault(tuple(t["senders"]), []).append(t)
        closed = max(-(-len(ts) // len(g)) for g, ts in groups.items()) * sizes.pop()
        assert greedy == opt == closed


def test_lpt_greedy_is_not_always_optimal_but_bruteforce_is():
    """Eq. 4 with unequal T_i is P||Cmax; the classical greedy is a 4/3-approximation.
    Sizes 3,3,2,2,2 on 2 identical senders: greedy 7, optimum 6 (R9)."""
    tasks = [dict(size=s, senders=[0, 1], receivers=[0]) for s in (3, 3, 2, 2, 2)]
    assert po.max_load(tasks, po.greedy_senders(tasks), 2) == 7
    assert po.bruteforce_optimum(tasks, 2) == 6


def test_message_table_and_pack():
    shape, sm, ss, dm, ds = (4, 4), (2, 2), "S01,R", (2, 2), "S0,R"       # Fig. 2 task 1
    D = np.arange(16, dtype=np.int32).reshape(shape)
    tasks = po.unit_tasks(shape, sm, ss, dm, ds)
    senders = po.greedy_senders(tasks)
    msgs = po.message_table(tasks, senders)
    # 4 senders x 2 receivers each, one slice per message
    assert [(s, r) for s, r, _ids, _n in msgs] == [(0, 0), (0, 1), (1, 0), (1, 1), (2, 2), (2, 3), (3, 2), (3, 3)]
    assert sum(n for *_x, n in msgs) == 16 * 2                         # size(D) * r_B
    src = [D[r:r + 1] for r in range(4)]
    packed = po.pack_messages(shape, sm, ss, tasks, senders, src)
    assert packed[0][2].tolist() == [0, 1, 2, 3] and packed[1][2].tolist() == [0, 1, 2, 3]
    assert packed[7][2].tolist() == [12, 13, 14, 15]


def test_spec_errors():
    with pytest.raises(po.SpecError):
        po.parse_spec("S0,S0", 2, 2)
    with pytest.raises(po.SpecError):
        po.parse_spec("S2,R", 2, 2)
    with pytest.raises(po.SpecError):
        po.parse_spec("S0", 2, 2)
    with pytest.raises(po.SpecError):
        po.parse_spec("S,R", 2, 2)
    with pytest.raises(po.SpecError):
        po.parse_spec("X0,R", 2, 2)
    assert po.parse_spec("RS^{01}R", 3, 2) == ((), (0, 1), ())
    assert po.parse_spec("(S0, S1, R)", 3, 2) == ((0,), (1,), ())
    assert po.parse_spec("RRR", 3, 2) == ((), (), ())


@settings(max_examples=40, deadline=None)
@given(st.sampled_from(LAYOUTS), st.integers(1, 3))
def test_lower_bound_scales(layout, mult):
    shape, sm, ss, dm, ds = layout
    shape = tuple(s * mult * (3 if mult == 3 else 1) for s in shape)
    try:
        tasks = po.unit_tasks(shape, sm, ss, dm, ds)
    except po.DivisError:
        return
    assert sum(t["size"] for t in tasks) == int(np.prod(shape))
