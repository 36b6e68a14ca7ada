"""S3.2 in the library (csrc/schedule.cpp, reshard_plan_ex / reshard_plan_schedule) against the
schedule oracle, on the CPU box (RS_HOST_ONLY plans).  The deterministic algorithms must agree with
the oracle decision by decision; the searches must be valid, and optimal when they finish."""
import numpy as np
import pytest
from hypothesis import given, settings, strategies as st

import table_interp as ti
from oracle import plan_oracle as po
from oracle import schedule_oracle as so
from paper_2211_05322_b200 import inputs
from paper_2211_05322_b200 import reshard as rs
from test_planner_host import LAYOUTS, _check_tables, _layouts, _plan

ALGS = [rs.RS_SCHED_NAIVE, rs.RS_SCHED_LOAD_BALANCE, rs.RS_SCHED_DFS, rs.RS_SCHED_GREEDY, rs.RS_SCHED_ENSEMBLE]
SHAPE = (64, 64, 32)


def _both(shape, e, sm, ss, dm, ds, alg, sdph, ddph, seed=0, trials=0, budget=0):
    p = _plan(shape, e, sm, ss, dm, ds, 0, dict(schedule=alg, src_devices_per_host=sdph, dst_devices_per_host=ddph,
                                                seed=seed, trials=trials, node_budget=budget))
    ht = so.host_tasks(po.unit_tasks(shape, sm, ss, dm, ds), e, sdph, ddph)
    return p, p.schedule(), ht


def _valid(p, sch, ht, sdph):
    """what must hold for every algorithm: Eq. 2, S_i per PAPER.md:175, Eq. 3, Eq. 1, device in host"""
    sh, order, start, info = sch["sender_host"], sch["order"], sch["start"], sch["info"]
    assert sorted(order) == list(range(len(ht)))
    assert all(sh[i] in ht[i]["n"] for i in range(len(ht)))
    S, end = so.start_times(ht, sh, order)
    assert S == start and end == info.makespan
    assert so.check_eq3(ht, sh, start)
    assert info.busiest_host_bytes == so.eq4_bound(ht, sh) <= info.makespan
    for i, sl in enumerate(p.slices()):
        assert sl["sender"] in sl["senders"] and sl["sender"] // sdph == sh[i]
    assert sum(p.sender_bytes()) == p.info.tensor_bytes and max(p.sender_bytes()) == p.info.max_sender_bytes


@pytest.mark.parametrize("case", [1, 2, 3, 4, 5, 7, 8, 9])
def test_table2_cases_agree_with_the_oracle(case):
    ss, ds, sm, dm = inputs.TABLE2[case]
    sdph, ddph = sm[-1], dm[-1]                              # a mesh row is a host
    for alg in ALGS:
        p, sch, ht = _both(SHAPE, 2, sm, ss, dm, ds, alg, sdph, ddph, seed=11, budget=20000)
        _valid(p, sch, ht, sdph)
        got = (sch["sender_host"], sch["order"])
        if alg == rs.RS_SCHED_NAIVE:
            assert got == tuple(map(list, so.naive(ht)))
            assert all(sl["sender"] == min(d for d in sl["senders"] if d // sdph == h)
                       for sl, h in zip(p.slices(), sch["sender_host"]))
        elif alg == rs.RS_SCHED_LOAD_BALANCE:
            assert got == tuple(map(list, so.load_balance_only(ht)))
        elif alg == rs.RS_SCHED_GREEDY:
            s, o, rounds = so.randomized_greedy(ht, seed=11)
            assert got == (s, o) and sch["info"].n_rounds == len(rounds)
        elif alg == rs.RS_SCHED_DFS:
            end, _s, _o, fin = so.dfs_with_pruning(ht, node_budget=20000)
            assert bool(sch["info"].dfs_finished) == fin
            if fin:
                assert sch["info"].makespan == end
        else:
            assert sch["info"].makespan == so.ensemble(ht, seed=11, node_budget=20000)[0]


def test_paper_ordering_naive_ge_balanced_ge_ensemble():
    """the shape of Fig. 8 as simulated makespans"""
    for case in (1, 2, 3, 4, 5, 7, 8, 9):
        ss, ds, sm, dm = inputs.TABLE2[case]
        m = [_both(SHAPE, 2, sm, ss, dm, ds, alg, sm[-1], dm[-1], budget=20000)[1]["info"].makespan
             for alg in (rs.RS_SCHED_NAIVE, rs.RS_SCHED_LOAD_BALANCE, rs.RS_SCHED_ENSEMBLE)]
        assert m[0] >= m[1] >= m[2]
        if case in (3, 4, 5, 9):
            assert m[1] > m[2]


@settings(max_examples=40, deadline=None)
@given(_layouts(), st.sampled_from([1, 2, 4]), st.sampled_from([1, 2, 3]), st.integers(0, 2 ** 40))
def test_random_layouts(layout, sdph, ddph, seed):
    shape, sm, ss, dm, ds, dtype, _tile = layout
    e = np.dtype(dtype).itemsize
    try:
        tasks = po.unit_tasks(shape, sm, ss, dm, ds)
    except po.DivisError:
        return
    for alg in ALGS:
        p, sch, ht = _both(shape, e, sm, ss, dm, ds, alg, sdph, ddph, seed=seed, trials=8, budget=3000)
        _valid(p, sch, ht, sdph)
        if alg == rs.RS_SCHED_LOAD_BALANCE:
            assert (sch["sender_host"], sch["order"]) == tuple(map(list, so.load_balance_only(ht)))
        if alg == rs.RS_SCHED_GREEDY:
            assert (sch["sender_host"], sch["order"]) == so.randomized_greedy(ht, seed, 8)[:2]
        if alg == rs.RS_SCHED_DFS and sch["info"].dfs_finished and len(tasks) <= 5:
            try:
                assert sch["info"].makespan == so.bruteforce(ht, limit=200000)[0]
            except ValueError:
                pass


def test_unequal_durations_dfs_is_optimal():
    """2-way x 3-way cuts: slices of 2 sizes; the finished search equals the brute-force optimum"""
    shape, sm, ss, dm, ds = (12, 6), (2, 3), "S0,R", (3, 2), "S0,R"
    p, sch, ht = _both(shape, 4, sm, ss, dm, ds, rs.RS_SCHED_DFS, 1, 1, budget=10 ** 6)
    assert len({t["T"] for t in ht}) > 1 and sch["info"].dfs_finished
    assert sch["info"].makespan == so.bruteforce(ht)[0]


@pytest.mark.parametrize("shape,sm,ss,dm,ds", LAYOUTS)
def test_scheduled_tables_replay_equals_oracle(shape, sm, ss, dm, ds):
    """the tables follow the schedule; the data result does not change (R10)"""
    for alg, dph in ((rs.RS_SCHED_ENSEMBLE, 1), (rs.RS_SCHED_GREEDY, 2), (rs.RS_SCHED_NAIVE, 4)):
        p = _check_tables(shape, np.int16, sm, ss, dm, ds,
                          opts=dict(schedule=alg, src_devices_per_host=dph, dst_devices_per_host=dph, seed=5))
        sch = p.schedule()
        tasks, _d, _t = ti.tables(p, rs.RS_OP_EXECUTE)
        # execute lists one task per slice in order of start time: recover each task's slice by its sender + offset
        starts = [sch["start"][i] for i in sorted(range(len(sch["start"])), key=lambda i: (sch["start"][i], sch["order"].index(i)))]
        assert starts == sorted(sch["start"]) and len(tasks) == p.info.n_slices
        by_start = sorted(range(p.info.n_slices), key=lambda i: (sch["start"][i], sch["order"].index(i)))
        assert [int(t["src_buf"]) for t in tasks] == [p.slice(i)["sender"] for i in by_start]


def test_unscheduled_plan_has_no_schedule_and_bad_options_fail():
    p = _plan((8, 8), 2, (2,), "S0,R", (2,), "R,S0")
    with pytest.raises(rs.ReshardError):
        p.schedule()
    with pytest.raises(rs.ReshardError):
        _plan((8, 8), 2, (2,), "S0,R", (2,), "R,S0", 0, dict(schedule=9))


@pytest.mark.parametrize("n", [96, 128])
@pytest.mark.parametrize("alg", [rs.RS_SCHED_DFS, rs.RS_SCHED_ENSEMBLE])
def test_thousands_of_unit_tasks_do_not_overflow_the_stack(n, alg):
    """n x n unit tasks (9216 / 16384) on 128-device meshes: the DFS is iterative and skipped above 4096 tasks
    (useless beyond ~20); the schedule is still valid (makespan >= the busiest host's bytes)"""
    p = rs.Plan((4 * n, 4 * n), 2, (n,), "S0,R", (n,), "R,S0", rs.RS_HOST_ONLY, dict(schedule=alg))
    info = p.schedule()["info"]
    assert p.info.n_slices == n * n and info.dfs_finished == 0 and info.dfs_nodes == 0
    assert info.makespan >= info.busiest_host_bytes > 0
    if alg == rs.RS_SCHED_ENSEMBLE:
        assert info.winner == rs.RS_SCHED_GREEDY


def test_deep_dfs_runs_inside_its_node_budget():
    """2500 unit tasks: the search descends 2500 levels on the heap and stops at the node budget"""
    p = rs.Plan((200, 200), 2, (50,), "S0,R", (50,), "R,S0", rs.RS_HOST_ONLY, dict(schedule=rs.RS_SCHED_DFS, node_budget=6000))
    info = p.schedule()["info"]
    assert info.dfs_finished == 0 and info.dfs_nodes == 6000 and info.makespan >= info.busiest_host_bytes
