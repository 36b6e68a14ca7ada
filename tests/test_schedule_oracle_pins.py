"""Pins of the schedule-side oracle (oracle/schedule_oracle.py): hand-computed
timelines, the facts the paper states about Table 2, brute force, and an independent statement of
Eq. 3."""
import itertools

import pytest
from hypothesis import given, settings, strategies as st

import golden_io
from oracle import plan_oracle as po
from oracle import schedule_oracle as so
from paper_2211_05322_b200 import inputs

G = golden_io.load("table2_schedule_facts.txt")
SHAPE = (64, 64, 32)                      # Table 2's (1024, 1024, 512) scaled by 1/16: same slices


def table2_hosts(case, e=2):
    ss, ds, sm, dm = inputs.TABLE2[case]
    tasks = po.unit_tasks(SHAPE, sm, ss, dm, ds)
    return so.host_tasks(tasks, e, sm[-1], dm[-1])      # a mesh row is a host


def span(ht, senders, order):
    S, end = so.start_times(ht, senders, order)
    assert so.check_eq3(ht, senders, S)
    return end


def test_splitmix64_public_vector():
    gamma = 0x9E3779B97F4A7C15
    assert [so.mix64(gamma), so.mix64(2 * gamma)] == G["splitmix64_seed0_out"]


def test_shuffled_is_a_deterministic_permutation():
    a = so.shuffled(range(20), 7, 3)
    assert sorted(a) == list(range(20)) and a == so.shuffled(range(20), 7, 3)
    assert a != so.shuffled(range(20), 7, 4) and a != list(range(20))


def test_hand_timeline_unequal_durations():
    ht = [dict(T=t, n=[s], m=[r]) for t, s, r in zip(G["hand_T"], G["hand_sender"], G["hand_receiver"])]
    senders = G["hand_sender"]
    S, end = so.start_times(ht, senders, [0, 1, 2])
    assert S == G["hand_order_abc_start"] and end == G["hand_order_abc_makespan"][0]
    S, end = so.start_times(ht, senders, [0, 2, 1])
    assert S == G["hand_order_acb_start"] and end == G["hand_order_acb_makespan"][0]
    assert so.bruteforce(ht)[0] == G["hand_order_acb_makespan"][0]


def test_case3_hand_timeline():
    ht = table2_hosts(3)
    T = ht[0]["T"]
    assert [(t["n"], t["m"]) for t in ht] == [([0], [0]), ([1], [0]), ([0], [1]), ([1], [1])]
    senders, order = so.naive(ht)
    S, end = so.start_times(ht, senders, order)
    assert [s // T for s in S] == G["case3_naive_start"] and end == G["case3_naive_makespan"][0] * T
    S, end = so.start_times(ht, senders, G["case3_best_order"])
    assert [s // T for s in S] == G["case3_best_start"] and end == G["case3_best_makespan"][0] * T


def test_paper_narrative_cases_1_2_8():
    """PAPER.md:320."""
    for case in (1, 8):
        ht = table2_hosts(case)
        T = ht[0]["T"]
        ends = {span(ht, *so.naive(ht)), span(ht, *so.load_balance_only(ht)), so.ensemble(ht)[0]}
        assert ends == {G["case%d_makespan" % case][0] * T}
    ht = table2_hosts(2)
    T = ht[0]["T"]
    s, o = so.naive(ht)
    assert set(s) == {0}                                   # "sends all tensors from the first node"
    assert span(ht, s, o) == G["case2_naive_makespan"][0] * T
    assert span(ht, *so.load_balance_only(ht)) == G["case2_balanced_makespan"][0] * T


@pytest.mark.parametrize("case", [3, 4, 5, 9])
def test_paper_narrative_congested_cases(case):
    """naive and load-balance-only are congested, the ensemble leaves no host idle."""
    ht = table2_hosts(case)
    T = ht[0]["T"]
    opt = G["case%d_optimum" % case][0] * T
    assert so.eq4_bound(ht) == opt
    assert span(ht, *so.naive(ht)) > opt
    assert span(ht, *so.load_balance_only(ht)) > opt
    end, s, o, _which = so.ensemble(ht, seed=1, node_budget=20000)
    assert end == opt and span(ht, s, o) == opt


def test_dfs_budget_fails_beyond_20_tasks_greedy_does_not():
    """PAPER.md:179 vs 195, on case 4 (64 unit tasks)."""
    ht = table2_hosts(4)
    assert len(ht) == 64
    end, s, o, finished = so.dfs_with_pruning(ht, node_budget=20000)
    assert not finished and end > so.eq4_bound(ht) and span(ht, s, o) == end
    s, o, rounds = so.randomized_greedy(ht, seed=3)
    assert span(ht, s, o) == so.eq4_bound(ht) and len(rounds) == 32
    assert all(len(r) == 2 for r in rounds)                # both sender and both receiver hosts busy


def test_closed_forms():
    # one receiver host shared by everything: fully serial whatever the order
    ht = [dict(T=t, n=[i], m=[0]) for i, t in enumerate([5, 3, 9, 1])]
    for order in itertools.permutations(range(4)):
        assert so.start_times(ht, [0, 1, 2, 3], order)[1] == 18
    # no common host at all: fully parallel
    ht = [dict(T=t, n=[i], m=[i]) for i, t in enumerate([5, 3, 9, 1])]
    for order in itertools.permutations(range(4)):
        assert so.start_times(ht, [0, 1, 2, 3], order)[1] == 9
    # multicast: one task to every receiver host blocks them all
    ht = [dict(T=4, n=[0], m=[0, 1, 2]), dict(T=2, n=[1], m=[1]), dict(T=3, n=[2], m=[2])]
    assert so.start_times(ht, [0, 1, 2], [0, 1, 2])[0] == [0, 4, 4]
    assert so.bruteforce(ht)[0] == 7


def test_check_eq3_rejects_overlap():
    ht = [dict(T=2, n=[0], m=[0]), dict(T=2, n=[0], m=[1]), dict(T=2, n=[1], m=[1])]
    assert so.check_eq3(ht, [0, 0, 1], [0, 2, 4])
    assert not so.check_eq3(ht, [0, 0, 1], [0, 1, 4])      # same sender host
    assert not so.check_eq3(ht, [0, 0, 1], [0, 2, 3])      # common receiver host
    assert so.check_eq3(ht, [0, 0, 1], [0, 2, 0])          # tasks 0 and 2 share nothing


host_task = st.builds(
    lambda T, n, m: dict(T=T, n=sorted(n), m=sorted(m)),
    st.integers(1, 6), st.sets(st.integers(0, 2), min_size=1, max_size=3), st.sets(st.integers(0, 2), min_size=1, max_size=2))


@settings(max_examples=60, deadline=None)
@given(st.lists(host_task, min_size=1, max_size=5), st.integers(0, 1000))
def test_algorithms_against_bruteforce(ht, seed):
    opt, s_opt, o_opt = so.bruteforce(ht)
    assert span(ht, s_opt, o_opt) == opt
    assert so.eq4_bound(ht) <= opt <= sum(t["T"] for t in ht)
    end, s, o, finished = so.dfs_with_pruning(ht, node_budget=10 ** 7)
    assert finished and end == opt and span(ht, s, o) == opt        # the search is exact when it finishes
    for s, o in (so.naive(ht), so.load_balance_only(ht), so.randomized_greedy(ht, seed)[:2]):
        assert span(ht, s, o) >= opt
    end_e, s, o, _w = so.ensemble(ht, seed, node_budget=10 ** 7)
    assert end_e == opt
    # any order of any valid assignment is feasible and never beats the optimum
    order = so.shuffled(range(len(ht)), seed, 0)
    assert span(ht, [t["n"][-1] for t in ht], order) >= opt


def test_randomized_greedy_rounds_are_conflict_free():
    ht = table2_hosts(9)
    s, o, rounds = so.randomized_greedy(ht, seed=5)
    assert sorted(o) == list(range(len(ht)))
    for r in rounds:
        hosts = [("s", s[i]) for i in r] + [("r", h) for i in r for h in ht[i]["m"]]
        assert len(hosts) == len(set(hosts))
