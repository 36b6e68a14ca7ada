"""Pins of the pipeline-schedule oracle (oracle/pipeline_oracle.py): the warm-up counts
the paper prints, a hand-written timeline, the textbook no-communication latency, and the properties S4
states about the two schedules."""
import pytest
from hypothesis import given, settings, strategies as st

import golden_io
from oracle import pipeline_oracle as pp

G = golden_io.load("pipeline_facts.txt")


def test_warmup_counts_the_paper_prints():
    S = G["n_stages"][0]
    assert [pp.warmup_count("1f1b", S, i, 100) for i in range(1, S + 1)] == G["warmup_1f1b"]
    assert [pp.warmup_count("eager", S, i, 100) for i in range(1, S + 1)] == G["warmup_eager"]
    assert [pp.warmup_count("eager", S, i, 4) for i in range(1, S + 1)] == [4, 4, 3, 1]       # capped at M (R28)
    for kind, want in (("1f1b", G["warmup_1f1b"]), ("eager", G["warmup_eager"])):
        for i in range(1, S + 1):
            ops = pp.stage_ops(kind, S, i, 16)
            assert [op for op, _m in ops[:want[i - 1] + 1]] == ["F"] * want[i - 1] + ["B"]
            assert sorted(m for op, m in ops if op == "F") == sorted(m for op, m in ops if op == "B") == list(range(16))


def test_hand_timeline():
    r = pp.simulate("1f1b", 2, 2, 1, 2, 1, 1)
    assert [r["start"][(1, op, m)] for op, m in r["ops"][1]] == G["hand_1f1b_stage1_start"]
    assert [r["start"][(2, op, m)] for op, m in r["ops"][2]] == G["hand_1f1b_stage2_start"]
    assert r["makespan"] == G["hand_1f1b_makespan"][0]


def test_no_communication_textbook_latency():
    S, M, f, b = G["n_stages"][0], G["example_micro_batches"][0], G["example_f"][0], G["example_b"][0]
    for kind in ("1f1b", "eager"):
        assert pp.simulate(kind, S, M, f, b, 0, 0)["makespan"] == G["example_no_comm_makespan"][0] == (M + S - 1) * (f + b)


@settings(max_examples=80, deadline=None)
@given(st.integers(1, 6), st.integers(1, 12), st.integers(1, 5), st.integers(1, 7), st.integers(0, 6), st.integers(0, 6))
def test_properties_section4_states(S, M, f, b, cf, cb):
    one = pp.simulate("1f1b", S, M, f, b, cf, cb)
    eag = pp.simulate("eager", S, M, f, b, cf, cb)
    blk = pp.simulate("1f1b", S, M, f, b, cf, cb, overlap=False)
    # equal when communication is free (and then = the textbook latency)
    z1, z2 = pp.simulate("1f1b", S, M, f, b, 0, 0), pp.simulate("eager", S, M, f, b, 0, 0)
    assert z1["makespan"] == z2["makespan"] == (M + S - 1) * (f + b)
    # communication only ever delays; eager never loses to 1F1B; hiding nothing is the slowest
    assert z1["makespan"] <= eag["makespan"] <= one["makespan"] <= blk["makespan"]
    # at most #stages more activations per stage, exactly S - i when M allows
    for i in range(1, S + 1):
        assert one["peak"][i] == min(M, S - i + 1) and eag["peak"][i] == min(M, 2 * (S - i) + 1)
        assert 0 <= eag["peak"][i] - one["peak"][i] <= S
    # every op ran once, after its input, in list order, and compute of a stage never overlaps itself
    for r in (one, eag, blk):
        for i in range(1, S + 1):
            t = 0
            for op, m in r["ops"][i]:
                assert r["start"][(i, op, m)] >= t
                t = r["end"][(i, op, m)]
                if op == "F" and i > 1:
                    assert r["start"][(i, op, m)] >= r["end"][(i - 1, "F", m)] + cf
                if op == "B":
                    assert r["start"][(i, op, m)] >= r["end"][(i, "F", m)]
                    if i < S:
                        assert r["start"][(i, op, m)] >= r["end"][(i + 1, "B", m)] + cb
            assert r["busy"][i] == M * (f + b)


def test_eager_hides_what_1f1b_cannot():
    """with communication, 1F1B pays per micro-batch, eager-1F1B only while filling and draining"""
    S, f, b, c = 4, 2, 4, 1
    d1 = pp.simulate("1f1b", S, 32, f, b, c, c)["makespan"] - pp.simulate("1f1b", S, 16, f, b, c, c)["makespan"]
    de = pp.simulate("eager", S, 32, f, b, c, c)["makespan"] - pp.simulate("eager", S, 16, f, b, c, c)["makespan"]
    assert de == 16 * (f + b) < d1                            # steady state of eager-1F1B is communication-free
    assert pp.simulate("eager", S, 32, f, b, c, c)["makespan"] - (32 + S - 1) * (f + b) \
        == pp.simulate("eager", S, 16, f, b, c, c)["makespan"] - (16 + S - 1) * (f + b)


def test_backward_weight_delaying():
    """the transfer leaves after the activation gradients; the weight gradients overlap it"""
    S, M, f, b, ba, c = 4, 16, 2, 4, 2, 2
    whole = pp.simulate("eager", S, M, f, b, c, c)
    split = pp.simulate("eager", S, M, f, b, c, c, b_act=ba, delay=0)
    assert split["makespan"] < whole["makespan"]
    for i in range(1, S + 1):
        ops = pp.stage_ops("eager", S, i, M, True, 1)
        assert sorted(m for op, m in ops if op == "BW") == list(range(M))
        for m in range(M):                                    # BW after its BA, one op later than with delay 0
            assert ops.index(("BW", m)) > ops.index(("BA", m))
        assert split["busy"][i] == M * (f + b)
    assert pp.least_delay("eager", S, 2, M, f, b, ba, 0) == 0
    assert pp.least_delay("eager", S, 2, M, f, b, ba, b - ba) == 0        # BW alone covers it
    assert pp.least_delay("eager", S, 2, M, f, b, ba, b - ba + 1) == 1    # needs one more op in between
