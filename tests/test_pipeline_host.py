"""S4 in the library (csrc/pipeline.cpp, reshard_pipeline_simulate) against the pipeline oracle: integer
ticks, so every start and end time must agree exactly."""
import pytest
from hypothesis import given, settings, strategies as st

from oracle import pipeline_oracle as pp
from paper_2211_05322_b200 import reshard as rs

KIND = {rs.RS_PIPE_F: "F", rs.RS_PIPE_B: "B", rs.RS_PIPE_BA: "BA", rs.RS_PIPE_BW: "BW"}
NAME = {rs.RS_PIPE_1F1B: "1f1b", rs.RS_PIPE_EAGER_1F1B: "eager"}


def _same(sched, S, M, f, b, cf, cb, overlap=True, ba=None, delay=0):
    got = rs.pipeline_simulate(sched, S, M, f, b, cf, cb, overlap, ba, delay)
    want = pp.simulate(NAME[sched], S, M, f, b, cf, cb, overlap, ba, delay)
    assert got["makespan"] == want["makespan"]
    for i in range(S):
        assert [(KIND[k], m) for k, m, _s, _e in got["ops"][i]] == want["ops"][i + 1]
        for k, m, s, e in got["ops"][i]:
            assert (s, e) == (want["start"][(i + 1, KIND[k], m)], want["end"][(i + 1, KIND[k], m)])
        assert got["peak"][i] == want["peak"][i + 1] and got["busy"][i] == want["busy"][i + 1]
        assert got["warmup"][i] == pp.warmup_count(NAME[sched], S, i + 1, M)
    return got


@settings(max_examples=120, deadline=None)
@given(st.sampled_from([rs.RS_PIPE_1F1B, rs.RS_PIPE_EAGER_1F1B]), st.integers(1, 7), st.integers(1, 14),
       st.lists(st.integers(1, 9), min_size=7, max_size=7), st.lists(st.integers(2, 12), min_size=7, max_size=7),
       st.integers(0, 9), st.integers(0, 9), st.booleans(), st.sampled_from([None, 0, 1, 2, 3]))
def test_library_timeline_equals_oracle(sched, S, M, f, b, cf, cb, overlap, delay):
    f, b = f[:S], b[:S]
    ba = None if delay is None else [x // 2 for x in b]
    _same(sched, S, M, f, b, cf, cb, overlap, ba, delay or 0)


def test_paper_shape_overlap_then_eager():
    """PAPER.md:330 in shape: 'Overlap' beats 'Broadcast' (no overlap), eager-1F1B adds to it; a handful of
    micro-batches leaves little to gain, many micro-batches a lot"""
    S, f, b, c = 4, 20, 40, 10
    for M, big in ((4, False), (64, True)):
        blocked = _same(rs.RS_PIPE_1F1B, S, M, f, b, c, c, overlap=False)["makespan"]
        overlap = _same(rs.RS_PIPE_1F1B, S, M, f, b, c, c)["makespan"]
        eager = _same(rs.RS_PIPE_EAGER_1F1B, S, M, f, b, c, c)["makespan"]
        ideal = (M + S - 1) * (f + b)
        assert ideal <= eager <= overlap <= blocked
        if big:
            assert eager < 1.05 * ideal and overlap > 1.2 * ideal
    assert _same(rs.RS_PIPE_1F1B, 4, 8, 1, 2, 0, 0)["makespan"] == _same(rs.RS_PIPE_EAGER_1F1B, 4, 8, 1, 2, 0, 0)["makespan"] == 33


def test_least_delay_and_bad_arguments():
    for stage in (1, 2, 3):
        for c in (0, 1, 2, 3, 5, 9):
            assert rs.pipeline_least_delay(rs.RS_PIPE_EAGER_1F1B, 4, stage, 16, 2, 4, 2, c) == pp.least_delay("eager", 4, stage, 16, 2, 4, 2, c)
    # a transfer no delay can cover: the oracle answers with its search limit 2 M, the library says so with -1
    assert pp.least_delay("eager", 4, 1, 4, 2, 4, 2, 10 ** 6) == 8
    assert rs.pipeline_least_delay(rs.RS_PIPE_EAGER_1F1B, 4, 1, 4, 2, 4, 2, 10 ** 6) == -1
    with pytest.raises(rs.ReshardError):
        rs.pipeline_simulate(rs.RS_PIPE_1F1B, 0, 4, 1, 2, 0, 0)
    with pytest.raises(rs.ReshardError):
        rs.pipeline_simulate(7, 2, 4, 1, 2, 0, 0)
    with pytest.raises(rs.ReshardError):
        rs.pipeline_simulate(rs.RS_PIPE_1F1B, 2, 4, 1, 2, 0, 0, bwd_act=3)          # longer than the whole backward
