"""Iteration latency of 1F1B vs eager-1F1B (PAPER.md S4) from the library's timeline simulator, relative to the
communication-free latency (M + S - 1)(f + b) -- the shape of Fig. 9 without a cluster.
Compute times are parameters (ticks); the transfer time is given as a fraction of the forward time.  Host only.

    python -m paper_2211_05322_b200.pipeline_report [n_stages] [n_micro_batches]
"""
import sys

from . import reshard as rs


def rows(S=4, M=32, f=100, b=200):
    out = []
    for pct in (0, 10, 25, 50, 100):
        c = f * pct // 100
        ideal = (M + S - 1) * (f + b)
        r = {"comm/fwd": pct}
        r["no overlap, 1F1B"] = rs.pipeline_simulate(rs.RS_PIPE_1F1B, S, M, f, b, c, c, overlap=False)["makespan"] / ideal
        r["overlap, 1F1B"] = rs.pipeline_simulate(rs.RS_PIPE_1F1B, S, M, f, b, c, c)["makespan"] / ideal
        e = rs.pipeline_simulate(rs.RS_PIPE_EAGER_1F1B, S, M, f, b, c, c)
        r["overlap, eager-1F1B"] = e["makespan"] / ideal
        d = rs.pipeline_least_delay(rs.RS_PIPE_EAGER_1F1B, S, 1, M, f, b, b // 2, c)
        r["+ weight delaying (least delay)"] = rs.pipeline_simulate(rs.RS_PIPE_EAGER_1F1B, S, M, f, b, c, c, bwd_act=b // 2,
                                                                   bw_delay=d)["makespan"] / ideal
        r["delay"] = d
        r["peak activations, stage 1 (1F1B / eager)"] = "%d / %d" % (
            rs.pipeline_simulate(rs.RS_PIPE_1F1B, S, M, f, b, c, c)["peak"][0], e["peak"][0])
        out.append(r)
    return out


if __name__ == "__main__":
    S = int(sys.argv[1]) if len(sys.argv) > 1 else 4
    M = int(sys.argv[2]) if len(sys.argv) > 2 else 32
    rws = rows(S, M)
    keys = list(rws[0])
    print("| " + " | ".join(keys) + " |")
    print("|" + "---|" * len(keys))
    for r in rws:
        print("| " + " | ".join(("%.3f" % r[k]) if isinstance(r[k], float) else str(r[k]) for k in keys) + " |")
