"""Simulated makespans (Eq. 1) of the paper's Table 2 cases under every S3.2 algorithm
of the library -- the shape of Fig. 8 without a network: T_i = slice bytes, a
mesh row is a host.  Host-only plans: runs on any machine with the library built.

    python -m paper_2211_05322_b200.schedule_report
"""
from . import inputs
from . import reshard as rs

ALGS = [("naive", rs.RS_SCHED_NAIVE), ("load balance only", rs.RS_SCHED_LOAD_BALANCE), ("DFS (200k nodes)", rs.RS_SCHED_DFS),
        ("randomized greedy", rs.RS_SCHED_GREEDY), ("ensemble", rs.RS_SCHED_ENSEMBLE)]


def rows(cases=(1, 2, 3, 4, 5, 7, 8, 9), e=2):
    out = []
    for c in cases:
        w = inputs.table2_workload(c)
        row = {"case": c, "spec": "%s -> %s" % (w.src_spec, w.dst_spec)}
        for name, alg in ALGS:
            p = rs.Plan(w.shape, e, w.src_mesh, w.src_spec, w.dst_mesh, w.dst_spec, rs.RS_HOST_ONLY,
                        dict(schedule=alg, src_devices_per_host=w.src_mesh[-1], dst_devices_per_host=w.dst_mesh[-1]))
            s = p.schedule()["info"]
            row["n_tasks"], row["bound"] = s.n_tasks, s.busiest_host_bytes
            row[name] = s.makespan
            p.close()
        out.append(row)
    return out


if __name__ == "__main__":
    names = [n for n, _ in ALGS]
    print("| case | specs | unit tasks | " + " | ".join(names) + " | busiest host (ensemble senders) |")
    print("|---|---|---|" + "---|" * (len(names) + 1))
    for r in rows():
        unit = r["bound"] / 1.0
        print("| %d | %s | %d | " % (r["case"], r["spec"], r["n_tasks"]) +
              " | ".join("%.2f" % (r[n] / unit) for n in names) + " | %d MiB |" % (r["bound"] >> 20))
