#!/usr/bin/env python
"""bench.py -- resharding GB/s (unique bytes read + bytes written) of the hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c4] [--impl ours|reference]

A STEP is one pass of the device rows of the hot path over one synthetic
tensor: reshard_execute, reshard_pack, reshard_unpack, one kernel launch each, back to back on one
stream.  The host rows a1..a5 (reshard_plan) run once before the timed region (SURVEY.md S8(d):
"plan once outside the timed region"); their time is reported as plan_ms.
value = algorithmic bytes of the three launches / step time, inputs resident in HBM.
e2e   = the same metric for reshard_execute_host: HOST (pinned) shards in, HOST shards out, copies
        inside the timed region.
One JSON line on stdout (rank 0).  Multi-GPU: "replicas only": every rank runs the same
task on its own GPU, no data-path collective; value = N x bytes / max-over-ranks time.
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "resharding GB/s (unique read+write bytes)"
NOMINAL_HBM_GBS = 8000.0          # BASELINE.json: "~8 TB/s"; the >=70 % bar refers to this
FALLBACK_HBM_GBS = 6650.0         # B200_PROFILING.md fallback if MEASURED_PEAKS.json is absent
# dram__bytes_read.sum + dram__bytes_write.sum of ONE rs_copy_* launch of reshard_execute, from the
# `ncu --set full` capture summarised in profiles/ (null for workloads without a capture)
NCU_TRAFFIC_BYTES = {            # profiles/r01_ncu_sweep.md (read + write, one reshard_execute launch)
    "c4": 1615138000 + 1562324000, "c2": 134619000 + 86010000, "u4": 1542835000 + 1459713000,
    "t2_9": 1078115000 + 4236157000,
    "sweep_P1_m8_1024MiB": 1076611000 + 1025437000, "sweep_P2_m8_1024MiB": 1077257000 + 4237063000,
    "sweep_P3_m8_1024MiB": 1076592000 + 1026159000, "sweep_P4_m8_1024MiB": 1076634000 + 1024245000,
    "sweep_P5_m8_1024MiB": 1076652000 + 8530394000, "sweep_P6_m8_1024MiB": 1076653000 + 1021720000,
}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c4", help="c4 (default, 1.5 GiB GPT activation), c2, c3, t2_<n>, sweep_<pair>_<m8|m4>_<MiB>MiB")
    ap.add_argument("--path", default="auto", choices=["auto", "lsu", "bulk", "shift"])
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="target CPU work of the oracle sample")
    ap.add_argument("--sweep", default=None, help="time execute/pack/unpack on a list of workloads instead of the step: "
                    "'configs' (c2,c3,c3i,c3ii,c4), 'pairs' (6 pairs x 2 mesh pairs x 1 MiB..4 GiB), 'table2', 'fig5' (1 sender -> n receivers), 'all', "
                    "or comma-separated workload names; one JSON line per workload")
    ap.add_argument("--strategies", action="store_true", help="with --sweep: also time RS_STRATEGY_SENDRECV and "
                    "RS_STRATEGY_ALLGATHER (PAPER.md S3.1) against the broadcast executor")
    ap.add_argument("--overlap", action="store_true", help="resharding beside compute (PAPER.md S4, on chip): reshard_execute "
                    "on a high-priority stream limited to max_ctas CTAs while torch.matmul (cuBLAS) runs on another stream")
    ap.add_argument("--group", action="store_true", help="many tensors across one stage boundary (PAPER.md:100): n copies of "
                    "--workload resharded by n launches against ONE launch of a reshard_plan_group")
    ap.add_argument("--sweep-md", default=None, help="also write the sweep as a markdown table to this file")
    return ap.parse_args()


def peak_hbm():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, torch copy_)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


# ------------------------------------------------------------------ oracle timing (CPU baseline / reference arm)

def oracle_sample(w, seconds, steps=1, warmup=0, one_core=False):
    """Time the oracle AS IT STANDS on a bounded sample of workload w: whole destination shards
    (devices 0, 1, ...) until about `seconds` of wall time, all host cores.  Source shards hold a
    cheap seeded byte pattern (the oracle's cost does not depend on values).  Returns dict."""
    import numpy as np
    from oracle import data_oracle as do
    from paper_2211_05322_b200 import inputs
    e = inputs.elem_bytes(w.dtype)
    ct = np.dtype({1: np.uint8, 2: np.int16, 4: np.int32, 8: np.int64}[e])
    cores = do.max_threads()
    n_src, n_dst = do.num_devices(w.src_mesh), do.num_devices(w.dst_mesh)
    lshape = do.local_shape(w.shape, w.src_mesh, w.src_spec)
    # only the lowest-index replica of each source tile is dereferenced: alias replicas of a tile
    bufs, src = {}, []
    for r in range(n_src):
        key = do.device_box(w.shape, w.src_mesh, w.src_spec, r)
        if key not in bufs:
            a = np.arange(int(np.prod(lshape)), dtype=np.int64)
            bufs[key] = ((a * 2654435761 + w.seed + r) >> 7).astype(ct).reshape(lshape)
        src.append(bufs[key])
    out = np.empty(do.local_shape(w.shape, w.dst_mesh, w.dst_spec), dtype=ct)
    shard_bytes = out.nbytes
    r_B = n_dst * shard_bytes / (int(np.prod(w.shape)) * e)           # destination replication
    per_shard_metric_bytes = shard_bytes * (1.0 + 1.0 / r_B)            # written + its share of the unique read
    times, shards_done = [], 0
    for it in range(warmup + steps):
        t0 = time.perf_counter()
        q = 0
        while True:
            do.reshard_device(w.shape, e, w.src_mesh, w.src_spec, w.dst_mesh, w.dst_spec, src, q % n_dst, ct,
                              n_threads=cores, out=out)
            q += 1
            if time.perf_counter() - t0 >= seconds:
                break
        dt = time.perf_counter() - t0
        if it >= warmup:
            times.append(dt / q)
            shards_done = q
    t = statistics.median(times)
    t1 = None
    if one_core:                                                       # also at 1 thread (one shard)
        t0 = time.perf_counter()
        do.reshard_device(w.shape, e, w.src_mesh, w.src_spec, w.dst_mesh, w.dst_spec, src, 0, ct, n_threads=1, out=out)
        t1 = time.perf_counter() - t0
    return {"value_1core": None if t1 is None else per_shard_metric_bytes / t1 / 1e9, "value": per_shard_metric_bytes / t / 1e9, "unit": "GB/s", "cores": cores, "kind": "oracle",
            "sample": "%d destination shards of %s computed in full (devices 0..%d cyclically, %.0f MiB each), %d threads, %.2f s per shard"
                      % (shards_done, w.name, n_dst - 1, shard_bytes / 2**20, cores, t),
            "seconds_per_shard": t, "shards": shards_done}


def run_reference(args):
    """--impl reference: the oracle on host cores, same metric/config; rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return 0
    from paper_2211_05322_b200 import inputs
    w = inputs.get_workload(args.workload)
    steps, warmup = max(1, args.steps), max(0, args.warmup)
    budget = 150.0                                                     # whole run within a few minutes
    per_step = max(1.0, min(args.cpu_seconds, budget / (steps + warmup)))
    r = oracle_sample(w, per_step, steps=steps, warmup=warmup)
    line = {"impl": "reference", "metric": METRIC, "value": r["value"], "unit": "GB/s", "n_gpus": args.gpus,
            "steps": steps, "warmup": warmup, "ms_per_step": r["seconds_per_shard"] * r["shards"] * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u8", "data": "synthetic",
            "config": _config(w, "cpu-oracle"), "gpu_launches": 0,
            "cpu_baseline": {k: r[k] for k in ("value", "unit", "cores", "kind", "sample")},
            "e2e": {"value": r["value"], "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))
    return 0


def _config(w, path):
    return {"workload": "%s: %s %s, src mesh %s spec (%s) -> dst mesh %s spec (%s)" % (
                w.name, w.dtype, list(w.shape), "x".join(map(str, w.src_mesh)), w.src_spec,
                "x".join(map(str, w.dst_mesh)), w.dst_spec),
            "step": "reshard_execute + reshard_pack + reshard_unpack (plan outside the timed region)",
            "executor": path, "l2": "inputs larger than L2 (no flush needed)", "parallelism": "replicas only"}


# ------------------------------------------------------------------ clocks

SMI_FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")


class ClockSampler:
    """nvidia-smi -lms 50 in the background while the timed region runs"""

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + SMI_FIELDS,
                                       "--format=csv,noheader,nounits", "-lms", "50"], stdout=self.f,
                                      stderr=subprocess.DEVNULL)
        except OSError:
            pass

    def n_samples(self):
        try:
            with open(self.f.name) as f:
                return sum(1 for _ in f)
        except OSError:
            return 0

    def stop(self):
        if self.p is not None:
            self.p.terminate()
            try:
                self.p.wait(timeout=5)
            except subprocess.TimeoutExpired:
                self.p.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        try:
            with open(self.f.name) as f:
                for line in f:
                    c = [x.strip() for x in line.split(",")]
                    if len(c) < 8:
                        continue
                    try:
                        sm.append(float(c[0])); mx.append(float(c[1]))
                    except ValueError:
                        continue
                    for name, v in zip(names, c[4:8]):
                        if v.lower().startswith("active"):
                            reasons.add(name)
            os.unlink(self.f.name)
        except OSError:
            pass
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "reasons": sorted(reasons), "samples": len(sm)}


# ------------------------------------------------------------------ our arm

def run_ours(args):
    import torch
    from paper_2211_05322_b200 import harness, inputs, multi
    from paper_2211_05322_b200 import reshard as rs

    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        multi.init("nccl", dev)

    def barrier():
        multi.barrier(torch.cuda.synchronize)

    w = inputs.get_workload(args.workload)
    flags = {"auto": rs.RS_PATH_AUTO, "lsu": rs.RS_PATH_LSU, "bulk": rs.RS_PATH_BULK, "shift": rs.RS_PATH_BULK_SHIFT}[args.path]
    t0 = time.perf_counter()
    plan = harness.make_plan(w, flags)                     # rows a1..a5, once, outside the timed region
    plan_ms = (time.perf_counter() - t0) * 1e3
    info = plan.info
    ops = [plan.op_info(o) for o in (rs.RS_OP_EXECUTE, rs.RS_OP_PACK, rs.RS_OP_UNPACK)]
    op_bytes = [o.read_bytes + o.write_bytes for o in ops]
    step_bytes = sum(op_bytes)

    D, src = harness.device_inputs(w, plan, dev)
    dst = harness.device_outputs(plan, D, dev)
    arena = torch.empty(info.arena_bytes, dtype=torch.uint8, device=dev)
    del D
    sp, dp, ap = harness.ptrs(src), harness.ptrs(dst), arena.data_ptr()
    stream = torch.cuda.current_stream()
    sh = stream.cuda_stream
    flush = None
    if step_bytes < (1 << 30):                              # working set comparable to the 126 MB L2: flush it
        flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev)

    K, W = max(1, args.steps), max(3, args.warmup)
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(K)]

    def step(e4=None):
        if flush is not None:
            flush.fill_(1)
        if e4: e4[0].record(stream)
        plan.execute(sp, dp, sh)
        if e4: e4[1].record(stream)
        plan.pack(sp, ap, sh)
        if e4: e4[2].record(stream)
        plan.unpack(ap, dp, sh)
        if e4: e4[3].record(stream)

    for _ in range(W):
        step()
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    n0 = rs.launch_count()
    barrier()
    for i in range(K):
        step(ev[i])
    barrier()
    launches = rs.launch_count() - n0
    if sampler is not None:
        t_end = time.perf_counter() + 2.0                   # short regions: keep the same load until >= 3 samples
        while sampler.n_samples() < 3 and time.perf_counter() < t_end:
            for _ in range(20):
                step()
            torch.cuda.synchronize()
        clocks = sampler.stop()
    if flush is None:
        total_ms = ev[0][0].elapsed_time(ev[-1][3])
    else:
        total_ms = sum(e[0].elapsed_time(e[3]) for e in ev)
    k_ms = [statistics.mean(e[j].elapsed_time(e[j + 1]) for e in ev) for j in range(3)]
    k_best = [min(e[j].elapsed_time(e[j + 1]) for e in ev) for j in range(3)]
    total_ms = multi.max_over_ranks(total_ms, dev)
    ms_per_step = total_ms / K
    value = multi.job_gbs(step_bytes, ms_per_step, world)

    # ---- end to end: host (pinned) shards in, host shards out, through reshard_execute_host
    e2e = None
    if not args.no_e2e:
        src_h = [torch.empty(s.shape, dtype=s.dtype).pin_memory() for s in src]
        for h, s in zip(src_h, src):
            h.copy_(s)
        dst_h = [torch.empty(d.shape, dtype=d.dtype).pin_memory() for d in dst]
        ws = torch.empty(plan.host_workspace_bytes(), dtype=torch.uint8, device=dev)
        shp, dhp = harness.ptrs(src_h), harness.ptrs(dst_h)
        up = down = 0
        for _ in range(2):
            c0 = rs.launch_count()
            up, down = plan.execute_host(shp, dhp, ws.data_ptr(), sh)
            n_slabs = rs.launch_count() - c0                 # one kernel launch per slab
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        n_e2e = max(1, args.e2e_steps)
        e0.record(stream)
        for _ in range(n_e2e):
            plan.execute_host(shp, dhp, ws.data_ptr(), sh)
            stream.synchronize()                            # the caller reads the result on the host
        e1.record(stream)
        barrier()
        e2e_ms = multi.max_over_ranks(e0.elapsed_time(e1) / n_e2e, dev)
        e2e = {"value": multi.job_gbs(op_bytes[0], e2e_ms, world), "unit": "GB/s", "h2d_bytes_per_step": up,
               "d2h_bytes_per_step": down, "ms_per_step": e2e_ms, "steps": n_e2e,
               "call": "reshard_execute_host (pinned host shards; H2D, kernel and D2H pipelined over %d slabs of dim 0)" % n_slabs}
        del src_h, dst_h, ws

    if rank != 0:
        multi.shutdown()
        return 0

    peak, peak_src = peak_hbm()
    names = ["reshard_execute", "reshard_pack", "reshard_unpack"]
    pname = {rs.RS_PATH_LSU: "rs_copy_lsu", rs.RS_PATH_BULK: "rs_copy_bulk", rs.RS_PATH_BULK_SHIFT: "rs_copy_bulk_shift"}
    kernels = {n: {"kernel": pname[o.path], "ms": k_ms[j], "best_ms": k_best[j], "bytes": op_bytes[j],
                   "GB/s": op_bytes[j] / (k_ms[j] * 1e-3) / 1e9, "grid": o.grid, "block": o.block,
                   "smem": o.smem_bytes, "tiles": o.n_tiles, "tile_bytes": o.tile_bytes}
               for j, (n, o) in enumerate(zip(names, ops))}
    achieved = kernels["reshard_execute"]["GB/s"]
    line = {"metric": METRIC, "value": value, "unit": "GB/s", "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "u8", "data": "synthetic", "config": _config(w, kernels["reshard_execute"]["kernel"]),
            "clocks": clocks, "gpu_launches": launches, "plan_ms": plan_ms,
            "pct_of_nominal_8TBs": 100.0 * achieved / NOMINAL_HBM_GBS,
            "roofline": {"bound": "hbm", "kernel": "reshard_execute (%s)" % kernels["reshard_execute"]["kernel"],
                         "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "peak_source": peak_src, "algorithmic_bytes": op_bytes[0],
                         "traffic": NCU_TRAFFIC_BYTES.get(w.name)},
            "kernels": kernels}
    if flush is not None:
        line["config"]["l2"] = "L2 flushed between steps (512 MiB fill); working set is L2-sized: effective GB/s"
    if e2e is not None:
        line["e2e"] = e2e
    if world == 1 and not args.no_cpu_baseline:
        r = oracle_sample(w, args.cpu_seconds, one_core=True)
        line["cpu_baseline"] = {k: r[k] for k in ("value", "unit", "cores", "kind", "sample", "value_1core")}
    print(json.dumps(line))
    multi.shutdown()
    return 0


# ------------------------------------------------------------------ sweep

def sweep_names(what):
    from paper_2211_05322_b200 import inputs
    cfg = ["c2", "c3", "c3i", "c3ii", "c4"]
    pairs = ["sweep_%s_%s_%dMiB" % (p, m, b >> 20) for p in inputs.SWEEP_PAIRS for m in inputs.SWEEP_MESHES
             for b in inputs.SWEEP_BYTES]
    t2 = ["t2_%d" % c for c in (1, 2, 3, 4, 5, 6, 7, 8, 9)]
    fig5 = ["fig5_%dx%d" % ab for ab in inputs.FIG5]
    return {"configs": cfg, "pairs": pairs, "table2": t2, "fig5": fig5, "all": cfg + pairs + t2}.get(what) or what.split(",")


def run_sweep(args):
    """Per workload: plan, then each of execute / pack / unpack timed alone with CUDA events on the
    launching stream (3 warm-up + --steps launches, L2 flushed before every launch when the
    operation moves < 1 GiB).  Buffer contents are irrelevant to a copy: shards are seeded bytes."""
    import torch
    from paper_2211_05322_b200 import harness, inputs
    from paper_2211_05322_b200 import reshard as rs
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    stream = torch.cuda.current_stream()
    sh = stream.cuda_stream
    peak, _ = peak_hbm()
    flags = {"auto": rs.RS_PATH_AUTO, "lsu": rs.RS_PATH_LSU, "bulk": rs.RS_PATH_BULK, "shift": rs.RS_PATH_BULK_SHIFT}[args.path]
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev)
    K = max(3, min(args.steps, 30))
    rows = []
    for name in sweep_names(args.sweep):
        w = inputs.get_workload(name)
        if args.strategies:                                 # a mesh row is a host: local all-gather per row
            plan = rs.Plan(w.shape, inputs.elem_bytes(w.dtype), w.src_mesh, w.src_spec, w.dst_mesh, w.dst_spec,
                           flags | rs.RS_WITH_STRATEGIES, dict(dst_devices_per_host=w.dst_mesh[-1]))
        else:
            plan = harness.make_plan(w, flags)
        info = plan.info
        g = torch.Generator(device=dev); g.manual_seed(w.seed % (1 << 31))
        def buf(n):
            t = torch.empty(n, dtype=torch.uint8, device=dev)
            t[: min(n, 1 << 26)].random_(0, 256, generator=g)
            return t
        src = [buf(info.src_shard_bytes) for _ in range(info.n_src)]
        dst = [torch.empty(info.dst_shard_bytes, dtype=torch.uint8, device=dev) for _ in range(info.n_dst)]
        arena = buf(info.arena_bytes)
        sp, dp, ap = harness.ptrs(src), harness.ptrs(dst), arena.data_ptr()
        calls = [("execute", rs.RS_OP_EXECUTE, lambda: plan.execute(sp, dp, sh)),
                 ("pack", rs.RS_OP_PACK, lambda: plan.pack(sp, ap, sh)),
                 ("unpack", rs.RS_OP_UNPACK, lambda: plan.unpack(ap, dp, sh))]
        if args.strategies:      # same result by the paper's other strategies; GB/s counts the USEFUL bytes (1 + r_B) like execute
            calls = [calls[0],
                     ("sendrecv", rs.RS_OP_EXECUTE, lambda: plan.execute_strategy(rs.RS_STRATEGY_SENDRECV, sp, dp, sh)),
                     ("allgather", rs.RS_OP_EXECUTE, lambda: plan.execute_strategy(rs.RS_STRATEGY_ALLGATHER, sp, dp, sh)),
                     ("allgather_local", rs.RS_OP_EXECUTE, lambda: plan.execute_strategy(rs.RS_STRATEGY_ALLGATHER_LOCAL, sp, dp, sh))]
        row = {"workload": name, "shape": list(w.shape), "src": "%s %s" % ("x".join(map(str, w.src_mesh)), w.src_spec),
               "dst": "%s %s" % ("x".join(map(str, w.dst_mesh)), w.dst_spec), "n_slices": info.n_slices,
               "tensor_bytes": info.tensor_bytes}
        for opname, op, call in calls:
            o = plan.op_info(op)
            nbytes = o.read_bytes + o.write_bytes
            do_flush = nbytes < (1 << 30)
            for _ in range(3):
                call()
            ts = []
            for _ in range(K):
                if do_flush:
                    flush.fill_(1)
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream); call(); e1.record(stream)
                e1.synchronize()
                ts.append(e0.elapsed_time(e1))
            med = statistics.median(ts)
            row[opname] = {"kernel": {rs.RS_PATH_BULK: "rs_copy_bulk", rs.RS_PATH_BULK_SHIFT: "rs_copy_bulk_shift"}.get(o.path, "rs_copy_lsu"), "bytes": nbytes,
                           "ms": med, "best_ms": min(ts), "GB/s": nbytes / med / 1e6, "frac_of_copy_peak": nbytes / med / 1e6 / peak,
                           "tiles": o.n_tiles, "tile_bytes": o.tile_bytes, "grid": o.grid, "l2_flushed": do_flush}
        plan.close()
        del src, dst, arena
        torch.cuda.empty_cache()
        # on-box ceiling: torch copy_ moving the same byte volume as execute (capped at 2 x 4 GiB)
        half = min(row["execute"]["bytes"] // 2, 4 << 30)
        a, b = torch.empty(half, dtype=torch.uint8, device=dev), torch.empty(half, dtype=torch.uint8, device=dev)
        for _ in range(3):
            b.copy_(a)
        ts = []
        for _ in range(K):
            if 2 * half < (1 << 30):
                flush.fill_(1)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream); b.copy_(a); e1.record(stream)
            e1.synchronize()
            ts.append(e0.elapsed_time(e1))
        row["torch_copy_same_volume_GB/s"] = 2 * half / statistics.median(ts) / 1e6
        del a, b
        torch.cuda.empty_cache()
        rows.append(row)
        print(json.dumps(row), flush=True)
    if args.sweep_md and args.strategies:
        with open(args.sweep_md, "w") as f:
            f.write("| workload | src -> dst | receivers per slice | broadcast ms (GB/s useful) | send/recv ms (x broadcast) | global all-gather ms (x broadcast) | local all-gather ms (x broadcast) | bytes moved: broadcast / others |\n")
            f.write("|---|---|---|---|---|---|---|---|\n")
            for r in rows:
                k = (r["execute"]["bytes"] - r["tensor_bytes"]) // r["tensor_bytes"]
                b = r["execute"]["ms"]
                f.write("| %s | %s -> %s | %d | %.3f (%.0f) | %.3f (%.2f) | %.3f (%.2f) | %.3f (%.2f) | %d / %d x size(D) |\n" % (
                    r["workload"], r["src"], r["dst"], k, b, r["execute"]["GB/s"], r["sendrecv"]["ms"], r["sendrecv"]["ms"] / b,
                    r["allgather"]["ms"], r["allgather"]["ms"] / b, r["allgather_local"]["ms"], r["allgather_local"]["ms"] / b,
                    1 + k, 2 * k))
        return 0
    if args.sweep_md:
        with open(args.sweep_md, "w") as f:
            f.write("| workload | tensor | src -> dst | slices | read + write (execute) | execute GB/s (frac of %.0f) | pack GB/s | unpack GB/s | torch copy_ same volume GB/s | kernel |\n" % peak)
            f.write("|---|---|---|---|---|---|---|---|---|---|\n")
            for r in rows:
                x = r["execute"]
                f.write("| %s | %s | %s -> %s | %d | %.0f + %.0f MiB | %.0f (%.3f) | %.0f | %.0f | %.0f | %s |\n" % (
                    r["workload"], r["shape"], r["src"], r["dst"], r["n_slices"], r["tensor_bytes"] / 2**20,
                    (x["bytes"] - r["tensor_bytes"]) / 2**20, x["GB/s"], x["frac_of_copy_peak"], r["pack"]["GB/s"],
                    r["unpack"]["GB/s"], r["torch_copy_same_volume_GB/s"], x["kernel"]))
    return 0


def run_overlap(args):
    """Per CTA cap: time N matmuls alone, M reshard_execute launches alone, then both started together on two
    streams (wall time on the device between a common start event and the later of the two end events).
    overlap gain = (t_gemm + t_reshard) / t_both: 1.0 = serialised, 2.0 = perfectly hidden."""
    import torch
    from paper_2211_05322_b200 import harness, inputs
    from paper_2211_05322_b200 import reshard as rs
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    w = inputs.get_workload(args.workload)
    n = 8192
    a = torch.randn(n, n, device=dev, dtype=torch.bfloat16)
    b = torch.randn(n, n, device=dev, dtype=torch.bfloat16)
    c = torch.empty(n, n, device=dev, dtype=torch.bfloat16)
    s_gemm = torch.cuda.Stream()
    s_copy = torch.cuda.Stream(priority=-1)                    # the copy's few CTAs get SMs as soon as they free up
    n_gemm, n_copy = 12, 16

    def timed(fn_g, fn_c):
        torch.cuda.synchronize()
        e0 = torch.cuda.Event(enable_timing=True)
        eg, ec = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(torch.cuda.current_stream())
        s_gemm.wait_event(e0); s_copy.wait_event(e0)
        if fn_c:
            with torch.cuda.stream(s_copy):
                fn_c()
                ec.record(s_copy)
        if fn_g:
            with torch.cuda.stream(s_gemm):
                fn_g()
                eg.record(s_gemm)
        torch.cuda.synchronize()
        return (e0.elapsed_time(eg) if fn_g else 0.0), (e0.elapsed_time(ec) if fn_c else 0.0)

    def gemms():
        for _ in range(n_gemm):
            torch.matmul(a, b, out=c)

    rows = []
    for cap in (0, 96, 64, 48, 32, 16):
        plan = rs.Plan(w.shape, inputs.elem_bytes(w.dtype), w.src_mesh, w.src_spec, w.dst_mesh, w.dst_spec, 0,
                       dict(max_ctas=cap))
        info = plan.info
        src = [torch.empty(info.src_shard_bytes, dtype=torch.uint8, device=dev) for _ in range(info.n_src)]
        dst = [torch.empty(info.dst_shard_bytes, dtype=torch.uint8, device=dev) for _ in range(info.n_dst)]
        sp, dp = harness.ptrs(src), harness.ptrs(dst)
        o = plan.op_info(rs.RS_OP_EXECUTE)

        def copies():
            for _ in range(n_copy):
                plan.execute(sp, dp, s_copy.cuda_stream)

        for _ in range(2):
            timed(gemms, copies)
        tg = statistics.median(timed(gemms, None)[0] for _ in range(5))
        tc = statistics.median(timed(None, copies)[1] for _ in range(5))
        both = [timed(gemms, copies) for _ in range(5)]
        tb = statistics.median(max(x) for x in both)
        nbytes = (o.read_bytes + o.write_bytes) * n_copy
        row = {"max_ctas": cap, "grid": o.grid, "gemm_alone_ms": tg, "reshard_alone_ms": tc, "both_ms": tb,
               "gemm_TFLOPs_alone": 2 * n ** 3 * n_gemm / tg / 1e9, "reshard_GBs_alone": nbytes / tc / 1e6,
               "gemm_TFLOPs_concurrent": 2 * n ** 3 * n_gemm / statistics.median(x[0] for x in both) / 1e9,
               "reshard_GBs_concurrent": nbytes / statistics.median(x[1] for x in both) / 1e6,
               "overlap_gain": (tg + tc) / tb, "workload": w.name}
        rows.append(row)
        print(json.dumps(row), flush=True)
        plan.close()
        del src, dst
    if args.sweep_md:
        with open(args.sweep_md, "w") as f:
            f.write("| max_ctas (grid) | reshard alone GB/s | GEMM alone TFLOP/s | concurrent: reshard GB/s | concurrent: GEMM TFLOP/s | both ms vs sum of alone ms | gain |\n")
            f.write("|---|---|---|---|---|---|---|\n")
            for r in rows:
                f.write("| %s (%d) | %.0f | %.0f | %.0f | %.0f | %.2f vs %.2f | %.2f |\n" % (
                    r["max_ctas"] or "library default", r["grid"], r["reshard_GBs_alone"], r["gemm_TFLOPs_alone"],
                    r["reshard_GBs_concurrent"], r["gemm_TFLOPs_concurrent"], r["both_ms"],
                    r["gemm_alone_ms"] + r["reshard_alone_ms"], r["overlap_gain"]))
    return 0


def run_group(args):
    """n tensors of the same layout pair: n x reshard_execute back to back against one grouped launch (CUDA events,
    L2 flushed before every timed region, median of --steps)."""
    import torch
    from paper_2211_05322_b200 import harness, inputs
    from paper_2211_05322_b200 import reshard as rs
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    stream = torch.cuda.current_stream()
    sh = stream.cuda_stream
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev)
    K = max(5, min(args.steps, 40))
    rows = []
    for name in args.workload.split(","):
        mixed = "+" in name                                  # a+b+c: ONE group of different workloads
        for n in ((len(name.split("+")),) if mixed else (1, 2, 4, 8)):
            ws = [inputs.get_workload(x) for x in name.split("+")] if mixed else [inputs.get_workload(name)] * n
            plans = [harness.make_plan(w) for w in ws]
            if sum(p.info.n_src for p in plans) > rs.RS_MAX_DEVICES or sum(p.info.n_dst for p in plans) > rs.RS_MAX_DEVICES:
                break
            src = [[torch.empty(p.info.src_shard_bytes, dtype=torch.uint8, device=dev) for _ in range(p.info.n_src)] for p in plans]
            dst = [[torch.empty(p.info.dst_shard_bytes, dtype=torch.uint8, device=dev) for _ in range(p.info.n_dst)] for p in plans]
            g = rs.Plan.group(plans)
            sp, dp = [harness.ptrs(x) for x in src], [harness.ptrs(x) for x in dst]
            gsp, gdp = [a for x in sp for a in x], [a for x in dp for a in x]

            def separate():
                for i in range(n):
                    plans[i].execute(sp[i], dp[i], sh)

            def grouped():
                g.execute(gsp, gdp, sh)

            res = {}
            for label, fn in (("separate", separate), ("grouped", grouped)):
                for _ in range(3):
                    fn()
                ts = []
                for _ in range(K):
                    flush.fill_(1)
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    e0.record(stream); fn(); e1.record(stream)
                    e1.synchronize()
                    ts.append(e0.elapsed_time(e1))
                res[label] = statistics.median(ts)
            nbytes = sum(p.info.unique_read_bytes + p.info.write_bytes for p in plans)
            row = {"workload": name, "tensors": n, "bytes": nbytes, "separate_us": res["separate"] * 1e3, "grouped_us": res["grouped"] * 1e3,
                   "separate_GBs": nbytes / res["separate"] / 1e6, "grouped_GBs": nbytes / res["grouped"] / 1e6,
                   "speedup": res["separate"] / res["grouped"]}
            rows.append(row)
            print(json.dumps(row), flush=True)
            g.close()
            for p in plans:
                p.close()
    if args.sweep_md:
        with open(args.sweep_md, "w") as f:
            f.write("| workload | tensors | bytes moved | n launches: us (GB/s) | one grouped launch: us (GB/s) | speedup |\n|---|---|---|---|---|---|\n")
            for r in rows:
                f.write("| %s | %d | %.1f MiB | %.1f (%.0f) | %.1f (%.0f) | %.2f |\n" % (r["workload"], r["tensors"], r["bytes"] / 2**20,
                        r["separate_us"], r["separate_GBs"], r["grouped_us"], r["grouped_GBs"], r["speedup"]))
    return 0


def main():
    args = parse_args()
    if args.group:
        return run_group(args)
    if args.overlap:
        return run_overlap(args)
    if args.sweep:
        return run_sweep(args)
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
