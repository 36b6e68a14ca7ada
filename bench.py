#!/usr/bin/env python
"""bench.py -- resharding GB/s (unique bytes read + bytes written) of the hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c4] [--impl ours|reference]

A STEP is one pass of the device rows of the hot path over one synthetic
tensor: reshard_execute, reshard_pack, reshard_unpack, one kernel launch each, back to back on one
stream.  The host rows a1..a5 (reshard_plan) run once before the timed region (SURVEY.md S8(d):
"plan once outside the timed region"); their time is reported as plan_ms (warm) / plan_ms_cold.
value = algorithmic bytes of the three launches / step time, inputs resident in HBM.
e2e   = the same metric for reshard_execute_host: HOST (pinned) shards in, HOST shards out, copies
        inside the timed region.
One JSON line on stdout (rank 0).  Multi-GPU: "replicas only": every rank runs the same
task on its own GPU, no data-path collective; value = N x bytes / max-over-ranks time.

Other modes (one JSON line per row, optional markdown with --md):
    --sweep LIST        execute / pack / unpack of each workload timed alone
    --roof              the roof of a 1-read + k-write stream on contiguous buffers (launch shapes swept)
    --group, --overlap, --strategies
    --ncu-summary name=report.ncu-rep ...   DRAM traffic of one captured launch per report -> CSV rows
    --sass              SASS opcode histogram of every kernel in libreshard.so (markdown)
    --report schedule|pipeline            the host-side tables of DESIGN.md S10
"""
import argparse
import csv
import io
import json
import math
import os
import re
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
L2_BYTES = 126 << 20
# tracked artefacts this file reads (written by `bench.py --ncu-summary` / `bench.py --roof --csv`)
TRAFFIC_CSV = os.path.join(ROOT, "profiles", "ncu_traffic.csv")
ROOF_CSV = os.path.join(ROOT, "profiles", "roof_1k.csv")
TUNING_FIELDS = ("bulk_warps", "bulk_stages", "bulk_lookahead", "bulk_tile_bytes", "bulk_ctas", "bulk_ctas_mcast", "shift_warps",
                 "shift_stages", "shift_lookahead", "shift_tile_bytes", "lsu_tile_bytes", "lsu_ctas_per_sm", "task_order",
                 "small_op_bytes_mib", "tiles_per_worker", "pace_permille", "no_pdl", "pace_burst", "pace_adapt", "ring_min_smem", "lsu_narrow", "shift_mode")


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c4", help="c4 (default, 1.5 GiB GPT activation), c2, c3, t2_<n>, sweep_<pair>_<m8|m4>_<MiB>MiB")
    ap.add_argument("--path", default="auto", choices=["auto", "lsu", "bulk", "shift", "tmap"])
    ap.add_argument("--mode", default="replicas", choices=["replicas", "sharded"], help="N > 1: 'replicas' (default, DESIGN.md S8: every rank runs "
                    "the whole task on its own GPU) or 'sharded' (the multi-process executor: virtual device r lives on rank r mod N, every "
                    "rank launches its share of the unit tasks and stores into its peers' shards through CUDA IPC; NCCL only for the barrier)")
    ap.add_argument("--tune", default="", help="rs_plan_opts.tuning overrides, e.g. bulk_ctas=148,bulk_warps=4 (A/B runs and ncu captures)")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="target CPU work of the oracle sample")
    ap.add_argument("--sweep", default=None, help="time execute/pack/unpack on a list of workloads instead of the step: "
                    "comma-separated workload names and/or the sets 'configs' (c2,c3,c3i,c3ii,c4), 'pairs' (6 pairs x 2 mesh pairs x "
                    "1 MiB..4 GiB), 'table2', 'fig5' (1 sender -> n receivers), 'all'; one JSON line per workload")
    ap.add_argument("--ops", default="execute,pack,unpack", help="with --sweep: which operations to time")
    ap.add_argument("--plain", action="store_true", help="with --sweep: every launch on its own between two events, one buffer set, no CUDA "
                    "graph (the protocol to run under ncu: -k regex:rs_copy -s 3 -c 1 captures the first timed launch)")
    ap.add_argument("--strategies", action="store_true", help="with --sweep: also time RS_STRATEGY_SENDRECV and "
                    "RS_STRATEGY_ALLGATHER (PAPER.md S3.1) against the broadcast executor")
    ap.add_argument("--roof", action="store_true", help="1 read + k writes on contiguous buffers, k = 1, 2, 4, 8: launch shapes swept, "
                    "beside torch copy_ / fill_ / sum and the read/write-rate model")
    ap.add_argument("--hot", action="store_true", help="with --sweep (operations >= 1 GiB moved): a burst of 24 bf16 8192^3 GEMMs before every timed launch, so that "
                    "the launch runs at the SM clock a training step leaves behind (power-limited, ~1.3-1.6 GHz) instead of the idle boost clock")
    ap.add_argument("--mix", default=None, help="reshard_execute of several workloads alternating in one stream (a,b[,c]) against each back to back alone")
    ap.add_argument("--overlap", action="store_true", help="resharding beside compute (PAPER.md S4, on chip): reshard_execute "
                    "on a high-priority stream limited to max_ctas CTAs while torch.matmul (cuBLAS) runs on another stream")
    ap.add_argument("--group", action="store_true", help="many tensors across one stage boundary (PAPER.md:100): n copies of "
                    "--workload resharded by n launches against ONE launch of a reshard_plan_group")
    ap.add_argument("--md", "--sweep-md", dest="md", default=None, help="also write the rows as a markdown table to this file")
    ap.add_argument("--csv", default=None, help="--roof: also write the best shape per k to this CSV (profiles/roof_1k.csv)")
    ap.add_argument("--ncu-summary", nargs="+", default=None, metavar="WORKLOAD:OP=REPORT",
                    help="summarise one-launch ncu reports into CSV rows (stdout); append them to profiles/ncu_traffic.csv")
    ap.add_argument("--sass", action="store_true", help="SASS opcode histogram per kernel of libreshard.so (markdown on stdout)")
    ap.add_argument("--report", default=None, choices=["schedule", "pipeline"], help="host-only tables of DESIGN.md S10")
    return ap.parse_args()


def parse_tune(text):
    out = {}
    for kv in filter(None, (text or "").split(",")):
        k, v = kv.split("=")
        if k not in TUNING_FIELDS:
            raise SystemExit("unknown tuning field %r (one of %s)" % (k, ", ".join(TUNING_FIELDS)))
        out[k] = int(v)
    return out


def peak_hbm():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, torch copy_)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def ncu_traffic(workload, op="execute"):
    """dram__bytes_read.sum + dram__bytes_write.sum of one launch of `op` on `workload`, from the tracked summary of
    the `ncu --set full` captures (profiles/ncu_traffic.csv, written by --ncu-summary; the last matching row wins).
    Returns (bytes or None, where it came from)."""
    try:
        with open(TRAFFIC_CSV) as f:
            rows = [r for r in csv.DictReader(f) if r["workload"] == workload and r["op"] == op]
    except OSError:
        return None, None
    if not rows:
        return None, None
    r = rows[-1]
    return int(r["dram_read_bytes"]) + int(r["dram_write_bytes"]), "profiles/ncu_traffic.csv: %s, captured at commit %s (%s us under ncu)" % (
        r["report"], r["commit"], r["duration_us"])


def roof_1k(k):
    """best measured GB/s of a contiguous 1-read + k-write stream (profiles/roof_1k.csv, written by --roof --csv)"""
    try:
        with open(ROOF_CSV) as f:
            for r in csv.DictReader(f):
                if int(r["k"]) == int(k):
                    return float(r["best_gbs"])
    except (OSError, KeyError, ValueError):
        pass
    return None


def git_commit():
    try:
        return subprocess.run(["git", "rev-parse", "--short", "HEAD"], capture_output=True, text=True, cwd=ROOT).stdout.strip() or "unknown"
    except OSError:
        return "unknown"


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
    t1 = tn = None
    if one_core:                                                       # also at 1 thread (one shard)
        t0 = time.perf_counter()
        do.reshard_device(w.shape, e, w.src_mesh, w.src_spec, w.dst_mesh, w.dst_spec, src, 0, ct, n_threads=1, out=out)
        t1 = time.perf_counter() - t0
        # context for the ratio: the same shard by numpy basic slicing of a global array (one memcpy-like
        # strided copy, 1 thread) -- what a run-wise CPU copy costs, as opposed to the element-by-element checker
        D = np.empty(w.shape, dtype=ct)
        lo, hi = do.device_box(w.shape, w.dst_mesh, w.dst_spec, 0)
        t0 = time.perf_counter()
        np.copyto(out[tuple(slice(0, b - a) for a, b in zip(lo, hi))], D[tuple(slice(a, b) for a, b in zip(lo, hi))])
        tn = time.perf_counter() - t0
        del D
    return {"value_1core": None if t1 is None else per_shard_metric_bytes / t1 / 1e9,
            "numpy_slicing_1core": None if tn is None else per_shard_metric_bytes / tn / 1e9,
            "value": per_shard_metric_bytes / t / 1e9, "unit": "GB/s", "cores": cores, "kind": "oracle",
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
            "config": _config(w), "executor": "cpu-oracle", "gpu_launches": 0,
            "cpu_baseline": {k: r[k] for k in ("value", "unit", "cores", "kind", "sample")},
            "e2e": {"value": r["value"], "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))
    return 0


def _config(w):
    """identical in both arms (the executor is a top-level key of the line, not part of the workload)"""
    return {"workload": "%s: %s %s, src mesh %s spec (%s) -> dst mesh %s spec (%s)" % (
                w.name, w.dtype, list(w.shape), "x".join(map(str, w.src_mesh)), w.src_spec,
                "x".join(map(str, w.dst_mesh)), w.dst_spec),
            "step": "reshard_execute + reshard_pack + reshard_unpack (plan outside the timed region)",
            "l2": "inputs larger than L2 (no flush needed)", "parallelism": "replicas only"}


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


# ------------------------------------------------------------------ timing protocols

_HEAT = None     # --hot: a burst of tensor-core GEMMs enqueued before every timed launch (the chip at its power-limited clocks)


def make_heater(torch, dev, n_gemms=24):
    n = 8192
    a = torch.randn(n, n, device=dev, dtype=torch.bfloat16)
    b = torch.randn(n, n, device=dev, dtype=torch.bfloat16)
    c = torch.empty(n, n, device=dev, dtype=torch.bfloat16)

    def heat():
        for _ in range(n_gemms):
            torch.matmul(a, b, out=c)
    for _ in range(8):
        heat()
    torch.cuda.synchronize()
    return heat


def time_each(call, stream, n, warm=3):
    """n launches, each between its own pair of CUDA events on the launching stream (operations much larger than
    L2: nothing to flush).  Returns (median ms, best ms)."""
    import torch
    for _ in range(warm):
        call()
    ts = []
    for _ in range(n):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        if _HEAT:
            _HEAT()
        e0.record(stream); call(); e1.record(stream)
        e1.synchronize()
        ts.append(e0.elapsed_time(e1))
    return statistics.median(ts), min(ts)


def time_rotating(calls, n_launches, reps=5):
    """Small operations (VERDICT r1 #2d): n_launches launches, rotating over len(calls) buffer sets whose total
    exceeds 2 x L2 (so no launch finds its data in L2), captured once into a CUDA graph and replayed between ONE pair
    of events: the time per launch is total / n_launches, free of the ~1 us event quantum and of the host's launch
    rate.  calls[i](stream_handle) enqueues the operation on buffer set i.  Returns (median ms, best ms) per launch."""
    import torch
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        for c in calls:                                         # warm-up: every set once (also loads the kernels)
            c(side.cuda_stream)
    side.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=side):
        s = torch.cuda.current_stream().cuda_stream
        for i in range(n_launches):
            calls[i % len(calls)](s)
    torch.cuda.synchronize()
    g.replay()
    torch.cuda.synchronize()
    ts = []
    st = torch.cuda.current_stream()
    for _ in range(reps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(st); g.replay(); e1.record(st)
        e1.synchronize()
        ts.append(e0.elapsed_time(e1) / n_launches)
    del g
    return statistics.median(ts), min(ts)


def n_sets_for(touched_bytes):
    return int(max(2, min(256, math.ceil(2.05 * L2_BYTES / max(1, touched_bytes)))))


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
    flags = {"auto": rs.RS_PATH_AUTO, "lsu": rs.RS_PATH_LSU, "bulk": rs.RS_PATH_BULK, "shift": rs.RS_PATH_BULK_SHIFT, "tmap": rs.RS_PATH_TMAP}[args.path]
    tune = parse_tune(args.tune)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    plan = harness.make_plan(w, flags, tune)               # rows a1..a5, once, outside the timed region
    plan_ms_cold = (time.perf_counter() - t0) * 1e3         # first plan of the process: CUDA module load included
    ts = []
    for _ in range(7):                                      # steady state: what a benchmark that re-plans would pay
        t0 = time.perf_counter()
        q = harness.make_plan(w, flags, tune)
        ts.append((time.perf_counter() - t0) * 1e3)
        q.close()
    plan_ms = statistics.median(ts)
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
    pname = {rs.RS_PATH_LSU: "rs_copy_lsu", rs.RS_PATH_BULK: "rs_copy_bulk", rs.RS_PATH_BULK_SHIFT: "rs_copy_bulk_shift", rs.RS_PATH_TMAP: "rs_copy_tmap"}
    kernels = {n: {"kernel": pname[o.path], "ms": k_ms[j], "best_ms": k_best[j], "bytes": op_bytes[j],
                   "GB/s": op_bytes[j] / (k_ms[j] * 1e-3) / 1e9, "grid": o.grid, "block": o.block,
                   "smem": o.smem_bytes, "tiles": o.n_tiles, "tile_bytes": o.tile_bytes, "table_bytes": o.table_bytes}
               for j, (n, o) in enumerate(zip(names, ops))}
    achieved = kernels["reshard_execute"]["GB/s"]
    traffic, traffic_src = ncu_traffic(w.name)
    line = {"metric": METRIC, "value": value, "unit": "GB/s", "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "u8", "data": "synthetic", "config": _config(w), "executor": kernels["reshard_execute"]["kernel"],
            "clocks": clocks, "gpu_launches": launches, "plan_ms": plan_ms, "plan_ms_cold": plan_ms_cold,
            "plan_table_bytes": sum(k["table_bytes"] for k in kernels.values()),
            "pct_of_nominal_8TBs": 100.0 * achieved / NOMINAL_HBM_GBS,
            "roofline": {"bound": "hbm", "kernel": "reshard_execute (%s)" % kernels["reshard_execute"]["kernel"],
                         "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "peak_source": peak_src, "algorithmic_bytes": op_bytes[0],
                         "traffic": traffic, "traffic_source": traffic_src},
            "kernels": kernels}
    if tune:
        line["tuning"] = tune
    if flush is not None:
        line["config"]["l2"] = "L2 flushed between steps (512 MiB fill); working set is L2-sized: effective GB/s"
    if e2e is not None:
        line["e2e"] = e2e
    if world == 1 and not args.no_cpu_baseline:
        r = oracle_sample(w, args.cpu_seconds, one_core=True)
        line["cpu_baseline"] = {k: r[k] for k in ("value", "unit", "cores", "kind", "sample", "value_1core", "numpy_slicing_1core")}
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
    sets = {"configs": cfg, "pairs": pairs, "table2": t2, "fig5": fig5, "all": cfg + pairs + t2}
    out = []
    for item in what.split(","):
        out += sets.get(item, [item])
    return out


def _release(torch):
    """give freed buffers back to the driver and let it finish with them: for some ms after a large cudaFree the device
    is busy with the freed pages (the first ~20 launches after a 36 GiB free ran at 5.0 TB/s instead of 6.5, the same
    launches after a 2 s wait at 6.5: profiles/r02_pacing.md part 5), which would be charged to the NEXT workload of a sweep"""
    torch.cuda.empty_cache()
    time.sleep(1.0)


def _buffers(torch, dev, n, nbytes, gen):
    """n device buffers of nbytes each (256-byte aligned slices of ONE allocation), seeded bytes"""
    pitch = (nbytes + 255) // 256 * 256
    flat = torch.empty(max(1, n * pitch), dtype=torch.uint8, device=dev)
    flat[: min(flat.numel(), 1 << 26)].random_(0, 256, generator=gen)
    return flat, [flat.data_ptr() + i * pitch for i in range(n)]


def run_sweep(args):
    """Per workload: plan, then each of execute / pack / unpack timed alone with CUDA events on the launching stream.
    Operations moving >= 1 GiB: 3 warm-up + --steps launches, each between its own events (median).  Smaller ones:
    time_rotating -- >= 50 launches per event pair over buffer sets totalling > 2 x L2, replayed from a CUDA graph.
    Buffer contents are irrelevant to a copy: shards are seeded bytes."""
    import torch
    from paper_2211_05322_b200 import harness, inputs
    from paper_2211_05322_b200 import reshard as rs
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    if args.hot:
        global _HEAT
        _HEAT = make_heater(torch, dev)
    stream = torch.cuda.current_stream()
    sh = stream.cuda_stream
    peak, _ = peak_hbm()
    flags = {"auto": rs.RS_PATH_AUTO, "lsu": rs.RS_PATH_LSU, "bulk": rs.RS_PATH_BULK, "shift": rs.RS_PATH_BULK_SHIFT, "tmap": rs.RS_PATH_TMAP}[args.path]
    tune = parse_tune(args.tune)
    K = max(3, min(args.steps, 30))
    want_ops = args.ops.split(",")
    rows = []
    for name in sweep_names(args.sweep):
        w = inputs.get_workload(name)
        opts = {}
        if tune:
            opts["tuning"] = tune
        if args.strategies:                                 # a mesh row is a host: local all-gather per row
            opts["dst_devices_per_host"] = w.dst_mesh[-1]
        plan = rs.Plan(w.shape, inputs.elem_bytes(w.dtype), w.src_mesh, w.src_spec, w.dst_mesh, w.dst_spec,
                       flags | (rs.RS_WITH_STRATEGIES if args.strategies else 0), opts or None)
        info = plan.info
        g = torch.Generator(device=dev); g.manual_seed(w.seed % (1 << 31))
        x_bytes = info.unique_read_bytes + info.write_bytes
        small = x_bytes < (1 << 30) and not args.plain
        n_sets = n_sets_for(x_bytes) if small else 1
        keep, sets = [], []
        for _ in range(n_sets):
            fs, sp = _buffers(torch, dev, info.n_src, info.src_shard_bytes, g)
            fd, dp = _buffers(torch, dev, info.n_dst, info.dst_shard_bytes, g)
            fa, ap = _buffers(torch, dev, 1, info.arena_bytes, g)
            keep += [fs, fd, fa]
            sets.append((sp, dp, ap[0]))
        calls = [("execute", rs.RS_OP_EXECUTE, lambda s, st: plan.execute(s[0], s[1], st)),
                 ("pack", rs.RS_OP_PACK, lambda s, st: plan.pack(s[0], s[2], st)),
                 ("unpack", rs.RS_OP_UNPACK, lambda s, st: plan.unpack(s[2], s[1], st))]
        calls = [c for c in calls if c[0] in want_ops]
        if args.strategies:      # same result by the paper's other strategies; GB/s counts the USEFUL bytes (1 + r_B) like execute
            calls = [calls[0],
                     ("sendrecv", rs.RS_OP_EXECUTE, lambda s, st: plan.execute_strategy(rs.RS_STRATEGY_SENDRECV, s[0], s[1], st)),
                     ("allgather", rs.RS_OP_EXECUTE, lambda s, st: plan.execute_strategy(rs.RS_STRATEGY_ALLGATHER, s[0], s[1], st)),
                     ("allgather_local", rs.RS_OP_EXECUTE, lambda s, st: plan.execute_strategy(rs.RS_STRATEGY_ALLGATHER_LOCAL, s[0], s[1], st))]
        r_B = info.write_bytes // max(1, info.unique_read_bytes)
        row = {"workload": name, "shape": list(w.shape), "src": "%s %s" % ("x".join(map(str, w.src_mesh)), w.src_spec),
               "dst": "%s %s" % ("x".join(map(str, w.dst_mesh)), w.dst_spec), "n_slices": info.n_slices,
               "tensor_bytes": info.tensor_bytes, "r_B": r_B,
               "protocol": ("CUDA graph of %d launches over %d buffer sets (> 2 x L2) between one event pair" % (max(50, 2 * n_sets), n_sets))
                           if small else "each launch between its own events, one buffer set (operation >> L2)"}
        if tune:
            row["tuning"] = tune
        for opname, op, call in calls:
            o = plan.op_info(op)
            nbytes = o.read_bytes + o.write_bytes
            if small:
                med, best = time_rotating([(lambda st, s=s, call=call: call(s, st)) for s in sets], max(50, 2 * n_sets))
            else:
                med, best = time_each(lambda call=call: call(sets[0], sh), stream, K)
            t0 = time.perf_counter()                          # host cost of one call (marshalling + launch, no synchronisation)
            for _ in range(100):
                call(sets[0], sh)
            host_us = (time.perf_counter() - t0) / 100 * 1e6
            torch.cuda.synchronize()
            row[opname] = {"host_us_per_call": host_us, "kernel": {rs.RS_PATH_BULK: "rs_copy_bulk", rs.RS_PATH_BULK_SHIFT: "rs_copy_bulk_shift", rs.RS_PATH_TMAP: "rs_copy_tmap"}.get(o.path, "rs_copy_lsu"), "bytes": nbytes,
                           "ms": med, "best_ms": best, "GB/s": nbytes / med / 1e6, "frac_of_copy_peak": nbytes / med / 1e6 / peak,
                           "tiles": o.n_tiles, "tile_bytes": o.tile_bytes, "grid": o.grid, "block": o.block, "table_bytes": o.table_bytes}
        roof = roof_1k(r_B)
        if roof and "execute" in row:
            row["execute"]["frac_of_1k_roof"] = row["execute"]["GB/s"] / roof
            row["roof_1k_GB/s"] = roof
        plan.close()
        del keep, sets
        _release(torch)
        # on-box ceiling: torch copy_ moving the same byte volume as execute (capped at 2 x 4 GiB), same protocol
        if not args.plain:
            half = min(x_bytes // 2, 4 << 30)
            pairs = [(torch.empty(half, dtype=torch.uint8, device=dev), torch.empty(half, dtype=torch.uint8, device=dev)) for _ in range(n_sets)]
            if small:
                med, _b = time_rotating([(lambda st, a=a, b=b: b.copy_(a)) for a, b in pairs], max(50, 2 * n_sets))
            else:
                med, _b = time_each(lambda: pairs[0][1].copy_(pairs[0][0]), stream, K)
            row["torch_copy_same_volume_GB/s"] = 2 * half / med / 1e6
            del pairs
            _release(torch)
        rows.append(row)
        print(json.dumps(row), flush=True)
    if args.md and args.strategies:
        with open(args.md, "w") as f:
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
    if args.md:
        with open(args.md, "w") as f:
            f.write("| workload | tensor | src -> dst | slices | read + write (execute) | execute us | execute GB/s (frac of %.0f) | frac of the 1 : k roof | pack GB/s | unpack GB/s | torch copy_ same volume GB/s | kernel, grid x block | table bytes |\n" % peak)
            f.write("|---|---|---|---|---|---|---|---|---|---|---|---|---|\n")
            for r in rows:
                x = r["execute"]
                f.write("| %s | %s | %s -> %s | %d | %.0f + %.0f MiB | %.2f | %.0f (%.3f) | %s | %s | %s | %.0f | %s, %d x %d | %d |\n" % (
                    r["workload"], r["shape"], r["src"], r["dst"], r["n_slices"], r["tensor_bytes"] / 2**20,
                    (x["bytes"] - r["tensor_bytes"]) / 2**20, x["ms"] * 1e3, x["GB/s"], x["frac_of_copy_peak"],
                    ("%.3f" % x["frac_of_1k_roof"]) if "frac_of_1k_roof" in x else "-",
                    ("%.0f" % r["pack"]["GB/s"]) if "pack" in r else "-", ("%.0f" % r["unpack"]["GB/s"]) if "unpack" in r else "-",
                    r.get("torch_copy_same_volume_GB/s", 0.0), x["kernel"], x["grid"], x["block"], x["table_bytes"]))
    return 0


# ------------------------------------------------------------------ the roof of a 1 : k stream

def run_roof(args):
    """What can this GPU sustain for 1 byte read + k bytes written, with NO layout in the way?  One contiguous
    source buffer, k contiguous destination buffers (a 1-D tensor, fully replicated on a k-device mesh: one unit
    task, one run), 1 GiB read per launch.  Swept: executor (TMA ring / registers), CTAs, warps per CTA, tile bytes.
    Beside it: torch copy_ (1 : 1), torch zero_ (pure write), torch sum (pure read), and the rate model
    t = read / R + write / W (one data bus per HBM channel: reads and writes do not overlap on it)."""
    import torch
    from paper_2211_05322_b200 import reshard as rs
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    stream = torch.cuda.current_stream()
    sh = stream.cuda_stream
    sms = torch.cuda.get_device_properties(dev).multi_processor_count
    K = max(5, min(args.steps, 15))
    n = 1 << 30
    src = torch.empty(n, dtype=torch.uint8, device=dev); src.random_(0, 256)
    dsts = [torch.empty(n, dtype=torch.uint8, device=dev) for _ in range(8)]
    rows = []
    # references
    med, best = time_each(lambda: dsts[0].copy_(src), stream, K)
    copy_gbs = 2 * n / med / 1e6
    med_w, _ = time_each(lambda: dsts[0].zero_(), stream, K)
    W = n / med_w / 1e6
    f32 = src.view(torch.float32)
    med_r, _ = time_each(lambda: f32.sum(), stream, K)
    R = n / med_r / 1e6
    refs = {"torch_copy_1to1_GB/s": copy_gbs, "torch_zero_pure_write_GB/s": W, "torch_sum_pure_read_GB/s": R}
    print(json.dumps({"references": refs}), flush=True)
    best_of = {}
    for k in (1, 2, 4, 8):
        shapes = []
        for ctas in sorted({sms * f // 148 for f in (64, 80, 96, 104, 112, 120, 128, 136, 148)}):
            for warps in (2, 4):
                for tile in (4096, 8192, 12288, 16384):
                    shapes.append(("bulk", dict(bulk_ctas=ctas, bulk_ctas_mcast=ctas, bulk_warps=warps, bulk_tile_bytes=tile)))
        for cps in (1, 2, 4):
            for tile in (8192, 16384, 32768):
                shapes.append(("lsu", dict(lsu_ctas_per_sm=cps, lsu_tile_bytes=tile)))
        shapes.append(("auto", {}))
        for path, tune in shapes:
            flags = {"bulk": rs.RS_PATH_BULK, "lsu": rs.RS_PATH_LSU, "auto": rs.RS_PATH_AUTO}[path]
            p = rs.Plan((n // 16,), 16, (1,), "R", (k,), "R", flags, dict(tuning=tune) if tune else None)
            o = p.op_info(rs.RS_OP_EXECUTE)
            sp, dp = [src.data_ptr()], [d.data_ptr() for d in dsts[:k]]
            med, bst = time_each(lambda: p.execute(sp, dp, sh), stream, K)
            nbytes = o.read_bytes + o.write_bytes
            row = {"k": k, "path": path, "tuning": tune, "grid": o.grid, "block": o.block, "tile_bytes": o.tile_bytes, "smem": o.smem_bytes,
                   "ms": med, "best_ms": bst, "GB/s": nbytes / med / 1e6}
            rows.append(row)
            print(json.dumps(row), flush=True)
            if path != "auto" and (k not in best_of or row["GB/s"] > best_of[k]["GB/s"]):
                best_of[k] = row
            p.close()
        med, _ = time_each(lambda: [d.copy_(src) for d in dsts[:k]], stream, K)          # k separate copies: k reads + k writes
        best_of[k]["k_torch_copies_useful_GB/s"] = (1 + k) * n / med / 1e6
        best_of[k]["model_GB/s"] = (1 + k) / (1.0 / R + k / W)
        best_of[k]["auto_GB/s"] = [r for r in rows if r["k"] == k and r["path"] == "auto"][0]["GB/s"]
    print(json.dumps({"best": best_of, "references": refs}), flush=True)
    if args.csv:
        with open(args.csv, "w") as f:
            f.write("k,best_gbs,path,grid,block,tile_bytes,auto_gbs,model_gbs,torch_copy_gbs,pure_write_gbs,pure_read_gbs,commit\n")
            for k, r in sorted(best_of.items()):
                f.write("%d,%.1f,%s,%d,%d,%d,%.1f,%.1f,%.1f,%.1f,%.1f,%s\n" % (k, r["GB/s"], r["path"], r["grid"], r["block"], r["tile_bytes"],
                                                                             r["auto_GB/s"], r["model_GB/s"], copy_gbs, W, R, git_commit()))
    if args.md:
        with open(args.md, "w") as f:
            f.write("References on this GPU (1 GiB buffers, median of %d, CUDA events): torch copy_ %.0f GB/s (read + write), torch zero_ %.0f GB/s "
                    "(pure write), torch sum %.0f GB/s (pure read).\n\n" % (K, copy_gbs, W, R))
            f.write("| k (1 read + k writes) | best GB/s | best shape | library default (AUTO) GB/s | AUTO / best | model (1+k)/(1/R + k/W) | k torch copy_ (useful bytes) |\n|---|---|---|---|---|---|---|\n")
            for k, r in sorted(best_of.items()):
                f.write("| %d | %.0f | %s, %d CTAs x %d threads, %d B tiles | %.0f | %.3f | %.0f | %.0f |\n" % (
                    k, r["GB/s"], r["path"], r["grid"], r["block"], r["tile_bytes"], r["auto_GB/s"], r["auto_GB/s"] / r["GB/s"], r["model_GB/s"],
                    r["k_torch_copies_useful_GB/s"]))
            f.write("\nEvery shape tried (GB/s; rows: CTAs x warps, columns: tile bytes), TMA ring executor:\n")
            for k in (1, 2, 4, 8):
                f.write("\nk = %d\n\n| CTAs x warps | 4096 | 8192 | 12288 | 16384 |\n|---|---|---|---|---|\n" % k)
                cells = {}
                for r in rows:
                    if r["k"] == k and r["path"] == "bulk":
                        cells.setdefault((r["tuning"]["bulk_ctas"], r["tuning"]["bulk_warps"]), {})[r["tuning"]["bulk_tile_bytes"]] = r["GB/s"]
                for (c, wp), d in sorted(cells.items()):
                    f.write("| %d x %d | %s |\n" % (c, wp, " | ".join("%.0f" % d.get(t, 0) for t in (4096, 8192, 12288, 16384))))
                f.write("\nregisters (rs_copy_lsu): " + ", ".join("%d CTAs/SM x %d B: %.0f" % (r["tuning"]["lsu_ctas_per_sm"], r["tuning"]["lsu_tile_bytes"], r["GB/s"])
                                                                 for r in rows if r["k"] == k and r["path"] == "lsu") + "\n")
    return 0


def run_sharded(args):
    """--mode sharded: ONE resharding task over N GPUs (strong scaling).  Virtual device r lives on rank r mod N; every
    rank executes the unit tasks whose sender it holds, writing local and peer-mapped (CUDA IPC -> NVLink) destination
    shards; no data-path collective.  A step = one reshard_execute launch per rank; time = max over ranks of the device
    time of K steps.  Not measurable on the 1-GPU boxes of this run (world 1 degenerates to the normal plan)."""
    import torch
    from paper_2211_05322_b200 import inputs, multi, sharded
    from paper_2211_05322_b200 import reshard as rs
    rank, world, local = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world == 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1"); os.environ.setdefault("MASTER_PORT", "29511")
        os.environ.setdefault("RANK", "0"); os.environ.setdefault("WORLD_SIZE", "1")
    multi.init("nccl", dev)
    w = inputs.get_workload(args.workload)
    e = inputs.elem_bytes(w.dtype)
    n_src, n_dst = 1, 1
    for m in w.src_mesh: n_src *= m
    for m in w.dst_mesh: n_dst *= m
    so, dow = sharded.round_robin_owner(n_src, world), sharded.round_robin_owner(n_dst, world)
    x = sharded.ShardedReshard(w.shape, e, w.src_mesh, w.src_spec, w.dst_mesh, w.dst_spec, so, dow, 0, dict(tuning=parse_tune(args.tune)) if args.tune else None)
    info = x.plan.info
    src_local = {r: torch.empty(info.src_shard_bytes, dtype=torch.uint8, device=dev).random_(0, 256) for r in range(n_src) if so[r] == rank}
    dst_local = {q: torch.empty(info.dst_shard_bytes, dtype=torch.uint8, device=dev) for q in range(n_dst) if dow[q] == rank}
    x.bind(src_local, dst_local)
    stream = torch.cuda.current_stream()
    K, W = max(1, args.steps), max(3, args.warmup)
    for _ in range(W):
        x.execute(stream.cuda_stream)
    x.wait()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    n0 = rs.launch_count()
    e0.record(stream)
    for _ in range(K):
        x.execute(stream.cuda_stream)
    e1.record(stream)
    x.wait()
    ms = multi.max_over_ranks(e0.elapsed_time(e1) / K, dev)
    total = info.unique_read_bytes + info.write_bytes
    peer = sum(1 for q in x.writes if dow[q] != rank)
    if rank == 0:
        print(json.dumps({"metric": METRIC, "value": total / (ms * 1e-3) / 1e9, "unit": "GB/s", "n_gpus": world, "steps": K, "warmup": W,
                          "ms_per_step": ms, "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "u8", "data": "synthetic",
                          "mode": "sharded", "config": dict(_config(w), step="reshard_execute, one launch per rank", parallelism="virtual device r on rank r mod N; peer stores through CUDA IPC"),
                          "gpu_launches": rs.launch_count() - n0, "rank0_bytes_per_step": x.my_bytes(), "rank0_peer_destinations": peer}))
    x.close()
    multi.shutdown()
    return 0


def run_mix(args):
    """--mix a,b[,c]: reshard_execute of DIFFERENT workloads alternating in ONE stream (a stage boundary carries tensors of several layouts),
    between one pair of CUDA events, against each workload launched back to back on its own.  One JSON line."""
    import torch
    from paper_2211_05322_b200 import harness, inputs
    from paper_2211_05322_b200 import reshard as rs
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    st = torch.cuda.current_stream().cuda_stream
    opts = dict(tuning=parse_tune(args.tune)) if args.tune else None
    items = []
    for name in args.mix.split(","):
        w = inputs.get_workload(name)
        plan = rs.Plan(w.shape, inputs.elem_bytes(w.dtype), w.src_mesh, w.src_spec, w.dst_mesh, w.dst_spec,
                       {"auto": rs.RS_PATH_AUTO, "lsu": rs.RS_PATH_LSU, "bulk": rs.RS_PATH_BULK, "shift": rs.RS_PATH_BULK_SHIFT, "tmap": rs.RS_PATH_TMAP}[args.path], opts)
        info = plan.info
        src = [torch.empty(info.src_shard_bytes, dtype=torch.uint8, device=dev) for _ in range(info.n_src)]
        dst = [torch.empty(info.dst_shard_bytes, dtype=torch.uint8, device=dev) for _ in range(info.n_dst)]
        o = plan.op_info(rs.RS_OP_EXECUTE)
        items.append((name, plan, harness.ptrs(src), harness.ptrs(dst), o.read_bytes + o.write_bytes, (src, dst), o))

    def rate(seq, rounds):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        for _ in range(rounds):
            for it in seq:
                it[1].execute(it[2], it[3], st)
        e1.record()
        torch.cuda.synchronize()
        return sum(it[4] for it in seq) * rounds / (e0.elapsed_time(e1) * 1e-3) / 1e9

    rounds = max(3, args.steps // 10)
    for _ in range(2):
        rate(items, 2)
    out = {"mix": args.mix, "protocol": "%d rounds of the listed launches alternating in one stream, one pair of CUDA events" % rounds,
           "alternating_GB/s": statistics.median(rate(items, rounds) for _ in range(5)),
           "each_alone_GB/s": {it[0]: statistics.median(rate([it], rounds * len(items)) for _ in range(5)) for it in items},
           "shapes": {it[0]: "%s %d x %d, %d B shared" % ({rs.RS_PATH_BULK: "rs_copy_bulk", rs.RS_PATH_BULK_SHIFT: "rs_copy_bulk_shift", rs.RS_PATH_TMAP: "rs_copy_tmap"}.get(it[6].path, "rs_copy_lsu"), it[6].grid, it[6].block, it[6].smem_bytes) for it in items},
           "tune": args.tune}
    print(json.dumps(out))
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
    if args.md:
        with open(args.md, "w") as f:
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
    if args.md:
        with open(args.md, "w") as f:
            f.write("| workload | tensors | bytes moved | n launches: us (GB/s) | one grouped launch: us (GB/s) | speedup |\n|---|---|---|---|---|---|\n")
            for r in rows:
                f.write("| %s | %d | %.1f MiB | %.1f (%.0f) | %.1f (%.0f) | %.2f |\n" % (r["workload"], r["tensors"], r["bytes"] / 2**20,
                        r["separate_us"], r["separate_GBs"], r["grouped_us"], r["grouped_GBs"], r["speedup"]))
    return 0


# ------------------------------------------------------------------ evidence tooling (runs on the CPU box)

_UNIT = {"Gbyte": 1e9, "Mbyte": 1e6, "Kbyte": 1e3, "byte": 1.0, "s": 1e6, "ms": 1e3, "us": 1.0, "ns": 1e-3}


def run_ncu_summary(args):
    """`ncu -i <report> --page raw --csv` of one-launch reports -> CSV rows on stdout (header first).  Append them to
    profiles/ncu_traffic.csv; bench.py reads roofline.traffic from there."""
    cols = ["workload", "op", "kernel", "grid", "block", "duration_us", "dram_read_bytes", "dram_write_bytes", "dram_throughput_pct",
            "dram_active_min_pct", "dram_active_max_pct", "warp_inst_executed", "commit", "report"]
    out_csv = csv.writer(sys.stdout, lineterminator="\n")
    out_csv.writerow(cols)
    for item in args.ncu_summary:
        key, path = item.rsplit("=", 1)
        workload, op = key.rsplit(":", 1) if ":" in key else (key, "execute")     # (x:... workload names hold colons)
        out = subprocess.run(["ncu", "-i", path, "--page", "raw", "--csv"], capture_output=True, text=True, check=True).stdout
        rows = list(csv.reader(io.StringIO(out)))
        hdr, units = rows[0], rows[1]
        launches = [r for r in rows[2:] if "rs_copy" in r[hdr.index("Kernel Name")]]
        if not launches:
            raise SystemExit("%s holds no rs_copy_* launch" % path)
        v = launches[0]

        def get(name, scale=True):
            if name not in hdr:
                return ""
            i = hdr.index(name)
            x = float(v[i].replace(",", ""))
            return x * _UNIT.get(units[i], 1.0) if scale else x
        dims = lambda s: int(re.findall(r"\d+", s)[0])
        out_csv.writerow([
            workload, op, v[hdr.index("Kernel Name")].split("(")[0], dims(v[hdr.index("Grid Size")]), dims(v[hdr.index("Block Size")]),
            "%.3f" % get("gpu__time_duration.sum"), int(get("dram__bytes_read.sum")), int(get("dram__bytes_write.sum")),
            "%.2f" % get("gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed", False),
            "%.2f" % get("dram__cycles_active.min.pct_of_peak_sustained_elapsed", False),      # least / most busy DRAM channel
            "%.2f" % get("dram__cycles_active.max.pct_of_peak_sustained_elapsed", False),
            int(get("smsp__inst_executed.sum", False) or 0), git_commit(), os.path.basename(path)])
    return 0


def run_sass(_args):
    """cuobjdump -sass libreshard.so -> per kernel: instruction count and the opcodes that prove (or disprove) the
    Blackwell copy engines: UBLKCP (cp.async.bulk), UTMALDG / UTMASTG (tensor-map TMA), SYNCS (mbarrier), PREEXIT / ACQBULK
    (griddepcontrol.launch_dependents / .wait: programmatic dependent launch), NANOSLEEP (rate matching), LDG / STG."""
    from paper_2211_05322_b200 import reshard as rs
    rs._lib()
    out = subprocess.run(["cuobjdump", "-sass", rs.LIB_PATH], capture_output=True, text=True, check=True).stdout
    kernels, cur = {}, None
    for line in out.splitlines():
        m = re.match(r"\s*Function : (\S+)", line)
        if m:
            cur = subprocess.run(["c++filt", m.group(1)], capture_output=True, text=True).stdout.strip().split("(")[0]
            kernels[cur] = {}
            continue
        m = re.match(r"\s*/\*[0-9a-f]{4}\*/\s+(?:@!?U?P\d+\s+)?([A-Z][A-Z0-9_.]*)", line)
        if m and cur:
            kernels[cur][m.group(1)] = kernels[cur].get(m.group(1), 0) + 1
    watch = ["UBLKCP", "UTMALDG", "UTMASTG", "SYNCS", "PREEXIT", "ACQBULK", "NANOSLEEP", "LDG", "STG", "LDS", "STS", "SHF", "IMAD", "BAR", "LDC", "UTC", "HMMA"]
    print("Command: `python bench.py --sass` (= `cuobjdump -sass paper_2211_05322_b200/libreshard.so`, opcode prefixes counted per kernel), commit %s.\n" % git_commit())
    print("| kernel | instructions | " + " | ".join(watch) + " |")
    print("|---|---|" + "---|" * len(watch))
    for name, ops in sorted(kernels.items()):
        print("| `%s` | %d | %s |" % (name, sum(ops.values()), " | ".join(str(sum(c for o, c in ops.items() if o.startswith(wd))) for wd in watch)))
    print("\nFull opcode lists (opcode: count):\n")
    for name, ops in sorted(kernels.items()):
        print("- `%s`: %s" % (name, ", ".join("%s %d" % (o, c) for o, c in sorted(ops.items(), key=lambda x: -x[1]) if c >= 1 and (
            any(o.startswith(wd) for wd in watch) or c >= 8))))
    return 0


def run_report(args):
    """Host-only tables of DESIGN.md S10 (no GPU): simulated makespans of Table 2 under every S3.2 algorithm (the shape
    of Fig. 8) and iteration latency of 1F1B vs eager-1F1B (the shape of Fig. 9)."""
    from paper_2211_05322_b200 import inputs
    from paper_2211_05322_b200 import reshard as rs
    if args.report == "schedule":
        algs = [("naive", rs.RS_SCHED_NAIVE), ("load balance only", rs.RS_SCHED_LOAD_BALANCE), ("DFS (200k nodes)", rs.RS_SCHED_DFS),
                ("randomized greedy", rs.RS_SCHED_GREEDY), ("ensemble", rs.RS_SCHED_ENSEMBLE)]
        print("| case | specs | unit tasks | " + " | ".join(n for n, _ in algs) + " | busiest host (ensemble senders) |")
        print("|---|---|---|" + "---|" * (len(algs) + 1))
        for c in (1, 2, 3, 4, 5, 7, 8, 9):
            w = inputs.table2_workload(c)
            res = {}
            for name, alg in algs:
                p = rs.Plan(w.shape, 2, w.src_mesh, w.src_spec, w.dst_mesh, w.dst_spec, rs.RS_HOST_ONLY,
                            dict(schedule=alg, src_devices_per_host=w.src_mesh[-1], dst_devices_per_host=w.dst_mesh[-1]))
                s = p.schedule()["info"]
                res[name], n_tasks, bound = s.makespan, s.n_tasks, s.busiest_host_bytes
                p.close()
            print("| %d | %s -> %s | %d | " % (c, w.src_spec, w.dst_spec, n_tasks) + " | ".join("%.2f" % (res[n] / bound) for n, _ in algs) + " | %d MiB |" % (bound >> 20))
        return 0
    S, M, f, b = 4, 32, 100, 200
    keys = ["comm/fwd %", "no overlap, 1F1B", "overlap, 1F1B", "overlap, eager-1F1B", "+ weight delaying (least delay)", "delay",
            "peak activations, stage 1 (1F1B / eager)"]
    print("| " + " | ".join(keys) + " |")
    print("|" + "---|" * len(keys))
    for pct in (0, 10, 25, 50, 100):
        c = f * pct // 100
        ideal = (M + S - 1) * (f + b)
        e = rs.pipeline_simulate(rs.RS_PIPE_EAGER_1F1B, S, M, f, b, c, c)
        d = max(0, rs.pipeline_least_delay(rs.RS_PIPE_EAGER_1F1B, S, 1, M, f, b, b // 2, c))
        vals = [pct, rs.pipeline_simulate(rs.RS_PIPE_1F1B, S, M, f, b, c, c, overlap=False)["makespan"] / ideal,
                rs.pipeline_simulate(rs.RS_PIPE_1F1B, S, M, f, b, c, c)["makespan"] / ideal, e["makespan"] / ideal,
                rs.pipeline_simulate(rs.RS_PIPE_EAGER_1F1B, S, M, f, b, c, c, bwd_act=b // 2, bw_delay=d)["makespan"] / ideal, d,
                "%d / %d" % (rs.pipeline_simulate(rs.RS_PIPE_1F1B, S, M, f, b, c, c)["peak"][0], e["peak"][0])]
        print("| " + " | ".join(("%.3f" % v) if isinstance(v, float) else str(v) for v in vals) + " |")
    return 0


def main():
    args = parse_args()
    if args.ncu_summary:
        return run_ncu_summary(args)
    if args.sass:
        return run_sass(args)
    if args.report:
        return run_report(args)
    if args.roof:
        return run_roof(args)
    if args.group:
        return run_group(args)
    if args.mix:
        return run_mix(args)
    if args.overlap:
        return run_overlap(args)
    if args.sweep:
        return run_sweep(args)
    if args.impl == "reference":
        return run_reference(args)
    if args.mode == "sharded":
        return run_sharded(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
