"""Pipeline-schedule oracle: 1F1B and eager-1F1B op orders and their timelines.

TEST INFRASTRUCTURE, NOT THE PRODUCT.  Pure Python, written from PAPER.md alone; shares no code
with paper_2211_05322_b200/ and neither imports the other.

What it follows (PAPER.md:<line>):
  1F1B warm-up          PAPER.md:209  "stage i runs forward computations for the first (#stages - i + 1)
                                      batches ... and enters the steady one-forward-one-backward phase
                                      after it is able to run the first backward computation"
  eager-1F1B warm-up    PAPER.md:209  "Stage i runs (2 x (#stages - i) + 1) forward computations and then
                                      enters the steady phase"
  data dependency       PAPER.md:205  compute of stage i, communication i -> i+1, compute of stage i+1 of
                                      the same micro-batch follow one another
  equal without comm    PAPER.md:211  "When there is no communication cost, the latencies of these two
                                      schedules are the same"
  memory                PAPER.md:213  eager-1F1B stores activations of more micro-batches: at most
                                      #stages x size_activation more per GPU
  backward weight delay PAPER.md:215-217 backward = gradients of activations, then gradients of weights;
                                      the cross-mesh communication only needs the first; the second is
                                      delayed "the least to cover all communications"
  no overlap baseline   PAPER.md:310  "Broadcast" = resharding without overlapping

Readings: R28 stages are numbered 1..S as in the paper, micro-batches 0..M-1; warm-up counts
are capped at M.  R29 a stage executes its op list strictly in order (no re-ordering at run time); an op
starts when the stage is free and its input has arrived.  R30 every stage boundary has one link per
direction; a transfer occupies its link for the communication time, transfers of one link run in the
order they were issued; with overlap the sender's compute continues, without overlap the
sender stage is busy until the transfer has finished ("cannot be overlapped").  R31 the
steady phase alternates one backward, one forward ("one-forward-one-backward ... after it is
able to run the first backward"), and the remaining backwards follow when the forwards run out.
R32 backward weight delaying: B = BA (activation gradients, duration b_act) then BW (weight gradients,
b - b_act); the backward transfer leaves after BA; BW is moved `delay` ops later in the stage's list
(delay 0: directly after BA, already overlapping the transfer); the cost model picks the least delay
whose intervening compute covers the communication time.

Pins: tests/test_pipeline_oracle_pins.py.
"""


def warmup_count(kind, n_stages, stage, n_micro):
    """number of forwards stage `stage` (1-based) runs before its first backward.  PAPER.md:209."""
    if kind == "1f1b":
        w = n_stages - stage + 1
    elif kind == "eager":
        w = 2 * (n_stages - stage) + 1
    else:
        raise ValueError(kind)
    return min(w, n_micro)                                   # R28


def stage_ops(kind, n_stages, stage, n_micro, split_backward=False, delay=0):
    """op list of one stage: tuples (op, micro_batch), op in 'F', 'B' (or 'BA', 'BW' when the backward is
    split).  Warm-up forwards, then one backward / one forward alternately, then the remaining backwards
    (R31).  With split_backward every 'B' becomes 'BA' and a 'BW' placed `delay` ops later (R32)."""
    w = warmup_count(kind, n_stages, stage, n_micro)
    ops = [("F", m) for m in range(w)]
    nf, nb = w, 0
    while nb < n_micro:
        ops.append(("B", nb))
        nb += 1
        if nf < n_micro:
            ops.append(("F", nf))
            nf += 1
    if not split_backward:
        return ops
    out, pending = [], []                                    # pending: [ops still to pass, micro_batch]
    for op, m in ops:
        for p in pending:
            p[0] -= 1
        if op == "B":
            out.append(("BA", m))
            pending.append([delay, m])
        else:
            out.append((op, m))
        while pending and pending[0][0] <= 0:
            out.append(("BW", pending.pop(0)[1]))
    out.extend(("BW", m) for _d, m in pending)
    return out


def peak_activations(ops):
    """most micro-batches whose forward has run and whose backward (activation gradients) has not."""
    live = peak = 0
    for op, _m in ops:
        if op == "F":
            live += 1
            peak = max(peak, live)
        elif op in ("B", "BA"):
            live -= 1
    return peak


def simulate(kind, n_stages, n_micro, f, b, c_fwd, c_bwd, overlap=True, b_act=None, delay=0):
    """Timeline of one training iteration.  f, b: forward / backward compute time of every stage (scalars or
    per-stage lists, stage 1 first); c_fwd / c_bwd: transfer time of one micro-batch across a stage boundary.
    b_act not None splits the backward (R32).  Returns dict(makespan, start, end, ops, peak, busy):
    start/end keyed by (stage, op, micro_batch); busy = per-stage compute time."""
    S, M = n_stages, n_micro
    fl = list(f) if isinstance(f, (list, tuple)) else [f] * S
    bl = list(b) if isinstance(b, (list, tuple)) else [b] * S
    split = b_act is not None
    bal = (list(b_act) if isinstance(b_act, (list, tuple)) else [b_act] * S) if split else None
    ops = {i: stage_ops(kind, S, i, M, split, delay) for i in range(1, S + 1)}
    dur = {}
    for i in range(1, S + 1):
        dur[(i, "F")] = fl[i - 1]
        dur[(i, "B")] = bl[i - 1]
        if split:
            dur[(i, "BA")] = bal[i - 1]
            dur[(i, "BW")] = bl[i - 1] - bal[i - 1]
    pos = {i: 0 for i in ops}                                 # next op of every stage
    free = {i: 0 for i in ops}                                # when the stage's compute is free
    link = {}                                                 # (boundary, direction) -> when the link is free
    arrive = {}                                               # (stage, 'F'|'B', m) -> when that op's input has arrived
    start, end = {}, {}
    grad = "BA" if split else "B"
    remaining = sum(len(v) for v in ops.values())
    while remaining:
        progressed = False
        for i in range(1, S + 1):
            while pos[i] < len(ops[i]):
                op, m = ops[i][pos[i]]
                if op == "F":
                    ready = 0 if i == 1 else arrive.get((i, "F", m))
                elif op == grad:
                    ready = end.get((i, "F", m)) if i == S else arrive.get((i, "B", m))
                    if ready is not None and end.get((i, "F", m)) is None:
                        ready = None
                else:                                         # BW: after its BA, no other input
                    ready = end.get((i, "BA", m))
                if ready is None:
                    break                                     # strictly in order (R29): wait for this op's input
                s = max(free[i], ready)
                e = s + dur[(i, op)]
                start[(i, op, m)], end[(i, op, m)] = s, e
                free[i] = e
                # the transfer this op feeds (R30)
                if op == "F" and i < S:
                    key, t = (i, "fwd"), c_fwd
                    ts = max(e, link.get(key, 0))
                    link[key] = ts + t
                    arrive[(i + 1, "F", m)] = ts + t
                    if not overlap:
                        free[i] = ts + t
                elif op == grad and i > 1:
                    key, t = (i - 1, "bwd"), c_bwd
                    ts = max(e, link.get(key, 0))
                    link[key] = ts + t
                    arrive[(i - 1, "B", m)] = ts + t
                    if not overlap:
                        free[i] = ts + t
                pos[i] += 1
                remaining -= 1
                progressed = True
        if not progressed:
            raise RuntimeError("schedule deadlocks: an op waits for an input that is never produced")
    busy = {i: sum(dur[(i, op)] for op, _m in ops[i]) for i in ops}
    return dict(makespan=max(end.values()), start=start, end=end, ops=ops, busy=busy,
                peak={i: peak_activations(ops[i]) for i in ops})


def least_delay(kind, n_stages, stage, n_micro, f, b, b_act, c_bwd):
    """PAPER.md:217 cost model: the least `delay` such that the compute a stage runs between BA(m) and the
    point where BW(m) is put back covers the backward transfer time; BW itself counts (delay 0 already
    overlaps b - b_act of it)."""
    for delay in range(0, 2 * n_micro + 1):
        ops = stage_ops(kind, n_stages, stage, n_micro, True, delay)
        # steady state: look at the first backward that is followed by a forward
        idx = [k for k, (op, _m) in enumerate(ops) if op == "BA"]
        if not idx:
            return 0
        k = idx[0]
        m = ops[k][1]
        covered = 0
        for op, mm in ops[k + 1:]:
            covered += {"F": f, "BA": b_act, "BW": b - b_act}[op]
            if op == "BW" and mm == m:
                break
        if covered >= c_bwd:
            return delay
    return 2 * n_micro
