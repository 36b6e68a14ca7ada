"""Schedule-side oracle: load balance AND order of the unit tasks (S3.2).

TEST INFRASTRUCTURE, NOT THE PRODUCT.  Pure Python (small inputs only), written from PAPER.md
alone; shares no code with paper_2211_05322_b200/ and neither imports the other.  It takes the
unit tasks of oracle/plan_oracle.py (dicts with size / senders / receivers) as input.

What it follows (PAPER.md:<line>):
  hosts               PAPER.md:149    "we perform load balancing and scheduling at host level":
                                      n_i = hosts holding a replica, m_i = hosts requiring the slice
  Eq. 1               PAPER.md:153    minimise max_i S_i + T_i
  Eq. 2               PAPER.md:155    n_i* in n_i
  Eq. 3               PAPER.md:157    tasks with the same sender host or a common receiver host do
                                      not overlap in time (garbled indices read as i, j: R14)
  per-host orders     PAPER.md:175    S_i = earliest time at which all preceding tasks have finished
                                      on the sender host and on every receiver host
  naive               PAPER.md:163    lowest-indexed sender, arbitrary (here: slice id) global order
  load balance only   PAPER.md:167-171, 318  Eq. 4 greedy; order = the order the greedy assigned in
  DFS with pruning    PAPER.md:173-179 search over sender choice and order, prune by the Eq. 4 bound
  randomized greedy   PAPER.md:181, 195 rounds of non-overlapping tasks covering the most hosts,
                                      each found by repeated random orderings
  ensemble            PAPER.md:318    run both, keep the better schedule

Readings: R7 T_i = slice bytes; R8 host = device id // devices_per_host (default 1:
every virtual device is its own host); R14 Eq. 3; R24 the randomized greedy keeps the Eq. 4
senders and draws its orderings from a counter-based generator (splitmix64 finaliser of
seed + counter; Fisher-Yates from the top); R25 the DFS explores (next task, sender host) pairs in
ascending (task id, host id) and stops after a node budget instead of a time budget.

Pins: tests/test_schedule_oracle_pins.py (hand-computed timelines of Table 2 cases 1, 2, 3, 8 as
the paper describes them at PAPER.md:282, 320; brute force over all orders x senders; the
independent pairwise Eq. 3 checker; Eq. 4 lower bound).
"""
import itertools

_M64 = (1 << 64) - 1


def mix64(x):
    """splitmix64 finaliser (same constants as the seeded input generator; restated, not imported)."""
    x &= _M64
    x ^= x >> 30
    x = (x * 0xBF58476D1CE4E5B9) & _M64
    x ^= x >> 27
    x = (x * 0x94D049BB133111EB) & _M64
    x ^= x >> 31
    return x


def shuffled(items, seed, counter):
    """Fisher-Yates from the top: for j = n-1 .. 1 swap a[j] with a[r_j mod (j+1)],
    r_j = mix64(seed + (counter << 20) + j)."""
    a = list(items)
    for j in range(len(a) - 1, 0, -1):
        k = mix64(seed + (counter << 20) + j) % (j + 1)
        a[j], a[k] = a[k], a[j]
    return a


def host_of(device, devices_per_host):
    return device // devices_per_host


def host_tasks(tasks, elem_bytes=1, src_devices_per_host=1, dst_devices_per_host=1):
    """unit tasks at host level: list of dict(T, n (sorted candidate sender hosts), m (sorted
    receiver hosts)).  PAPER.md:149."""
    out = []
    for t in tasks:
        n = sorted({host_of(d, src_devices_per_host) for d in t["senders"]})
        m = sorted({host_of(d, dst_devices_per_host) for d in t["receivers"]})
        out.append(dict(T=t["size"] * elem_bytes, n=n, m=m))
    return out


def start_times(ht, senders, order):
    """walk the tasks in `order`; S_i = max over the sender host and the receiver
    hosts of the time their previous task finished.  Returns (S list indexed by task, makespan)."""
    free_s, free_r = {}, {}
    S = [None] * len(ht)
    end = 0
    for i in order:
        assert senders[i] in ht[i]["n"], "Eq. 2 violated"
        s = free_s.get(senders[i], 0)
        for h in ht[i]["m"]:
            s = max(s, free_r.get(h, 0))
        S[i] = s
        f = s + ht[i]["T"]
        free_s[senders[i]] = f
        for h in ht[i]["m"]:
            free_r[h] = f
        end = max(end, f)
    assert all(x is not None for x in S), "order must list every task once"
    return S, end


def check_eq3(ht, senders, S):
    """independent statement of Eq. 3: every pair of tasks with the same sender host or a common
    receiver host occupies disjoint open intervals."""
    for i, j in itertools.combinations(range(len(ht)), 2):
        if senders[i] == senders[j] or set(ht[i]["m"]) & set(ht[j]["m"]):
            a0, a1, b0, b1 = S[i], S[i] + ht[i]["T"], S[j], S[j] + ht[j]["T"]
            if a0 < b1 and b0 < a1:
                return False
    return True


def eq4_bound(ht, senders=None):
    """lower bound on Eq. 1 'measured by the sum of task durations on a single device':
    receiver hosts' totals are fixed; sender hosts' totals need the assignment (else the best
    case: every replica group spread perfectly)."""
    load = {}
    for i, t in enumerate(ht):
        for h in t["m"]:
            load[("r", h)] = load.get(("r", h), 0) + t["T"]
        if senders is not None:
            load[("s", senders[i])] = load.get(("s", senders[i]), 0) + t["T"]
    lb = max(load.values())
    lb = max(lb, max(t["T"] for t in ht))
    return lb


# ------------------------------------------------------------------ the four algorithms

def naive(ht):
    """lowest-indexed sender, global order = slice id."""
    senders = [t["n"][0] for t in ht]
    order = list(range(len(ht)))
    return senders, order


def load_balance_only(ht):
    """PAPER.md:171 + 318: Eq. 4 greedy (descending T_i, lightest candidate host, ties lowest id);
    the order is the one the greedy walked the tasks in."""
    order = sorted(range(len(ht)), key=lambda i: (-ht[i]["T"], i))
    load, senders = {}, [None] * len(ht)
    for i in order:
        s = min(ht[i]["n"], key=lambda h: (load.get(h, 0), h))
        senders[i] = s
        load[s] = load.get(s, 0) + ht[i]["T"]
    return senders, order


def bruteforce(ht, limit=3_000_000):
    """optimum of Eq. 1-3 by enumerating every sender assignment and every global order."""
    n = len(ht)
    count = 1
    for t in ht:
        count *= len(t["n"])
    for k in range(2, n + 1):
        count *= k
    if count > limit:
        raise ValueError("too many schedules to enumerate")
    best = None
    for senders in itertools.product(*[t["n"] for t in ht]):
        for order in itertools.permutations(range(n)):
            _S, end = start_times(ht, senders, order)
            if best is None or end < best[0]:
                best = (end, list(senders), list(order))
    return best


def dfs_with_pruning(ht, node_budget=200_000):
    """PAPER.md:173-179.  Incumbent = load_balance_only.  A node fixes the next task of the global
    order and its sender host; a branch is cut when max(partial makespan, Eq. 4 bound of the partial
    assignment) >= incumbent.  Returns (makespan, senders, order, finished)."""
    n = len(ht)
    senders0, order0 = load_balance_only(ht)
    _S, best_end = start_times(ht, senders0, order0)
    best = [best_end, list(senders0), list(order0)]
    recv_total = {}
    for t in ht:
        for h in t["m"]:
            recv_total[h] = recv_total.get(h, 0) + t["T"]
    floor = max(max(recv_total.values()), max(t["T"] for t in ht))
    nodes = [0]
    finished = [True]

    senders, order, used = [None] * n, [], [False] * n
    free_s, free_r, send_load = {}, {}, {}

    def rec(cur_end):
        if best[0] <= floor:
            return
        if nodes[0] >= node_budget:
            finished[0] = False
            return
        nodes[0] += 1
        if len(order) == n:
            if cur_end < best[0]:
                best[0], best[1], best[2] = cur_end, list(senders), list(order)
            return
        for i in range(n):
            if used[i]:
                continue
            for h in ht[i]["n"]:
                s = free_s.get(h, 0)
                for r in ht[i]["m"]:
                    s = max(s, free_r.get(r, 0))
                f = s + ht[i]["T"]
                new_load = send_load.get(h, 0) + ht[i]["T"]
                if max(cur_end, f, new_load, floor) >= best[0]:
                    continue
                saved = (free_s.get(h), [free_r.get(r) for r in ht[i]["m"]])
                free_s[h] = f
                for r in ht[i]["m"]:
                    free_r[r] = f
                send_load[h] = new_load
                used[i] = True; senders[i] = h; order.append(i)
                rec(max(cur_end, f))
                order.pop(); used[i] = False; senders[i] = None
                send_load[h] = new_load - ht[i]["T"]
                if saved[0] is None:
                    del free_s[h]
                else:
                    free_s[h] = saved[0]
                for r, v in zip(ht[i]["m"], saved[1]):
                    if v is None:
                        del free_r[r]
                    else:
                        free_r[r] = v

    rec(0)
    return best[0], best[1], best[2], finished[0]


def randomized_greedy(ht, seed=0, trials=32):
    """PAPER.md:181, 195.  Senders = Eq. 4 greedy.  Repeat: draw `trials` random orderings of the
    remaining tasks (ascending id, then shuffled); walking an ordering, select every task that
    shares no sender host and no receiver host with those already selected; keep the selection
    involving the most hosts (first such trial on ties); it becomes the next round.  The global
    order is the concatenation of the rounds (each in ascending id)."""
    senders, _o = load_balance_only(ht)
    remaining = list(range(len(ht)))
    rounds, counter = [], 0
    while remaining:
        best_sel, best_score = None, -1
        for _ in range(trials):
            perm = shuffled(remaining, seed, counter)
            counter += 1
            used, sel = set(), []
            for i in perm:
                H = {("s", senders[i])} | {("r", h) for h in ht[i]["m"]}
                if not (H & used):
                    sel.append(i)
                    used |= H
            if len(used) > best_score:
                best_sel, best_score = sel, len(used)
        rounds.append(sorted(best_sel))
        chosen = set(best_sel)
        remaining = [i for i in remaining if i not in chosen]
    order = [i for r in rounds for i in r]
    return senders, order, rounds


def ensemble(ht, seed=0, trials=32, node_budget=200_000):
    """'We run both algorithms and choose the better result'.  Ties keep the DFS."""
    end_d, s_d, o_d, _fin = dfs_with_pruning(ht, node_budget)
    s_g, o_g, _rounds = randomized_greedy(ht, seed, trials)
    _S, end_g = start_times(ht, s_g, o_g)
    if end_g < end_d:
        return end_g, s_g, o_g, "greedy"
    return end_d, s_d, o_d, "dfs"
