"""CPU oracle of the scheduling-policy simulator — TEST INFRASTRUCTURE, NOT THE PRODUCT (see oracle/dit_oracle.py's header
for who may import it).  Plain, slow, obviously-correct Python: lists, sorts and an event heap; shares no code with
paper_2606_13501_b200/csrc/sim.cu.

What it is: PAPER.md:297-315 (§5.4 scheduling policies, §5.5 simulator and cost model) followed step by step — a request
is a chain of n_steps denoising tasks; a task runs on `degree` ranks for cost(shape, degree) seconds,
"cost-model completion events" replace worker execution; when two consecutive tasks of a request run on
different rank sets its state migrates first.  Every tie-break is DESIGN.md reading R39:
events are processed in order of (time, completions before arrivals, request index); lowest index wins ties between
groups / ranks; EDF orders by (deadline, arrival, index); SRTF by (remaining work, arrival, index).

Pins (tests/test_sim.py): one request alone finishes at arrival + n_steps x cost; a FIFO pair on one group; the EDF degree
choice by hand; SRTF's order on a hand-made trace; conservation laws on random traces (no rank runs two tasks at once, every
task runs exactly once and after its predecessor, busy time = sum of task durations).
"""
from __future__ import annotations

import heapq
import math

FCFS, SRTF, EDF = 0, 1, 2


def _cost(table, c, p):
    if (c, p) not in table:
        raise KeyError(f"cost table has no entry for class {c}, degree {p}")
    return table[(c, p)]


def simulate(cfg: dict, table: dict, requests: list, trace: list | None = None):
    """cfg: policy, n_ranks, fcfs_group, state_mb (list per class), relayout_gbps, timeout_s.
    table: {(shape_class, degree): step seconds}.  requests: list of dicts shape_class, n_steps, arrival_s, deadline_s
    (arrival non-decreasing).  Returns (results, summary); `trace` (optional list) receives one tuple per executed task:
    (request, step, start, end, ranks tuple)."""
    n = len(requests)
    R = cfg["n_ranks"]
    policy = cfg["policy"]
    gbps = cfg.get("relayout_gbps", 0.0)
    timeout = cfg.get("timeout_s", 0.0)

    def mig_time(r):
        return cfg["state_mb"][requests[r]["shape_class"]] * 1e6 / (gbps * 1e9) if gbps > 0 else 0.0

    done = [0] * n            # completed tasks
    started = [0] * n         # started tasks
    last_set = [None] * n     # rank set of the previous task (FCFS: group index; EDF: tuple of ranks; SRTF: rank)
    run_set = [None] * n
    finish = [math.nan] * n
    busy_s = [0.0] * n
    n_mig = [0] * n
    max_deg = [0] * n
    events = []               # (time, kind, request): kind 0 = completion, 1 = arrival
    for r, q in enumerate(requests):
        heapq.heappush(events, (q["arrival_s"], 1, r))
    n_events = 0

    def start(r, now, ranks, set_id, degree):
        c = requests[r]["shape_class"]
        mig = mig_time(r) if (last_set[r] is not None and last_set[r] != set_id) else 0.0
        if mig > 0.0 or (last_set[r] is not None and last_set[r] != set_id):
            n_mig[r] += 1
        dur = mig + _cost(table, c, degree)
        end = now + dur
        run_set[r] = set_id
        started[r] += 1
        busy_s[r] += degree * dur
        max_deg[r] = max(max_deg[r], degree)
        heapq.heappush(events, (end, 0, r))
        if trace is not None:
            trace.append((r, started[r] - 1, now, end, tuple(ranks)))
        return end

    if policy == FCFS:
        g = cfg["fcfs_group"]
        G = R // g
        queue = [[] for _ in range(G)]
        busy = [False] * G
        free_at = [0.0] * G

        def ready(r, now):
            c = requests[r]["shape_class"]
            best, best_w = 0, None
            for j in range(G):
                w = max(free_at[j] - now, 0.0) if busy[j] else 0.0
                for q in queue[j]:
                    w += _cost(table, requests[q]["shape_class"], g)
                if best_w is None or w < best_w:
                    best, best_w = j, w
            queue[best].append(r)

        def dispatch(now):
            for j in range(G):
                if not busy[j] and queue[j]:
                    r = queue[j].pop(0)
                    busy[j] = True
                    free_at[j] = start(r, now, range(j * g, (j + 1) * g), j, g)

        def complete(r, now):
            busy[run_set[r]] = False
    elif policy == SRTF:
        owner = [None] * n
        busy = [False] * R
        free_at = [0.0] * R
        waiting = [False] * n     # has a ready, not yet started task

        def ready(r, now):
            if owner[r] is None:
                best, best_w = 0, None
                for k in range(R):
                    w = max(free_at[k] - now, 0.0) if busy[k] else 0.0
                    for q in range(n):
                        if owner[q] == k and done[q] < requests[q]["n_steps"]:
                            w += (requests[q]["n_steps"] - started[q]) * _cost(table, requests[q]["shape_class"], 1)
                    if best_w is None or w < best_w:
                        best, best_w = k, w
                owner[r] = best
            waiting[r] = True

        def dispatch(now):
            for k in range(R):
                if busy[k]:
                    continue
                cand = [q for q in range(n) if owner[q] == k and waiting[q]]
                if not cand:
                    continue
                r = min(cand, key=lambda q: ((requests[q]["n_steps"] - done[q]) * _cost(table, requests[q]["shape_class"], 1),
                                             requests[q]["arrival_s"], q))
                waiting[r] = False
                busy[k] = True
                free_at[k] = start(r, now, (k,), k, 1)

        def complete(r, now):
            busy[run_set[r]] = False
    elif policy == EDF:
        busy = [False] * R
        ready_set = []
        degrees = {}
        for (c, p) in sorted(table):
            degrees.setdefault(c, []).append(p)

        def ready(r, now):
            ready_set.append(r)

        def dispatch(now):
            while True:
                free = [k for k in range(R) if not busy[k]]
                if not free or not ready_set:
                    return
                r = min(ready_set, key=lambda q: (requests[q]["deadline_s"], requests[q]["arrival_s"], q))
                c = requests[r]["shape_class"]
                cands = [p for p in degrees.get(c, []) if p <= len(free)]
                if not cands:
                    raise KeyError(f"cost table has no degree <= {len(free)} for class {c}")
                choice = cands[-1]
                for p in cands:                              # smallest degree predicted to meet the deadline
                    sid = tuple(free[:p])
                    mig = mig_time(r) if (last_set[r] is not None and last_set[r] != sid) else 0.0
                    if now + mig + (requests[r]["n_steps"] - done[r]) * _cost(table, c, p) <= requests[r]["deadline_s"]:
                        choice = p
                        break
                ranks = tuple(free[:choice])
                ready_set.remove(r)
                for k in ranks:
                    busy[k] = True
                start(r, now, ranks, ranks, choice)

        def complete(r, now):
            for k in run_set[r]:
                busy[k] = False
    else:
        raise ValueError(f"policy {policy}")

    while events:
        now, kind, r = heapq.heappop(events)
        if kind == 0:
            n_events += 1
            complete(r, now)
            last_set[r] = run_set[r]
            done[r] += 1
            if done[r] == requests[r]["n_steps"]:
                finish[r] = now
            else:
                ready(r, now)
        else:
            ready(r, now)
        dispatch(now)

    results = []
    for r, q in enumerate(requests):
        lat = finish[r] - q["arrival_s"]
        failed = bool(timeout > 0 and lat > timeout)
        results.append(dict(finish_s=finish[r], busy_rank_s=busy_s[r], n_migrations=n_mig[r], max_degree=max_deg[r],
                            met_deadline=int((not failed) and finish[r] <= q["deadline_s"]), failed=int(failed)))
    lats = sorted(res["finish_s"] - q["arrival_s"] for res, q in zip(results, requests) if not res["failed"])
    makespan = (max(res["finish_s"] for res in results) - min(q["arrival_s"] for q in requests)) if n else 0.0
    summary = dict(
        makespan_s=makespan,
        throughput_rps=len(lats) / makespan if makespan > 0 else 0.0,
        mean_latency_s=(sum(res["finish_s"] - q["arrival_s"] for res, q in zip(results, requests) if not res["failed"]) / len(lats)) if lats else 0.0,
        p95_latency_s=lats[max(0, math.ceil(0.95 * len(lats)) - 1)] if lats else 0.0,
        slo_attainment=sum(res["met_deadline"] for res in results) / n if n else 0.0,
        utilisation=sum(res["busy_rank_s"] for res in results) / (R * makespan) if makespan > 0 else 0.0,
        n_events=n_events)
    return results, summary
