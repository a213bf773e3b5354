"""Scheduling-policy simulator + cost model (include/dit_sim.h).  CPU only.
(i) pins of the Python oracle (oracle/sim_oracle.py) against hand-computed traces and conservation laws; (ii) the C++
simulator in libdit_b200.so against the oracle, request by request, bit for bit (same arithmetic in the same order)."""
import math

import pytest

from oracle import sim_oracle as S
from paper_2606_13501_b200 import binding as B
from paper_2606_13501_b200 import synth

TABLE = {(0, 1): 0.010, (0, 2): 0.006, (0, 4): 0.004, (1, 1): 0.050, (1, 2): 0.027, (1, 4): 0.015, (1, 8): 0.009,
         (2, 1): 0.200, (2, 2): 0.104, (2, 4): 0.055, (2, 8): 0.031}


def _cfg(policy, **kw):
    d = dict(policy=policy, n_ranks=4, fcfs_group=2, state_mb=[4.0, 16.0, 40.0], relayout_gbps=50.0, timeout_s=0.0)
    d.update(kw)
    return d


def _req(c, n, a, d):
    return dict(shape_class=c, n_steps=n, arrival_s=a, deadline_s=d)


# ------------------------------------------------------------------------------------------ oracle pins
def test_single_request_closed_forms():
    for pol, deg in ((S.FCFS, 2), (S.SRTF, 1)):
        res, summ = S.simulate(_cfg(pol), TABLE, [_req(1, 20, 3.0, 99.0)])
        assert res[0]["finish_s"] == pytest.approx(3.0 + 20 * TABLE[(1, deg)], abs=1e-12)
        assert res[0]["n_migrations"] == 0 and res[0]["max_degree"] == deg and res[0]["met_deadline"] == 1
        assert summ["n_events"] == 20 and summ["mean_latency_s"] == pytest.approx(20 * TABLE[(1, deg)])
    # EDF, loose deadline: the SMALLEST degree predicted to meet it (1), all the way
    res, _ = S.simulate(_cfg(S.EDF), TABLE, [_req(1, 20, 3.0, 8.0)])
    assert res[0]["max_degree"] == 1 and res[0]["finish_s"] == pytest.approx(3.0 + 20 * 0.05, abs=1e-12) and res[0]["n_migrations"] == 0
    # impossible deadline: nothing meets it, so the largest degree that fits the 4 free ranks, all the way
    res, _ = S.simulate(_cfg(S.EDF), TABLE, [_req(1, 20, 3.0, 3.01)])
    assert res[0]["max_degree"] == 4 and res[0]["finish_s"] == pytest.approx(3.0 + 20 * 0.015, abs=1e-12)
    assert res[0]["busy_rank_s"] == pytest.approx(4 * 20 * 0.015) and res[0]["met_deadline"] == 0
    # tight deadline 3.6: degree 1 would end at 4.0, degree 2 at 3.54 -> 2.  The choice is re-evaluated at every trajectory
    # boundary: after i steps at degree 2, degree 1 (on rank 0 alone: another rank set, so one migration of
    # 16 MB / 50 GB/s = 0.32 ms) meets the deadline once 3 + 0.027 i + 0.00032 + 0.05 (20 - i) <= 3.6, i.e. from i = 18
    res, _ = S.simulate(_cfg(S.EDF), TABLE, [_req(1, 20, 3.0, 3.6)])
    assert res[0]["max_degree"] == 2 and res[0]["n_migrations"] == 1
    assert res[0]["finish_s"] == pytest.approx(3.0 + 18 * 0.027 + 16.0e6 / 50e9 + 2 * 0.05, abs=1e-12)
    assert res[0]["busy_rank_s"] == pytest.approx(2 * 18 * 0.027 + 16.0e6 / 50e9 + 2 * 0.05)


def test_fcfs_fifo_and_group_assignment_by_hand():
    # one group of 2 ranks: two requests interleave step by step in ready order (task-level FIFO)
    tr = []
    reqs = [_req(0, 2, 0.0, 9.0), _req(0, 2, 0.001, 9.0)]
    res, _ = S.simulate(_cfg(S.FCFS, n_ranks=2), TABLE, reqs, trace=tr)
    c = TABLE[(0, 2)]
    assert [(t[0], t[1]) for t in tr] == [(0, 0), (1, 0), (0, 1), (1, 1)]
    assert res[0]["finish_s"] == pytest.approx(3 * c) and res[1]["finish_s"] == pytest.approx(4 * c)
    # two groups: the second request goes to the idle group and both run undisturbed, never migrating
    res, _ = S.simulate(_cfg(S.FCFS, n_ranks=4), TABLE, reqs)
    assert res[0]["finish_s"] == pytest.approx(2 * c) and res[1]["finish_s"] == pytest.approx(0.001 + 2 * c)
    assert res[0]["n_migrations"] == 0 and res[1]["n_migrations"] == 0


def test_srtf_runs_the_shortest_remaining_work_first():
    # one rank, a long request is running when two more arrive: at its next trajectory boundary the rank takes the request
    # with the least remaining work (the short late-comer), then the other short one, the long one last
    reqs = [_req(2, 3, 0.0, 99.0), _req(0, 4, 0.01, 99.0), _req(0, 2, 0.02, 99.0)]
    tr = []
    res, _ = S.simulate(_cfg(S.SRTF, n_ranks=1), TABLE, reqs, trace=tr)
    assert [t[0] for t in tr] == [0, 2, 2, 1, 1, 1, 1, 0, 0]
    assert res[2]["finish_s"] == pytest.approx(0.2 + 2 * 0.01) and res[1]["finish_s"] == pytest.approx(0.2 + 6 * 0.01)
    assert res[0]["finish_s"] == pytest.approx(3 * 0.2 + 6 * 0.01)


def test_edf_orders_ready_tasks_by_deadline():
    # one rank; the policy runs after EVERY event (R39), so request 0's first task starts the moment it arrives; from then
    # on, at every trajectory boundary, the ready task with the earliest deadline runs: 1, 1, 2, 2, then 0's second task
    reqs = [_req(1, 2, 0.0, 50.0), _req(1, 2, 0.0, 0.2), _req(1, 2, 0.0, 30.0)]
    tr = []
    res, _ = S.simulate(_cfg(S.EDF, n_ranks=1), TABLE, reqs, trace=tr)
    assert [t[0] for t in tr] == [0, 1, 1, 2, 2, 0]
    assert res[1]["finish_s"] == pytest.approx(3 * 0.05) and res[1]["met_deadline"] == 1
    assert res[0]["finish_s"] == pytest.approx(6 * 0.05)


def test_edf_deadline_beats_arrival_and_migration_enters_the_degree_choice():
    # the earlier DEADLINE wins although the request arrived later (R39: order by (deadline, arrival, index))
    reqs = [_req(1, 2, 0.0, 50.0), _req(1, 2, 0.01, 0.5)]
    tr = []
    S.simulate(_cfg(S.EDF, n_ranks=1), TABLE, reqs, trace=tr)
    assert [t[0] for t in tr] == [0, 1, 1, 0]
    # the predicted finish of a candidate degree includes the migration it would cause: with a slow
    # re-layout (16 MB at 0.16 GB/s = 0.1 s) leaving degree 2 for degree 1 never meets 3.6 (3 + 0.027 i + 0.1 + 0.05 (20 - i)
    # <= 3.6 needs i >= 21.7), so the request stays on its two ranks: 20 x 0.027, no migration, deadline met.  (Without the
    # migration term it would switch after 18 steps and finish at 3.686.)
    res, _ = S.simulate(_cfg(S.EDF, relayout_gbps=0.16), TABLE, [_req(1, 20, 3.0, 3.6)])
    assert res[0]["n_migrations"] == 0 and res[0]["max_degree"] == 2 and res[0]["met_deadline"] == 1
    assert res[0]["finish_s"] == pytest.approx(3.0 + 20 * 0.027, abs=1e-12)
    # a change of rank set is counted as a migration even when it costs no time (no re-layout bandwidth given): degree 1 meets
    # the deadline once 3 + 0.027 i + 0.05 (20 - i) <= 3.6, i.e. from i = 18
    res, _ = S.simulate(_cfg(S.EDF, relayout_gbps=0.0), TABLE, [_req(1, 20, 3.0, 3.6)])
    assert res[0]["n_migrations"] == 1 and res[0]["finish_s"] == pytest.approx(3.0 + 18 * 0.027 + 2 * 0.05, abs=1e-12)


def test_summary_statistics_and_timeouts_by_hand():
    # 20 requests of 1..20 steps, one rank each (SRTF places a new request on the least-loaded rank): latency_i = 0.01 i
    reqs = [_req(0, i + 1, 0.0, 0.01 * (i + 1) + (1e-9 if i % 2 == 0 else -1e-3)) for i in range(20)]
    res, summ = S.simulate(_cfg(S.SRTF, n_ranks=20), TABLE, reqs)
    for i, r in enumerate(res):
        assert r["finish_s"] == pytest.approx(0.01 * (i + 1), abs=1e-12) and r["failed"] == 0
        assert r["met_deadline"] == (1 if i % 2 == 0 else 0)
    assert summ["p95_latency_s"] == pytest.approx(0.19, abs=1e-12)          # 19th of 20 sorted latencies (ceil(0.95 n))
    assert summ["mean_latency_s"] == pytest.approx(0.105, abs=1e-12)
    assert summ["makespan_s"] == pytest.approx(0.20, abs=1e-12) and summ["throughput_rps"] == pytest.approx(100.0)
    assert summ["slo_attainment"] == pytest.approx(0.5)
    assert summ["utilisation"] == pytest.approx(sum(0.01 * (i + 1) for i in range(20)) / (20 * 0.20))
    # a timeout of 0.155 s fails the five requests of 16..20 steps: they leave the latency statistics and miss their SLO
    res, summ = S.simulate(_cfg(S.SRTF, n_ranks=20, timeout_s=0.155), TABLE, reqs)
    assert [r["failed"] for r in res] == [0] * 15 + [1] * 5
    assert summ["p95_latency_s"] == pytest.approx(0.15, abs=1e-12) and summ["mean_latency_s"] == pytest.approx(0.08, abs=1e-12)
    assert summ["slo_attainment"] == pytest.approx(8 / 20)                   # the even-indexed ones among the first 15
    assert summ["throughput_rps"] == pytest.approx(15 / 0.20)


def _random_trace(seed, n, classes=3, rate=40.0):
    u = synth.uniform01(seed, "sim.trace", 4 * n).tolist()
    t, reqs = 0.0, []
    for i in range(n):
        t += -math.log(u[4 * i]) / rate
        c = int(u[4 * i + 1] * classes)
        steps = 4 + int(u[4 * i + 2] * 28)
        alpha = (2.0, 2.5, 3.5)[c]
        reqs.append(_req(c, steps, t, t + alpha * steps * TABLE[(c, 1)] * (0.3 + u[4 * i + 3])))
    return reqs


@pytest.mark.parametrize("policy", [S.FCFS, S.SRTF, S.EDF])
def test_conservation_laws_on_random_traces(policy):
    reqs = _random_trace(3, 60)
    tr = []
    cfg = _cfg(policy, n_ranks=8, fcfs_group=2)
    res, summ = S.simulate(cfg, TABLE, reqs, trace=tr)
    # every task exactly once, in order, after its predecessor and after the arrival
    per = {}
    for r, step, t0, t1, ranks in tr:
        per.setdefault(r, []).append((step, t0, t1))
    for r, q in enumerate(reqs):
        steps = sorted(per[r])
        assert [s_[0] for s_ in steps] == list(range(q["n_steps"]))
        assert steps[0][1] >= q["arrival_s"] - 1e-12
        for a, b in zip(steps, steps[1:]):
            assert b[1] >= a[2] - 1e-12
        assert res[r]["finish_s"] == pytest.approx(steps[-1][2])
    # no rank runs two tasks at once
    by_rank = {}
    for r, step, t0, t1, ranks in tr:
        for k in ranks:
            by_rank.setdefault(k, []).append((t0, t1))
    for k, iv in by_rank.items():
        iv.sort()
        for a, b in zip(iv, iv[1:]):
            assert b[0] >= a[1] - 1e-12, f"rank {k} runs two tasks at once"
    # busy time = sum of task durations x degree; utilisation <= 1
    assert sum(x["busy_rank_s"] for x in res) == pytest.approx(sum((t1 - t0) * len(rk) for _, _, t0, t1, rk in tr))
    assert 0 < summ["utilisation"] <= 1 + 1e-12 and summ["n_events"] == len(tr) == sum(q["n_steps"] for q in reqs)


# ------------------------------------------------------------------------------------------ C++ vs oracle
@pytest.mark.parametrize("policy", [S.FCFS, S.SRTF, S.EDF])
@pytest.mark.parametrize("seed,n,ranks,group,rate", [(1, 40, 4, 2, 30.0), (2, 120, 8, 4, 80.0), (5, 200, 8, 1, 200.0), (7, 25, 1, 1, 5.0)])
def test_library_simulator_matches_oracle(lib, policy, seed, n, ranks, group, rate):
    reqs = _random_trace(seed, n, rate=rate)
    cfg = _cfg(policy, n_ranks=ranks, fcfs_group=group, timeout_s=3.0)
    ro, so = S.simulate(cfg, TABLE, reqs)
    rl, sl = B.dit_sim_run(cfg, TABLE, reqs)
    for a, b in zip(ro, rl):
        assert a == b, (a, b)                                  # finish times etc. bit for bit
    for k in so:
        assert sl[k] == so[k] or sl[k] == pytest.approx(so[k], rel=1e-15), k


def test_library_simulator_on_the_hand_made_scenarios(lib):
    """The scenarios the oracle is pinned on by hand, through the library: slow / absent re-layout bandwidth in EDF's degree
    choice, deadline-before-arrival order, timeouts in the summary."""
    cases = [(_cfg(S.EDF, n_ranks=1), [_req(1, 2, 0.0, 50.0), _req(1, 2, 0.01, 0.5)]),
             (_cfg(S.EDF, relayout_gbps=0.16), [_req(1, 20, 3.0, 3.6)]),
             (_cfg(S.EDF, relayout_gbps=0.0), [_req(1, 20, 3.0, 3.6)]),
             (_cfg(S.EDF), [_req(1, 20, 3.0, 3.6)]),
             (_cfg(S.SRTF, n_ranks=20, timeout_s=0.155), [_req(0, i + 1, 0.0, 0.01 * (i + 1) + (1e-9 if i % 2 == 0 else -1e-3)) for i in range(20)])]
    for cfg, reqs in cases:
        ro, so = S.simulate(cfg, TABLE, reqs)
        rl, sl = B.dit_sim_run(cfg, TABLE, reqs)
        assert ro == rl
        for k in so:
            assert sl[k] == so[k] or sl[k] == pytest.approx(so[k], rel=1e-15), k


def test_library_simulator_rejects_bad_input(lib):
    with pytest.raises(B.DitError, match="no entry"):
        B.dit_sim_run(_cfg("fcfs", fcfs_group=4), {(0, 1): 0.01}, [_req(0, 2, 0.0, 1.0)])
    with pytest.raises(B.DitError, match="arrives before"):
        B.dit_sim_run(_cfg("srtf"), TABLE, [_req(0, 2, 1.0, 2.0), _req(0, 2, 0.5, 2.0)])
    with pytest.raises(B.DitError, match="divide"):
        B.dit_sim_run(_cfg("fcfs", n_ranks=4, fcfs_group=3), TABLE, [_req(0, 2, 0.0, 1.0)])
    res, summ = B.dit_sim_run(_cfg("edf"), TABLE, [])
    assert res == [] and summ["n_events"] == 0
