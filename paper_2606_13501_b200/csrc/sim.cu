// sim.cu — step-time cost model + scheduling-policy simulator (include/dit_sim.h).  Host code only (compiled with the rest of
// the library so that one .so carries the whole C ABI), reading R39.
// Event-driven: a min-heap of (time, completion-before-arrival, request) events; after every event the policy dispatches.
// Rank sets are 64-bit masks (n_ranks <= 64); the cost table is a dense [class][degree] array.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <queue>
#include <vector>

#include "../../include/dit_sim.h"
#include "common.cuh"

namespace {

constexpr int MAX_CLASSES = 16, MAX_DEGREE = 64;

struct Event {
  double t;
  int kind;   // 0 = completion, 1 = arrival
  int req;
  bool operator>(const Event& o) const {
    if (t != o.t) return t > o.t;
    if (kind != o.kind) return kind > o.kind;
    return req > o.req;
  }
};

struct Sim {
  const dit_sim_config& cfg;
  const dit_sim_request* rq;
  int n;
  double cost[MAX_CLASSES][MAX_DEGREE + 1];   // < 0: no entry
  std::vector<int> done, started, n_mig, max_deg;
  std::vector<uint64_t> last_set, run_set;    // rank masks (FCFS: 1 << group; SRTF: 1 << rank); 0 = none yet
  std::vector<double> finish, busy_s;
  std::priority_queue<Event, std::vector<Event>, std::greater<Event>> ev;
  bool bad = false;   // a needed (class, degree) was missing

  Sim(const dit_sim_config& c, const dit_sim_request* r, int n_) : cfg(c), rq(r), n(n_) {
    done.assign(n, 0); started.assign(n, 0); n_mig.assign(n, 0); max_deg.assign(n, 0);
    last_set.assign(n, 0); run_set.assign(n, 0); finish.assign(n, NAN); busy_s.assign(n, 0.0);
  }
  double c_of(int cls, int deg) {
    const double v = (deg >= 1 && deg <= MAX_DEGREE) ? cost[cls][deg] : -1.0;
    if (v < 0) { bad = true; dit::set_error("dit_sim_run: cost table has no entry for class %d, degree %d", cls, deg); return 1.0; }
    return v;
  }
  double mig_time(int r) const {
    return cfg.relayout_gbps > 0 ? cfg.state_mb[rq[r].shape_class] * 1e6 / (cfg.relayout_gbps * 1e9) : 0.0;
  }
  double start(int r, double now, uint64_t set, int degree) {
    const bool moved = last_set[r] != 0 && last_set[r] != set;
    const double mig = moved ? mig_time(r) : 0.0;
    if (moved) ++n_mig[r];
    const double dur = mig + c_of(rq[r].shape_class, degree);
    const double end = now + dur;
    run_set[r] = set;
    ++started[r];
    busy_s[r] += degree * dur;
    max_deg[r] = std::max(max_deg[r], degree);
    ev.push(Event{end, 0, r});
    return end;
  }
};

}  // namespace

extern "C" dit_status dit_sim_run(const dit_sim_config* cfg, const dit_cost_entry* table, int32_t n_entries,
                                  const dit_sim_request* requests, int32_t n_requests, dit_sim_result* results,
                                  dit_sim_summary* summary) {
  using dit::set_error;
  DIT_REQUIRE(cfg && cfg->struct_size == (int)sizeof(dit_sim_config), DIT_ERR_INVALID_ARG, "dit_sim_config.struct_size mismatch");
  DIT_REQUIRE(cfg->n_ranks >= 1 && cfg->n_ranks <= 64 && cfg->n_classes >= 1 && cfg->n_classes <= MAX_CLASSES, DIT_ERR_INVALID_ARG,
              "n_ranks %d (1..64), n_classes %d (1..16)", cfg->n_ranks, cfg->n_classes);
  DIT_REQUIRE(cfg->policy >= DIT_POLICY_FCFS && cfg->policy <= DIT_POLICY_EDF, DIT_ERR_INVALID_ARG, "policy %d", cfg->policy);
  DIT_REQUIRE(n_requests >= 0 && (n_requests == 0 || (requests && results)) && (n_entries == 0 || table), DIT_ERR_INVALID_ARG, "NULL argument");
  if (cfg->policy == DIT_POLICY_FCFS)
    DIT_REQUIRE(cfg->fcfs_group >= 1 && cfg->n_ranks % cfg->fcfs_group == 0, DIT_ERR_INVALID_ARG, "fcfs_group %d must divide n_ranks %d",
                cfg->fcfs_group, cfg->n_ranks);
  Sim s(*cfg, requests, n_requests);
  for (int c = 0; c < MAX_CLASSES; ++c) for (int p = 0; p <= MAX_DEGREE; ++p) s.cost[c][p] = -1.0;
  for (int i = 0; i < n_entries; ++i) {
    DIT_REQUIRE(table[i].shape_class >= 0 && table[i].shape_class < cfg->n_classes && table[i].degree >= 1 && table[i].degree <= MAX_DEGREE &&
                    table[i].step_s > 0, DIT_ERR_INVALID_ARG, "cost entry %d is malformed", i);
    s.cost[table[i].shape_class][table[i].degree] = table[i].step_s;
  }
  for (int r = 0; r < n_requests; ++r) {
    DIT_REQUIRE(requests[r].shape_class >= 0 && requests[r].shape_class < cfg->n_classes && requests[r].n_steps >= 1, DIT_ERR_INVALID_ARG,
                "request %d: shape_class %d, n_steps %d", r, requests[r].shape_class, requests[r].n_steps);
    DIT_REQUIRE(r == 0 || requests[r].arrival_s >= requests[r - 1].arrival_s, DIT_ERR_INVALID_ARG, "request %d arrives before request %d", r, r - 1);
    s.ev.push(Event{requests[r].arrival_s, 1, r});
  }
  const int n = n_requests, R = cfg->n_ranks, policy = cfg->policy;
  const int g = cfg->policy == DIT_POLICY_FCFS ? cfg->fcfs_group : 1;
  const int G = R / g;
  // FCFS: per group a FIFO queue;  SRTF: per rank an owner list;  EDF: one ready list
  std::vector<std::vector<int>> queue(policy == DIT_POLICY_FCFS ? G : 0);
  std::vector<char> busy(64, 0);
  std::vector<double> free_at(64, 0.0);
  std::vector<int> owner(n, -1);
  std::vector<char> waiting(n, 0);
  std::vector<int> ready_set;
  std::vector<int> degs[MAX_CLASSES];
  for (int c = 0; c < cfg->n_classes; ++c)
    for (int p = 1; p <= MAX_DEGREE; ++p)
      if (s.cost[c][p] >= 0) degs[c].push_back(p);

  auto ready = [&](int r, double now) {
    if (policy == DIT_POLICY_FCFS) {
      int best = 0;
      double best_w = 0;
      for (int j = 0; j < G; ++j) {
        double w = busy[j] ? std::max(free_at[j] - now, 0.0) : 0.0;
        for (int q : queue[j]) w += s.c_of(requests[q].shape_class, g);
        if (j == 0 || w < best_w) { best = j; best_w = w; }
      }
      queue[best].push_back(r);
    } else if (policy == DIT_POLICY_SRTF) {
      if (owner[r] < 0) {
        int best = 0;
        double best_w = 0;
        for (int k = 0; k < R; ++k) {
          double w = busy[k] ? std::max(free_at[k] - now, 0.0) : 0.0;
          for (int q = 0; q < n; ++q)
            if (owner[q] == k && s.done[q] < requests[q].n_steps) w += (requests[q].n_steps - s.started[q]) * s.c_of(requests[q].shape_class, 1);
          if (k == 0 || w < best_w) { best = k; best_w = w; }
        }
        owner[r] = best;
      }
      waiting[r] = 1;
    } else {
      ready_set.push_back(r);
    }
  };
  auto dispatch = [&](double now) {
    if (policy == DIT_POLICY_FCFS) {
      for (int j = 0; j < G; ++j)
        if (!busy[j] && !queue[j].empty()) {
          const int r = queue[j].front();
          queue[j].erase(queue[j].begin());
          busy[j] = 1;
          free_at[j] = s.start(r, now, 1ull << j, g);
        }
    } else if (policy == DIT_POLICY_SRTF) {
      for (int k = 0; k < R; ++k) {
        if (busy[k]) continue;
        int pick = -1;
        double pw = 0;
        for (int q = 0; q < n; ++q) {
          if (owner[q] != k || !waiting[q]) continue;
          const double w = (requests[q].n_steps - s.done[q]) * s.c_of(requests[q].shape_class, 1);
          if (pick < 0 || w < pw || (w == pw && requests[q].arrival_s < requests[pick].arrival_s)) { pick = q; pw = w; }
        }
        if (pick < 0) continue;
        waiting[pick] = 0;
        busy[k] = 1;
        free_at[k] = s.start(pick, now, 1ull << k, 1);
      }
    } else {
      for (;;) {
        int free_ranks[64], nf = 0;
        for (int k = 0; k < R; ++k) if (!busy[k]) free_ranks[nf++] = k;
        if (nf == 0 || ready_set.empty()) return;
        int pi = 0;
        for (int i = 1; i < (int)ready_set.size(); ++i) {
          const dit_sim_request &a = requests[ready_set[i]], &b = requests[ready_set[pi]];
          if (a.deadline_s < b.deadline_s || (a.deadline_s == b.deadline_s && (a.arrival_s < b.arrival_s ||
              (a.arrival_s == b.arrival_s && ready_set[i] < ready_set[pi])))) pi = i;
        }
        const int r = ready_set[pi], c = requests[r].shape_class;
        int choice = -1;
        bool met = false;
        for (int p : degs[c]) {
          if (p > nf) break;
          uint64_t sid = 0;
          for (int i = 0; i < p; ++i) sid |= 1ull << free_ranks[i];
          const double mig = (s.last_set[r] != 0 && s.last_set[r] != sid) ? s.mig_time(r) : 0.0;
          if (!met) choice = p;                        // the largest that fits, unless a smaller one meets the deadline
          if (!met && now + mig + (requests[r].n_steps - s.done[r]) * s.c_of(c, p) <= requests[r].deadline_s) met = true;
        }
        if (choice < 0) { s.bad = true; set_error("dit_sim_run: cost table has no degree <= %d for class %d", nf, c); return; }
        uint64_t sid = 0;
        for (int i = 0; i < choice; ++i) { sid |= 1ull << free_ranks[i]; busy[free_ranks[i]] = 1; }
        ready_set.erase(ready_set.begin() + pi);
        s.start(r, now, sid, choice);
      }
    }
  };
  int64_t n_events = 0;
  while (!s.ev.empty() && !s.bad) {
    const Event e = s.ev.top();
    s.ev.pop();
    const int r = e.req;
    if (e.kind == 0) {
      ++n_events;
      const uint64_t set = s.run_set[r];
      if (policy == DIT_POLICY_EDF) { for (int k = 0; k < R; ++k) if ((set >> k) & 1) busy[k] = 0; }
      else { for (int k = 0; k < 64; ++k) if ((set >> k) & 1) busy[k] = 0; }
      s.last_set[r] = set;
      if (++s.done[r] == requests[r].n_steps) s.finish[r] = e.t;
      else ready(r, e.t);
    } else {
      ready(r, e.t);
    }
    dispatch(e.t);
  }
  if (s.bad) return DIT_ERR_INVALID_ARG;
  std::vector<double> lats;
  double lat_sum = 0, busy_sum = 0, last_finish = 0, first_arrival = n ? requests[0].arrival_s : 0;
  int met = 0;
  for (int r = 0; r < n; ++r) {
    const double lat = s.finish[r] - requests[r].arrival_s;
    const bool failed = cfg->timeout_s > 0 && lat > cfg->timeout_s;
    results[r].finish_s = s.finish[r];
    results[r].busy_rank_s = s.busy_s[r];
    results[r].n_migrations = s.n_mig[r];
    results[r].max_degree = s.max_deg[r];
    results[r].failed = failed ? 1 : 0;
    results[r].met_deadline = (!failed && s.finish[r] <= requests[r].deadline_s) ? 1 : 0;
    met += results[r].met_deadline;
    if (!failed) { lats.push_back(lat); lat_sum += lat; }
    busy_sum += s.busy_s[r];
    last_finish = r == 0 ? s.finish[r] : std::max(last_finish, s.finish[r]);
    first_arrival = std::min(first_arrival, requests[r].arrival_s);
  }
  if (summary) {
    std::sort(lats.begin(), lats.end());
    const double makespan = n ? last_finish - first_arrival : 0.0;
    summary->makespan_s = makespan;
    summary->throughput_rps = makespan > 0 ? lats.size() / makespan : 0.0;
    summary->mean_latency_s = lats.empty() ? 0.0 : lat_sum / lats.size();
    summary->p95_latency_s = lats.empty() ? 0.0 : lats[std::max<int64_t>(0, (int64_t)std::ceil(0.95 * lats.size()) - 1)];
    summary->slo_attainment = n ? (double)met / n : 0.0;
    summary->utilisation = makespan > 0 ? busy_sum / (R * makespan) : 0.0;
    summary->n_events = n_events;
  }
  return DIT_OK;
}
