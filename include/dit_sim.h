/* dit_sim.h — step-time cost model + scheduling-policy simulator (host only; part of libdit_b200.so).
 *
 * SURVEY.md §8(f) item 3; PAPER.md:297-315 (§5.4 "Scheduling Policies", §5.5 "Simulator and Cost Model").  The paper's
 * simulator "replaces worker execution with cost-model completion events while preserving task readiness, dependency
 * updates, resource allocation, and policy invocation"; its cost model is "populated from profiled task latencies indexed by
 * model, task type, request shape, and parallel configuration".  Here the profiled latencies are this
 * library's measured dit_step times (bench.py --workload sim feeds them in), a request is a chain of n_steps denoising
 * tasks, a task runs on `degree` ranks for cost(shape, degree) seconds, and when two consecutive tasks of a
 * request run on different rank sets the request's state is migrated first: state_mb / relayout_gbps.
 * Encoder / VAE stages are not modelled ("denoising dominates").  DESIGN.md reading R39 fixes every tie-break.
 *
 * Policies:
 *   DIT_POLICY_FCFS  "FCFS with workload-aware group assignment": the ranks form n_ranks / fcfs_group fixed groups; a task
 *                    that becomes ready is appended to the FIFO queue of the group with the lowest estimated queued
 *                    workload (time until free + queued task costs); every task runs at degree fcfs_group.
 *   DIT_POLICY_SRTF  "SRTF with per-rank local queues": a request is assigned, on arrival, to the rank with the lowest
 *                    estimated queued workload (remaining work of the requests it owns); a free rank runs, among its own
 *                    requests with a ready task, the one with the shortest remaining trajectory work; degree 1.
 *   DIT_POLICY_EDF   "EDF with best-fit parallelism": ready tasks are taken earliest deadline first; the smallest degree
 *                    (among the table's degrees that fit the free ranks) predicted to meet the deadline is chosen, else the
 *                    largest that fits; re-evaluated at every trajectory boundary.
 */
#ifndef DIT_SIM_B200_H
#define DIT_SIM_B200_H

#include <stdint.h>

#include "dit.h"

#ifdef __cplusplus
extern "C" {
#endif

typedef enum { DIT_POLICY_FCFS = 0, DIT_POLICY_SRTF = 1, DIT_POLICY_EDF = 2 } dit_policy;

typedef struct {
  int32_t shape_class; /* index of the request shape (S / M / L ...) */
  int32_t degree;      /* parallel degree P (ranks used by one task) */
  double step_s;       /* profiled latency of one denoising step at (shape_class, degree), seconds */
} dit_cost_entry;

typedef struct {
  int32_t shape_class;
  int32_t n_steps;   /* denoising tasks of the trajectory (>= 1) */
  double arrival_s;  /* non-decreasing over the request array */
  double deadline_s; /* absolute: a + alpha_c T_c + allowance */
} dit_sim_request;

typedef struct {
  int32_t struct_size;
  int32_t policy;        /* dit_policy */
  int32_t n_ranks;       /* GPUs of the simulated server (1..64) */
  int32_t fcfs_group;    /* FCFS: ranks per group (divides n_ranks; its degree must be in the cost table) */
  int32_t n_classes;     /* shape classes (<= 16) */
  double state_mb[16];   /* per class: bytes/1e6 of inter-step state that a migration moves */
  double relayout_gbps;  /* migration bandwidth, GB/s (<= 0: migrations are free) */
  double timeout_s;      /* client timeout; a request whose latency exceeds it counts as failed; <= 0: none */
} dit_sim_config;

typedef struct {
  double finish_s;        /* completion time of the last task */
  double busy_rank_s;     /* sum over its tasks of degree x (migration + step) */
  int32_t n_migrations;   /* tasks that started on another rank set than their predecessor */
  int32_t max_degree;
  int32_t met_deadline;   /* finish <= deadline and not timed out */
  int32_t failed;         /* timed out */
} dit_sim_result;

typedef struct {
  double makespan_s;      /* last finish - first arrival */
  double throughput_rps;  /* completed (not failed) requests / makespan */
  double mean_latency_s;  /* over completed requests */
  double p95_latency_s;   /* nearest-rank 95th percentile over completed requests */
  double slo_attainment;  /* met_deadline / all requests (failures count as violations) */
  double utilisation;     /* sum busy_rank_s / (n_ranks x makespan) */
  int64_t n_events;       /* completion events processed */
} dit_sim_summary;

/* Runs the trace to completion.  results [n_requests], summary may be NULL.  Errors (negative dit_status, message via
 * dit_last_error(NULL)): a (class, degree) needed but missing from the table, arrivals out of order, bad config. */
dit_status dit_sim_run(const dit_sim_config* cfg, const dit_cost_entry* table, int32_t n_entries,
                       const dit_sim_request* requests, int32_t n_requests, dit_sim_result* results,
                       dit_sim_summary* summary);

#ifdef __cplusplus
}
#endif
#endif /* DIT_SIM_B200_H */
