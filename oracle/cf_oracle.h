/*
 * cf_oracle.h -- TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, sequential CPU oracle for the request-level plan-evaluation hot path of
 * arxiv/paper_2512_14098 (Cornfigurator), Algorithm 2 phase 3 and
 * section 4.3 "Request-level simulation", under the fixed model of
 * BASELINE.json `north_star` (integer microseconds, Philox4x32-10, Lindley / Kiefer-Wolfowitz)
 * and the readings R1..R19 listed in DESIGN.md.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * call this. It shares no code, header, table or constant generator with the CUDA path under
 * paper_2512_14098_b200/csrc; the struct layouts below are the oracle's own.
 *
 * Parity status: every function below is pinned by tests/test_oracle_*.py (Random123 known-answer
 * vectors, queueing closed forms, exact D/D/c cases, brute-force event simulators on tiny inputs,
 * invariants; the phase-1/2/selection functions by hand-worked examples, closed forms, brute force
 * and the identity "Monte Carlo = simulation with unlimited replicas": tests/test_oracle_phases.py).
 * Nothing here is "parity unpinned"; the modelling choices R2/R6/R7 are pinned to
 * independent brute-force simulators of the same discipline.
 *
 * All pointers are HOST pointers. All functions are deterministic and thread-safe.
 */
#ifndef CF_ORACLE_H
#define CF_ORACLE_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* status codes (the oracle's own numbering happens to follow the same convention: 0 ok, <0 error) */
#define ORC_OK 0
#define ORC_ERR_ARG (-1)
#define ORC_ERR_RANGE (-2)
#define ORC_ERR_PLAN (-3)
#define ORC_ERR_TABLE (-4)

/* Tail-refined integer quantile table (R3): levels*2^log2_cells + 1 entries,
 * non-decreasing, >= 0. */
typedef struct {
  uint32_t levels, log2_cells;
  const int32_t* q;
} orc_qtab;

/* Model graph + workload (model definition, workload with fractions pi_t). */
typedef struct {
  uint32_t n_comp, n_types, n_req, n_trials; /* C<=8, T<=8, 1<=N<=2^24, K>=1 */
  const uint8_t* type_mask;    /* [T] bit i => type visits component i (topological index) */
  const uint32_t* type_thresh; /* [T] cumulative mix, Q32, non-decreasing; last is catch-all */
  const uint16_t* svc_tab;     /* [C*T] table id for (component i, type t) at i*T+t        */
  const orc_qtab* tabs;        /* service tables, int32 microseconds                       */
  uint32_t n_tabs;
  orc_qtab arr_tab;            /* unit-mean inter-arrival gap, Q16                         */
  const uint8_t* edges;        /* [2*n_edges] (u,v) pairs, component DAG                   */
  uint32_t n_edges;
  int64_t edge_delay_us;       /* PAPER.md:322; added between consecutive visited stages   */
  const uint16_t* cpu_tab;     /* [C*T] table id of the CPU pre-processing time of (i, t), 0xffff = none;
                                  NULL = no component has any (R24) */
  uint32_t join_mode;          /* 0: a request visits its stages one after another (R7); 1: fork-join along
                                  the DAG edges (R25): a stage starts when all its predecessor
                                  stages on the request's subgraph have finished */
  uint32_t order_mode;         /* 0: every stage serves its visitors in request-index order (R2);
                                  1: in the order in which they reach the stage, ties by index -- textbook
                                  FCFS (R27) */
} orc_graph;

/* P physical plans, each an ordered list of stages = (component bitmask, replica count). */
typedef struct {
  uint32_t n_plans, max_stages;
  const uint8_t* n_stages;    /* [P] */
  const uint8_t* stage_mask;  /* [P*max_stages] */
  const uint16_t* stage_c;    /* [P*max_stages] */
  /* Routing between alternative paths (R26). max_routes == 0: none, a
   * request visits every stage that holds one of its components. Else 1..4 routes per (plan,
   * type): the request draws a route with the cumulative probabilities route_cum (Q32, the last
   * route takes the rest) and visits the stages of route_mask (a bitmask over the plan's stages)
   * that hold one of its components. Stage masks may then overlap across stages; along every
   * route they must cover the type's components exactly once. */
  uint32_t max_routes;
  const uint8_t* route_mask;  /* [P*T*max_routes] */
  const uint32_t* route_cum;  /* [P*T*max_routes] */
} orc_plans;

typedef struct {
  const int64_t* L_us;      /* [T] latency target */
  const uint32_t* att_num;  /* [T] attainment target numerator   */
  const uint32_t* att_den;  /* [T]                   denominator */
} orc_slo;

/* Philox4x32-10 (Salmon et al., SC'11); ctr[4], key[2] -> out[4]. */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);

/* Integer table sampling, R3. */
int64_t orc_qtab_sample(const orc_qtab* tab, uint32_t u);

/* Validate graph/plans; returns ORC_OK or the first error found. */
int32_t orc_validate(const orc_graph* g, const orc_plans* pl);

/* One simulation per (plan p, rate r, trial k). Outputs:
 *   out_counts  [P][R][K][T][2] = {cnt_t, hits_t}
 *   out_dep_sum [P][R][K]  sum of final departures mod 2^64     (may be NULL)
 *   out_makespan[P][R][K]  max final departure                   (may be NULL)
 *   out_sim_status [P][R][K] 0 ok, ORC_ERR_RANGE if the sim was out of range (then its outputs
 *                  are all zero)                                  (may be NULL)
 * Returns ORC_OK, a validation error, or ORC_ERR_RANGE if any sim was out of range.
 * n_threads > 1 splits the sims over std::thread (timing only; results identical). */
int32_t orc_eval_plans(const orc_graph* g, const orc_plans* pl, const uint32_t* rate_mrps,
                       uint32_t R, const orc_slo* slo, uint64_t seed, uint32_t variant,
                       uint32_t* out_counts, uint64_t* out_dep_sum, int64_t* out_makespan,
                       int32_t* out_sim_status, int32_t n_threads);

/* Integer rate bisection per plan ("highest request rate that the plan can
 * support"; R12, R18). Outputs: out_rate_mrps[P], out_goodput_mrps[P][T],
 * out_counts[P][K][T][2] at the returned rate (may be NULL). */
int32_t orc_goodput_bisect(const orc_graph* g, const orc_plans* pl, const uint32_t* rate_hi_mrps,
                           uint32_t n_steps, const orc_slo* slo, uint64_t seed, uint32_t variant,
                           uint32_t* out_rate_mrps, uint32_t* out_goodput_mrps,
                           uint32_t* out_counts, int32_t n_threads);

/* Trace of one sim: system arrival, final departure, type of every request ([N] each). */
int32_t orc_trace_sim(const orc_graph* g, const orc_plans* pl, uint32_t plan, uint32_t rate_mrps,
                      uint32_t trial, uint64_t seed, uint32_t variant, int64_t* out_arrival,
                      int64_t* out_departure, uint8_t* out_type);

/* Materialised request stream (C<=6): for variant v in [variant_lo, variant_lo+n_variants),
 * trial k, request n a 32-byte record {uint64 cu | (type<<56), int32 svc[6]} where cu is the
 * cumulative Q16 gap and svc[i] is the sampled service of component i if the request's type
 * visits i, else 0. out has n_variants*K*N records. */
int32_t orc_materialize_stream(const orc_graph* g, uint64_t seed, uint32_t variant_lo,
                               uint32_t n_variants, void* out);

/* ---- the cheap phases around the simulation (cf_oracle_phases.cpp; SURVEY.md 8(f) NEXT-1..3) ---- */

/* Mean of the distribution a quantile table induces, Q16 (R21). */
uint64_t orc_qtab_mean_q16(const orc_qtab* tab);

/* Phase 1, flow-based throughput estimation (Algorithm 2 l.1-5).
 * out_rate_mrps[P] = min(floor(R_d * alpha_num / alpha_den), 1e9); optional out_bound_mrps[P] = R_d
 * (capped at 1e9), out_bottleneck[P] (stage index, 0xff: no demand anywhere), out_redundant[P]. */
int32_t orc_flow_bound(const orc_graph* g, const orc_plans* pl, uint32_t alpha_num,
                       uint32_t alpha_den, uint32_t* out_rate_mrps, uint32_t* out_bound_mrps,
                       uint8_t* out_bottleneck, uint8_t* out_redundant);

/* Phase 2, latency estimation with Monte Carlo (Algorithm 2 l.6-11).
 * rate_mrps[P] = the incoming rate alpha R_d of each plan. out_counts[P][K][T][2] (may be NULL),
 * out_goodput_mrps[P][T]. */
int32_t orc_mc_latency(const orc_graph* g, const orc_plans* pl, const uint32_t* rate_mrps,
                       const orc_slo* slo, uint64_t seed, uint32_t variant, uint32_t* out_counts,
                       uint32_t* out_goodput_mrps);

/* Pareto pruning of goodput vectors and the default selection policy (Algorithm 2 l.12, 16-18,
 * PAPER.md:251-259, 286-288). goodput[P][T], alive[P] or NULL; out_pruned[P]. */
int32_t orc_pareto_select(const uint32_t* goodput, uint32_t P, uint32_t T, const uint8_t* alive,
                          uint8_t* out_pruned, uint32_t* out_best, uint32_t* out_n_survivors);

#ifdef __cplusplus
}
#endif
#endif
