/*
 * cf.h -- C ABI of the B200-native plan-evaluation hot path (libcf_b200.so).
 *
 * What it computes: for many candidate deployment plans at once, the per-request-type SLO-hit
 * counts (hence goodput, "the throughput of type-t requests that meet their latency target",
 * PAPER.md:139) of arxiv/paper_2512_14098's request-level simulation phase (Algorithm 2 l.13-15,
 * PAPER.md:252-255; sec. 4.3). One independent discrete simulation runs per
 * (plan p, arrival rate r, trial k): requests of each type follow their path through the plan's
 * ordered stages and queue at a c-replica executor pool at every visited stage (Lindley recursion
 * for c = 1, Kiefer-Wolfowitz free-time multiset for c > 1). The exact integer model -- Philox4x32-10
 * counters, integer quantile tables, rounding -- is written out in DESIGN.md ("Algorithm", readings
 * R1..R19); results are bit-exact with the CPU oracle under oracle/.
 *
 * Conventions
 *  - No floating point crosses this ABI. Times are int64 microseconds, services int32 microseconds,
 *    rates uint32 milli-requests/s, gaps Q16 (65536 == one mean inter-arrival gap).
 *  - "host" pointers are read during the call only (descriptors, tables, plan lists: small).
 *    "dev" pointers are CUDA device pointers (e.g. torch.Tensor.data_ptr()); the caller owns all
 *    device memory. The only thing the library keeps between calls is a host-side cache (pinned
 *    memory, at most 16 entries, LRU) of what cf_eval_plans* / cf_goodput_bisect* derive from their
 *    host descriptors -- the launch schedule and the descriptor bytes they upload -- so that a call
 *    repeated with byte-identical descriptors skips that work and its upload is a true asynchronous
 *    copy. The cache never changes a result; cf_cache_clear() releases it.
 *  - Every compute call takes a cudaStream_t (as void*), enqueues its work on it and returns
 *    without synchronising (host-side scheduling happens before the first launch; the FIRST call
 *    with given descriptors also allocates pinned memory, which may synchronise the device;
 *    cf_trace_sim, cf_materialize_stream, cf_flow_bound and cf_mc_latency stage their small
 *    descriptors through a pageable copy, which synchronises with the stream). Scratch comes
 *    from the caller's `workspace` (dev, >= cf_workspace_bytes(), 256-byte aligned); it must stay
 *    untouched until the stream work has finished. Distinct streams + distinct workspaces are
 *    thread-safe; no call reads or writes library-wide state.
 *  - Return value: CF_OK or a negative cf_status. Argument errors are detected on the host before
 *    anything is enqueued. Conditions that depend on device data (a rate outside [1, 1e9] mrps, or
 *    arrivals that would exceed 2^62 us, R17) are detected on the device: that
 *    simulation's outputs are all zero and a sticky CF_ERR_RANGE is recorded in the workspace,
 *    readable with cf_workspace_status().
 */
#ifndef CF_H
#define CF_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  CF_OK = 0,
  CF_ERR_ARG = -1,   /* null pointer, size out of bounds, bad table id                         */
  CF_ERR_RANGE = -2, /* overflow guard (services, edge delay, rate, arrival horizon, c, smem)  */
  CF_ERR_PLAN = -3,  /* c = 0, masks overlap / miss a used component, order violates a DAG edge */
  CF_ERR_TABLE = -4, /* quantile table decreasing, negative, or of unsupported shape            */
  CF_ERR_CUDA = -5,  /* a CUDA runtime call failed                                              */
  CF_ERR_WORKSPACE = -6 /* workspace NULL, misaligned or smaller than cf_workspace_bytes()     */
} cf_status;

/* Tail-refined integer quantile table (R3; stands for a latency profile "sampled from
 * profiling results"). levels*2^log2_cells + 1 entries, non-decreasing, >= 0.
 * Level k < levels-1 covers quantiles [1-2^-k, 1-2^-(k+1)), the last level [1-2^-(levels-1), 1);
 * each level has 2^log2_cells equal cells; entry (k,m) is the quantile at the left edge of cell m;
 * the final entry closes the last cell. 1 <= levels <= 32, log2_cells <= 16. q: host. */
typedef struct {
  uint32_t levels, log2_cells;
  const int32_t* q;
} cf_qtab;

/* Model definition graph + workload. All pointers host. */
typedef struct {
  uint32_t n_comp, n_types, n_req, n_trials; /* C<=8, T<=8, 1<=N<=2^24 requests per sim, K trials */
  const uint8_t* type_mask;    /* [T] bit i: type visits component i; components in topological order */
  const uint32_t* type_thresh; /* [T] cumulative mix pi_t in Q32, non-decreasing; last entry ignored */
  const uint16_t* svc_tab;     /* [C*T] id of the service table of (component i, type t) at i*T+t   */
  const cf_qtab* tabs;         /* [n_tabs] service tables, entries int32 microseconds              */
  uint32_t n_tabs;
  cf_qtab arr_tab;             /* unit-mean inter-arrival gap, entries Q16                         */
  const uint8_t* edges;        /* [2*n_edges] (u,v): component u feeds component v (validation)    */
  uint32_t n_edges;
  int64_t edge_delay_us;       /* PAPER.md:322; added between consecutive visited stages; [0,2^31) */
  const uint16_t* cpu_tab;     /* [C*T] id of the CPU pre-processing time table of (i, t), 0xffff = none; or
                                  NULL. CPU-GPU overlap of PAPER.md:318-320 (R24): a request that
                                  finds the stage's earliest-free replica idle pays CPU + GPU time (svc_tab is
                                  the GPU time), a request that queued pays GPU time alone. Such graphs run on
                                  the 64-bit kernel and cannot be materialised as a stream (CF_ERR_ARG).    */
  uint32_t join_mode;          /* 0: a request visits its stages one after another in the plan's order (R7).
                                  1: fork-join along `edges` (R25; Fig. 1, encoders
                                  feeding the LLM): a request reaches a stage when every predecessor stage --
                                  one holding a component u of the request with an edge (u, v) into a
                                  component v of the request on that stage -- has finished, plus
                                  edge_delay_us; with no predecessor at its system arrival; it is done when
                                  its last stage is. 64-bit kernel only; no stream; cf_mc_latency then returns
                                  the critical path of every request (per-plan kernel).                     */
  uint32_t order_mode;         /* 0: every stage serves its visitors in request-index order (R2).
                                  1: in the order in which they REACH the stage, ties by request index --
                                  textbook FCFS at every node (R27). Runs on
                                  the arrival-order kernel: one warp per simulation, stage by stage, over
                                  48 N bytes of workspace per simulation in flight (52 N with cpu_tab) plus
                                  80 N K bytes of request records; cf_workspace_bytes asks for 3552
                                  simulations in flight (fewer if that exceeds 16 GiB): the warps a B200 holds
                                  at once.
                                  Replicas per stage <= 256; no stream. With join_mode = 1 a slot holds 64 N
                                  bytes more (the departure of every request from every stage).            */
} cf_graph;

/* P physical plans; plan p is an ORDERED list of n_stages[p] stages, stage s = (bitmask of the
 * components colocated on that node, replica count c >= 1) (nodes/executors: PAPER.md:127,199-221).
 * Masks are disjoint within a plan and cover every component some type uses. All pointers host. */
typedef struct {
  uint32_t n_plans, max_stages; /* max_stages <= 8 */
  const uint8_t* n_stages;      /* [P] */
  const uint8_t* stage_mask;    /* [P*max_stages] */
  const uint16_t* stage_c;      /* [P*max_stages] */
  /* Routing between alternative paths ("routing probabilities ... between alternative
   * parallel paths in the logical plan"; R26). max_routes = 0 (and NULL pointers): none.
   * Else 1..4 routes per (plan, type): a request of type t draws route r with the cumulative
   * probabilities route_cum (Q32, non-decreasing; the last route takes the rest; Philox block 0,
   * word 2) and visits the stages of bitmask route_mask (bit s = stage s) that hold one of its
   * components. Stage masks may then overlap across stages; along every route they must serve
   * each component of the type exactly once, in an order the DAG allows. Routed plans cannot be
   * evaluated on a materialised stream; cf_mc_latency follows each request's drawn route (per-plan
   * kernel over shared request records instead of the plan-independent histogram). */
  uint32_t max_routes;
  const uint8_t* route_mask;    /* [P*T*max_routes] */
  const uint32_t* route_cum;    /* [P*T*max_routes] */
} cf_plans;

/* Per-type latency targets L_t and the attainment target used by the rate
 * bisection (R12): feasible iff hits_t*att_den[t] >= att_num[t]*cnt_t for all t. host. */
typedef struct {
  const int64_t* L_us;     /* [T] */
  const uint32_t* att_num; /* [T] (bisection only; may be NULL for cf_eval_plans) */
  const uint32_t* att_den; /* [T] */
} cf_slo;

/* Upper bound of the scratch any call below needs for (graph, plans, R rates per plan). */
size_t cf_workspace_bytes(const cf_graph* g, const cf_plans* pl, uint32_t R);

/* cf_eval_plans: simulate every (plan p, rate r, trial k), p<P, r<R, k<K.
 *   rate_mrps    dev [P*R]  arrival rate of (p,r) in milli-requests/s, valid range [1, 1e9]
 *   seed         Philox key; variant = Philox counter word 3 (decorrelates streams, R4)
 *   out_counts   dev [P][R][K][T][2] = {cnt_t, hits_t}: requests of type t, and those with
 *                sojourn D_n - A_n <= L_t (F_{t,d}(L_t) = hits_t/cnt_t)
 *   out_dep_sum  dev [P][R][K] sum of final departures mod 2^64, or NULL
 *   out_makespan dev [P][R][K] max final departure (R10), or NULL                               */
int32_t cf_eval_plans(const cf_graph* g, const cf_plans* pl, const uint32_t* rate_mrps, uint32_t R,
                      const cf_slo* slo, uint64_t seed, uint32_t variant, uint32_t* out_counts,
                      uint64_t* out_dep_sum, int64_t* out_makespan, void* workspace,
                      size_t workspace_bytes, void* stream);

/* cf_goodput_bisect: per plan, n_steps steps of integer bisection on the rate (PAPER.md:340
 * "the highest request rate that the plan can support"), entirely on the device: lo = 0,
 * hi = rate_hi_mrps[p] (exclusive); mid = lo + (hi-lo)/2; mid == lo -> no-op; else run the K trials
 * at mid, pool counts, feasible -> lo = mid else hi = mid (R12, R18).
 *   rate_hi_mrps     dev [P]
 *   out_rate_mrps    dev [P]     rate* = final lo
 *   out_goodput_mrps dev [P][T]  floor(rate* * hits_t / (N*K)), hits pooled at rate* (R10)
 *   out_counts       dev [P][K][T][2] counts at rate* (zeros if rate* = 0), or NULL               */
int32_t cf_goodput_bisect(const cf_graph* g, const cf_plans* pl, const uint32_t* rate_hi_mrps,
                          uint32_t n_steps, const cf_slo* slo, uint64_t seed, uint32_t variant,
                          uint32_t* out_rate_mrps, uint32_t* out_goodput_mrps, uint32_t* out_counts,
                          void* workspace, size_t workspace_bytes, void* stream);

/* Materialised request stream (north_star "request stream materialised in HBM"), C <= 6 only.
 * Record (32 bytes, 16-byte aligned): { uint64 cu | (type << 56) ; int32 svc[6] } where cu is the
 * cumulative Q16 gap up to and including the request and svc[i] the sampled service of component i
 * if the request's type visits i, else 0. Layout [n_variants][K][N]; variant index vi holds Philox
 * variant variant_lo + vi. cf_stream_bytes = n_variants*K*N*32. */
size_t cf_stream_bytes(const cf_graph* g, uint32_t n_variants);
size_t cf_materialize_workspace_bytes(const cf_graph* g, uint32_t n_variants); /* scratch of the call below */
int32_t cf_materialize_stream(const cf_graph* g, uint64_t seed, uint32_t variant_lo,
                              uint32_t n_variants, void* out_stream /* dev */, void* workspace,
                              size_t workspace_bytes, void* stream);

/* As cf_eval_plans / cf_goodput_bisect, but requests are read from a materialised stream instead
 * of being drawn in registers; results are bit-identical to the in-register calls with
 * variant = variant_lo + plan_variant. plan_variant: host [P] index in [0,n_variants) of the
 * stream variant plan p reads, or NULL for p % n_variants. */
int32_t cf_eval_plans_stream(const cf_graph* g, const cf_plans* pl, const uint32_t* rate_mrps,
                             uint32_t R, const cf_slo* slo, const void* stream_records /* dev */,
                             uint32_t n_variants, const uint32_t* plan_variant,
                             uint32_t* out_counts, uint64_t* out_dep_sum, int64_t* out_makespan,
                             void* workspace, size_t workspace_bytes, void* stream);
int32_t cf_goodput_bisect_stream(const cf_graph* g, const cf_plans* pl,
                                 const uint32_t* rate_hi_mrps, uint32_t n_steps, const cf_slo* slo,
                                 const void* stream_records /* dev */, uint32_t n_variants,
                                 const uint32_t* plan_variant, uint32_t* out_rate_mrps,
                                 uint32_t* out_goodput_mrps, uint32_t* out_counts, void* workspace,
                                 size_t workspace_bytes, void* stream);

/* Parity/debug: per-request trace of one simulation (plan, rate, trial): system arrival A_n,
 * final departure D_n and type, dev [N] each (any may be NULL). rate_mrps is a host value. */
int32_t cf_trace_sim(const cf_graph* g, const cf_plans* pl, uint32_t plan, uint32_t rate_mrps,
                     uint32_t trial, uint64_t seed, uint32_t variant, int64_t* out_arrival,
                     int64_t* out_departure, uint8_t* out_type, void* workspace,
                     size_t workspace_bytes, void* stream);

/* Synchronises `stream`, reads the sticky device status of the last call that used `workspace`
 * and returns it (CF_OK, CF_ERR_RANGE, or CF_ERR_CUDA). */
int32_t cf_workspace_status(const void* workspace, void* stream);

/* The simulation runs on a 32-bit fast kernel (times as uint32 offsets from a per-tile origin,
 * DESIGN.md 5.2) followed by the 64-bit kernel over exactly those simulations that left the 32-bit
 * window; results are bit-identical either way. cf_workspace_wide_count synchronises `stream` and
 * returns how many simulations of the last call on `workspace` were redone by the 64-bit kernel
 * (>= 0), or a negative cf_status. (Test and tuning hooks that force one path or the other live in
 * cf_debug.h; they are per-call arguments, not library state.) */
int64_t cf_workspace_wide_count(const void* workspace, void* stream);

/* Bench bookkeeping: synchronises `stream` and copies to out_probes (host, [n_plans]) how many
 * probes (simulated rates) lay on the bisection path of each plan in the last cf_goodput_bisect*
 * call on `workspace` (steps whose bracket had already closed are no-ops and do not count). */
int32_t cf_bisect_probes(const void* workspace, uint32_t n_plans, uint32_t* out_probes, void* stream);

/* ---- the cheap phases around the simulation (Algorithm 2 phases 1-2 and selection) --------------
 * They run on the device so that alpha R_d, goodput vectors and survivor flags pass from phase to
 * phase without leaving HBM. Integer definitions: DESIGN.md readings R20-R23. */

/* Scratch of cf_flow_bound / cf_mc_latency for (graph, plans); of cf_pareto_select. */
size_t cf_aux_workspace_bytes(const cf_graph* g, const cf_plans* pl);
size_t cf_pareto_workspace_bytes(void);

/* Phase 1, flow-based throughput estimation (Algorithm 2 l.1-5; sec. 4.3
 * PAPER.md:274-276). A node's demand per arriving request is sum_t pi_t * (mean service of type t on
 * the node's components), from the exact means of the quantile tables; "the node whose aggregate
 * demand first reaches its capacity is the bottleneck, and the aggregate request rate R_d at which
 * this occurs is plan d's maximum throughput"; "plans that configure a node with more capacity than
 * the node's aggregate demand are redundant".
 *   out_rate_mrps  dev [P]  min(floor(R_d * alpha_num / alpha_den), 1e9): the rate alpha R_d the later
 *                           phases evaluate; usable as cf_goodput_bisect's rate_hi_mrps
 *   out_bound_mrps dev [P]  R_d in milli-requests/s, capped at 1e9, or NULL
 *   out_bottleneck dev [P]  index of the bottleneck stage (lowest on ties; 0xff: no stage has demand), or NULL
 *   out_redundant  dev [P]  1 iff some stage with >= 2 replicas still sustains R_d with one fewer, or
 *                           has no demand at all (R22), or NULL
 * alpha_den >= 1. */
int32_t cf_flow_bound(const cf_graph* g, const cf_plans* pl, uint32_t alpha_num, uint32_t alpha_den,
                      uint32_t* out_rate_mrps, uint32_t* out_bound_mrps, uint8_t* out_bottleneck,
                      uint8_t* out_redundant, void* workspace, size_t workspace_bytes, void* stream);

/* Phase 2, latency estimation with Monte Carlo (Algorithm 2 l.6-11; sec. 4.3
 * PAPER.md:278): the K x N sampled requests of the simulation (same Philox counters, R4) are routed
 * through every plan; a request's latency is the sum of its sampled processing latencies along its
 * path plus edge_delay_us per hop; "queuing not modeled". F_{t,d}(L_t) = hits_t / cnt_t.
 *   rate_mrps        dev [P]  incoming rate alpha R_d of each plan (e.g. cf_flow_bound's out_rate_mrps)
 *   out_counts       dev [P][K][T][2] = {cnt_t, hits_t}, or NULL
 *   out_goodput_mrps dev [P][T] floor(rate * hits_t / (N K)), hits pooled over trials
 *                    (G_{t,d} = alpha R_d pi_t F_{t,d}(L_t), Algorithm 2 l.11, with the sampled mix) */
int32_t cf_mc_latency(const cf_graph* g, const cf_plans* pl, const uint32_t* rate_mrps, const cf_slo* slo,
                      uint64_t seed, uint32_t variant, uint32_t* out_counts, uint32_t* out_goodput_mrps,
                      void* workspace, size_t workspace_bytes, void* stream);

/* Pareto pruning of per-type goodput vectors and the default selection policy (Algorithm 2 l.12,
 * 16-18; sec. 4.3). Plan p is pruned iff it is not live or some
 * live plan q has G_q[t] >= G_p[t] for all t and G_q[t] > G_p[t] for one t (equal vectors do not
 * prune each other, R23). The policy picks the live plan with the largest sum_t G[t] (lowest index
 * on ties); it is never a pruned plan.
 *   goodput_mrps dev [P][T] (e.g. cf_mc_latency's or cf_goodput_bisect's output), T <= 8
 *   alive        dev [P] 0/1, or NULL (all live): chains the phases' survivor sets
 *   out_pruned   dev [P]; out_best dev [1] (0xffffffff if no plan is live) or NULL;
 *   out_n_survivors dev [1] or NULL */
int32_t cf_pareto_select(const uint32_t* goodput_mrps, uint32_t n_plans, uint32_t n_types,
                         const uint8_t* alive, uint8_t* out_pruned, uint32_t* out_best,
                         uint32_t* out_n_survivors, void* workspace, size_t workspace_bytes, void* stream);

/* cf_pareto_select for callers that cannot provide scratch because they cannot allocate device memory
 * (code under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc): same arguments
 * without the workspace, same results. Its scratch is a fixed array inside the library,
 * (32 + CF_PARETO_STATIC_MAX_PLANS) x 8 bytes = 512.25 KiB that every GPU which loads the library holds
 * until the process exits; n_plans > CF_PARETO_STATIC_MAX_PLANS returns CF_ERR_RANGE (and says so on
 * stderr) before anything is enqueued. The call allocates nothing (no cudaMalloc / cudaFree): three
 * kernel launches on `stream`, which must belong to the current device. All calls on a device share
 * the array: calls that may overlap on the GPU (different streams, concurrent graph branches) race on
 * it -- keep them on one stream or order them with events. */
#define CF_PARETO_STATIC_MAX_PLANS 65536u
uint32_t cf_pareto_static_max_plans(void);
int32_t cf_pareto_select_static(const uint32_t* goodput_mrps, uint32_t n_plans, uint32_t n_types,
                                const uint8_t* alive, uint8_t* out_pruned, uint32_t* out_best,
                                uint32_t* out_n_survivors, void* stream);

/* Releases the host-side cache of prepared calls (waits for uploads still in flight). */
void cf_cache_clear(void);

const char* cf_strerror(int32_t status);

#ifdef __cplusplus
}
#endif
#endif
