/*
 * cf_oracle_phases.cpp -- TEST INFRASTRUCTURE ONLY (see cf_oracle.h).
 *
 * Plain CPU statements of the cheap phases around the request-level simulation (SURVEY.md 8(f)
 * NEXT-1..3), in the paper's order and notation:
 *   phase 1, flow-based throughput estimation: Algorithm 2 l.1-5 and sec. 4.3
 *            "Network flow-based throughput estimation";
 *   phase 2, latency estimation with Monte Carlo: Algorithm 2 l.6-12 and sec. 4.3
 *            "Latency estimation with Monte Carlo";
 *   pruning + selection: Algorithm 2 l.12, 16-18, sec. 4.3.
 * Integer model and readings R20..R23: DESIGN.md section 3. Every loop is the definition written
 * out: no tables of partial results, no sorting, no early exits.
 *
 * Uses orc_philox4x32_10 / orc_qtab_sample of cf_oracle.cpp through their C interface only.
 */
#include "cf_oracle.h"

#include <algorithm>
#include <vector>

namespace {

typedef unsigned __int128 u128;


const uint64_t RATE_MAX = 1000000000ull;  /* largest valid rate, milli-requests/s (R5) */

/* Probability weight of type t in Q32 (R20): the type draw picks the first t with u < thresh[t],
 * else T-1, so P(t) = (thresh[t] - thresh[t-1]) / 2^32 and the last type takes the rest. */
uint64_t type_weight_q32(const orc_graph* g, uint32_t t) {
  const uint64_t hi = (t + 1 == g->n_types) ? (1ull << 32) : (uint64_t)g->type_thresh[t];
  const uint64_t lo = (t == 0) ? 0ull : (uint64_t)g->type_thresh[t - 1];
  return hi > lo ? hi - lo : 0ull;
}

/* Aggregate demand of stage (node) `mask` per arriving request, microseconds in Q16 (R21):
 * "the demands of all types passing through it are summed":
 * D = floor( sum_t w_t * sum_{i in mask & M_t} mean_q16(table of (i,t)) / 2^32 ). */
uint64_t stage_demand_q16(const orc_graph* g, uint8_t mask) {
  u128 D = 0;
  for (uint32_t t = 0; t < g->n_types; ++t) {
    uint64_t mu = 0;
    for (uint32_t i = 0; i < g->n_comp; ++i)
      if (((mask & g->type_mask[t]) >> i) & 1)
        mu += orc_qtab_mean_q16(&g->tabs[g->svc_tab[i * g->n_types + t]]);
    D += (u128)type_weight_q32(g, t) * mu;
  }
  return (uint64_t)(D >> 32);
}

/* R26: with routing, type t loads stage s of plan p only on the routes that include it:
 * D = floor( sum_t sum_r floor(w_t * q_{t,r} / 2^32) * sum_{i in mask & M_t} mean_q16(i,t) / 2^32 ),
 * q_{t,r} the route's probability in Q32 (the last route takes the rest). */
uint64_t routed_stage_demand_q16(const orc_graph* g, const orc_plans* pl, uint32_t p, uint32_t s) {
  const uint32_t T = g->n_types, MR = pl->max_routes;
  const uint8_t mask = pl->stage_mask[p * pl->max_stages + s];
  u128 D = 0;
  for (uint32_t t = 0; t < T; ++t) {
    uint64_t mu = 0;
    for (uint32_t i = 0; i < g->n_comp; ++i)
      if (((mask & g->type_mask[t]) >> i) & 1)
        mu += orc_qtab_mean_q16(&g->tabs[g->svc_tab[i * T + t]]);
    for (uint32_t r = 0; r < MR; ++r) {
      const size_t at = ((size_t)p * T + t) * MR + r;
      if (!((pl->route_mask[at] >> s) & 1)) continue;
      const uint64_t hi = (r + 1 == MR) ? (1ull << 32) : (uint64_t)pl->route_cum[at];
      const uint64_t lo = (r == 0) ? 0ull : (uint64_t)pl->route_cum[at - 1];
      const uint64_t q = hi > lo ? hi - lo : 0ull;
      const uint64_t pr = (uint64_t)(((u128)type_weight_q32(g, t) * q) >> 32);
      D += (u128)pr * mu;
    }
  }
  return (uint64_t)(D >> 32);
}

uint64_t demand_of(const orc_graph* g, const orc_plans* pl, uint32_t p, uint32_t s) {
  return pl->max_routes ? routed_stage_demand_q16(g, pl, p, s)
                        : stage_demand_q16(g, pl->stage_mask[p * pl->max_stages + s]);
}

/* Rate (milli-requests/s) at which c replicas saturate under demand Dq (Q16 us per request):
 * c / (Dq / 65536 us) requests per us = c * 65536 * 1e9 / Dq milli-requests per second. */
uint64_t saturation_mrps(uint64_t c, uint64_t Dq) { return c * 65536ull * 1000000000ull / Dq; }

}  // namespace

extern "C" {

/* Mean of the distribution a table induces, Q16 (R21): cell (k,m) has probability
 * w_k / 2^B (w_k = 2^-(k+1) below the cap level, 2^-(L-1) on it) and mean (q_i + q_{i+1}) / 2
 * (the sample is linear in the 16-bit fraction; its sub-unit floor is ignored). */
uint64_t orc_qtab_mean_q16(const orc_qtab* tab) {
  const uint32_t L = tab->levels, B = tab->log2_cells;
  u128 acc = 0; /* mean * 2^(L+B) */
  for (uint32_t k = 0; k < L; ++k) {
    uint64_t Tk = 0;
    for (uint32_t m = 0; m < (1u << B); ++m) {
      const size_t i = ((size_t)k << B) + m;
      Tk += (uint64_t)tab->q[i] + (uint64_t)tab->q[i + 1];
    }
    const uint32_t e = (k + 2 <= L) ? (L - 2 - k) : 0; /* w_k * 2^(L-1) = 2^e */
    acc += (u128)Tk << e;
  }
  const uint32_t s = L + B;
  return (uint64_t)(s >= 16 ? (acc >> (s - 16)) : (acc << (16 - s)));
}

/* Phase 1 (Algorithm 2 l.2-5): per plan the bottleneck node, R_d = the aggregate rate that
 * saturates it, the evaluated rate alpha * R_d and the redundant-capacity verdict
 * (R22: some node keeps at least R_d with one executor fewer, or has executors but no demand).
 * out_bottleneck: stage index, 0xff if no stage has any demand (then R_d is capped at 1e9). */
int32_t orc_flow_bound(const orc_graph* g, const orc_plans* pl, uint32_t alpha_num,
                       uint32_t alpha_den, uint32_t* out_rate_mrps, uint32_t* out_bound_mrps,
                       uint8_t* out_bottleneck, uint8_t* out_redundant) {
  if (int32_t rc = orc_validate(g, pl)) return rc;
  if (alpha_den == 0 || !out_rate_mrps) return ORC_ERR_ARG;
  for (uint32_t p = 0; p < pl->n_plans; ++p) {
    const uint32_t V = pl->n_stages[p];
    uint64_t R = UINT64_MAX;
    uint8_t bott = 0xff;
    for (uint32_t s = 0; s < V; ++s) {
      const uint64_t Dq = demand_of(g, pl, p, s);
      if (Dq == 0) continue; /* nothing flows through this node */
      const uint64_t r = saturation_mrps(pl->stage_c[p * pl->max_stages + s], Dq);
      if (r < R) { R = r; bott = (uint8_t)s; } /* the node whose demand first reaches capacity */
    }
    bool redundant = false;
    for (uint32_t s = 0; s < V; ++s) {
      const uint64_t c = pl->stage_c[p * pl->max_stages + s];
      if (c < 2) continue;
      const uint64_t Dq = demand_of(g, pl, p, s);
      if (Dq == 0 || saturation_mrps(c - 1, Dq) >= R) redundant = true;
    }
    const uint64_t bound = std::min<uint64_t>(R, RATE_MAX);
    out_rate_mrps[p] = (uint32_t)std::min<uint64_t>(bound * alpha_num / alpha_den, RATE_MAX);
    if (out_bound_mrps) out_bound_mrps[p] = (uint32_t)bound;
    if (out_bottleneck) out_bottleneck[p] = bott;
    if (out_redundant) out_redundant[p] = redundant ? 1 : 0;
  }
  return ORC_OK;
}

/* Phase 2 (Algorithm 2 l.6-11): every plan sees the same K x N sampled requests (the draws of
 * cf_oracle.cpp's simulate: common random numbers, R4); a request's latency is the sum of its
 * sampled processing latencies along its path plus the transfer delay per hop,
 * "queuing not modeled"; F_{t,d}(L_t) = hits_t / cnt_t and
 * G_{t,d} = floor(rate_d * hits_t / (N K)) (= alpha R_d * pi_t * F_{t,d}(L_t) with the sampled mix, R10).
 * With routes (R26) the path is the drawn route's; with fork-join (R25) the latency is the critical
 * path: a stage starts when its predecessor stages have finished (+ the delay of that edge). */
int32_t orc_mc_latency(const orc_graph* g, const orc_plans* pl, const uint32_t* rate_mrps,
                       const orc_slo* slo, uint64_t seed, uint32_t variant, uint32_t* out_counts,
                       uint32_t* out_goodput_mrps) {
  if (int32_t rc = orc_validate(g, pl)) return rc;
  if (!rate_mrps || !slo || !slo->L_us || !out_goodput_mrps) return ORC_ERR_ARG;
  const uint32_t C = g->n_comp, T = g->n_types, N = g->n_req, K = g->n_trials;
  const uint32_t key[2] = {(uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32)};
  for (uint32_t p = 0; p < pl->n_plans; ++p) {
    const uint8_t* smask = pl->stage_mask + (size_t)p * pl->max_stages;
    std::vector<uint64_t> pooled_hits(T, 0);
    for (uint32_t k = 0; k < K; ++k) {
      std::vector<uint32_t> cnt(T, 0), hits(T, 0);
      for (uint32_t n = 0; n < N; ++n) {
        uint32_t ctr[4] = {n, k, 0, variant}, b0[4];
        orc_philox4x32_10(ctr, key, b0);
        uint32_t t = T - 1;
        for (uint32_t tt = 0; tt < T; ++tt)
          if (b0[1] < g->type_thresh[tt]) { t = tt; break; }
        const uint8_t tm = g->type_mask[t];
        uint8_t route = 0xff; /* R26: the stages of the route this request drew */
        if (pl->max_routes > 0) {
          const uint32_t MR = pl->max_routes;
          uint32_t r = MR - 1;
          for (uint32_t rr = 0; rr < MR; ++rr)
            if (b0[2] < pl->route_cum[((size_t)p * T + t) * MR + rr]) { r = rr; break; }
          route = pl->route_mask[((size_t)p * T + t) * MR + r];
        }
        int64_t svc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
        for (uint32_t i = 0; i < C; ++i)
          if ((tm >> i) & 1) {
            uint32_t c2[4] = {n, k, 1 + i / 4, variant}, b[4];
            orc_philox4x32_10(c2, key, b);
            svc[i] = orc_qtab_sample(&g->tabs[g->svc_tab[i * T + t]], b[i % 4]);
            if (g->cpu_tab && g->cpu_tab[i * T + t] != 0xffff) { /* R24: nobody queues, so every executor is idle */
              uint32_t c3[4] = {n, k, 3 + i / 4, variant};
              orc_philox4x32_10(c3, key, b);
              svc[i] += orc_qtab_sample(&g->tabs[g->cpu_tab[i * T + t]], b[i % 4]);
            }
          }
        int64_t lat = 0; /* accumulated latency since the request's arrival, no waiting */
        bool first = true;
        int64_t done[8];
        bool visited[8] = {false, false, false, false, false, false, false, false};
        for (uint32_t s = 0; s < pl->n_stages[p]; ++s) {
          const uint8_t m = smask[s] & tm;
          if (m == 0 || !((route >> s) & 1)) continue;
          int64_t x; /* when the request reaches stage s */
          if (g->join_mode) { /* R25: after its last predecessor stage, plus that edge's delay */
            x = 0;
            for (uint32_t sp = 0; sp < s; ++sp) {
              if (!visited[sp]) continue;
              bool feeds = false;
              for (uint32_t e = 0; e < g->n_edges; ++e)
                if ((((smask[sp] & tm) >> g->edges[2 * e]) & 1) && ((m >> g->edges[2 * e + 1]) & 1)) feeds = true;
              if (feeds) x = std::max(x, done[sp] + g->edge_delay_us);
            }
          } else {
            x = lat + (first ? 0 : g->edge_delay_us);
          }
          first = false;
          for (uint32_t i = 0; i < C; ++i)
            if ((m >> i) & 1) x += svc[i];
          done[s] = x;
          visited[s] = true;
          lat = g->join_mode ? std::max(lat, x) : x; /* R25: done when the last branch is */
        }
        cnt[t]++;
        if (lat <= slo->L_us[t]) hits[t]++;
      }
      for (uint32_t t = 0; t < T; ++t) {
        pooled_hits[t] += hits[t];
        if (out_counts) {
          out_counts[(((size_t)p * K + k) * T + t) * 2 + 0] = cnt[t];
          out_counts[(((size_t)p * K + k) * T + t) * 2 + 1] = hits[t];
        }
      }
    }
    for (uint32_t t = 0; t < T; ++t)
      out_goodput_mrps[(size_t)p * T + t] =
          (uint32_t)(((u128)rate_mrps[p] * pooled_hits[t]) / ((uint64_t)N * K));
  }
  return ORC_OK;
}

/* Pruning and selection (Algorithm 2 l.12, 16-17): plan p is Pareto-suboptimal iff some live plan q
 * has G_q[t] >= G_p[t] for every type and G_q[t] > G_p[t] for one (R23: equal vectors do not prune
 * each other); the default policy picks the live plan with the largest sum of goodput across types
 * (lowest index on ties). alive == NULL: every plan is live. out_pruned[p] = 1 for plans that were
 * not live or are suboptimal. out_best = UINT32_MAX if nothing is live. */
int32_t orc_pareto_select(const uint32_t* goodput, uint32_t P, uint32_t T, const uint8_t* alive,
                          uint8_t* out_pruned, uint32_t* out_best, uint32_t* out_n_survivors) {
  if (!goodput || !out_pruned || P < 1 || T < 1 || T > 8) return ORC_ERR_ARG;
  uint32_t survivors = 0, best = UINT32_MAX;
  uint64_t best_sum = 0;
  for (uint32_t p = 0; p < P; ++p) {
    bool pruned = alive && !alive[p];
    for (uint32_t q = 0; q < P && !pruned; ++q) {
      if (q == p || (alive && !alive[q])) continue;
      bool ge_all = true, gt_any = false;
      for (uint32_t t = 0; t < T; ++t) {
        if (goodput[(size_t)q * T + t] < goodput[(size_t)p * T + t]) ge_all = false;
        if (goodput[(size_t)q * T + t] > goodput[(size_t)p * T + t]) gt_any = true;
      }
      if (ge_all && gt_any) pruned = true;
    }
    out_pruned[p] = pruned ? 1 : 0;
    if (alive && !alive[p]) continue;
    survivors += pruned ? 0 : 1;
    uint64_t sum = 0;
    for (uint32_t t = 0; t < T; ++t) sum += goodput[(size_t)p * T + t];
    if (best == UINT32_MAX || sum > best_sum) { best = p; best_sum = sum; }
  }
  if (out_best) *out_best = best;
  if (out_n_survivors) *out_n_survivors = survivors;
  return ORC_OK;
}

}  // extern "C"
