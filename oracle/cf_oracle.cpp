/*
 * cf_oracle.cpp -- TEST INFRASTRUCTURE ONLY (see cf_oracle.h).
 *
 * Sequential reference simulator. It follows, step by step and in the paper's order,
 *   - PAPER.md:280-286 (sec. 4.3 "Request-level simulation": run the workload at a given rate
 *     through a physical plan, produce per-type throughput and latency CDF),
 *   - PAPER.md:255 (Algorithm 2 l.15, G = R * F(L_t)), PAPER.md:322 (per-edge transfer delay),
 *   - PAPER.md:340 (maximum achievable goodput = highest supported rate),
 * with the fixed model BASELINE.json `north_star` prescribes where the paper is silent:
 * integer microseconds, counter-based Philox4x32-10 draws, Lindley D_n = max(A_n, D_{n-1}) + S_n
 * and the Kiefer-Wolfowitz sorted-vector recursion for c replicas. Readings R1..R19: DESIGN.md.
 *
 * Deliberately plain: one loop over requests, one loop over stages, a std::vector per stage that
 * is re-sorted after every update. No blocking, fusion, scan or shared generation of draws.
 */
#include "cf_oracle.h"

#include <algorithm>
#include <cstring>
#include <thread>
#include <vector>

namespace {

/* ---- Philox4x32-10, Salmon/Moraes/Dror/Shaw SC'11 (north_star's generator) ------------------ */
const uint32_t PHILOX_M0 = 0xD2511F53u, PHILOX_M1 = 0xCD9E8D57u;
const uint32_t PHILOX_W0 = 0x9E3779B9u, PHILOX_W1 = 0xBB67AE85u;

void philox(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1,
            uint32_t out[4]) {
  for (int round = 0; round < 10; ++round) {
    uint64_t p0 = (uint64_t)PHILOX_M0 * c0;
    uint64_t p1 = (uint64_t)PHILOX_M1 * c2;
    uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
    uint32_t n1 = (uint32_t)p1;
    uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
    uint32_t n3 = (uint32_t)p0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += PHILOX_W0; k1 += PHILOX_W1; /* key schedule between rounds */
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* ---- DESIGN.md R3: integer sample from a tail-refined quantile table ------------------------ */
int count_leading_ones(uint32_t u) {
  int k = 0;
  while (k < 32 && ((u >> (31 - k)) & 1u)) ++k;
  return k;
}

int64_t qtab_sample(const orc_qtab& tab, uint32_t u) {
  const int L = (int)tab.levels, B = (int)tab.log2_cells;
  int k = std::min(count_leading_ones(u), L - 1);
  /* drop the k leading ones and (below the cap level) the terminating zero; 32-bit, zero-filled */
  int drop = (k < L - 1) ? (k + 1) : (L - 1);
  uint32_t r = (drop >= 32) ? 0u : (u << drop);
  uint32_t m = (B == 0) ? 0u : (r >> (32 - B));  /* cell inside the level        */
  uint32_t f = (r >> (16 - B)) & 0xffffu;        /* 16-bit fraction inside cell  */
  uint32_t i = ((uint32_t)k << B) + m;
  int64_t q0 = tab.q[i], q1 = tab.q[i + 1];
  return q0 + (((q1 - q0) * (int64_t)f) >> 16);
}

size_t qtab_entries(const orc_qtab& t) { return ((size_t)t.levels << t.log2_cells) + 1; }

int32_t check_qtab(const orc_qtab& t) {
  if (t.q == nullptr || t.levels < 1 || t.levels > 32 || t.log2_cells > 16) return ORC_ERR_TABLE;
  size_t n = qtab_entries(t);
  if (t.q[0] < 0) return ORC_ERR_TABLE;
  for (size_t i = 1; i < n; ++i)
    if (t.q[i] < t.q[i - 1]) return ORC_ERR_TABLE;
  return ORC_OK;
}

const int64_t RANGE_LIMIT = (int64_t)1 << 62; /* DESIGN.md R17: arrivals must stay below 2^62 */

int32_t validate(const orc_graph* g, const orc_plans* pl) {
  if (!g || !pl) return ORC_ERR_ARG;
  const uint32_t C = g->n_comp, T = g->n_types;
  if (C < 1 || C > 8 || T < 1 || T > 8) return ORC_ERR_ARG;
  if (g->n_req < 1 || g->n_req > (1u << 24) || g->n_trials < 1) return ORC_ERR_ARG;
  if (!g->type_mask || !g->type_thresh || !g->svc_tab || !g->tabs || g->n_tabs < 1)
    return ORC_ERR_ARG;
  if (g->n_edges > 0 && !g->edges) return ORC_ERR_ARG;
  if (g->order_mode > 1) return ORC_ERR_ARG;
  for (uint32_t t = 0; t < T; ++t) {
    if (g->type_mask[t] >> C) return ORC_ERR_ARG;
    if (t > 0 && g->type_thresh[t] < g->type_thresh[t - 1]) return ORC_ERR_ARG;
  }
  for (uint32_t e = 0; e < g->n_edges; ++e)
    if (g->edges[2 * e] >= C || g->edges[2 * e + 1] >= C) return ORC_ERR_ARG;
  for (uint32_t i = 0; i < C; ++i)
    for (uint32_t t = 0; t < T; ++t) {
      if (((g->type_mask[t] >> i) & 1) && g->svc_tab[i * T + t] >= g->n_tabs) return ORC_ERR_ARG;
      if (g->cpu_tab && ((g->type_mask[t] >> i) & 1) && g->cpu_tab[i * T + t] != 0xffff &&
          g->cpu_tab[i * T + t] >= g->n_tabs)
        return ORC_ERR_ARG;
    }
  for (uint32_t j = 0; j < g->n_tabs; ++j)
    if (int32_t rc = check_qtab(g->tabs[j])) return rc;
  if (int32_t rc = check_qtab(g->arr_tab)) return rc;
  if (g->edge_delay_us < 0 || g->edge_delay_us >= ((int64_t)1 << 31)) return ORC_ERR_RANGE;
  /* R17: the largest possible service of a request (all components) must fit int32 */
  int64_t worst = 0;
  for (uint32_t i = 0; i < C; ++i) {
    int64_t mx = 0;
    for (uint32_t t = 0; t < T; ++t)
      if ((g->type_mask[t] >> i) & 1) {
        const orc_qtab& tb = g->tabs[g->svc_tab[i * T + t]];
        int64_t both = tb.q[qtab_entries(tb) - 1];
        if (g->cpu_tab && g->cpu_tab[i * T + t] != 0xffff) { /* R24: CPU + GPU time of an idle executor */
          const orc_qtab& tc = g->tabs[g->cpu_tab[i * T + t]];
          both += tc.q[qtab_entries(tc) - 1];
        }
        mx = std::max<int64_t>(mx, both);
      }
    worst += mx;
  }
  if (worst > INT32_MAX) return ORC_ERR_RANGE;

  if (pl->n_plans < 1 || pl->max_stages < 1 || pl->max_stages > 8) return ORC_ERR_ARG;
  if (!pl->n_stages || !pl->stage_mask || !pl->stage_c) return ORC_ERR_ARG;
  uint8_t used = 0;
  for (uint32_t t = 0; t < T; ++t) used |= g->type_mask[t];
  if (pl->max_routes > 4 || (pl->max_routes > 0 && (!pl->route_mask || !pl->route_cum))) return ORC_ERR_ARG;
  for (uint32_t p = 0; p < pl->n_plans && pl->max_routes > 0; ++p) { /* R26: plans with routing */
    const uint32_t V = pl->n_stages[p], MR = pl->max_routes;
    if (V < 1 || V > pl->max_stages) return ORC_ERR_PLAN;
    uint8_t all = 0;
    for (uint32_t s = 0; s < V; ++s) {
      const uint8_t m = pl->stage_mask[p * pl->max_stages + s];
      if (m == 0 || (m >> C) || pl->stage_c[p * pl->max_stages + s] < 1) return ORC_ERR_PLAN;
      all |= m;
    }
    if (used & ~all) return ORC_ERR_PLAN;
    for (uint32_t t = 0; t < T; ++t)
      for (uint32_t r = 0; r < MR; ++r) {
        const size_t at = ((size_t)p * T + t) * MR + r;
        if (r > 0 && pl->route_cum[at] < pl->route_cum[at - 1]) return ORC_ERR_PLAN;
        uint8_t seen = 0;
        int stage_of[8];
        for (int i = 0; i < 8; ++i) stage_of[i] = -1;
        for (uint32_t s = 0; s < V; ++s) {
          if (!((pl->route_mask[at] >> s) & 1)) continue;
          const uint8_t m = pl->stage_mask[p * pl->max_stages + s] & g->type_mask[t];
          if (m & seen) return ORC_ERR_PLAN; /* a component served twice along the route */
          seen |= m;
          for (uint32_t i = 0; i < C; ++i)
            if ((m >> i) & 1) stage_of[i] = (int)s;
        }
        if (seen != g->type_mask[t]) return ORC_ERR_PLAN; /* the route misses a component of the type */
        for (uint32_t e = 0; e < g->n_edges; ++e) {
          int su = stage_of[g->edges[2 * e]], sv = stage_of[g->edges[2 * e + 1]];
          if (su >= 0 && sv >= 0 && su > sv) return ORC_ERR_PLAN;
        }
      }
  }
  for (uint32_t p = 0; p < pl->n_plans && pl->max_routes == 0; ++p) {
    uint32_t V = pl->n_stages[p];
    if (V < 1 || V > pl->max_stages) return ORC_ERR_PLAN;
    uint8_t seen = 0;
    int stage_of[8];
    for (int i = 0; i < 8; ++i) stage_of[i] = -1;
    for (uint32_t s = 0; s < V; ++s) {
      uint8_t m = pl->stage_mask[p * pl->max_stages + s];
      if (m == 0 || (m >> C)) return ORC_ERR_PLAN;
      if (m & seen) return ORC_ERR_PLAN; /* overlap */
      seen |= m;
      if (pl->stage_c[p * pl->max_stages + s] < 1) return ORC_ERR_PLAN;
      for (uint32_t i = 0; i < C; ++i)
        if ((m >> i) & 1) stage_of[i] = (int)s;
    }
    if (used & ~seen) return ORC_ERR_PLAN; /* a used component has no stage */
    for (uint32_t e = 0; e < g->n_edges; ++e) {
      int su = stage_of[g->edges[2 * e]], sv = stage_of[g->edges[2 * e + 1]];
      if (su >= 0 && sv >= 0 && su > sv) return ORC_ERR_PLAN; /* order violates the DAG */
    }
  }
  return ORC_OK;
}

struct SimOut {
  uint32_t cnt[8], hits[8];
  uint64_t dep_sum;
  int64_t makespan;
  int32_t status;
};

/* One simulation with ARRIVAL-ORDER service (orc_graph.order_mode = 1; R27, SURVEY.md 8(f)
 * NEXT-4 "true stage-arrival-order FCFS", the discipline reading R2 departs from): every stage
 * serves its visitors in the order in which they REACH the stage, ties by request index -- textbook
 * FCFS at a c-server node. The plan's stages are in topological order and a request only moves
 * forward, so the arrivals at stage s are known once stages 0..s-1 are done: the stages are
 * processed one after another, each over all its visitors sorted by (arrival at the stage, index).
 * Same draws, same arrival times, same per-visit rule (Kiefer-Wolfowitz, idle/busy R24, hop delay
 * R9, routes R26, fork-join R25: a request reaches a stage when its predecessor stages are done) as
 * simulate(); only the order of service differs. */
void simulate_fcfs(const orc_graph* g, const orc_plans* pl, uint32_t p, uint32_t rate_mrps, uint32_t k,
                   const orc_slo* slo, uint64_t seed, uint32_t variant, SimOut* out,
                   int64_t* trace_arr, int64_t* trace_dep, uint8_t* trace_type) {
  std::memset(out, 0, sizeof(*out));
  const uint32_t C = g->n_comp, T = g->n_types, N = g->n_req;
  const uint32_t V = pl->n_stages[p];
  const uint8_t* smask = pl->stage_mask + (size_t)p * pl->max_stages;
  const uint16_t* sc = pl->stage_c + (size_t)p * pl->max_stages;
  if (rate_mrps < 1 || rate_mrps > 1000000000u) {
    out->status = ORC_ERR_RANGE;
    return;
  }
  const int64_t period_us = (int64_t)((1000000000ull + rate_mrps / 2) / rate_mrps);
  const uint32_t k0 = (uint32_t)(seed & 0xffffffffu), k1 = (uint32_t)(seed >> 32);
  /* the requests of the trial: the draws of simulate(), kept per request */
  std::vector<int64_t> A(N), x(N), svc((size_t)N * 8, 0), cpu((size_t)N * 8, 0);
  std::vector<uint8_t> type(N), route(N, 0xff), hops(N, 0), visited(N, 0);
  std::vector<int64_t> done(g->join_mode ? (size_t)N * 8 : 0, 0); /* R25: departure of request n from stage s */
  uint64_t CU = 0;
  for (uint32_t n = 0; n < N; ++n) {
    uint32_t b0[4];
    philox(n, k, 0, variant, k0, k1, b0);
    CU += (uint64_t)qtab_sample(g->arr_tab, b0[0]);
    unsigned __int128 wide = (unsigned __int128)CU * (uint64_t)period_us + 32768u;
    if (wide >= (unsigned __int128)RANGE_LIMIT) { /* R17 */
      out->status = ORC_ERR_RANGE;
      return;
    }
    A[n] = (int64_t)((CU * (uint64_t)period_us + 32768u) >> 16);
    uint32_t t = T - 1;
    for (uint32_t tt = 0; tt < T; ++tt)
      if (b0[1] < g->type_thresh[tt]) { t = tt; break; }
    type[n] = (uint8_t)t;
    if (pl->max_routes > 0) { /* R26 */
      const uint32_t MR = pl->max_routes;
      uint32_t r = MR - 1;
      for (uint32_t rr = 0; rr < MR; ++rr)
        if (b0[2] < pl->route_cum[((size_t)p * T + t) * MR + rr]) { r = rr; break; }
      route[n] = pl->route_mask[((size_t)p * T + t) * MR + r];
    }
    for (uint32_t i = 0; i < C; ++i)
      if ((g->type_mask[t] >> i) & 1) {
        uint32_t b[4];
        philox(n, k, 1 + i / 4, variant, k0, k1, b);
        svc[(size_t)n * 8 + i] = qtab_sample(g->tabs[g->svc_tab[i * T + t]], b[i % 4]);
        if (g->cpu_tab && g->cpu_tab[i * T + t] != 0xffff) { /* R24 */
          philox(n, k, 3 + i / 4, variant, k0, k1, b);
          cpu[(size_t)n * 8 + i] = qtab_sample(g->tabs[g->cpu_tab[i * T + t]], b[i % 4]);
        }
      }
    x[n] = A[n]; /* a request that visits no stage leaves at once (R14) */
  }
  for (uint32_t s = 0; s < V; ++s) { /* stages in the plan's (topological) order */
    std::vector<std::pair<int64_t, uint32_t>> order; /* (arrival at stage s, request index) */
    for (uint32_t n = 0; n < N; ++n) {
      const uint8_t m = smask[s] & g->type_mask[type[n]];
      if (m == 0 || !((route[n] >> s) & 1)) continue;
      if (g->join_mode) { /* R25: after every predecessor stage, plus that edge's delay; else at A_n */
        int64_t a = A[n];
        for (uint32_t sp = 0; sp < s; ++sp) {
          if (!((visited[n] >> sp) & 1)) continue;
          bool feeds = false;
          for (uint32_t e = 0; e < g->n_edges; ++e)
            if ((((smask[sp] & g->type_mask[type[n]]) >> g->edges[2 * e]) & 1) && ((m >> g->edges[2 * e + 1]) & 1)) feeds = true;
          if (feeds) a = std::max(a, done[(size_t)n * 8 + sp] + g->edge_delay_us);
        }
        order.emplace_back(a, n);
        continue;
      }
      order.emplace_back(x[n] + (hops[n] ? g->edge_delay_us : 0), n); /* R9: a hop delay after the first visit */
    }
    std::sort(order.begin(), order.end()); /* first come, first served; ties: lower index */
    std::vector<int64_t> F(sc[s], 0); /* free times of the c replicas, sorted ascending */
    for (const auto& e : order) {
      const int64_t a = e.first;
      const uint32_t n = e.second;
      const uint8_t m = smask[s] & g->type_mask[type[n]];
      int64_t S = 0, S_cpu = 0;
      for (uint32_t i = 0; i < C; ++i)
        if ((m >> i) & 1) { S += svc[(size_t)n * 8 + i]; S_cpu += cpu[(size_t)n * 8 + i]; }
      const int64_t f = F[0];
      int64_t d;
      if (f <= a) d = a + S_cpu + S; /* idle executor: CPU + GPU time */
      else d = f + S;                /* busy: GPU time alone */
      if (g->join_mode) { /* done when the last branch is */
        done[(size_t)n * 8 + s] = d;
        visited[n] |= (uint8_t)(1u << s);
        x[n] = std::max(x[n], d);
      } else {
        x[n] = d;
      }
      hops[n]++;
      F[0] = d;
      std::sort(F.begin(), F.end());
    }
  }
  for (uint32_t n = 0; n < N; ++n) {
    const uint32_t t = type[n];
    out->cnt[t]++;
    if (x[n] - A[n] <= slo->L_us[t]) out->hits[t]++;
    out->dep_sum += (uint64_t)x[n];
    out->makespan = std::max(out->makespan, x[n]);
    if (trace_arr) trace_arr[n] = A[n];
    if (trace_dep) trace_dep[n] = x[n];
    if (trace_type) trace_type[n] = (uint8_t)t;
  }
}

/* One simulation, SURVEY.md 8(c) / DESIGN.md "Algorithm", literally.
 * trace_*: optional [N] outputs. */
void simulate(const orc_graph* g, const orc_plans* pl, uint32_t p, uint32_t rate_mrps, uint32_t k,
              const orc_slo* slo, uint64_t seed, uint32_t variant, SimOut* out,
              int64_t* trace_arr, int64_t* trace_dep, uint8_t* trace_type) {
  if (g->order_mode) { /* R27: arrival-order service, stage by stage */
    simulate_fcfs(g, pl, p, rate_mrps, k, slo, seed, variant, out, trace_arr, trace_dep, trace_type);
    return;
  }
  std::memset(out, 0, sizeof(*out));
  const uint32_t C = g->n_comp, T = g->n_types, N = g->n_req;
  const uint32_t V = pl->n_stages[p];
  const uint8_t* smask = pl->stage_mask + (size_t)p * pl->max_stages;
  const uint16_t* sc = pl->stage_c + (size_t)p * pl->max_stages;
  if (rate_mrps < 1 || rate_mrps > 1000000000u) { /* R5/R17 */
    out->status = ORC_ERR_RANGE;
    return;
  }
  const int64_t period_us = (int64_t)((1000000000ull + rate_mrps / 2) / rate_mrps);
  const uint32_t k0 = (uint32_t)(seed & 0xffffffffu), k1 = (uint32_t)(seed >> 32);

  std::vector<std::vector<int64_t>> F(V); /* free times per stage, kept sorted ascending */
  for (uint32_t s = 0; s < V; ++s) F[s].assign(sc[s], 0);

  uint64_t CU = 0;
  for (uint32_t n = 0; n < N; ++n) {
    uint32_t b0[4];
    philox(n, k, 0, variant, k0, k1, b0);
    CU += (uint64_t)qtab_sample(g->arr_tab, b0[0]); /* first request arrives after one gap */
    unsigned __int128 wide = (unsigned __int128)CU * (uint64_t)period_us + 32768u;
    if (wide >= (unsigned __int128)RANGE_LIMIT) { /* R17: sim out of range -> all-zero outputs */
      std::memset(out, 0, sizeof(*out));
      out->status = ORC_ERR_RANGE;
      return;
    }
    const int64_t A = (int64_t)((CU * (uint64_t)period_us + 32768u) >> 16);
    uint32_t t = T - 1;
    for (uint32_t tt = 0; tt < T; ++tt)
      if (b0[1] < g->type_thresh[tt]) { t = tt; break; }
    const uint8_t tm = g->type_mask[t];
    uint8_t route = 0xff; /* R26: the stages this request may visit */
    if (pl->max_routes > 0) {
      const uint32_t MR = pl->max_routes;
      uint32_t r = MR - 1;
      for (uint32_t rr = 0; rr < MR; ++rr)
        if (b0[2] < pl->route_cum[((size_t)p * T + t) * MR + rr]) { r = rr; break; }
      route = pl->route_mask[((size_t)p * T + t) * MR + r];
    }
    int64_t svc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    int64_t cpu[8] = {0, 0, 0, 0, 0, 0, 0, 0}; /* R24: CPU pre-processing time, paid only at an idle executor */
    for (uint32_t i = 0; i < C; ++i)
      if ((tm >> i) & 1) {
        uint32_t b[4];
        philox(n, k, 1 + i / 4, variant, k0, k1, b);
        svc[i] = qtab_sample(g->tabs[g->svc_tab[i * T + t]], b[i % 4]);
        if (g->cpu_tab && g->cpu_tab[i * T + t] != 0xffff) {
          philox(n, k, 3 + i / 4, variant, k0, k1, b);
          cpu[i] = qtab_sample(g->tabs[g->cpu_tab[i * T + t]], b[i % 4]);
        }
      }
    int64_t x = A;
    bool first = true;
    int64_t done[8]; /* R25: departure of the request from every stage it has visited so far */
    bool visited[8] = {false, false, false, false, false, false, false, false};
    int64_t last = A;
    for (uint32_t s = 0; s < V; ++s) { /* stages in the plan's order */
      const uint8_t m = smask[s] & tm;
      if (m == 0 || !((route >> s) & 1)) continue;
      if (g->join_mode) {
        /* fork-join (Fig. 1: encoders feed the LLM): the request reaches stage s
         * when every predecessor stage -- one holding a component u of the request with a DAG
         * edge (u, v) into a component v of the request on stage s -- has finished, plus the
         * transfer delay of that edge; with no predecessor, at its system arrival. */
        x = A;
        for (uint32_t sp = 0; sp < s; ++sp) {
          if (!visited[sp]) continue;
          bool feeds = false;
          for (uint32_t e = 0; e < g->n_edges; ++e) {
            const uint32_t u = g->edges[2 * e], v = g->edges[2 * e + 1];
            if (((smask[sp] & tm) >> u) & 1 && ((m >> v) & 1)) feeds = true;
          }
          if (feeds) x = std::max(x, done[sp] + g->edge_delay_us);
        }
        first = true; /* the hop delay has been applied per edge above */
      }
      int64_t S = 0, S_cpu = 0;
      for (uint32_t i = 0; i < C; ++i)
        if ((m >> i) & 1) { S += svc[i]; S_cpu += cpu[i]; }
      if (!first) x += g->edge_delay_us;
      first = false;
      const int64_t f = F[s][0]; /* earliest-free replica */
      /* "When a request arrives at an idle multimodal encoder executor, it
       * experiences the full CPU + GPU time. However, when the encoder is already busy, CPU
       * preprocessing happens while the request is in the queue, and processing time reduces to
       * GPU time alone" -- idle: the executor is free at the request's arrival (f <= x). */
      if (f <= x) x = x + S_cpu + S;
      else x = f + S;
      done[s] = x;
      visited[s] = true;
      last = std::max(last, x);
      F[s][0] = x;
      std::sort(F[s].begin(), F[s].end());
    }
    if (g->join_mode) x = last; /* R25: the request is done when its last branch is */
    out->cnt[t]++;
    if (x - A <= slo->L_us[t]) out->hits[t]++;
    out->dep_sum += (uint64_t)x;
    out->makespan = std::max(out->makespan, x);
    if (trace_arr) trace_arr[n] = A;
    if (trace_dep) trace_dep[n] = x;
    if (trace_type) trace_type[n] = (uint8_t)t;
  }
}

template <class Fn>
void parallel_for(size_t n, int n_threads, Fn fn) {
  if (n_threads <= 1 || n <= 1) {
    for (size_t i = 0; i < n; ++i) fn(i);
    return;
  }
  std::vector<std::thread> th;
  size_t nt = std::min<size_t>((size_t)n_threads, n);
  for (size_t w = 0; w < nt; ++w)
    th.emplace_back([=] {
      for (size_t i = w; i < n; i += nt) fn(i);
    });
  for (auto& t : th) t.join();
}

}  // namespace

extern "C" {

void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  philox(ctr[0], ctr[1], ctr[2], ctr[3], key[0], key[1], out);
}

int64_t orc_qtab_sample(const orc_qtab* tab, uint32_t u) { return qtab_sample(*tab, u); }

int32_t orc_validate(const orc_graph* g, const orc_plans* pl) { return validate(g, pl); }

int32_t orc_eval_plans(const orc_graph* g, const orc_plans* pl, const uint32_t* rate_mrps,
                       uint32_t R, const orc_slo* slo, uint64_t seed, uint32_t variant,
                       uint32_t* out_counts, uint64_t* out_dep_sum, int64_t* out_makespan,
                       int32_t* out_sim_status, int32_t n_threads) {
  if (int32_t rc = validate(g, pl)) return rc;
  if (!rate_mrps || R < 1 || !slo || !slo->L_us || !out_counts) return ORC_ERR_ARG;
  const uint32_t P = pl->n_plans, K = g->n_trials, T = g->n_types;
  const size_t n_sims = (size_t)P * R * K;
  std::vector<int32_t> status(n_sims, 0);
  parallel_for(n_sims, n_threads, [&](size_t sim) {
    const uint32_t k = (uint32_t)(sim % K);
    const uint32_t r = (uint32_t)((sim / K) % R);
    const uint32_t p = (uint32_t)(sim / ((size_t)K * R));
    SimOut o;
    simulate(g, pl, p, rate_mrps[(size_t)p * R + r], k, slo, seed, variant, &o, nullptr, nullptr,
             nullptr);
    for (uint32_t t = 0; t < T; ++t) {
      out_counts[(sim * T + t) * 2 + 0] = o.cnt[t];
      out_counts[(sim * T + t) * 2 + 1] = o.hits[t];
    }
    if (out_dep_sum) out_dep_sum[sim] = o.dep_sum;
    if (out_makespan) out_makespan[sim] = o.makespan;
    status[sim] = o.status;
  });
  int32_t rc = ORC_OK;
  for (size_t i = 0; i < n_sims; ++i) {
    if (out_sim_status) out_sim_status[i] = status[i];
    if (status[i]) rc = ORC_ERR_RANGE;
  }
  return rc;
}

int32_t orc_goodput_bisect(const orc_graph* g, const orc_plans* pl, const uint32_t* rate_hi_mrps,
                           uint32_t n_steps, const orc_slo* slo, uint64_t seed, uint32_t variant,
                           uint32_t* out_rate_mrps, uint32_t* out_goodput_mrps,
                           uint32_t* out_counts, int32_t n_threads) {
  if (int32_t rc = validate(g, pl)) return rc;
  if (!rate_hi_mrps || !slo || !slo->L_us || !slo->att_num || !slo->att_den || !out_rate_mrps ||
      !out_goodput_mrps)
    return ORC_ERR_ARG;
  const uint32_t P = pl->n_plans, K = g->n_trials, T = g->n_types, N = g->n_req;
  std::vector<int32_t> prc(P, 0);
  parallel_for(P, n_threads, [&](size_t p) {
    uint32_t lo = 0, hi = rate_hi_mrps[p];
    std::vector<SimOut> at_lo(K), probe(K);
    for (uint32_t k = 0; k < K; ++k) std::memset(&at_lo[k], 0, sizeof(SimOut));
    for (uint32_t step = 0; step < n_steps; ++step) {
      const uint32_t mid = lo + (hi - lo) / 2;
      if (mid == lo) continue; /* bracket closed: the step is a no-op */
      bool in_range = true;
      uint64_t cnt[8] = {0}, hits[8] = {0};
      for (uint32_t k = 0; k < K; ++k) {
        simulate(g, pl, (uint32_t)p, mid, k, slo, seed, variant, &probe[k], nullptr, nullptr,
                 nullptr);
        if (probe[k].status) in_range = false;
        for (uint32_t t = 0; t < T; ++t) { cnt[t] += probe[k].cnt[t]; hits[t] += probe[k].hits[t]; }
      }
      bool feasible = in_range; /* R18: an out-of-range probe counts as infeasible */
      if (!in_range) prc[p] = ORC_ERR_RANGE;
      for (uint32_t t = 0; t < T && feasible; ++t)
        if (cnt[t] > 0 && hits[t] * (uint64_t)slo->att_den[t] < (uint64_t)slo->att_num[t] * cnt[t])
          feasible = false;
      if (feasible) { lo = mid; at_lo = probe; } else { hi = mid; }
    }
    out_rate_mrps[p] = lo;
    for (uint32_t t = 0; t < T; ++t) {
      uint64_t h = 0;
      for (uint32_t k = 0; k < K; ++k) h += at_lo[k].hits[t];
      out_goodput_mrps[p * T + t] = (uint32_t)(((uint64_t)lo * h) / ((uint64_t)N * K));
    }
    if (out_counts)
      for (uint32_t k = 0; k < K; ++k)
        for (uint32_t t = 0; t < T; ++t) {
          out_counts[(((size_t)p * K + k) * T + t) * 2 + 0] = at_lo[k].cnt[t];
          out_counts[(((size_t)p * K + k) * T + t) * 2 + 1] = at_lo[k].hits[t];
        }
  });
  for (uint32_t p = 0; p < P; ++p)
    if (prc[p]) return prc[p];
  return ORC_OK;
}

int32_t orc_trace_sim(const orc_graph* g, const orc_plans* pl, uint32_t plan, uint32_t rate_mrps,
                      uint32_t trial, uint64_t seed, uint32_t variant, int64_t* out_arrival,
                      int64_t* out_departure, uint8_t* out_type) {
  if (int32_t rc = validate(g, pl)) return rc;
  if (plan >= pl->n_plans || trial >= g->n_trials) return ORC_ERR_ARG;
  /* trace does not need an SLO; use a zero one */
  int64_t L[8] = {0};
  orc_slo slo = {L, nullptr, nullptr};
  SimOut o;
  simulate(g, pl, plan, rate_mrps, trial, &slo, seed, variant, &o, out_arrival, out_departure,
           out_type);
  return o.status;
}

int32_t orc_materialize_stream(const orc_graph* g, uint64_t seed, uint32_t variant_lo,
                               uint32_t n_variants, void* out) {
  if (!g || !out || g->n_comp < 1 || g->n_comp > 6 || g->n_types < 1 || g->n_types > 8 || g->cpu_tab)
    return ORC_ERR_ARG; /* the 32-byte record has no room for CPU times (R24) */
  const uint32_t C = g->n_comp, T = g->n_types, N = g->n_req, K = g->n_trials;
  const uint32_t k0 = (uint32_t)(seed & 0xffffffffu), k1 = (uint32_t)(seed >> 32);
  uint8_t* dst = (uint8_t*)out;
  for (uint32_t vi = 0; vi < n_variants; ++vi) {
    const uint32_t variant = variant_lo + vi;
    for (uint32_t k = 0; k < K; ++k) {
      uint64_t CU = 0;
      for (uint32_t n = 0; n < N; ++n) {
        uint32_t b0[4];
        philox(n, k, 0, variant, k0, k1, b0);
        CU += (uint64_t)qtab_sample(g->arr_tab, b0[0]);
        uint32_t t = T - 1;
        for (uint32_t tt = 0; tt < T; ++tt)
          if (b0[1] < g->type_thresh[tt]) { t = tt; break; }
        int32_t svc[6] = {0, 0, 0, 0, 0, 0};
        for (uint32_t i = 0; i < C; ++i)
          if ((g->type_mask[t] >> i) & 1) {
            uint32_t b[4];
            philox(n, k, 1 + i / 4, variant, k0, k1, b);
            svc[i] = (int32_t)qtab_sample(g->tabs[g->svc_tab[i * T + t]], b[i % 4]);
          }
        uint64_t head = CU | ((uint64_t)t << 56);
        std::memcpy(dst, &head, 8);
        std::memcpy(dst + 8, svc, 24);
        dst += 32;
      }
    }
  }
  return ORC_OK;
}

}  // extern "C"
