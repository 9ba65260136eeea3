// cf_aux.cuh -- kernels of the cheap phases around the request-level simulation (sm_100a):
//   phase 1  flow-based throughput estimation, Algorithm 2 l.1-5:
//            exact table means -> demand of every possible node (component mask) -> per plan the
//            bottleneck node, R_d, alpha R_d and the redundant-capacity verdict;
//   phase 2  Monte-Carlo latency estimation, Algorithm 2 l.6-11;
//   pruning + selection, Algorithm 2 l.12, 16-18.
// Integer model: DESIGN.md readings R20-R23. All of it is HBM/latency-trivial next to phase 3; the
// point of running it on the device is that rate_hi, goodput vectors and the survivor set never
// leave HBM between the phases.
//
// B200-first restructuring of phase 2: with common random numbers (R4) and service tables that do
// not depend on the plan, a request's accumulated latency depends on the plan only through the
// number of hops h between the stages it visits: latency = (sum of its component services) + h * delay.
// So the K x N sampled requests are drawn ONCE into a histogram hits[k][t][h], h = 0..7, and every
// plan then reads its answer with one lookup per type: 10^6 plans cost one pass over 2 M requests
// plus 8 M lookups, where a per-plan loop (the oracle, the paper's 17.6 us per plan) redraws them.
#pragma once
#include "cf_device.cuh"

namespace cfk {

struct U128 {
  uint64_t lo, hi;
};
__device__ __forceinline__ void u128_add(U128& a, uint64_t lo, uint64_t hi) {
  a.lo += lo;
  a.hi += hi + (a.lo < lo ? 1ull : 0ull);
}
__device__ __forceinline__ void u128_add_shl(U128& a, uint64_t v, uint32_t e) {  // a += v << e, e < 64
  u128_add(a, v << e, e ? v >> (64u - e) : 0ull);
}
__device__ __forceinline__ void u128_add_mul(U128& a, uint64_t x, uint64_t y) {  // a += x * y
  u128_add(a, x * y, __umul64hi(x, y));
}
// floor((hi:lo) / d) for a quotient that fits 64 bits (hi < d): binary long division
__device__ __forceinline__ uint64_t u128_div(uint64_t hi, uint64_t lo, uint64_t d) {
  if (hi == 0) return lo / d;
  uint64_t q = 0, r = hi;
  for (int i = 63; i >= 0; --i) {
    const bool top = (r >> 63) != 0;
    r = (r << 1) | ((lo >> i) & 1ull);
    if (top || r >= d) { r -= d; q |= 1ull << i; }
  }
  return q;
}

struct AuxParams {
  uint32_t C, T, N, K, P, MS;
  uint32_t type_thresh[8];
  uint8_t type_mask[8];
  DevTab svc_tab[64];   // [i*8 + t]
  DevTab cpu_tab[64];   // [i*8 + t] CPU pre-processing time (R24); levels == 0: none
  uint32_t tab_id[64];  // table id of (i, t): index into mean_q16
  const int32_t* qpool;
  const DevTab* tabs;   // [n_tabs]
  uint32_t n_tabs;
  int64_t L_us[8];
  int64_t edge_delay;
  uint32_t seed_lo, seed_hi, variant;
  uint32_t alpha_num, alpha_den;
  const uint8_t* n_stages;    // [P]
  const uint8_t* stage_mask;  // [P*MS]
  const uint16_t* stage_c;    // [P*MS]
  uint32_t max_routes;        // R26: 0 = none
  const uint8_t* route_mask;  // [P*T*max_routes]
  const uint32_t* route_cum;  // [P*T*max_routes]
  uint64_t* mean_q16;         // [n_tabs]
  uint64_t* demand_q16;       // [256] demand of the node with component mask m
  uint32_t* hist;             // [K][8][9]: hits for h = 0..7 hops, [8] = requests of the type
  uint32_t join;              // R25: fork-join along the DAG edges (generic Monte-Carlo kernel)
  uint8_t edge_to[8];         // edge_to[u] = bitmask of the components v with a DAG edge (u, v)
};

// ---- phase 1 -----------------------------------------------------------------------------------
// R21: mean of the distribution a table induces, Q16. One block per table; level k's cell sums are
// reduced by the block, thread 0 accumulates mean * 2^(L+B) in 128 bits.
__global__ void __launch_bounds__(256) flow_tabmean_kernel(const __grid_constant__ AuxParams prm) {
  __shared__ uint64_t part[8];
  const DevTab tb = prm.tabs[blockIdx.x];
  const uint32_t L = tb.levels, B = tb.log2_cells;
  const int32_t* q = prm.qpool + tb.off;
  U128 acc{0, 0};
  for (uint32_t k = 0; k < L; ++k) {
    uint64_t s = 0;
    for (uint32_t m = threadIdx.x; m < (1u << B); m += 256) {
      const size_t i = ((size_t)k << B) + m;
      s += (uint64_t)(uint32_t)q[i] + (uint64_t)(uint32_t)q[i + 1];
    }
#pragma unroll
    for (int d = 16; d >= 1; d >>= 1) s += __shfl_xor_sync(0xffffffffu, s, d);
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
      uint64_t Tk = 0;
      for (int w = 0; w < 8; ++w) Tk += part[w];
      u128_add_shl(acc, Tk, (k + 2 <= L) ? (L - 2 - k) : 0u);  // w_k * 2^(L-1)
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    const uint32_t s = L + B;
    uint64_t r;
    if (s >= 16) {
      const uint32_t sh = s - 16;  // <= 32
      r = sh ? ((acc.lo >> sh) | (acc.hi << (64u - sh))) : acc.lo;
    } else {
      r = acc.lo << (16 - s);
    }
    prm.mean_q16[blockIdx.x] = r;
  }
}

// R20/R21: aggregate demand per arriving request of the node holding component set m, Q16 us
__global__ void __launch_bounds__(256) flow_demand_kernel(const __grid_constant__ AuxParams prm) {
  const uint32_t m = threadIdx.x;  // one thread per component mask
  U128 D{0, 0};
  for (uint32_t t = 0; t < prm.T; ++t) {
    const uint64_t hi = (t + 1 == prm.T) ? (1ull << 32) : (uint64_t)prm.type_thresh[t];
    const uint64_t lo = t == 0 ? 0ull : (uint64_t)prm.type_thresh[t - 1];
    const uint64_t w = hi > lo ? hi - lo : 0ull;
    uint64_t mu = 0;
    for (uint32_t i = 0; i < prm.C; ++i)
      if (((m & prm.type_mask[t]) >> i) & 1u) mu += prm.mean_q16[prm.tab_id[i * 8 + t]];
    u128_add_mul(D, w, mu);
  }
  prm.demand_q16[m] = (D.lo >> 32) | (D.hi << 32);
}

__device__ __forceinline__ uint64_t saturation_mrps(uint64_t c, uint64_t Dq) {
  return c * 65536ull * 1000000000ull / Dq;
}

// R26: demand of stage s of plan p when types reach it only on some of their routes
__device__ __forceinline__ uint64_t routed_demand_q16(const AuxParams& prm, uint32_t p, uint32_t s) {
  const uint32_t mask = prm.stage_mask[(size_t)p * prm.MS + s], MR = prm.max_routes;
  U128 D{0, 0};
  for (uint32_t t = 0; t < prm.T; ++t) {
    const uint64_t thi = (t + 1 == prm.T) ? (1ull << 32) : (uint64_t)prm.type_thresh[t];
    const uint64_t tlo = t == 0 ? 0ull : (uint64_t)prm.type_thresh[t - 1];
    const uint64_t w = thi > tlo ? thi - tlo : 0ull;
    uint64_t mu = 0;
    for (uint32_t i = 0; i < prm.C; ++i)
      if (((mask & prm.type_mask[t]) >> i) & 1u) mu += prm.mean_q16[prm.tab_id[i * 8 + t]];
    for (uint32_t r = 0; r < MR; ++r) {
      const size_t at = ((size_t)p * prm.T + t) * MR + r;
      if (!((prm.route_mask[at] >> s) & 1u)) continue;
      const uint64_t hi = (r + 1 == MR) ? (1ull << 32) : (uint64_t)prm.route_cum[at];
      const uint64_t lo = r == 0 ? 0ull : (uint64_t)prm.route_cum[at - 1];
      const uint64_t q = hi > lo ? hi - lo : 0ull;
      // floor(w * q / 2^32): w, q <= 2^32, so the product needs 65 bits at most
      const uint64_t pl = w * q, ph = __umul64hi(w, q);
      const uint64_t pr = (pl >> 32) | (ph << 32);
      u128_add_mul(D, pr, mu);
    }
  }
  return (D.lo >> 32) | (D.hi << 32);
}

__global__ void __launch_bounds__(128)
flow_plan_kernel(const __grid_constant__ AuxParams prm, uint32_t* out_rate, uint32_t* out_bound,
                 uint8_t* out_bottleneck, uint8_t* out_redundant) {
  const uint32_t p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= prm.P) return;
  const uint32_t V = prm.n_stages[p];
  uint64_t R = UINT64_MAX;
  uint32_t bott = 0xffu;
  for (uint32_t s = 0; s < V; ++s) {
    const uint64_t Dq = prm.max_routes ? routed_demand_q16(prm, p, s) : prm.demand_q16[prm.stage_mask[(size_t)p * prm.MS + s]];
    if (Dq == 0) continue;
    const uint64_t r = saturation_mrps(prm.stage_c[(size_t)p * prm.MS + s], Dq);
    if (r < R) { R = r; bott = s; }
  }
  bool redundant = false;  // R22
  for (uint32_t s = 0; s < V; ++s) {
    const uint64_t c = prm.stage_c[(size_t)p * prm.MS + s];
    if (c < 2) continue;
    const uint64_t Dq = prm.max_routes ? routed_demand_q16(prm, p, s) : prm.demand_q16[prm.stage_mask[(size_t)p * prm.MS + s]];
    if (Dq == 0 || saturation_mrps(c - 1, Dq) >= R) redundant = true;
  }
  const uint64_t bound = R < 1000000000ull ? R : 1000000000ull;
  const uint64_t rate = bound * prm.alpha_num / prm.alpha_den;
  out_rate[p] = (uint32_t)(rate < 1000000000ull ? rate : 1000000000ull);
  if (out_bound) out_bound[p] = (uint32_t)bound;
  if (out_bottleneck) out_bottleneck[p] = (uint8_t)bott;
  if (out_redundant) out_redundant[p] = redundant ? 1 : 0;
}

// ---- phase 2 -----------------------------------------------------------------------------------
// one thread per sampled request (n, trial k): the draws of the simulation kernels' producer
__global__ void __launch_bounds__(256) mc_hist_kernel(const __grid_constant__ AuxParams prm) {
  __shared__ uint32_t h_s[8 * 9];
  for (int i = threadIdx.x; i < 72; i += 256) h_s[i] = 0;
  __syncthreads();
  const uint32_t n = blockIdx.x * 256 + threadIdx.x, trial = blockIdx.y;
  if (n < prm.N) {
    const uint4 b0 = philox4x32_10(n, trial, 0, prm.variant, prm.seed_lo, prm.seed_hi);
    uint32_t t = prm.T - 1;
    for (int tt = (int)prm.T - 2; tt >= 0; --tt)
      if (b0.y < prm.type_thresh[tt]) t = tt;
    const uint32_t tm = prm.type_mask[t];
    int64_t total = 0;  // sum of the request's component services (every component sits on one stage)
    if (tm & 0x0fu) {
      const uint4 b1 = philox4x32_10(n, trial, 1, prm.variant, prm.seed_lo, prm.seed_hi);
      if (tm & 1u) total += qtab_sample(prm.qpool, prm.svc_tab[0 * 8 + t], b1.x);
      if (tm & 2u) total += qtab_sample(prm.qpool, prm.svc_tab[1 * 8 + t], b1.y);
      if (tm & 4u) total += qtab_sample(prm.qpool, prm.svc_tab[2 * 8 + t], b1.z);
      if (tm & 8u) total += qtab_sample(prm.qpool, prm.svc_tab[3 * 8 + t], b1.w);
    }
    if (tm & 0xf0u) {
      const uint4 b2 = philox4x32_10(n, trial, 2, prm.variant, prm.seed_lo, prm.seed_hi);
      if (tm & 16u) total += qtab_sample(prm.qpool, prm.svc_tab[4 * 8 + t], b2.x);
      if (tm & 32u) total += qtab_sample(prm.qpool, prm.svc_tab[5 * 8 + t], b2.y);
      if (tm & 64u) total += qtab_sample(prm.qpool, prm.svc_tab[6 * 8 + t], b2.z);
      if (tm & 128u) total += qtab_sample(prm.qpool, prm.svc_tab[7 * 8 + t], b2.w);
    }
    // R24: nobody queues, so every executor is idle at every arrival: CPU time on top (blocks 3 + i/4)
    uint32_t lo = 0, hi = 0;
    for (uint32_t i = 0; i < prm.C; ++i)
      if (((tm >> i) & 1u) && prm.cpu_tab[i * 8 + t].levels) { if (i < 4) lo = 1; else hi = 1; }
    if (lo) {
      const uint4 b3 = philox4x32_10(n, trial, 3, prm.variant, prm.seed_lo, prm.seed_hi);
      const uint32_t u[4] = {b3.x, b3.y, b3.z, b3.w};
      for (uint32_t i = 0; i < 4 && i < prm.C; ++i)
        if (((tm >> i) & 1u) && prm.cpu_tab[i * 8 + t].levels) total += qtab_sample(prm.qpool, prm.cpu_tab[i * 8 + t], u[i]);
    }
    if (hi) {
      const uint4 b4 = philox4x32_10(n, trial, 4, prm.variant, prm.seed_lo, prm.seed_hi);
      const uint32_t u[4] = {b4.x, b4.y, b4.z, b4.w};
      for (uint32_t i = 4; i < prm.C; ++i)
        if (((tm >> i) & 1u) && prm.cpu_tab[i * 8 + t].levels) total += qtab_sample(prm.qpool, prm.cpu_tab[i * 8 + t], u[i - 4]);
    }
    atomicAdd(&h_s[t * 9 + 8], 1u);
    const int64_t L = prm.L_us[t];
#pragma unroll
    for (int h = 0; h < 8; ++h)
      if (total + (int64_t)h * prm.edge_delay <= L) atomicAdd(&h_s[t * 9 + h], 1u);
  }
  __syncthreads();
  for (int i = threadIdx.x; i < 72; i += 256)
    if (h_s[i]) atomicAdd(&prm.hist[(size_t)trial * 72 + i], h_s[i]);
}

__global__ void __launch_bounds__(128)
mc_plan_kernel(const __grid_constant__ AuxParams prm, const uint32_t* rate_mrps, uint32_t* out_counts,
               uint32_t* out_goodput) {
  const uint32_t p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= prm.P) return;
  const uint32_t V = prm.n_stages[p];
  const uint64_t rate = rate_mrps[p], nk = (uint64_t)prm.N * prm.K;
  for (uint32_t t = 0; t < prm.T; ++t) {
    uint32_t nvis = 0;
    for (uint32_t s = 0; s < V; ++s)
      if (prm.stage_mask[(size_t)p * prm.MS + s] & prm.type_mask[t]) ++nvis;
    const uint32_t h = nvis ? nvis - 1 : 0;  // hops between the visited stages
    uint64_t hits = 0;
    for (uint32_t k = 0; k < prm.K; ++k) {
      const uint32_t c = prm.hist[(size_t)k * 72 + t * 9 + 8], hh = prm.hist[(size_t)k * 72 + t * 9 + h];
      hits += hh;
      if (out_counts) {
        out_counts[(((size_t)p * prm.K + k) * prm.T + t) * 2 + 0] = c;
        out_counts[(((size_t)p * prm.K + k) * prm.T + t) * 2 + 1] = hh;
      }
    }
    out_goodput[(size_t)p * prm.T + t] = (uint32_t)u128_div(__umul64hi(rate, hits), rate * hits, nk);
  }
}

// Phase 2 for plans whose latency is not "services + hops x delay of the type": routed plans (R26: the
// path depends on the request's route draw against the PLAN's probabilities) and fork-join graphs
// (R25: the latency is the critical path over the request's stages). One block per (plan, trial)
// walks the trial's request records (drawn once per call by the kernels of cf_fcfs.cuh, shared by
// all plans: common random numbers) and accumulates every request's latency without queueing.
template <int CMAX, bool HAS_CPU>
__global__ void __launch_bounds__(256)
mc_generic_kernel(const __grid_constant__ AuxParams prm, const uint4* __restrict__ records,
                  unsigned long long* pooled_hits, uint32_t* out_counts) {
  constexpr int kW = CompRec<CMAX, HAS_CPU>::kWords;
  constexpr int kB = CompRec<CMAX, HAS_CPU>::kBase;
  __shared__ uint32_t cnt_s[8][2];
  __shared__ uint8_t smask_s[8], feeds_s[8][8], rmask_s[8][4];
  __shared__ uint32_t rcum_s[8][4];
  const uint32_t p = blockIdx.x, k = blockIdx.y, tid = threadIdx.x, lane = tid & 31u;
  const uint32_t V = prm.n_stages[p], MR = prm.max_routes;
  if (tid < 16) cnt_s[tid >> 1][tid & 1] = 0;
  if (tid < 8) smask_s[tid] = tid < V ? prm.stage_mask[(size_t)p * prm.MS + tid] : 0;
  if (tid < 32 && MR) {
    const uint32_t t = tid >> 2, r = tid & 3u;
    const bool has = t < prm.T && r < MR;
    rcum_s[t][r] = has ? prm.route_cum[((size_t)p * prm.T + t) * MR + r] : 0xffffffffu;
    rmask_s[t][r] = has ? prm.route_mask[((size_t)p * prm.T + t) * MR + r] : 0;
  }
  __syncthreads();
  if (tid < 64) {  // feeds[t][s]: the stages before s holding a component of type t with an edge into one on s
    const uint32_t t = tid >> 3, s = tid & 7u, tm = prm.type_mask[t];
    uint32_t pm = 0;
    const uint32_t ms = smask_s[s] & tm;
    for (uint32_t sp = 0; sp < s; ++sp) {
      const uint32_t mp = smask_s[sp] & tm;
      for (uint32_t u = 0; u < prm.C; ++u)
        if (((mp >> u) & 1u) && (prm.edge_to[u] & ms)) pm |= 1u << sp;
    }
    feeds_s[t][s] = (uint8_t)pm;
  }
  __syncthreads();
  const int64_t delay = prm.edge_delay;
  const uint4* recs = records + (size_t)k * prm.N * kW;
  for (uint32_t base = 0; base < prm.N; base += 256) {
    const uint32_t n = base + tid;
    const bool valid = n < prm.N;
    const uint4* src = recs + (size_t)min(n, prm.N - 1u) * kW;
    const uint4 w0 = __ldg(src), w1 = __ldg(src + 1);
    uint4 w2 = make_uint4(0, 0, 0, 0);
    if (CMAX > 6) w2 = __ldg(src + 2);
    const uint32_t t = w0.y >> 24, tm = prm.type_mask[t];
    int64_t svc[8];
    svc[0] = (int32_t)w0.z; svc[1] = (int32_t)w0.w; svc[2] = (int32_t)w1.x; svc[3] = (int32_t)w1.y;
    svc[4] = (int32_t)w1.z; svc[5] = (int32_t)w1.w; svc[6] = (int32_t)w2.x; svc[7] = (int32_t)w2.y;
    if (HAS_CPU) {  // R24: nobody queues, so every executor is idle at every arrival
      const uint4 c0 = __ldg(src + kB), c1 = __ldg(src + kB + 1);
      svc[0] += (int32_t)c0.x; svc[1] += (int32_t)c0.y; svc[2] += (int32_t)c0.z; svc[3] += (int32_t)c0.w;
      svc[4] += (int32_t)c1.x; svc[5] += (int32_t)c1.y; svc[6] += (int32_t)c1.z; svc[7] += (int32_t)c1.w;
    }
    uint32_t rmask = 0xffu;
    if (MR) {  // R26: first route with u < cum, the last one takes the rest
      uint32_t r = MR - 1u;
      for (int rr = (int)MR - 2; rr >= 0; --rr)
        if (w2.z < rcum_s[t][rr]) r = (uint32_t)rr;
      rmask = rmask_s[t][r];
    }
    int64_t lat = 0, fin[8];
    uint32_t vm = 0;
#pragma unroll
    for (int s = 0; s < 8; ++s) {
      fin[s] = 0;
      const uint32_t m = smask_s[s] & tm;
      if (m != 0u && ((rmask >> s) & 1u)) {
        int64_t x;
        if (prm.join) {  // R25: after the last predecessor stage, plus that edge's delay
          x = 0;
          const uint32_t pm = feeds_s[t][s] & vm;
#pragma unroll
          for (int sp = 0; sp < s; ++sp)
            if ((pm >> sp) & 1u) x = max(x, fin[sp] + delay);
        } else {
          x = lat + (vm ? delay : 0);
        }
#pragma unroll
        for (int i = 0; i < CMAX; ++i)
          if ((m >> i) & 1u) x += svc[i];
        fin[s] = x;
        vm |= 1u << s;
        lat = prm.join ? max(lat, x) : x;
      }
    }
    const bool hit = valid && lat <= prm.L_us[t];
    for (uint32_t tt = 0; tt < prm.T; ++tt) {
      const uint32_t mc = __ballot_sync(0xffffffffu, valid && t == tt);
      const uint32_t mh = __ballot_sync(0xffffffffu, hit && t == tt);
      if (lane == 0 && mc) { atomicAdd(&cnt_s[tt][0], __popc(mc)); if (mh) atomicAdd(&cnt_s[tt][1], __popc(mh)); }
    }
  }
  __syncthreads();
  if (tid < prm.T) {
    if (out_counts) {
      out_counts[(((size_t)p * prm.K + k) * prm.T + tid) * 2 + 0] = cnt_s[tid][0];
      out_counts[(((size_t)p * prm.K + k) * prm.T + tid) * 2 + 1] = cnt_s[tid][1];
    }
    atomicAdd(&pooled_hits[(size_t)p * prm.T + tid], (unsigned long long)cnt_s[tid][1]);
  }
}

__global__ void __launch_bounds__(128)
mc_generic_final_kernel(const __grid_constant__ AuxParams prm, const uint32_t* rate_mrps,
                        const unsigned long long* pooled_hits, uint32_t* out_goodput) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= prm.P * prm.T) return;
  const uint64_t rate = rate_mrps[i / prm.T], hits = pooled_hits[i], nk = (uint64_t)prm.N * prm.K;
  out_goodput[i] = (uint32_t)u128_div(__umul64hi(rate, hits), rate * hits, nk);
}

// ---- pruning and selection -----------------------------------------------------------------------
// scratch: [0] = max over live plans of (sum of goodput + 1), 0 if none is live
__global__ void pareto_init_kernel(unsigned long long* scratch, uint32_t* out_best, uint32_t* out_n) {
  scratch[0] = 0ull;
  if (out_best) *out_best = 0xffffffffu;
  if (out_n) *out_n = 0u;
}

// one thread per plan p; candidate dominators q staged through shared memory 256 at a time (R23)
template <int T>
__global__ void __launch_bounds__(256)
pareto_dom_kernel(const uint32_t* __restrict__ G, uint32_t P, const uint8_t* __restrict__ alive,
                  uint8_t* out_pruned, uint32_t* out_n, unsigned long long* scratch) {
  __shared__ uint32_t gq[256 * T];
  __shared__ uint8_t lq[256];
  const uint32_t p = blockIdx.x * 256 + threadIdx.x;
  uint32_t gp[T];
  bool live = p < P && (!alive || alive[p]);
  uint64_t sum = 0;
#pragma unroll
  for (int t = 0; t < T; ++t) {
    gp[t] = p < P ? G[(size_t)p * T + t] : 0u;
    sum += gp[t];
  }
  bool dominated = false;
  for (uint32_t q0 = 0; q0 < P; q0 += 256) {
    __syncthreads();
    const uint32_t q = q0 + threadIdx.x;
    lq[threadIdx.x] = q < P && (!alive || alive[q]);
#pragma unroll
    for (int t = 0; t < T; ++t) gq[threadIdx.x * T + t] = q < P ? G[(size_t)q * T + t] : 0u;
    __syncthreads();
    if (live && !dominated) {
      const uint32_t nq = min(256u, P - q0);
      for (uint32_t j = 0; j < nq; ++j) {
        bool ge_all = lq[j] != 0, gt_any = false;
#pragma unroll
        for (int t = 0; t < T; ++t) {
          const uint32_t v = gq[j * T + t];
          ge_all = ge_all && v >= gp[t];
          gt_any = gt_any || v > gp[t];
        }
        dominated = dominated || (ge_all && gt_any);  // q == p: gt_any is false
      }
    }
  }
  if (p < P) {
    out_pruned[p] = (!live || dominated) ? 1 : 0;
    if (live) atomicMax(scratch, (unsigned long long)(sum + 1ull));
  }
  const uint32_t surv = __syncthreads_count(live && !dominated);
  if (threadIdx.x == 0 && surv && out_n) atomicAdd(out_n, surv);
}

// default policy: the live plan with the largest sum of goodput, lowest index on ties
template <int T>
__global__ void __launch_bounds__(256)
pareto_best_kernel(const uint32_t* __restrict__ G, uint32_t P, const uint8_t* __restrict__ alive,
                   const unsigned long long* scratch, uint32_t* out_best) {
  const uint32_t p = blockIdx.x * 256 + threadIdx.x;
  if (p >= P || (alive && !alive[p])) return;
  uint64_t sum = 0;
#pragma unroll
  for (int t = 0; t < T; ++t) sum += G[(size_t)p * T + t];
  if (sum + 1ull == scratch[0]) atomicMin(out_best, p);
}

}  // namespace cfk
