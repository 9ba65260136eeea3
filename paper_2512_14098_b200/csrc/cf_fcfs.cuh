// cf_fcfs.cuh -- arrival-order service at every stage (cf_graph.order_mode = 1; R27,
// SURVEY.md 8(f) NEXT-4 "true stage-arrival-order FCFS via segmented sort") for sm_100a.
//
// A stage that serves in ARRIVAL order cannot be advanced request by request: whether request n is
// next at stage s depends on when later requests get there. But the plan's stages are in topological
// order and a request only moves forward, so every arrival at stage s is known once stages 0..s-1 are
// done. One WARP runs one simulation, stage by stage, over scratch arrays in HBM (x[n] = the time at
// which request n leaves the last stage it has visited so far):
//   phase 0   the request stream, one request per lane (the producer code of the other kernels, hence
//             the same draws): x[n] = A_n;
//   per stage gather   the visitors of the stage, compacted with ballots: (arrival = x[n] + hop
//                      delay, n) and, by request, the summed service (and CPU time, R24) at the stage;
//             sort     the pairs by (arrival, n) -- a bitonic network over the warp's segment, skipped
//                      when the arrivals are already in order (every first stage);
//             serve    the Kiefer-Wolfowitz recursion in that order with the LANES AS REPLICAS: the
//                      sorted free-time vector of the stage lives one element per lane (CPL elements
//                      per lane for c > 32); replace-min = one ballot (where does the new departure
//                      go) and one shuffle (everything below it moves down a lane);
//   last      per-type counts and hits, checksum, makespan from x[n] - A_n (stream drawn once more).
// All times are absolute int64. Results are bit-identical to the oracle's order_mode = 1.
#pragma once
#include "cf_device.cuh"

namespace cfk {

constexpr int kFcfsWarps = 4;
constexpr uint32_t kAll = 0xffffffffu;

__device__ __forceinline__ bool pair_greater(int64_t ka, uint32_t ia, int64_t kb, uint32_t ib) {
  return ka > kb || (ka == kb && ia > ib);
}

// bitonic sort of (key, idx)[0..m_pad) ascending by (key, idx); m_pad a power of two; one warp
__device__ __forceinline__ void warp_bitonic_sort(int64_t* key, uint32_t* idx, uint32_t m_pad, int lane) {
  for (uint32_t k = 2; k <= m_pad; k <<= 1) {
    for (uint32_t j = k >> 1; j > 0; j >>= 1) {
      for (uint32_t t = lane; t < (m_pad >> 1); t += 32) {
        const uint32_t i = ((t & ~(j - 1u)) << 1) | (t & (j - 1u)), l = i | j;
        const bool up = (i & k) == 0u;
        const int64_t ki = key[i], kl = key[l];
        const uint32_t ii = idx[i], il = idx[l];
        if (pair_greater(ki, ii, kl, il) == up) {
          key[i] = kl; key[l] = ki;
          idx[i] = il; idx[l] = ii;
        }
      }
      __syncwarp();
    }
  }
}

// One replace-min of the Kiefer-Wolfowitz recursion on a sorted free-time vector spread over the
// warp: element e = j * 32 + lane lives in F[j] of that lane; elements >= c hold +inf.
// Arrival a, service S, CPU time Sc (R24: paid when the earliest-free replica is idle at a).
template <int CPL>
__device__ __forceinline__ int64_t kw_step(int64_t (&F)[CPL], int64_t a, int32_t S, int32_t Sc, int lane) {
  const int64_t f0 = __shfl_sync(kAll, F[0], 0);
  const int64_t D = (f0 <= a) ? a + (int64_t)Sc + (int64_t)S : f0 + (int64_t)S;
  uint32_t cnt = 0;
#pragma unroll
  for (int j = 0; j < CPL; ++j) cnt += __popc(__ballot_sync(kAll, F[j] <= D));
  const uint32_t q = cnt - 1u;  // D's place once the minimum is gone (F[0] <= D always)
#pragma unroll
  for (int j = 0; j < CPL; ++j) {
    int64_t next = __shfl_sync(kAll, F[j], (lane + 1) & 31);
    int64_t wrap = kInf;
    if (j + 1 < CPL) wrap = __shfl_sync(kAll, F[j + 1 < CPL ? j + 1 : j], 0);
    if (lane == 31) next = wrap;
    const uint32_t e = (uint32_t)(j * 32 + lane);
    F[j] = e < q ? next : (e == q ? D : F[j]);
  }
  return D;
}

template <int CMAX, bool HAS_CPU, int CPL>
__global__ void __launch_bounds__(kFcfsWarps * 32)
cf_fcfs_kernel(const __grid_constant__ KParams prm, const __grid_constant__ FcfsParams fp) {
  constexpr int kW = CompRec<CMAX, HAS_CPU>::kWords;
  constexpr int kB = CompRec<CMAX, HAS_CPU>::kBase;
  __shared__ __align__(16) uint4 rec_buf[kFcfsWarps][32 * kW];
  __shared__ uint64_t chunk_tot[kFcfsWarps];
  __shared__ uint32_t cnt_dummy[8];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t wid = blockIdx.x * kFcfsWarps + warp;
  if (wid >= fp.n_slots) return;  // nothing below synchronises the block
  uint8_t* slot_mem = fp.scratch + (size_t)wid * fp.slot_bytes;
  int64_t* xs = reinterpret_cast<int64_t*>(slot_mem);
  int64_t* key = reinterpret_cast<int64_t*>(slot_mem + fp.off_key);
  uint32_t* idx = reinterpret_cast<uint32_t*>(slot_mem + fp.off_idx);
  int32_t* sv = reinterpret_cast<int32_t*>(slot_mem + fp.off_sv);
  int32_t* scpu = reinterpret_cast<int32_t*>(slot_mem + fp.off_scpu);
  const int64_t delay = prm.edge_delay;
  const uint32_t lt_mask = (1u << lane) - 1u;

  for (uint32_t sim = wid; sim < fp.n_sims; sim += fp.n_slots) {
    uint32_t pr, trial, plan;
    if (fp.only_plan != 0xffffffffu) { plan = fp.only_plan; pr = plan; trial = prm.trial_base; }
    else { pr = sim / prm.k_launch; trial = prm.trial_base + sim % prm.k_launch; plan = pr / fp.R; }
    const uint32_t topo_id = prm.plan_topo[plan];
    const TopoDesc topo = prm.topos[topo_id];
    const uint32_t rate = prm.rates[pr];
    const size_t slot = (size_t)pr * prm.K + trial;
    const uint32_t variant = prm.variant_lo;
    bool rate_bad = false, skip = false;
    uint32_t period = 1;
    if (rate < 1u || rate > 1000000000u) {
      if (prm.bisect_mode && rate == 0u) skip = true; else rate_bad = true;
    } else {
      period = (1000000000u + rate / 2u) / rate;
    }
    uint32_t my_cnt = 0, my_hits = 0;  // lane t: requests / hits of type t
    uint64_t dep_sum = 0, last_cu = 0;
    int64_t makespan = 0;
    bool bad = rate_bad;

    // one chunk of the request stream: this lane's request n0 + lane (type, visited stages, services)
    struct Req { uint32_t t, vm; uint64_t cu; int32_t svc[8]; int32_t cpu[8]; bool valid; };
    uint64_t cu_base = 0;
    auto draw = [&](uint32_t n0) {
      Req r;
      produce_chunk_philox<CMAX, HAS_CPU>(prm, n0, trial, variant, rec_buf[warp], &chunk_tot[warp], cnt_dummy, lane);
      __syncwarp();
      const uint4* src = rec_buf[warp] + lane * kW;
      const uint4 w0 = src[0], w1 = src[1];
      uint4 w2 = make_uint4(0, 0, 0, 0);
      if (CMAX > 6) w2 = src[2];
      r.valid = n0 + lane < prm.N;
      r.cu = (((uint64_t)(w0.y & 0x00ffffffu) << 32) | w0.x) + cu_base;
      r.t = w0.y >> 24;
      r.svc[0] = (int32_t)w0.z; r.svc[1] = (int32_t)w0.w; r.svc[2] = (int32_t)w1.x; r.svc[3] = (int32_t)w1.y;
      r.svc[4] = (int32_t)w1.z; r.svc[5] = (int32_t)w1.w; r.svc[6] = (int32_t)w2.x; r.svc[7] = (int32_t)w2.y;
#pragma unroll
      for (int i = 0; i < 8; ++i) r.cpu[i] = 0;
      if (HAS_CPU) {
        const uint4 c0 = src[kB], c1 = src[kB + 1];
        r.cpu[0] = (int32_t)c0.x; r.cpu[1] = (int32_t)c0.y; r.cpu[2] = (int32_t)c0.z; r.cpu[3] = (int32_t)c0.w;
        r.cpu[4] = (int32_t)c1.x; r.cpu[5] = (int32_t)c1.y; r.cpu[6] = (int32_t)c1.z; r.cpu[7] = (int32_t)c1.w;
      }
      const uint32_t tm = prm.type_mask[r.t];
      const uint32_t rmask = CMAX > 6 ? route_stages(prm, topo_id, r.t, w2.z) : 0xffu;  // R26
      r.vm = 0;
#pragma unroll
      for (int s = 0; s < 8; ++s)
        if (s < topo.n_stages && (topo.mask[s] & tm) && ((rmask >> s) & 1u)) r.vm |= 1u << s;
      cu_base += chunk_tot[warp];
      __syncwarp();
      return r;
    };

    if (!skip && !bad) {
      // ---- phase 0: x[n] = A_n -------------------------------------------------------------------
      cu_base = 0;
      for (uint32_t n0 = 0; n0 < prm.N; n0 += 32) {
        const Req r = draw(n0);
        const int n_here = (int)min(32u, prm.N - n0);
        last_cu = __shfl_sync(kAll, r.cu, n_here - 1);
        if (r.valid) xs[n0 + lane] = (int64_t)((r.cu * (uint64_t)period + 32768ull) >> 16);
      }
      const uint64_t hi = __umul64hi(last_cu, (uint64_t)period);
      const uint64_t lo = last_cu * (uint64_t)period;
      if (hi != 0 || lo >= (1ull << 62) - 32768ull) bad = true;  // R17
    }
    if (!skip && !bad) {
      __syncwarp();
      for (uint32_t s = 0; s < topo.n_stages; ++s) {
        // ---- gather the visitors of stage s ------------------------------------------------------
        const uint32_t sm = topo.mask[s];
        uint32_t M = 0;
        cu_base = 0;
        for (uint32_t n0 = 0; n0 < prm.N; n0 += 32) {
          const Req r = draw(n0);
          const bool vis = r.valid && ((r.vm >> s) & 1u);
          int32_t S = 0, Sc = 0;
#pragma unroll
          for (int i = 0; i < CMAX; ++i) {
            S += ((sm >> i) & 1u) ? r.svc[i] : 0;
            if (HAS_CPU) Sc += ((sm >> i) & 1u) ? r.cpu[i] : 0;
          }
          const uint32_t b = __ballot_sync(kAll, vis);
          if (vis) {
            const uint32_t n = n0 + lane, pos = M + __popc(b & lt_mask);
            const bool first = (r.vm & ((1u << s) - 1u)) == 0u;
            key[pos] = xs[n] + (first ? 0 : delay);  // R9: a hop delay after the first visit
            idx[pos] = n;
            sv[n] = S;
            if (HAS_CPU) scpu[n] = Sc;
          }
          M += __popc(b);
        }
        __syncwarp();
        if (M == 0) continue;
        // ---- order of service: (arrival, index) ---------------------------------------------------
        bool unsorted = false;
        for (uint32_t i = lane; i + 1 < M; i += 32) unsorted = unsorted || key[i] > key[i + 1];
        if (__any_sync(kAll, unsorted)) {
          uint32_t m_pad = 2;
          while (m_pad < M) m_pad <<= 1;
          for (uint32_t i = M + lane; i < m_pad; i += 32) { key[i] = kInf; idx[i] = 0xffffffffu; }
          __syncwarp();
          warp_bitonic_sort(key, idx, m_pad, lane);
        }
        // ---- serve in that order, lanes as replicas -------------------------------------------------
        const uint32_t c = prm.plan_c[plan * 8 + s];
        int64_t F[CPL];
#pragma unroll
        for (int j = 0; j < CPL; ++j) F[j] = (uint32_t)(j * 32 + lane) < c ? 0 : kInf;
        for (uint32_t base = 0; base < M; base += 32) {
          const uint32_t e = base + lane;
          const int here = (int)min(32u, M - base);
          int64_t a = 0, d = 0;
          uint32_t n = 0;
          int32_t S = 0, Sc = 0;
          if (e < M) {
            a = key[e];
            n = idx[e];
            S = sv[n];
            if (HAS_CPU) Sc = scpu[n];
          }
          for (int j = 0; j < here; ++j) {
            const int64_t aj = __shfl_sync(kAll, a, j);
            const int32_t Sj = __shfl_sync(kAll, S, j);
            const int32_t Scj = HAS_CPU ? __shfl_sync(kAll, Sc, j) : 0;
            const int64_t D = kw_step<CPL>(F, aj, Sj, Scj, lane);
            if (lane == j) d = D;
          }
          if (e < M) xs[n] = d;
        }
        __syncwarp();
      }
      // ---- last: a8 over x[n] - A_n ------------------------------------------------------------------
      cu_base = 0;
      const bool traced = fp.only_plan != 0xffffffffu;
      for (uint32_t n0 = 0; n0 < prm.N; n0 += 32) {
        const Req r = draw(n0);
        const int64_t A = (int64_t)((r.cu * (uint64_t)period + 32768ull) >> 16);
        const int64_t x = r.valid ? xs[n0 + lane] : 0;
        if (traced && r.valid) {
          if (prm.tr_arrival) prm.tr_arrival[n0 + lane] = A;
          if (prm.tr_departure) prm.tr_departure[n0 + lane] = x;
          if (prm.tr_type) prm.tr_type[n0 + lane] = (uint8_t)r.t;
        }
        const bool hit = r.valid && (x - A) <= prm.L_us[r.t];
        for (uint32_t tt = 0; tt < prm.T; ++tt) {
          const uint32_t m = __ballot_sync(kAll, r.valid && r.t == tt);
          const uint32_t h = __ballot_sync(kAll, hit && r.t == tt);
          if ((uint32_t)lane == tt) { my_cnt += __popc(m); my_hits += __popc(h); }
        }
        if (r.valid) {
          dep_sum += (uint64_t)x;
          makespan = x > makespan ? x : makespan;
        }
      }
#pragma unroll
      for (int dd = 16; dd >= 1; dd >>= 1) {
        dep_sum += __shfl_xor_sync(kAll, dep_sum, dd);
        const int64_t o = __shfl_xor_sync(kAll, makespan, dd);
        makespan = o > makespan ? o : makespan;
      }
    }
    const bool zero = bad || skip;
    if (lane == 0 && bad) atomicMin(prm.status, -2);
    if ((uint32_t)lane < prm.T) {
      uint32_t* oc = prm.out_counts + slot * prm.T * 2;
      oc[2 * lane + 0] = zero ? 0u : my_cnt;
      oc[2 * lane + 1] = zero ? 0u : my_hits;
    }
    if (lane == 0) {
      if (prm.out_dep_sum) prm.out_dep_sum[slot] = zero ? 0ull : dep_sum;
      if (prm.out_makespan) prm.out_makespan[slot] = zero ? 0ll : makespan;
      if (prm.flags) prm.flags[slot] = 0;
    }
    __syncwarp();
  }
}

}  // namespace cfk
