// cf_scan.cuh -- the Lindley recursion as a max-plus scan across requests,
// for calls in which every stage of every plan has ONE replica (sm_100a). See DESIGN.md 5.6.
//
// With c = 1 a stage is max-plus linear: request n maps the previous departure D to
// f_n(D) = max(D + a_n, b_n) with a_n = S_n, b_n = (arrival at the stage) + S_n, and the identity
// (0, -inf) for a request that skips the stage; f_m after f_n is (a_n + a_m, max(b_n + a_m, b_m)).
// One WARP runs one simulation, one request per lane, 32 requests per step:
//   a1-a3  each lane draws its own request (Philox4x32-10 in registers, integer table lookups) or
//          reads its 32-byte record of the materialised stream with two coalesced 128-bit loads;
//          a warp inclusive sum of the Q16 gaps gives CU_n, A_n = (CU_n * period + 2^15) >> 16;
//   a4-a7  for every stage in plan order: an inclusive warp scan (5 shuffle steps on the 64-bit
//          pair (a, b)) composes the chunk's maps, the carry D_prev of the stage is applied,
//          visitors take the result as their arrival at the next stage (+ edge delay), and lane
//          31's result is the next chunk's carry;
//   a8     ballots give the per-type request and hit counts of the chunk (lane t keeps type t's).
// All times are absolute int64: there is no window and no fixup. Results are bit-identical to the
// thread-per-simulation kernels (same draws, same integer arithmetic, index-order service).
#pragma once
#include "cf_device.cuh"

namespace cfk {

constexpr int kScanWarps = 4;
constexpr int64_t kNegInf = INT64_MIN / 2;

template <int CMAX>
__global__ void __launch_bounds__(kScanWarps * 32)
cf_scan_kernel(const __grid_constant__ KParams prm, const uint32_t* __restrict__ plan_topo,
               const uint32_t* __restrict__ plan_var, uint32_t R, uint32_t n_sims) {
  __shared__ __align__(16) uint4 stage_buf[kScanWarps][32 * CompRec<CMAX>::kWords];
  __shared__ uint64_t chunk_tot[kScanWarps];
  __shared__ uint32_t cnt_dummy[8];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t sim = blockIdx.x * kScanWarps + warp;  // = pr * k_launch + trial index
  if (sim >= n_sims) return;                            // no block-wide barrier below
  const uint32_t pr = sim / prm.k_launch, trial = prm.trial_base + sim % prm.k_launch;
  const uint32_t plan = pr / R;
  const TopoDesc topo = prm.topos[plan_topo[plan]];
  const uint32_t rate = prm.rates[pr];
  const size_t slot = (size_t)pr * prm.K + trial;
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
  if (!skip) {
    const uint32_t vi = plan_var ? plan_var[plan] : 0u;
    const uint32_t variant = prm.variant_lo + vi;
    int64_t carry[8];  // departure of the stage's last visitor so far (all replicas free at 0)
#pragma unroll
    for (int s = 0; s < 8; ++s) carry[s] = 0;
    uint64_t cu_base = 0;
    const int64_t delay = prm.edge_delay;
    for (uint32_t n0 = 0; n0 < prm.N; n0 += 32) {
      const bool valid = n0 + lane < prm.N;
      const int n_here = (int)min(32u, prm.N - n0);
      uint4 w0 = make_uint4(0, 0, 0, 0), w1 = w0, w2 = w0;
      uint64_t cu;
      if (prm.stream == nullptr) {  // a1-a3 in registers (the shared producer code: identical draws)
        produce_chunk_philox<CMAX>(prm, n0, trial, variant, stage_buf[warp], &chunk_tot[warp], cnt_dummy, lane);
        __syncwarp();
        const uint4* src = stage_buf[warp] + lane * CompRec<CMAX>::kWords;
        w0 = src[0]; w1 = src[1];
        if (CMAX > 6) w2 = src[2];
        cu = (((uint64_t)(w0.y & 0x00ffffffu) << 32) | w0.x) + cu_base;
        cu_base += chunk_tot[warp];
        __syncwarp();
      } else {  // a10: two coalesced 128-bit loads per request
        if (valid) {
          const uint4* src = prm.stream + ((size_t)(vi * prm.K + trial) * prm.N + n0 + lane) * 2;
          w0 = __ldg(src); w1 = __ldg(src + 1);
        }
        cu = ((uint64_t)(w0.y & 0x00ffffffu) << 32) | w0.x;
      }
      last_cu = __shfl_sync(0xffffffffu, cu, n_here - 1);
      int32_t svc[8];
      svc[0] = (int32_t)w0.z; svc[1] = (int32_t)w0.w; svc[2] = (int32_t)w1.x; svc[3] = (int32_t)w1.y;
      svc[4] = (int32_t)w1.z; svc[5] = (int32_t)w1.w; svc[6] = (int32_t)w2.x; svc[7] = (int32_t)w2.y;
      const uint32_t t = w0.y >> 24;
      const uint32_t tm = prm.type_mask[t];
      const int64_t A = (int64_t)((cu * (uint64_t)period + 32768ull) >> 16);  // a3
      int64_t x = A;
      bool first = true;
#pragma unroll
      for (int s = 0; s < 8; ++s) {
        if (s < topo.n_stages) {  // warp-uniform
          const uint32_t sm = topo.mask[s];
          const bool vis = valid && (sm & tm) != 0;
          int64_t S = 0;
#pragma unroll
          for (int i = 0; i < CMAX; ++i) S += ((sm >> i) & 1u) ? svc[i] : 0;  // a4 (R6)
          if (vis && !first) x += delay;                                      // a7 (R9)
          if (vis) first = false;
          int64_t a = vis ? S : 0, b = vis ? x + S : kNegInf;                // f_n, or the identity
#pragma unroll
          for (int d = 1; d < 32; d <<= 1) {  // a5: inclusive max-plus scan, earlier maps first
            const int64_t ao = __shfl_up_sync(0xffffffffu, a, d), bo = __shfl_up_sync(0xffffffffu, b, d);
            if (lane >= d) {
              const int64_t bb = bo + a;
              b = bb > b ? bb : b;
              a = ao + a;
            }
          }
          const int64_t viaD = carry[s] + a;
          const int64_t D = viaD > b ? viaD : b;  // departure of the last visitor at or before this lane
          if (vis) x = D;
          carry[s] = __shfl_sync(0xffffffffu, D, 31);
        }
      }
      if (valid && plan == prm.tr_plan && sim % prm.k_launch == 0) {  // cf_trace_sim through this kernel (R = 1)
        if (prm.tr_arrival) prm.tr_arrival[n0 + lane] = A;
        if (prm.tr_departure) prm.tr_departure[n0 + lane] = x;
        if (prm.tr_type) prm.tr_type[n0 + lane] = (uint8_t)t;
      }
      // a8
      const bool hit = valid && (x - A) <= prm.L_us[t];
      for (uint32_t tt = 0; tt < prm.T; ++tt) {
        const uint32_t m = __ballot_sync(0xffffffffu, valid && t == tt);
        const uint32_t h = __ballot_sync(0xffffffffu, hit && t == tt);
        if ((uint32_t)lane == tt) { my_cnt += __popc(m); my_hits += __popc(h); }
      }
      if (valid) {
        dep_sum += (uint64_t)x;
        makespan = x > makespan ? x : makespan;
      }
    }
#pragma unroll
    for (int d = 16; d >= 1; d >>= 1) {
      dep_sum += __shfl_xor_sync(0xffffffffu, dep_sum, d);
      const int64_t o = __shfl_xor_sync(0xffffffffu, makespan, d);
      makespan = o > makespan ? o : makespan;
    }
  }
  // DESIGN.md R17: the arrival horizon CU_N * period + 2^15 must stay below 2^62
  bool bad = rate_bad;
  if (!bad && !skip) {
    const uint64_t hi = __umul64hi(last_cu, (uint64_t)period);
    const uint64_t lo = last_cu * (uint64_t)period;
    if (hi != 0 || lo >= (1ull << 62) - 32768ull) bad = true;
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
}

}  // namespace cfk
