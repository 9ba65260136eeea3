// cf_fcfs.cuh -- arrival-order service at every stage (cf_graph.order_mode = 1; R27,
// SURVEY.md 8(f) NEXT-4 "true stage-arrival-order FCFS via segmented sort") for sm_100a.
//
// A stage that serves in ARRIVAL order cannot be advanced request by request: whether request n is
// next at stage s depends on when later requests get there. But the plan's stages are in topological
// order and a request only moves forward, so every arrival at stage s is known once stages 0..s-1 are
// done. The request stream of every trial is drawn ONCE per call into HBM records (common random
// numbers, R4: every simulation of a trial reads the same records; two small kernels, the producer
// code of the other kernels, hence the same draws). Then one WARP runs one simulation, stage by stage,
// over scratch arrays in HBM (x[n] = the time at which request n leaves the last stage it has visited):
//   phase 0   x[n] = A_n;
//   per stage gather   the visitors of the stage, compacted with ballots: (arrival = x[n] + hop
//                      delay, n) and, by request, the summed service (and CPU time, R24) at the stage;
//             sort     by (arrival, request index). Visitors whose first stage this is arrive at A_n:
//                      they are in order as they come and form a run of their own; the others get an LSD
//                      radix sort, 8 bits a pass over the bits in which their keys differ (match.any
//                      ranks a chunk of 32 keys), skipped when they too are in order; a warp-level merge
//                      (each lane ranks its pair in the other run's 32-pair window) joins the two runs;
//             serve    the Kiefer-Wolfowitz recursion in that order with the LANES AS REPLICAS: the
//                      sorted free-time vector of the stage lives one element per lane (CPL consecutive
//                      elements per lane for c > 32); replace-min is F'[e] = min(F[e+1], max(F[e], D)):
//                      two shuffles a visit, one max and one min per element, no search for the
//                      insertion point. A batch of 32 visits whose
//                      times span less than 2^32 us runs on 32-bit offsets from the batch's first
//                      arrival (free times before it are clamped to it: exact, they are "idle");
//   last      per-type counts and hits, checksum, makespan from x[n] - A_n.
// All times are int64. Results are bit-identical to the oracle's order_mode = 1.
#pragma once
#include "cf_device.cuh"

namespace cfk {

constexpr int kFcfsWarps = 4;
constexpr uint32_t kAll = 0xffffffffu;
constexpr uint32_t kInf32 = 0xffffffffu;

// ---- the request records of the call's trials -------------------------------------------------------
// pass 1: gap totals of every segment of chunks_per_seg chunks (Philox block 0 + the arrival table only)
__global__ void __launch_bounds__(kFcfsWarps * 32)
cf_fcfs_totals_kernel(const __grid_constant__ KParams prm, const __grid_constant__ FcfsParams fp) {
  const int lane = threadIdx.x & 31;
  const uint32_t gw = blockIdx.x * kFcfsWarps + (threadIdx.x >> 5);
  if (gw >= prm.k_launch * fp.n_seg) return;
  const uint32_t ti = gw / fp.n_seg, seg = gw % fp.n_seg, trial = prm.trial_base + ti;
  const uint32_t n_chunks = (prm.N + 31u) / 32u;
  const uint32_t c0 = seg * fp.chunks_per_seg, c1 = min(c0 + fp.chunks_per_seg, n_chunks);
  uint64_t total = 0;
  for (uint32_t ch = c0; ch < c1; ++ch) {
    const uint32_t n = ch * 32u + lane;
    if (n < prm.N) {
      const uint4 b0 = philox4x32_10(n, trial, 0, prm.variant_lo, prm.seed_lo, prm.seed_hi);
      total += (uint32_t)qtab_sample(prm.qpool, prm.arr_tab, b0.x);
    }
  }
#pragma unroll
  for (int d = 16; d >= 1; d >>= 1) total += __shfl_xor_sync(kAll, total, d);
  if (lane == 0) fp.seg_tot[(size_t)ti * fp.n_seg + seg] = total;
}

// pass 2: the records of a segment, cumulative gaps made absolute with the totals of the segments before
template <int CMAX, bool HAS_CPU>
__global__ void __launch_bounds__(kFcfsWarps * 32)
cf_fcfs_records_kernel(const __grid_constant__ KParams prm, const __grid_constant__ FcfsParams fp) {
  constexpr int kW = CompRec<CMAX, HAS_CPU>::kWords;
  __shared__ __align__(16) uint4 rec_buf[kFcfsWarps][32 * kW];
  __shared__ uint64_t chunk_tot[kFcfsWarps];
  __shared__ uint32_t cnt_dummy[8];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t gw = blockIdx.x * kFcfsWarps + warp;
  if (gw >= prm.k_launch * fp.n_seg) return;
  const uint32_t ti = gw / fp.n_seg, seg = gw % fp.n_seg, trial = prm.trial_base + ti;
  const uint32_t n_chunks = (prm.N + 31u) / 32u;
  const uint32_t c0 = seg * fp.chunks_per_seg, c1 = min(c0 + fp.chunks_per_seg, n_chunks);
  uint64_t base = 0;
  for (uint32_t s = lane; s < seg; s += 32) base += fp.seg_tot[(size_t)ti * fp.n_seg + s];
#pragma unroll
  for (int d = 16; d >= 1; d >>= 1) base += __shfl_xor_sync(kAll, base, d);
  for (uint32_t ch = c0; ch < c1; ++ch) {
    produce_chunk_philox<CMAX, HAS_CPU>(prm, ch * 32u, trial, prm.variant_lo, rec_buf[warp], &chunk_tot[warp], cnt_dummy, lane);
    __syncwarp();
    const uint32_t n = ch * 32u + lane;
    if (n < prm.N) {
      const uint4* src = rec_buf[warp] + lane * kW;
      uint4* dst = fp.records + ((size_t)ti * prm.N + n) * kW;
      uint4 w0 = src[0];
      const uint64_t cu = (((uint64_t)(w0.y & 0x00ffffffu) << 32) | w0.x) + base;
      w0.x = (uint32_t)cu;
      w0.y = (uint32_t)(cu >> 32) | (w0.y & 0xff000000u);
      dst[0] = w0;
#pragma unroll
      for (int w = 1; w < kW; ++w) dst[w] = src[w];
    }
    base += chunk_tot[warp];
    __syncwarp();
  }
}

// ---- stable LSD radix sort of (key, idx)[0..M) by the key bits [0, bits): one warp, 8 bits a pass --------
// Returns the buffer (0 / 1) that holds the sorted pairs. cnt: 256 shared counters of this warp.
__device__ __forceinline__ int warp_radix_sort(int64_t* const (&key)[2], uint32_t* const (&idx)[2], uint32_t M,
                                               uint32_t bits, uint32_t* cnt, int lane) {
  const uint32_t lt_mask = (1u << lane) - 1u;
  int cur = 0;
  for (uint32_t shift = 0; shift < bits; shift += 8) {
    const int64_t* ks = key[cur];
    const uint32_t* is = idx[cur];
    int64_t* kd = key[cur ^ 1];
    uint32_t* id = idx[cur ^ 1];
#pragma unroll
    for (int k = 0; k < 8; ++k) cnt[lane * 8 + k] = 0;
    __syncwarp();
    // (the segment streams from HBM and a warp has nothing else to hide the round trip with: every
    //  loop below loads the NEXT group of 4 chunks of 32 before it works on the current one)
    int64_t kn[4];
    uint32_t in[4];
    auto fetch_keys = [&](uint32_t b0) {
#pragma unroll
      for (int r = 0; r < 4; ++r) {
        const uint32_t i = b0 + (uint32_t)r * 32u + lane;
        kn[r] = i < M ? ks[i] : 0;
      }
    };
    fetch_keys(0);
    for (uint32_t base = 0; base < M; base += 128) {  // histogram of the digit
      int64_t kc[4];
#pragma unroll
      for (int r = 0; r < 4; ++r) kc[r] = kn[r];
      if (base + 128 < M) fetch_keys(base + 128);
#pragma unroll
      for (int r = 0; r < 4; ++r) {
        const uint32_t i = base + (uint32_t)r * 32u + lane;
        if (base + (uint32_t)r * 32u >= M) break;
        const bool valid = i < M;
        const uint32_t d = valid ? (uint32_t)((uint64_t)kc[r] >> shift) & 255u : 0x100u + lane;
        const uint32_t m = __match_any_sync(kAll, d);
        if (valid && (m & lt_mask) == 0u) cnt[d] += __popc(m);  // the lowest lane of each digit group
        __syncwarp();
      }
    }
    {  // exclusive scan of the 256 counters, 8 per lane
      uint32_t v[8], s = 0;
#pragma unroll
      for (int k = 0; k < 8; ++k) { v[k] = cnt[lane * 8 + k]; s += v[k]; }
      uint32_t incl = s;
#pragma unroll
      for (int dd = 1; dd < 32; dd <<= 1) {
        const uint32_t o = __shfl_up_sync(kAll, incl, dd);
        if (lane >= dd) incl += o;
      }
      uint32_t run = incl - s;
#pragma unroll
      for (int k = 0; k < 8; ++k) { cnt[lane * 8 + k] = run; run += v[k]; }
    }
    __syncwarp();
    auto fetch_pairs = [&](uint32_t b0) {
#pragma unroll
      for (int r = 0; r < 4; ++r) {
        const uint32_t i = b0 + (uint32_t)r * 32u + lane;
        kn[r] = i < M ? ks[i] : 0;
        in[r] = i < M ? is[i] : 0u;
      }
    };
    fetch_pairs(0);
    for (uint32_t base = 0; base < M; base += 128) {  // stable scatter, a chunk of 32 at a time
      int64_t kc[4];
      uint32_t ic[4];
#pragma unroll
      for (int r = 0; r < 4; ++r) { kc[r] = kn[r]; ic[r] = in[r]; }
      if (base + 128 < M) fetch_pairs(base + 128);
#pragma unroll
      for (int r = 0; r < 4; ++r) {
        const uint32_t i = base + (uint32_t)r * 32u + lane;
        if (base + (uint32_t)r * 32u >= M) break;
        const bool valid = i < M;
        const uint32_t d = valid ? (uint32_t)((uint64_t)kc[r] >> shift) & 255u : 0x100u + lane;
        const uint32_t m = __match_any_sync(kAll, d);
        const uint32_t off = valid ? cnt[d] : 0u;
        __syncwarp();
        if (valid && (m & lt_mask) == 0u) cnt[d] = off + __popc(m);
        __syncwarp();
        if (valid) {
          const uint32_t pos = off + __popc(m & lt_mask);
          kd[pos] = kc[r];
          id[pos] = ic[r];
        }
      }
    }
    __syncwarp();
    cur ^= 1;
  }
  return cur;
}

// ---- merge of two sorted runs of (key, idx) pairs, ordered by (key, idx): one warp ------------------------
// Each step holds the next 32 pairs of either run, one per lane; a lane ranks its pair against the other
// run's window with a binary search over lanes (shuffles); the 32 smallest pairs of the two windows are
// the next 32 of the merged order (a pair that all 32 of the other window precede is not among them).
__device__ __forceinline__ bool pair_less(int64_t ka, uint32_t ia, int64_t kb, uint32_t ib) {
  return ka < kb || (ka == kb && ia < ib);
}
__device__ __forceinline__ uint32_t rank_in_window(int64_t wk, uint32_t wi, int64_t k, uint32_t i) {
  uint32_t lo = 0, hi = 32;  // number of window pairs (sorted across the lanes) that precede (k, i)
#pragma unroll
  for (int it = 0; it < 6; ++it) {
    const uint32_t mid = (lo + hi) >> 1;
    const int64_t mk = __shfl_sync(kAll, wk, (int)(mid & 31u));
    const uint32_t mi = __shfl_sync(kAll, wi, (int)(mid & 31u));
    if (lo < hi) {
      if (pair_less(mk, mi, k, i)) lo = mid + 1u; else hi = mid;
    }
  }
  return lo;
}
// The runs stream from HBM through a ring of kRing pairs per run in shared memory: a chunk of 32 is loaded
// into registers as soon as the ring has room for it and stored two steps later, so no step waits for a
// load it has just issued (a run gives at most 32 pairs a step: the ring is always 3 chunks ahead).
constexpr uint32_t kRing = 256;
struct MergePend { int64_t k; uint32_t i, pos; bool v; };
__device__ __forceinline__ void warp_merge(const int64_t* Ak, const uint32_t* Ai, uint32_t MA, const int64_t* Bk,
                                           const uint32_t* Bi, uint32_t MB, int64_t* Ok, uint32_t* Oi,
                                           int64_t* ringk, uint32_t* ringi, int lane) {  // rings: [2][kRing]
  int64_t* rak = ringk; int64_t* rbk = ringk + kRing;
  uint32_t* rai = ringi; uint32_t* rbi = ringi + kRing;
  for (uint32_t t = lane; t < min(MA, kRing); t += 32) { rak[t] = Ak[t]; rai[t] = Ai[t]; }
  for (uint32_t t = lane; t < min(MB, kRing); t += 32) { rbk[t] = Bk[t]; rbi[t] = Bi[t]; }
  uint32_t ta = min(MA, kRing), tb = min(MB, kRing);  // pairs of the run issued so far
  MergePend pa0{0, 0, 0, false}, pa1 = pa0, pb0 = pa0, pb1 = pa0;
  __syncwarp();
  uint32_t i = 0, j = 0, o = 0;
  const uint32_t M = MA + MB;
  while (o < M) {
    MergePend na_{0, 0, 0, false}, nb_ = na_;
    if (ta < MA && ta - i <= kRing - 32u) {  // room for [ta, ta + 32): its slots hold pairs already consumed
      na_.v = true; na_.pos = ta;
      if (ta + lane < MA) { na_.k = Ak[ta + lane]; na_.i = Ai[ta + lane]; }
      ta += 32u;
    }
    if (tb < MB && tb - j <= kRing - 32u) {
      nb_.v = true; nb_.pos = tb;
      if (tb + lane < MB) { nb_.k = Bk[tb + lane]; nb_.i = Bi[tb + lane]; }
      tb += 32u;
    }
    const bool av = i + lane < MA, bv = j + lane < MB;
    const uint32_t sa = (i + lane) & (kRing - 1u), sb = (j + lane) & (kRing - 1u);
    const int64_t ak = av ? rak[sa] : kInf, bk = bv ? rbk[sb] : kInf;
    const uint32_t ai = av ? rai[sa] : 0xffffffffu, bi = bv ? rbi[sb] : 0xffffffffu;
    const uint32_t pa = (uint32_t)lane + rank_in_window(bk, bi, ak, ai);
    const uint32_t pb = (uint32_t)lane + rank_in_window(ak, ai, bk, bi);
    const bool ea = av && pa < 32u, eb = bv && pb < 32u;
    if (ea) { Ok[o + pa] = ak; Oi[o + pa] = ai; }
    if (eb) { Ok[o + pb] = bk; Oi[o + pb] = bi; }
    const uint32_t na = __popc(__ballot_sync(kAll, ea)), nb = __popc(__ballot_sync(kAll, eb));
    i += na; j += nb; o += na + nb;
    __syncwarp();  // every lane has read its window: slots of consumed pairs may be overwritten
    if (pa0.v) { const uint32_t t = (pa0.pos + lane) & (kRing - 1u); rak[t] = pa0.k; rai[t] = pa0.i; }
    if (pb0.v) { const uint32_t t = (pb0.pos + lane) & (kRing - 1u); rbk[t] = pb0.k; rbi[t] = pb0.i; }
    pa0 = pa1; pa1 = na_; pb0 = pb1; pb1 = nb_;
    __syncwarp();
  }
  __syncwarp();
}

// ---- Kiefer-Wolfowitz on a sorted free-time vector spread over the warp ----------------------------------
// Lane l holds elements l * CPL .. l * CPL + CPL - 1 in F[0..CPL); elements >= c hold +inf. One visit with
// arrival a, service S, CPU time Sc (R24: paid when the earliest-free replica is idle at a): departure D, then
// the minimum leaves and D enters: F'[e] = min(F[e+1], max(F[e], D)) (F sorted, F[0] <= D). The serve loop
// costs two shuffles on the vector whatever CPL is: the minimum from lane 0 and the neighbour's first element.
template <int CPL, bool HAS_CPU, typename TT>
__device__ __forceinline__ TT kw_visit(TT (&F)[CPL], TT a, uint32_t S, uint32_t Sc, TT inf, int lane) {
  const TT f0 = __shfl_sync(kAll, F[0], 0);
  TT next = __shfl_sync(kAll, F[0], (lane + 1) & 31);
  if (lane == 31) next = inf;
  TT D;
  if (HAS_CPU) D = (f0 <= a) ? a + (TT)Sc + (TT)S : f0 + (TT)S;
  else D = (f0 > a ? f0 : a) + (TT)S;
#pragma unroll
  for (int j = 0; j < CPL; ++j) {
    const TT nx = j + 1 < CPL ? F[j + 1 < CPL ? j + 1 : j] : next;
    const TT up = F[j] > D ? F[j] : D;
    F[j] = nx < up ? nx : up;
  }
  return D;
}

template <int CMAX, bool HAS_CPU, int CPL>
__global__ void __launch_bounds__(kFcfsWarps * 32, 6)
cf_fcfs_kernel(const __grid_constant__ KParams prm, const __grid_constant__ FcfsParams fp) {
  constexpr int kW = CompRec<CMAX, HAS_CPU>::kWords;
  constexpr int kB = CompRec<CMAX, HAS_CPU>::kBase;
  __shared__ uint32_t cnt_s[kFcfsWarps][256];
  __shared__ int64_t ringk_s[kFcfsWarps][2 * kRing];
  __shared__ uint32_t ringi_s[kFcfsWarps][2 * kRing];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t wid = blockIdx.x * kFcfsWarps + warp;
  if (wid >= fp.n_slots) return;  // nothing below synchronises the block
  uint8_t* slot_mem = fp.scratch + (size_t)wid * fp.slot_bytes;
  int64_t* xs = reinterpret_cast<int64_t*>(slot_mem);
  // key / idx [0], [1]: the visitors that come from an earlier stage (the radix sort ping-pongs between them, the
  // merge writes into the free one); [2]: the visitors whose first stage this is (their arrival is A_n: in order)
  int64_t* const key[2] = {reinterpret_cast<int64_t*>(slot_mem + fp.off_key[0]), reinterpret_cast<int64_t*>(slot_mem + fp.off_key[1])};
  uint32_t* const idx[2] = {reinterpret_cast<uint32_t*>(slot_mem + fp.off_idx[0]), reinterpret_cast<uint32_t*>(slot_mem + fp.off_idx[1])};
  int64_t* const keyF = reinterpret_cast<int64_t*>(slot_mem + fp.off_key[2]);
  uint32_t* const idxF = reinterpret_cast<uint32_t*>(slot_mem + fp.off_idx[2]);
  int32_t* sv = reinterpret_cast<int32_t*>(slot_mem + fp.off_sv);
  int32_t* scpu = reinterpret_cast<int32_t*>(slot_mem + fp.off_scpu);
  auto done_of = [&](uint32_t s) { return reinterpret_cast<int64_t*>(slot_mem + fp.off_done + (size_t)s * fp.done_stride); };
  const bool join = prm.join != 0;  // R25: a request reaches a stage when its predecessor stages are done
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
    bool rate_bad = false, skip = false;
    uint32_t period = 1;
    if (rate < 1u || rate > 1000000000u) {
      if (prm.bisect_mode && rate == 0u) skip = true; else rate_bad = true;
    } else {
      period = (1000000000u + rate / 2u) / rate;
    }
    uint32_t my_cnt = 0, my_hits = 0;  // lane t: requests / hits of type t
    uint64_t dep_sum = 0;
    int64_t makespan = 0;
    bool bad = rate_bad;
    const uint4* recs = fp.records + (size_t)(trial - prm.trial_base) * prm.N * kW;

    // this lane's request n0 + lane: type, visited stages, A_n, services
    struct Req { uint32_t t, vm; uint64_t cu; int32_t svc[8]; int32_t cpu[8]; bool valid; };
    auto load = [&](uint32_t n0, bool want_svc) {
      Req r;
      r.valid = n0 + lane < prm.N;
      const uint4* src = recs + (size_t)min(n0 + lane, prm.N - 1u) * kW;
      const uint4 w0 = __ldg(src);
      uint4 w1 = make_uint4(0, 0, 0, 0), w2 = w1;
      if (want_svc) w1 = __ldg(src + 1);
      if (CMAX > 6) w2 = __ldg(src + 2);
      r.cu = ((uint64_t)(w0.y & 0x00ffffffu) << 32) | w0.x;
      r.t = w0.y >> 24;
      r.svc[0] = (int32_t)w0.z; r.svc[1] = (int32_t)w0.w; r.svc[2] = (int32_t)w1.x; r.svc[3] = (int32_t)w1.y;
      r.svc[4] = (int32_t)w1.z; r.svc[5] = (int32_t)w1.w; r.svc[6] = (int32_t)w2.x; r.svc[7] = (int32_t)w2.y;
#pragma unroll
      for (int i = 0; i < 8; ++i) r.cpu[i] = 0;
      if (HAS_CPU && want_svc) {
        const uint4 c0 = __ldg(src + kB), c1 = __ldg(src + kB + 1);
        r.cpu[0] = (int32_t)c0.x; r.cpu[1] = (int32_t)c0.y; r.cpu[2] = (int32_t)c0.z; r.cpu[3] = (int32_t)c0.w;
        r.cpu[4] = (int32_t)c1.x; r.cpu[5] = (int32_t)c1.y; r.cpu[6] = (int32_t)c1.z; r.cpu[7] = (int32_t)c1.w;
      }
      const uint32_t tm = prm.type_mask[r.t];
      const uint32_t rmask = CMAX > 6 ? route_stages(prm, topo_id, r.t, w2.z) : 0xffu;  // R26
      r.vm = 0;
#pragma unroll
      for (int s = 0; s < 8; ++s)
        if (s < topo.n_stages && (topo.mask[s] & tm) && ((rmask >> s) & 1u)) r.vm |= 1u << s;
      return r;
    };

    if (!skip && !bad) {  // R17: the arrival horizon CU_N * period + 2^15 must stay below 2^62
      const uint4 wl = __ldg(recs + (size_t)(prm.N - 1u) * kW);
      const uint64_t last_cu = ((uint64_t)(wl.y & 0x00ffffffu) << 32) | wl.x;
      const uint64_t hi = __umul64hi(last_cu, (uint64_t)period);
      const uint64_t lo = last_cu * (uint64_t)period;
      if (hi != 0 || lo >= (1ull << 62) - 32768ull) bad = true;
    }
    if (!skip && !bad) {
      // ---- phase 0: x[n] = A_n -------------------------------------------------------------------
#pragma unroll 4
      for (uint32_t n = lane; n < prm.N; n += 32) {
        const uint4 w0 = __ldg(recs + (size_t)n * kW);
        const uint64_t cu = ((uint64_t)(w0.y & 0x00ffffffu) << 32) | w0.x;
        xs[n] = (int64_t)((cu * (uint64_t)period + 32768ull) >> 16);
      }
      __syncwarp();
      for (uint32_t s = 0; s < topo.n_stages; ++s) {
        // ---- gather the visitors of stage s ------------------------------------------------------
        const uint32_t sm = topo.mask[s];
        uint32_t M = 0, MF = 0;  // visitors from an earlier stage / visitors that start here
        bool unsorted = false;
        int64_t kmin = kInf, kmax = 0, prev_last = 0;
        Req r_nx = load(0, true);
        int64_t x_nx = lane < prm.N ? xs[lane] : 0;
        for (uint32_t n0 = 0; n0 < prm.N; n0 += 32) {
          const Req r = r_nx;
          const int64_t x_cur = x_nx;
          if (n0 + 32 < prm.N) {
            r_nx = load(n0 + 32, true);
            if (n0 + 32 + lane < prm.N) x_nx = xs[n0 + 32 + lane];
          }
          const bool vis = r.valid && ((r.vm >> s) & 1u);
          int32_t S = 0, Sc = 0;
#pragma unroll
          for (int i = 0; i < CMAX; ++i) {
            S += ((sm >> i) & 1u) ? r.svc[i] : 0;
            if (HAS_CPU) Sc += ((sm >> i) & 1u) ? r.cpu[i] : 0;
          }
          // a visitor with no earlier stage (fork-join: no predecessor stage) arrives at A_n: those are in
          // order as they come and go to their own run; only the others may need sorting
          bool first = (r.vm & ((1u << s) - 1u)) == 0u;
          uint32_t pm = 0;
          if (join && vis) {
            pm = prm.topo_pred[topo_id * 64u + r.t * 8u + s] & r.vm;
            first = pm == 0u;
          }
          const uint32_t bf = __ballot_sync(kAll, vis && first);
          const uint32_t b = __ballot_sync(kAll, vis && !first);
          int64_t a = 0;
          if (vis) {
            const uint32_t n = n0 + lane;
            a = x_cur + (first ? 0 : delay);  // R9: a hop delay after the first visit
            if (join) {  // R25: after every predecessor stage of the request, plus that edge's delay; else at A_n
              a = (int64_t)((r.cu * (uint64_t)period + 32768ull) >> 16);
              while (pm) {
                const uint32_t sp = (uint32_t)__ffs((int)pm) - 1u;
                pm &= pm - 1u;
                const int64_t dsp = done_of(sp)[n] + delay;
                a = dsp > a ? dsp : a;
              }
            }
            if (first) {
              const uint32_t pos = MF + __popc(bf & lt_mask);
              keyF[pos] = a;
              idxF[pos] = n;
            } else {
              const uint32_t pos = M + __popc(b & lt_mask);
              key[0][pos] = a;
              idx[0][pos] = n;
              kmin = a < kmin ? a : kmin;
              kmax = a > kmax ? a : kmax;
            }
            sv[n] = S;
            if (HAS_CPU) scpu[n] = Sc;
          }
          if (b) {  // in order? every such visitor against the one before it (the previous chunk's last for the first)
            const uint32_t below = b & lt_mask;
            const int src = below ? 31 - __clz((int)below) : 0;
            const int64_t pa = __shfl_sync(kAll, a, src);
            if (vis && !first && (below ? pa : prev_last) > a && (below || M > 0)) unsorted = true;
            prev_last = __shfl_sync(kAll, a, 31 - __clz((int)b));
          }
          M += __popc(b);
          MF += __popc(bf);
        }
        __syncwarp();
        if (M + MF == 0) continue;
        // ---- order of service: by arrival, ties by index -----------------------------------------------
        int cur = 0;
        if (__any_sync(kAll, unsorted)) {
#pragma unroll
          for (int dd = 16; dd >= 1; dd >>= 1) {
            const int64_t o1 = __shfl_xor_sync(kAll, kmin, dd), o2 = __shfl_xor_sync(kAll, kmax, dd);
            kmin = o1 < kmin ? o1 : kmin;
            kmax = o2 > kmax ? o2 : kmax;
          }
          const uint32_t bits = 64u - (uint32_t)__clzll((long long)(kmin ^ kmax));  // keys agree above these bits
          cur = warp_radix_sort(key, idx, M, bits, cnt_s[warp], lane);
        }
        const int64_t* ks = key[cur];
        const uint32_t* is = idx[cur];
        if (M == 0) {
          ks = keyF; is = idxF;
        } else if (MF != 0) {  // two sorted runs -> one
          warp_merge(keyF, idxF, MF, key[cur], idx[cur], M, key[cur ^ 1], idx[cur ^ 1], ringk_s[warp], ringi_s[warp], lane);
          ks = key[cur ^ 1]; is = idx[cur ^ 1];
        }
        M += MF;
        // ---- serve in that order, lanes as replicas -------------------------------------------------
        const uint32_t c = prm.plan_c[plan * 8 + s];
        int64_t F[CPL];
#pragma unroll
        for (int j = 0; j < CPL; ++j) F[j] = (uint32_t)(lane * CPL + j) < c ? 0 : kInf;
        // the sorted pairs are loaded two batches ahead, the services they point to one batch ahead
        int64_t a_n1 = 0, a_n2 = 0;
        uint32_t n_n1 = 0, n_n2 = 0, S_n1 = 0, Sc_n1 = 0;
        if ((uint32_t)lane < M) { a_n1 = ks[lane]; n_n1 = is[lane]; S_n1 = (uint32_t)sv[n_n1]; if (HAS_CPU) Sc_n1 = (uint32_t)scpu[n_n1]; }
        if (32u + lane < M) { a_n2 = ks[32u + lane]; n_n2 = is[32u + lane]; }
        for (uint32_t base = 0; base < M; base += 32) {
          const uint32_t e = base + lane;
          const int here = (int)min(32u, M - base);
          const int64_t a = a_n1;
          const uint32_t n = n_n1, S = S_n1, Sc = Sc_n1;
          int64_t d = 0;
          a_n1 = a_n2; n_n1 = n_n2;
          if (e + 32 < M) { S_n1 = (uint32_t)sv[n_n1]; if (HAS_CPU) Sc_n1 = (uint32_t)scpu[n_n1]; }
          if (e + 64 < M) { a_n2 = ks[e + 64]; n_n2 = is[e + 64]; }
          // 32-bit body if every time of the batch fits an offset from its first arrival
          const int64_t a0 = __shfl_sync(kAll, a, 0), a_last = __shfl_sync(kAll, a, here - 1);
          int64_t fm = 0;  // the largest free time: element c - 1 of the sorted vector
#pragma unroll
          for (int j = 0; j < CPL; ++j) {
            const int64_t v = __shfl_sync(kAll, F[j], (int)((c - 1u) / CPL));
            if ((uint32_t)j == (c - 1u) % CPL) fm = v;
          }
          const uint32_t work = (e < M) ? S + Sc : 0u;
          const bool big = __any_sync(kAll, work >= (1u << 26));
          const uint64_t sum = __reduce_add_sync(kAll, min(work, 1u << 26));
          const int64_t top = fm > a_last ? fm : a_last;
          if (!big && (uint64_t)(top - a0) + sum < 0xfffffff0ull) {
            uint32_t G[CPL];
#pragma unroll
            for (int j = 0; j < CPL; ++j) G[j] = F[j] == kInf ? kInf32 : (uint32_t)((F[j] > a0 ? F[j] : a0) - a0);
            const uint32_t a32 = (uint32_t)(a - a0);
            uint32_t d32 = 0;
            for (int j = 0; j < here; ++j) {
              const uint32_t aj = __shfl_sync(kAll, a32, j), Sj = __shfl_sync(kAll, S, j);
              const uint32_t Scj = HAS_CPU ? __shfl_sync(kAll, Sc, j) : 0u;
              const uint32_t D = kw_visit<CPL, HAS_CPU, uint32_t>(G, aj, Sj, Scj, kInf32, lane);
              if (lane == j) d32 = D;
            }
#pragma unroll
            for (int j = 0; j < CPL; ++j) F[j] = G[j] == kInf32 ? kInf : a0 + (int64_t)G[j];
            d = a0 + (int64_t)d32;
          } else {
            for (int j = 0; j < here; ++j) {
              const int64_t aj = __shfl_sync(kAll, a, j);
              const uint32_t Sj = __shfl_sync(kAll, S, j);
              const uint32_t Scj = HAS_CPU ? __shfl_sync(kAll, Sc, j) : 0u;
              const int64_t D = kw_visit<CPL, HAS_CPU, int64_t>(F, aj, Sj, Scj, kInf, lane);
              if (lane == j) d = D;
            }
          }
          if (e < M) {
            if (join) {  // the request is done when its last branch is
              done_of(s)[n] = d;
              const int64_t xo = xs[n];
              xs[n] = d > xo ? d : xo;
            } else {
              xs[n] = d;
            }
          }
        }
        __syncwarp();
      }
      // ---- last: a8 over x[n] - A_n ------------------------------------------------------------------
      const bool traced = fp.only_plan != 0xffffffffu;
      uint4 w_nx = __ldg(recs + (size_t)min((uint32_t)lane, prm.N - 1u) * kW);
      int64_t xf_nx = (uint32_t)lane < prm.N ? xs[lane] : 0;
      for (uint32_t n0 = 0; n0 < prm.N; n0 += 32) {
        struct { bool valid; uint32_t t; uint64_t cu; } r;
        r.valid = n0 + lane < prm.N;
        r.t = w_nx.y >> 24;
        r.cu = ((uint64_t)(w_nx.y & 0x00ffffffu) << 32) | w_nx.x;
        const int64_t x = r.valid ? xf_nx : 0;
        if (n0 + 32 < prm.N) {
          w_nx = __ldg(recs + (size_t)min(n0 + 32 + lane, prm.N - 1u) * kW);
          if (n0 + 32 + lane < prm.N) xf_nx = xs[n0 + 32 + lane];
        }
        const int64_t A = (int64_t)((r.cu * (uint64_t)period + 32768ull) >> 16);
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
