// cf_device.cuh -- device code of libcf_b200 (sm_100a). See DESIGN.md "Kernels".
//
// Mapping:
//   * one THREAD per simulation (plan, rate, trial); a CTA holds simulations that share the trial
//     and the Philox variant, hence (common random numbers, R4) the same request stream;
//   * the CTA draws that stream ONCE per tile (a1 Philox4x32-10, a2 table lookup, a3 type + gap
//     prefix sum) into shared memory -- or copies it from the materialised HBM stream (a10) -- and
//     every thread then walks the tile sequentially;
//   * each warp holds simulations of one plan topology; it turns 32 component-level records into
//     stage-level records (a4) once per chunk, so the per-request loop sees only {cu, type, S[s]};
//   * a5/a6: the free-time multiset of a c-replica stage is a binary min-heap of int64 per thread,
//     root in a register, nodes 2..c+1 in shared memory as sibling pairs interleaved by lane (one
//     conflict-free LDS.128 per level); c = 1 degenerates to the Lindley recursion, no memory traffic;
//   * a7 hand-off is the running x; a8 counters are packed per-type byte fields flushed per chunk.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace cfk {

// warps per thread block: a template parameter of the kernels (4 or 8, chosen by the schedule)
constexpr int kMaxWarpsPerCta = 8;
constexpr int kTile = 128;              // requests per CTA tile
constexpr int kChunks = kTile / 32;     // 32-request chunks per tile
constexpr int64_t kInf = INT64_MAX;

struct DevTab {
  uint32_t off;  // index of entry 0 in the int32 pool
  uint32_t levels, log2_cells, pad;
};

struct TopoDesc {  // one plan topology = ordered stage masks
  uint8_t n_stages;
  uint8_t mask[8];
  uint8_t pad[7];
};

// R26: routing table of a topology: per type up to 4 routes = (cumulative probability Q32, bitmask
// over the topology's stages the route may visit); the last route is the catch-all
struct TopoRoutes {
  uint32_t cum[8][4];
  uint8_t mask[8][4];
};

struct SimDesc {
  uint32_t plan;  // plan index (for replica counts)
  uint32_t pr;    // p*R + r : index into the rate array; output slot is pr*K + k
};

struct WarpDesc {
  uint32_t sim_begin, n_lanes, topo;
  uint32_t variant;     // stream variant of this warp's simulations (materialised stream: a block may mix variants)
  uint32_t heap_off;    // byte offset of this warp's heap region in the CTA heap arena (64-bit kernel)
  uint32_t heap_off32;  // same for the 32-bit kernel (4-ary heap of uint32 quads)
  uint32_t heap_rows32; // 512-byte rows of that region
};

struct CtaDesc {
  uint32_t warp_begin, n_warps, variant, heap_bytes, heap_bytes32;
};

// Heap storage of one c-replica stage of one lane: floor(c/2) sibling pairs (nodes 2i, 2i+1), one
// 512-byte row per pair (32 lanes x 16 B). A lane's stages follow one another, so a warp's region
// is 512 B x max over its lanes of sum_s floor(c_s/2).
__host__ __device__ __forceinline__ uint32_t heap_pairs(uint32_t c) { return c >> 1; }
// 32-bit kernel: 4-ary heap, root in a register, nodes 1..c-1 in ceil((c-1)/4) quads (16 B per lane)
__host__ __device__ __forceinline__ uint32_t heap_quads(uint32_t c) { return (c + 2) >> 2; }

struct KParams {
  uint32_t C, T, N, K;
  uint32_t type_thresh[8];
  uint8_t type_mask[8];
  DevTab svc_tab[64];  // [i*8 + t]
  DevTab cpu_tab[64];  // [i*8 + t] CPU pre-processing time (R24); levels == 0: none
  DevTab arr_tab;
  const int32_t* qpool;
  int64_t L_us[8];
  int64_t edge_delay;
  uint32_t seed_lo, seed_hi;
  // request source: in-register Philox (stream == nullptr, Philox variant = variant_lo + cta.variant)
  // or materialised records [variant][K][N] x 32 B
  const uint4* stream;
  uint32_t variant_lo;
  uint32_t bisect_mode;  // rate 0 means "skip this simulation" instead of a range error
  uint32_t trial_base;   // trial = trial_base + blockIdx.x % k_launch (cf_trace_sim runs one trial)
  uint32_t k_launch;     // trials per launch; CTA = blockIdx.x / k_launch (heavy CTAs first)
  // schedule
  const CtaDesc* ctas;
  const WarpDesc* warps;
  const SimDesc* sims;
  const TopoDesc* topos;
  const uint16_t* plan_c;  // [P*8]
  const uint32_t* plan_topo;  // [P] topology of each plan   (scan kernel)
  const uint32_t* plan_var;   // [P] stream variant of each plan
  const uint32_t* rates;   // [P*R]
  // outputs
  uint32_t* out_counts;    // [PR][K][T][2]
  uint64_t* out_dep_sum;   // [PR][K] or null
  int64_t* out_makespan;   // [PR][K] or null
  int32_t* status;         // sticky device status; status[1] = simulations sent to the 64-bit kernel
  // 32-bit fast path (cf_rel32.cuh): flags[slot] = 1 <=> the simulation left the 32-bit window and
  // must be redone by the 64-bit kernel, which then runs with fixup = 1 and touches only those.
  uint8_t* flags;          // [PR][K] or null
  uint32_t fixup;
  int64_t* tr_arrival;     // trace (single simulation) or null
  int64_t* tr_departure;
  uint8_t* tr_type;
  uint32_t tr_plan;        // the traced plan (scan kernel: the warp whose simulation is written out)
  uint32_t has_cpu;        // some (component, type) has a CPU pre-processing table (R24): 64-bit kernel only
  uint32_t max_routes;     // R26: 0 = no routing tables; else routes per (topology, type)
  const TopoRoutes* topo_routes;  // [topology]
  uint32_t join;           // fork-join routing along the DAG edges (R25): 64-bit kernel only
  const uint8_t* topo_pred;  // join: [topology][type 8][stage 8] bitmask of the stage's predecessor stages
};

// Arrival-order kernels (cf_fcfs.cuh, R27): one warp per simulation in flight.
// Request records of the call's trials (drawn once, shared by every simulation of a trial):
//   records[(trial - trial_base) * N + n] = CompRec<CMAX, HAS_CPU> words with the ABSOLUTE cumulative gap.
// Scratch of one simulation in flight (byte offsets inside its slot; x at 0):
//   x int64[N] | key int64[N] x 3 | idx u32[N] x 3 (two for the radix sort to ping-pong, one for the visitors
//   that are in order by construction) | sv i32[N] | scpu i32[N]
//   | fork-join (R25): done int64[8][N], the departure of request n from stage s
struct FcfsParams {
  uint8_t* scratch;
  unsigned long long slot_bytes;
  uint4* records;
  unsigned long long* seg_tot;  // [trial][segment] sum of the gaps of a segment of chunks
  uint32_t n_seg, chunks_per_seg;
  uint32_t n_slots;    // warps (simulations in flight); simulation i runs on warp i mod n_slots
  uint32_t R;          // rates per plan
  uint32_t n_sims;     // P * R * k_launch, or 1 with only_plan
  uint32_t only_plan;  // cf_trace_sim: the one plan to run (R = 1); 0xffffffff = all
  uint32_t off_key[3], off_idx[3], off_sv, off_scpu;
  uint32_t off_done, done_stride;  // fork-join: byte offset of done[0], bytes between done[s] and done[s+1]
};

// ------------------------------------------------------------------------------------------------
// a1: Philox4x32-10 (Salmon et al. SC'11), counter (n, trial, block, variant), key = seed
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                               uint32_t k0, uint32_t k1) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint64_t p0 = (uint64_t)0xD2511F53u * c0;
    const uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
    const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
    const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
    c1 = (uint32_t)p1;
    c3 = (uint32_t)p0;
    c0 = n0;
    c2 = n2;
    k0 += 0x9E3779B9u;
    k1 += 0xBB67AE85u;
  }
  return make_uint4(c0, c1, c2, c3);
}

// ------------------------------------------------------------------------------------------------
// a2: integer sample from a tail-refined quantile table (R3)
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ int32_t qtab_sample(const int32_t* __restrict__ pool, const DevTab tb,
                                               uint32_t u) {
  const uint32_t L1 = tb.levels - 1, B = tb.log2_cells;
  const uint32_t k = min((uint32_t)__clz((int)~u), L1);  // leading ones, capped at the last level
  const uint32_t drop = (k < L1) ? k + 1 : L1;           // <= 31 because levels <= 32
  const uint32_t r = u << drop;
  const uint32_t m = (r >> 1) >> (31 - B);               // top B bits (B may be 0)
  const uint32_t f = (r >> (16 - B)) & 0xffffu;
  const int32_t* q = pool + tb.off + (k << B) + m;
  const int32_t q0 = __ldg(q), q1 = __ldg(q + 1);
  return q0 + (int32_t)(((int64_t)(q1 - q0) * (int64_t)f) >> 16);
}

// R26: stages the request of type t with route draw u may visit on topology `topo` (0xff: no routing)
__device__ __forceinline__ uint32_t route_stages(const KParams& prm, uint32_t topo, uint32_t t, uint32_t u) {
  if (prm.max_routes == 0u) return 0xffu;
  const TopoRoutes* tr = prm.topo_routes + topo;
  uint32_t r = prm.max_routes - 1u;
  for (int rr = (int)prm.max_routes - 2; rr >= 0; --rr)
    if (u < __ldg(&tr->cum[t][rr])) r = (uint32_t)rr;  // first route with u < cum
  return __ldg(&tr->mask[t][r]);
}

__device__ __forceinline__ uint64_t warp_inclusive_sum(uint64_t v, int lane) {
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const uint64_t o = __shfl_up_sync(0xffffffffu, v, d);
    if (lane >= d) v += o;
  }
  return v;
}

// Component-level record of one request in shared memory (and, for C <= 6, in the HBM stream):
//   w0.x,w0.y = cu (56 bit) | type << 56 ; w0.z,w0.w,w1.* = svc[0..5] ; (C > 6: w2.x,w2.y = svc[6..7])
// In-register mode cu is relative to the start of the 32-request chunk; the consumer adds the base.
// HAS_CPU (R24, 64-bit kernel only): two more words hold the CPU pre-processing times cpu[0..7]
template <int CMAX, bool HAS_CPU = false>
struct CompRec {
  static constexpr int kBase = (CMAX <= 6) ? 2 : 3;  // uint4 words
  static constexpr int kWords = kBase + (HAS_CPU ? 2 : 0);
};

// Stage-level record a warp builds for its topology: cu (absolute) | type<<56, then S[s] per stage
// (-1 = stage not visited by this request's type).
template <int VMAX, bool HAS_CPU = false, bool JOIN = false>
struct StageRec {
  static constexpr int kBase = (VMAX <= 2) ? 1 : (VMAX <= 6 ? 2 : 3);
  static constexpr int kCpu = HAS_CPU ? (VMAX <= 4 ? 1 : 2) : 0;  // + summed CPU time per stage
  static constexpr int kWords = kBase + kCpu + (JOIN ? 1 : 0);    // + predecessor masks of the stages (R25)
};

// ------------------------------------------------------------------------------------------------
// Producer: chunk `chunk` (32 requests starting at n0) of the tile, one request per lane.
// ------------------------------------------------------------------------------------------------
template <int CMAX, bool HAS_CPU = false>
__device__ __forceinline__ void produce_chunk_philox(const KParams& prm, uint32_t n0, uint32_t trial,
                                                     uint32_t variant, uint4* tile_chunk,
                                                     uint64_t* chunk_total, uint32_t* cnt_s,
                                                     int lane) {
  const uint32_t n = n0 + lane;
  const bool valid = n < prm.N;
  uint32_t gap = 0, t = 0, route_u = 0;
  int32_t svc[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) svc[i] = 0;
  if (valid) {
    const uint4 b0 = philox4x32_10(n, trial, 0, variant, prm.seed_lo, prm.seed_hi);
    gap = (uint32_t)qtab_sample(prm.qpool, prm.arr_tab, b0.x);
    route_u = b0.z;  // R26: the route draw (block 0, word 2)
    t = prm.T - 1;
    for (int tt = (int)prm.T - 2; tt >= 0; --tt)
      if (b0.y < prm.type_thresh[tt]) t = tt;  // first tt with u < thresh[tt]
    const uint32_t tm = prm.type_mask[t];
    if (tm & 0x0fu) {
      const uint4 b1 = philox4x32_10(n, trial, 1, variant, prm.seed_lo, prm.seed_hi);
      if (tm & 1u) svc[0] = qtab_sample(prm.qpool, prm.svc_tab[0 * 8 + t], b1.x);
      if (tm & 2u) svc[1] = qtab_sample(prm.qpool, prm.svc_tab[1 * 8 + t], b1.y);
      if (tm & 4u) svc[2] = qtab_sample(prm.qpool, prm.svc_tab[2 * 8 + t], b1.z);
      if (tm & 8u) svc[3] = qtab_sample(prm.qpool, prm.svc_tab[3 * 8 + t], b1.w);
    }
    if (tm & 0xf0u) {
      const uint4 b2 = philox4x32_10(n, trial, 2, variant, prm.seed_lo, prm.seed_hi);
      if (tm & 16u) svc[4] = qtab_sample(prm.qpool, prm.svc_tab[4 * 8 + t], b2.x);
      if (tm & 32u) svc[5] = qtab_sample(prm.qpool, prm.svc_tab[5 * 8 + t], b2.y);
      if (CMAX > 6) {
        if (tm & 64u) svc[6] = qtab_sample(prm.qpool, prm.svc_tab[6 * 8 + t], b2.z);
        if (tm & 128u) svc[7] = qtab_sample(prm.qpool, prm.svc_tab[7 * 8 + t], b2.w);
      }
    }
    atomicAdd(&cnt_s[t], 1u);
  }
  int32_t cpu[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) cpu[i] = 0;
  if (HAS_CPU && valid) {  // R24: CPU times from Philox blocks 3 + i/4, word i % 4
    const uint32_t tm = prm.type_mask[t];
    bool lo = false, hi = false;
#pragma unroll
    for (int i = 0; i < CMAX; ++i) {
      const bool has = ((tm >> i) & 1u) && prm.cpu_tab[i * 8 + t].levels != 0u;
      if (i < 4) lo = lo || has; else hi = hi || has;
    }
    if (lo) {
      const uint4 b3 = philox4x32_10(n, trial, 3, variant, prm.seed_lo, prm.seed_hi);
      const uint32_t u[4] = {b3.x, b3.y, b3.z, b3.w};
#pragma unroll
      for (int i = 0; i < 4 && i < CMAX; ++i)
        if (((tm >> i) & 1u) && prm.cpu_tab[i * 8 + t].levels) cpu[i] = qtab_sample(prm.qpool, prm.cpu_tab[i * 8 + t], u[i]);
    }
    if (hi) {
      const uint4 b4 = philox4x32_10(n, trial, 4, variant, prm.seed_lo, prm.seed_hi);
      const uint32_t u[4] = {b4.x, b4.y, b4.z, b4.w};
#pragma unroll
      for (int i = 4; i < CMAX; ++i)
        if (((tm >> i) & 1u) && prm.cpu_tab[i * 8 + t].levels) cpu[i] = qtab_sample(prm.qpool, prm.cpu_tab[i * 8 + t], u[i - 4]);
    }
  }
  const uint64_t cu = warp_inclusive_sum((uint64_t)gap, lane);  // relative to the chunk start
  if (lane == 31) *chunk_total = cu;
  uint4* dst = tile_chunk + lane * CompRec<CMAX, HAS_CPU>::kWords;
  dst[0] = make_uint4((uint32_t)cu, (uint32_t)(cu >> 32) | (t << 24), (uint32_t)svc[0], (uint32_t)svc[1]);
  dst[1] = make_uint4((uint32_t)svc[2], (uint32_t)svc[3], (uint32_t)svc[4], (uint32_t)svc[5]);
  if (CMAX > 6) dst[2] = make_uint4((uint32_t)svc[6], (uint32_t)svc[7], route_u, 0u);  // routed calls use this record
  if (HAS_CPU) {
    constexpr int kB = CompRec<CMAX, HAS_CPU>::kBase;
    dst[kB] = make_uint4((uint32_t)cpu[0], (uint32_t)cpu[1], (uint32_t)cpu[2], (uint32_t)cpu[3]);
    dst[kB + 1] = make_uint4((uint32_t)cpu[4], (uint32_t)cpu[5], (uint32_t)cpu[6], (uint32_t)cpu[7]);
  }
}

// ------------------------------------------------------------------------------------------------
// Producer of one CTA tile (kTile requests) into buffer tile_idx & 1: in-register Philox draws
// (a1-a3) or a copy of the materialised stream (a10). Shared by both simulation kernels.
// ------------------------------------------------------------------------------------------------
template <int CMAX, int WARPS, bool HAS_CPU = false>
__device__ __forceinline__ void produce_tile(const KParams& prm, uint32_t cta_variant, uint32_t trial,
                                             uint32_t variant, uint32_t tile_idx, uint4* tiles,
                                             uint64_t* totals, uint32_t* cnt_s, int tid, int warp,
                                             int lane) {
  const uint32_t buf = tile_idx & 1u;
  uint4* tb = tiles + buf * kTile * CompRec<CMAX, HAS_CPU>::kWords;
  const uint32_t n0 = tile_idx * kTile;
  if (prm.stream == nullptr) {
    for (int ch = warp; ch < kChunks; ch += WARPS)
      produce_chunk_philox<CMAX, HAS_CPU>(prm, n0 + ch * 32, trial, variant,
                                          tb + ch * 32 * CompRec<CMAX, HAS_CPU>::kWords,
                                          totals + buf * kChunks + ch, cnt_s, lane);
  } else {
    // a10: copy kTile 32-byte records (2 x uint4 each) from the materialised stream; cu is absolute
    const uint4* src = prm.stream + ((size_t)(cta_variant * prm.K + trial) * prm.N + n0) * 2;
    const uint32_t n_words = min((uint32_t)kTile, prm.N - n0) * 2u;
    for (uint32_t w = tid; w < n_words; w += WARPS * 32) {
      const uint4 v = __ldg(src + w);
      tb[w] = v;
      if ((w & 1u) == 0u) atomicAdd(&cnt_s[v.y >> 24], 1u);
    }
    if (tid < kChunks) totals[buf * kChunks + tid] = 0;
  }
}

// ------------------------------------------------------------------------------------------------
// Min-heap replace-min (a6). root = current minimum (register). Nodes 2..c live in shared memory as
// sibling pairs: pair i = nodes (2i, 2i+1) at hb + (i-1)*512 (+ lane*16 folded into hb), fetched
// with one LDS.128; if c is even, node c+1 holds +inf. Top-down sift of the new value x.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void heap_replace_min(uint8_t* smem, int64_t& root, uint32_t hb,
                                                 uint32_t c, int64_t x) {
  if (c < 2) {
    root = x;
    return;
  }
  longlong2 pr = *reinterpret_cast<const longlong2*>(smem + hb);
  bool bl = pr.y < pr.x;
  int64_t m = bl ? pr.y : pr.x;
  if (x <= m) {
    root = x;
    return;
  }
  root = m;
  uint32_t i = 2u + (bl ? 1u : 0u);            // the hole (node index)
  uint32_t hole = hb + (bl ? 8u : 0u);         // its byte address
  while (2u * i <= c) {
    const uint32_t pa = hb + (i - 1u) * 512u;  // pair i = children of node i
    pr = *reinterpret_cast<const longlong2*>(smem + pa);
    bl = pr.y < pr.x;
    m = bl ? pr.y : pr.x;
    if (x <= m) break;
    *reinterpret_cast<int64_t*>(smem + hole) = m;
    hole = pa + (bl ? 8u : 0u);
    i = 2u * i + (bl ? 1u : 0u);
  }
  *reinterpret_cast<int64_t*>(smem + hole) = x;
}

// ------------------------------------------------------------------------------------------------
// The simulation kernel. grid = (CTAs of this launch, K trials); block = kThreads.
// Dynamic shared memory: [tiles 2 x kTile x CompRec][chunk totals][cnt][L][warp stage buffers][heaps]
// ------------------------------------------------------------------------------------------------
template <int VMAX, int CMAX, int WARPS, bool HAS_CPU = false, bool JOIN = false>
struct SmemLayout {
  static constexpr uint32_t kCompRecBytes = CompRec<CMAX, HAS_CPU>::kWords * 16;
  static constexpr uint32_t kStageRecBytes = StageRec<VMAX, HAS_CPU, JOIN>::kWords * 16;
  static constexpr uint32_t tiles = 0;
  static constexpr uint32_t totals = tiles + 2 * kTile * kCompRecBytes;
  static constexpr uint32_t cnt = totals + 2 * kChunks * 8;
  static constexpr uint32_t lus = cnt + 8 * 4;
  static constexpr uint32_t wbuf = lus + 8 * 8;
  static constexpr uint32_t heaps = wbuf + WARPS * 32 * kStageRecBytes;
  static constexpr uint32_t fixed_bytes = heaps;
};

// HAS_CPU: the CPU-GPU overlap rule of PAPER.md:318-320 (R24): a request that finds the earliest-free
// replica idle pays its CPU pre-processing time on top of the GPU time, a queued one GPU time alone
// JOIN: fork-join routing (R25): a request reaches a stage when all its predecessor stages have
// finished (+ the edge delay each), and is done when its last branch is
template <int VMAX, int CMAX, bool HAS_DELAY, int WARPS, bool HAS_CPU = false, bool JOIN = false>
__global__ void __launch_bounds__(WARPS * 32)
cf_sim_kernel(const __grid_constant__ KParams prm, uint32_t cta_base) {
  using SL = SmemLayout<VMAX, CMAX, WARPS, HAS_CPU, JOIN>;
  constexpr int kCW = CompRec<CMAX, HAS_CPU>::kWords, kSW = StageRec<VMAX, HAS_CPU, JOIN>::kWords;
  extern __shared__ __align__(16) uint8_t smem[];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint32_t trial = prm.trial_base + blockIdx.x % prm.k_launch;
  const CtaDesc cta = prm.ctas[cta_base + blockIdx.x / prm.k_launch];
  const uint32_t variant = prm.variant_lo + cta.variant;

  uint4* tiles = reinterpret_cast<uint4*>(smem + SL::tiles);
  uint64_t* totals = reinterpret_cast<uint64_t*>(smem + SL::totals);
  uint32_t* cnt_s = reinterpret_cast<uint32_t*>(smem + SL::cnt);
  int64_t* L_s = reinterpret_cast<int64_t*>(smem + SL::lus);
  uint4* wbuf = reinterpret_cast<uint4*>(smem + SL::wbuf) + warp * 32 * kSW;

  if (tid < 8) {
    cnt_s[tid] = 0;
    L_s[tid] = prm.L_us[tid];
  }
  // a10: with a materialised stream every warp reads the records of its own (variant, trial) straight
  // from HBM, one request per lane (two 128-bit loads); no shared tile
  const bool streamed = prm.stream != nullptr;
  uint32_t my_cnt = 0;  // streamed: lane t counts the requests of type t

  // ---- per-lane simulation state -------------------------------------------------------------
  const bool warp_active = warp < (int)cta.n_warps;
  WarpDesc wd;
  TopoDesc topo;
  uint32_t period = 1, pr = 0, sim_c[VMAX], hb[VMAX];
  bool lane_live = false, rate_bad = false, skip = false;
  int64_t root[VMAX];
#pragma unroll
  for (int s = 0; s < VMAX; ++s) { root[s] = 0; sim_c[s] = 1; hb[s] = 0; }
  if (warp_active) {
    wd = prm.warps[cta.warp_begin + warp];
    topo = prm.topos[wd.topo];
    lane_live = lane < (int)wd.n_lanes;
    const SimDesc sd = prm.sims[wd.sim_begin + (lane_live ? lane : 0)];  // idle lanes mirror lane 0
    pr = sd.pr;
    const uint32_t rate = prm.rates[pr];
    if (rate < 1u || rate > 1000000000u) {
      if (prm.bisect_mode && rate == 0u) skip = true; else rate_bad = true;
    } else {
      period = (1000000000u + rate / 2u) / rate;
    }
    uint32_t row = 0;  // this lane's stages are laid out one after another
#pragma unroll
    for (int s = 0; s < VMAX; ++s) {
      if (s < topo.n_stages) {
        sim_c[s] = prm.plan_c[sd.plan * 8 + s];
        hb[s] = SL::heaps + wd.heap_off + row * 512u + lane * 16u;
        const uint32_t np = heap_pairs(sim_c[s]);
        for (uint32_t j = 0; j < np; ++j) {
          const bool sentinel = (j + 1 == np) && !(sim_c[s] & 1u);  // node c+1 closes an even heap
          *reinterpret_cast<longlong2*>(smem + hb[s] + j * 512u) = make_longlong2(0, sentinel ? kInf : 0);
        }
        row += np;
      }
    }
  }
  // Nothing to do for this CTA? (bisection: every plan's bracket has closed, rate 0; fixup pass:
  // no simulation of this CTA left the 32-bit window)
  bool wanted = warp_active && lane_live && !skip;
  if (prm.fixup) wanted = wanted && prm.flags[(size_t)pr * prm.K + trial] != 0;
  const bool write_out = prm.fixup ? wanted : (warp_active && lane_live);
  if (!__syncthreads_or(wanted)) {
    if (write_out) {  // all-skip CTA: the contract still wants zeros
      const size_t slot = (size_t)pr * prm.K + trial;
      for (uint32_t t = 0; t < 2 * prm.T; ++t) prm.out_counts[slot * prm.T * 2 + t] = 0u;
      if (prm.out_dep_sum) prm.out_dep_sum[slot] = 0ull;
      if (prm.out_makespan) prm.out_makespan[slot] = 0ll;
      if (rate_bad) atomicMin(prm.status, -2);
    }
    return;
  }
  uint32_t hits[8];
#pragma unroll
  for (int t = 0; t < 8; ++t) hits[t] = 0;
  uint64_t dep_sum = 0, cu_base = 0, last_cu = 0;
  int64_t makespan = 0;
  const int64_t delay = prm.edge_delay;
  const bool tracing = prm.tr_arrival != nullptr || prm.tr_departure != nullptr || prm.tr_type != nullptr;

  // ---- producer for one tile -----------------------------------------------------------------
  const uint32_t n_tiles = (prm.N + kTile - 1) / kTile;
  auto produce = [&](uint32_t tile_idx) {
    produce_tile<CMAX, WARPS, HAS_CPU>(prm, cta.variant, trial, variant, tile_idx, tiles, totals, cnt_s, tid, warp, lane);
  };

  __syncthreads();
  if (!streamed) produce(0);
  __syncthreads();
  const uint4* wsrc = streamed && warp_active ? prm.stream + (size_t)(wd.variant * prm.K + trial) * prm.N * 2 : nullptr;

  // a warp none of whose lanes has work (closed brackets; fixup pass: no flagged lane) only helps
  // producing the tiles
  const bool consume = __any_sync(0xffffffffu, wanted);
  for (uint32_t tile_idx = 0; tile_idx < n_tiles; ++tile_idx) {
    if (!streamed && tile_idx + 1 < n_tiles) produce(tile_idx + 1);
    if (consume) {
      const uint32_t buf = tile_idx & 1u;
      const uint4* tb = tiles + buf * kTile * kCW;
      const uint32_t n0 = tile_idx * kTile;
#pragma unroll 1
      for (int ch = 0; ch < kChunks; ++ch) {
        const uint32_t nc0 = n0 + ch * 32;
        if (nc0 >= prm.N) break;
        const int n_here = (int)min(32u, prm.N - nc0);
        // ---- a4: component-level -> stage-level records for this warp's topology -------------
        {
          const uint4* src = tb + (ch * 32 + lane) * kCW;
          uint4 w0 = make_uint4(0u, 0u, 0u, 0u), w1 = w0;
          if (!streamed) {
            w0 = src[0]; w1 = src[1];
          } else if (lane < n_here) {
            w0 = __ldg(wsrc + (size_t)(nc0 + lane) * 2);
            w1 = __ldg(wsrc + (size_t)(nc0 + lane) * 2 + 1);
          }
          int32_t svc[8];
          svc[0] = (int32_t)w0.z; svc[1] = (int32_t)w0.w; svc[2] = (int32_t)w1.x;
          svc[3] = (int32_t)w1.y; svc[4] = (int32_t)w1.z; svc[5] = (int32_t)w1.w;
          svc[6] = 0; svc[7] = 0;
          uint32_t route_u = 0;
          if (CMAX > 6) { const uint4 w2 = src[2]; svc[6] = (int32_t)w2.x; svc[7] = (int32_t)w2.y; route_u = w2.z; }
          const uint32_t t = w0.y >> 24;
          const uint32_t rmask = CMAX > 6 ? route_stages(prm, wd.topo, t, route_u) : 0xffu;  // R26
          if (streamed)
            for (uint32_t tt = 0; tt < prm.T; ++tt) {
              const uint32_t b = __ballot_sync(0xffffffffu, lane < n_here && t == tt);
              if ((uint32_t)lane == tt) my_cnt += __popc(b);
            }
          const uint64_t cu = (((uint64_t)(w0.y & 0x00ffffffu) << 32) | w0.x) + cu_base;
          const uint32_t tm = prm.type_mask[t];
          int32_t cpu[8];
#pragma unroll
          for (int i = 0; i < 8; ++i) cpu[i] = 0;
          if (HAS_CPU) {
            const uint4 c0 = src[CompRec<CMAX, HAS_CPU>::kBase], c1 = src[CompRec<CMAX, HAS_CPU>::kBase + 1];
            cpu[0] = (int32_t)c0.x; cpu[1] = (int32_t)c0.y; cpu[2] = (int32_t)c0.z; cpu[3] = (int32_t)c0.w;
            cpu[4] = (int32_t)c1.x; cpu[5] = (int32_t)c1.y; cpu[6] = (int32_t)c1.z; cpu[7] = (int32_t)c1.w;
          }
          int32_t S[VMAX], Sc[VMAX];
#pragma unroll
          for (int s = 0; s < VMAX; ++s) {
            const uint32_t sm = (s < topo.n_stages) ? topo.mask[s] : 0u;
            int32_t acc = 0, accc = 0;
#pragma unroll
            for (int i = 0; i < CMAX; ++i) {
              acc += ((sm >> i) & 1u) ? svc[i] : 0;
              accc += ((sm >> i) & 1u) ? cpu[i] : 0;
            }
            S[s] = ((sm & tm) && ((rmask >> s) & 1u)) ? acc : -1;
            Sc[s] = accc;
          }
          uint4* dst = wbuf + lane * kSW;
          if (JOIN) {  // the predecessor masks of this topology's stages for the request's type
            const uint2 pm = *reinterpret_cast<const uint2*>(prm.topo_pred + ((size_t)wd.topo * 8 + t) * 8);
            dst[StageRec<VMAX, HAS_CPU, JOIN>::kBase + StageRec<VMAX, HAS_CPU, JOIN>::kCpu] = make_uint4(pm.x, pm.y, 0u, 0u);
          }
          if (HAS_CPU) {
            constexpr int kB = StageRec<VMAX, HAS_CPU>::kBase;
            dst[kB] = make_uint4((uint32_t)Sc[0], (uint32_t)Sc[VMAX > 1 ? 1 : 0], (uint32_t)Sc[VMAX > 2 ? 2 : 0],
                                 (uint32_t)Sc[VMAX > 3 ? 3 : 0]);
            if (VMAX > 4)
              dst[kB + 1] = make_uint4((uint32_t)Sc[VMAX > 4 ? 4 : 0], (uint32_t)Sc[VMAX > 5 ? 5 : 0],
                                       (uint32_t)Sc[VMAX > 6 ? 6 : 0], (uint32_t)Sc[VMAX > 7 ? 7 : 0]);
          }
          const uint32_t hi = (uint32_t)(cu >> 32) | (t << 24);
          if (VMAX <= 2) {
            dst[0] = make_uint4((uint32_t)cu, hi, (uint32_t)S[0], (uint32_t)S[VMAX > 1 ? 1 : 0]);
          } else {
            dst[0] = make_uint4((uint32_t)cu, hi, (uint32_t)S[0], (uint32_t)S[1]);
            dst[1] = make_uint4((uint32_t)S[2], (uint32_t)S[VMAX > 3 ? 3 : 0], (uint32_t)S[VMAX > 4 ? 4 : 0],
                                (uint32_t)S[VMAX > 5 ? 5 : 0]);
            if (VMAX > 6) dst[2] = make_uint4((uint32_t)S[VMAX > 6 ? 6 : 0], (uint32_t)S[VMAX > 7 ? 7 : 0], 0u, 0u);
          }
        }
        __syncwarp();
        // ---- the per-request loop: every lane runs its own simulation over the same 32 requests
        uint64_t hp = 0;  // per-type hit counters of this chunk, one byte each
#pragma unroll 1
        for (int r = 0; r < n_here; ++r) {
          const uint4* rp = wbuf + r * kSW;
          const uint4 w0 = rp[0];
          int32_t Sc[VMAX];
#pragma unroll
          for (int s = 0; s < VMAX; ++s) Sc[s] = 0;
          if (HAS_CPU) {
            constexpr int kB = StageRec<VMAX, HAS_CPU>::kBase;
            const uint4 c0 = rp[kB];
            Sc[0] = (int32_t)c0.x;
            if (VMAX > 1) Sc[1] = (int32_t)c0.y;
            if (VMAX > 2) Sc[2] = (int32_t)c0.z;
            if (VMAX > 3) Sc[3] = (int32_t)c0.w;
            if (VMAX > 4) {
              const uint4 c1 = rp[kB + 1];
              Sc[4] = (int32_t)c1.x;
              if (VMAX > 5) Sc[5] = (int32_t)c1.y;
              if (VMAX > 6) Sc[6] = (int32_t)c1.z;
              if (VMAX > 7) Sc[7] = (int32_t)c1.w;
            }
          }
          int32_t S[VMAX];
          S[0] = (int32_t)w0.z;
          if (VMAX > 1) S[1] = (int32_t)w0.w;
          if (VMAX > 2) {
            const uint4 w1 = rp[1];
            S[2] = (int32_t)w1.x;
            if (VMAX > 3) S[3] = (int32_t)w1.y;
            if (VMAX > 4) S[4] = (int32_t)w1.z;
            if (VMAX > 5) S[5] = (int32_t)w1.w;
          }
          if (VMAX > 6) {
            const uint4 w2 = rp[2];
            S[6] = (int32_t)w2.x;
            if (VMAX > 7) S[7] = (int32_t)w2.y;
          }
          const uint32_t t = w0.y >> 24;
          const uint64_t cu = ((uint64_t)(w0.y & 0x00ffffffu) << 32) | w0.x;
          // a3: A = (CU * period + 2^15) >> 16
          const int64_t A = (int64_t)((cu * (uint64_t)period + 32768ull) >> 16);
          int64_t x = A;
          bool first = true;
          int64_t xs[VMAX], last = A;  // JOIN: departures of the visited stages so far
          uint64_t pmask = 0;
          if (JOIN) {
            const uint4 pw = rp[StageRec<VMAX, HAS_CPU, JOIN>::kBase + StageRec<VMAX, HAS_CPU, JOIN>::kCpu];
            pmask = ((uint64_t)pw.y << 32) | pw.x;
          }
#pragma unroll
          for (int s = 0; s < VMAX; ++s) {
            if (S[s] >= 0) {
              if (JOIN) {
                x = A;
                const uint32_t pm = (uint32_t)(pmask >> (8 * s)) & 0xffu;
#pragma unroll
                for (int sp = 0; sp < s; ++sp)
                  if (((pm >> sp) & 1u) && S[sp] >= 0) { const int64_t a = xs[sp] + delay; x = a > x ? a : x; }
              } else if (HAS_DELAY) { if (!first) x += delay; first = false; }
              const int64_t f = root[s];
              if (HAS_CPU) x = (f <= x) ? x + (int64_t)Sc[s] : f;  // idle: CPU + GPU; queued: GPU alone (R24)
              else x = x > f ? x : f;                              // a5/a6: start at max(arrival, earliest free)
              x += (int64_t)S[s];
              heap_replace_min(smem, root[s], hb[s], sim_c[s], x);
              if (JOIN) { xs[s] = x; last = x > last ? x : last; }
            }
          }
          if (JOIN) x = last;
          // a8
          const bool hit = (x - A) <= L_s[t];
          hp += (uint64_t)(hit ? 1u : 0u) << (t * 8u);
          dep_sum += (uint64_t)x;
          makespan = x > makespan ? x : makespan;
          last_cu = cu;
          if (tracing && warp == 0 && lane == 0) {
            const uint32_t n = nc0 + r;
            if (prm.tr_arrival) prm.tr_arrival[n] = A;
            if (prm.tr_departure) prm.tr_departure[n] = x;
            if (prm.tr_type) prm.tr_type[n] = (uint8_t)t;
          }
        }
#pragma unroll
        for (int t = 0; t < 8; ++t) hits[t] += (uint32_t)(hp >> (8 * t)) & 0xffu;
        __syncwarp();
        if (!streamed) cu_base += totals[buf * kChunks + ch];
      }
    }
    __syncthreads();
  }

  // ---- outputs ---------------------------------------------------------------------------------
  uint32_t cnt_out[8];
#pragma unroll
  for (int t = 0; t < 8; ++t) cnt_out[t] = streamed ? __shfl_sync(0xffffffffu, my_cnt, t) : cnt_s[t];
  if (write_out) {
    // DESIGN.md R17: the arrival horizon CU_N * period + 2^15 must stay below 2^62
    bool bad = rate_bad;
    if (!bad && !skip) {
      const uint64_t hi = __umul64hi(last_cu, (uint64_t)period);
      const uint64_t lo = last_cu * (uint64_t)period;
      if (hi != 0 || lo >= (1ull << 62) - 32768ull) bad = true;
    }
    if (bad) atomicMin(prm.status, -2);
    const bool zero = bad || skip;
    const size_t slot = (size_t)pr * prm.K + trial;
    uint32_t* oc = prm.out_counts + slot * prm.T * 2;
    for (uint32_t t = 0; t < prm.T; ++t) {
      oc[2 * t + 0] = zero ? 0u : cnt_out[t];
      oc[2 * t + 1] = zero ? 0u : hits[t];
    }
    if (prm.out_dep_sum) prm.out_dep_sum[slot] = zero ? 0ull : dep_sum;
    if (prm.out_makespan) prm.out_makespan[slot] = zero ? 0ll : makespan;
  }
}

}  // namespace cfk
