// cf_rel32.cuh -- the fast path of the simulation kernel (sm_100a). See DESIGN.md section 5.
//
// Same mapping as cf_device.cuh (one thread per simulation, CTA-shared request tiles, per-warp
// stage records), re-coded so that the Kiefer-Wolfowitz heaps -- where the time goes -- work on
// 32-bit keys:
//
//   * every time inside a tile of kTile requests is an offset from a per-lane TILE ORIGIN O = the
//     system arrival of the last request of the previous tile. a3: A_n - O = (r0 + d_n*period) >> 16
//     with d_n the tile-relative cumulative gap (u32) and r0 the low 16 bits of CU_prev*period + 2^15:
//     one IMAD.WIDE and one funnel shift. The running departure x is a 64-bit offset (waits are
//     unbounded under overload);
//   * every stage of every lane has its own 64-bit STAGE BASE (an offset from O); the free times
//     of its c replicas are 30-bit keys relative to that base: the root in the lane's state record,
//     nodes 1..c-1 in a 4-ary min-heap of quads (16 B per lane, interleaved by lane: one
//     conflict-free LDS.128 fetches all four children). A stored key is (key << 2) | slot, so the
//     minimum of the four packed words is the minimum key AND names its slot: no index arithmetic;
//   * the per-request record lists only the stages the request visits (stage ids + services), so a
//     stage that is not visited costs nothing; per-lane stage state lives in shared memory;
//   * a8: hit <=> x - (A_n - O) <= min(L_t, 2^32-1) (a sojourn of 2^32 us or more under a clamped
//     target leaves the fast path); per-type hit counters are byte fields of two 32-bit words
//     flushed every 4 chunks.
//
// At every tile boundary the origin moves forward and every stage base moves to
// max(earliest free time of the stage, new origin); keys below the new base are clamped to it.
// Clamping at the origin is exact: every later request reaches every stage at or after its own
// system arrival >= origin, so a replica that is free before the origin is simply "free"
// (max(arrival, F) = arrival either way) -- DESIGN.md 5.2.
//
// A lane whose arrivals are sparse (an arrival 2^29 us or more past its origin) moves its own origin
// to that arrival in the middle of a tile (same exact rebase), so any rate down to 1 mrps stays here.
//
// A lane leaves the fast path when a key does not fit 30 bits (free times of ONE stage more than
// 17.9 minutes apart), a tile spans >= 2^32 gap units, the rate is outside [1, 1e9] or the R17
// horizon is exceeded. It then sets flags[slot] and writes nothing; the 64-bit kernel of
// cf_device.cuh runs in fixup mode over exactly those simulations. Results are bit-identical.
#pragma once
#include <type_traits>

#include "cf_device.cuh"

namespace cfk {

constexpr uint32_t kInf32 = 0xffffffffu;
constexpr uint32_t kFull = 0xffffffffu;
constexpr uint32_t kKeyLimit = (1u << 30) - 4u;  // keys must stay below this

// Stage-level record of the fast kernel (a warp builds 32 of them per chunk for its topology):
//   w0 = { d (tile-relative cumulative gap, Q16), min(L_t, 2^32-1), hit increment for types 0..3,
//          hit increment for types 4..7 }   (one byte field per type; 0 if L_t < 0)
//   w1 = { stage ids of visits 0..3 (one byte each, 0xff = end), of visits 4..7, S_0, S_1 }
//   w2 = { S_2 .. S_5 },  w3 = { S_6, S_7, -, - }        (S_j = service of the j-th visit)
template <int VMAX>
struct StageRec32 {
  static constexpr int kWords = VMAX <= 2 ? 2 : (VMAX <= 6 ? 3 : 4);
};

// Per-lane, per-stage state record (16 B): { base_lo, base_hi, root key, hb | nq << 18 }: hb = shared
// address of the lane's top heap quad (18 bits; the record's own address when nq == 0, so that the
// request loop can load "the top quad" unconditionally), nq = number of quads
constexpr uint32_t kHbMask = 0x3ffffu;
// PW (materialised stream, a10): no block-shared tile; every warp owns a ring of two 32-record
// chunks (32-byte records) filled by cp.async.bulk behind two mbarriers, and its own type counts
template <int VMAX, int CMAX, int WARPS, bool PW = false>
struct SmemLayout32 {
  static constexpr uint32_t kCompRecBytes = CompRec<CMAX>::kWords * 16;
  static constexpr uint32_t kStageRecBytes = StageRec32<VMAX>::kWords * 16;
  static constexpr uint32_t tiles = 0;   // PW: [warp][2][32] x 32 B
  static constexpr uint32_t totals = tiles + (PW ? WARPS * 2 * 32 * 32 : 2 * kTile * kCompRecBytes);  // PW: [warp][2] mbarriers
  static constexpr uint32_t cnt = totals + (PW ? WARPS * 2 * 8 : 2 * kChunks * 8);                      // PW: [warp][8]
  static constexpr uint32_t l32 = cnt + (PW ? WARPS * 8 * 4 : 8 * 4);
  static constexpr uint32_t inc = l32 + 8 * 4;  // 8 x {lo, hi}
  static constexpr uint32_t wbuf = inc + 8 * 8;
  static constexpr uint32_t state = wbuf + WARPS * 32 * kStageRecBytes;  // [warp][stage][lane] x 16 B
  static constexpr uint32_t heaps = state + WARPS * VMAX * 512;
  static constexpr uint32_t fixed_bytes = heaps;
};

__device__ __forceinline__ uint64_t mad_wide_u32(uint32_t a, uint32_t b, uint64_t c) {
  uint64_t d;
  asm("mad.wide.u32 %0, %1, %2, %3;" : "=l"(d) : "r"(a), "r"(b), "l"(c));
  return d;
}

// explicit shared-window accesses (32-bit shared addresses: no generic-address arithmetic)
__device__ __forceinline__ uint4 lds128(uint32_t a) {
  uint4 v;
  asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(a) : "memory");
  return v;
}
// volatile: ptxas keeps the load where it is written (ahead of the arithmetic that hides its latency)
__device__ __forceinline__ uint4 lds128v(uint32_t a) {
  uint4 v;
  asm volatile("ld.volatile.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(a) : "memory");
  return v;
}
__device__ __forceinline__ void sts128(uint32_t a, uint4 v) {
  asm volatile("st.shared.v4.u32 [%0], {%1,%2,%3,%4};" ::"r"(a), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
__device__ __forceinline__ void sts32(uint32_t a, uint32_t v) {
  asm volatile("st.shared.u32 [%0], %1;" ::"r"(a), "r"(v) : "memory");
}

// ------------------------------------------------------------------------------------------------
// a6: replace-min on a 4-ary min-heap of packed keys. The root key (node 0) is passed in/out in a
// register; quad g holds the children 4g+1..4g+4 of node g at hb + g*512 (lane*16 folded into hb),
// each stored as (key << 2) | slot; nodes >= c hold +inf. nq = heap_quads(c) >= 1.
// Returns the new root key.
// ------------------------------------------------------------------------------------------------
// slot bits of a packed key; opaque to the compiler, which otherwise derives the hole address and the
// child offset from the packed word by separate shift/mask chains (8 instructions per level instead of 4)
__device__ __forceinline__ uint32_t slot_of(uint32_t m) {
  uint32_t k;
  asm("and.b32 %0, %1, 3;" : "=r"(k) : "r"(m));
  return k;
}
__device__ __forceinline__ uint32_t heap4_replace_min(uint32_t hb, uint32_t nq512, uint32_t key, uint4 q) {
  const uint32_t xk = key << 2;  // q = the top quad (at hb), loaded by the caller ahead of time
  uint32_t m = min(min(q.x, q.y), min(q.z, q.w));
  if (xk <= m) return key;  // x <= every child
  const uint32_t new_root = m >> 2;
  uint32_t k = slot_of(m);
  uint32_t hole = hb + 4u * k;       // byte address of the hole; its slot is k
  uint32_t rel = k * 512u + 512u;    // 512 * node index of the hole = byte offset of its children quad
  while (rel < nq512) {
    const uint32_t qa = hb + rel;
    q = lds128(qa);
    m = min(min(q.x, q.y), min(q.z, q.w));
    if (xk <= m) break;
    sts32(hole, (m & ~3u) | k);      // the smallest child moves up into the hole (slot k)
    k = slot_of(m);
    hole = qa + 4u * k;
    rel = 4u * rel + (k * 512u + 512u);
  }
  sts32(hole, xk | k);
  return new_root;
}

// ---- per-warp bulk copies of stream chunks (sm_90+ bulk async copy: one instruction per chunk) -----
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_load(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "CF_WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra CF_DONE_%=;\n"
      "bra CF_WAIT_%=;\n"
      "CF_DONE_%=:\n"
      "}" ::"r"(bar), "r"(parity) : "memory");
}

// packed key p of slot k -> rebased by sh4 = shift << 2 (clamped at 0); +inf stays +inf
__device__ __forceinline__ uint32_t rebase_packed(uint32_t p, uint32_t sh4, uint32_t k) {
  const uint32_t v = (max(p, sh4) - sh4) | k;
  return p == kInf32 ? kInf32 : v;
}

// T8: more than 4 request types (a second word of hit-counter byte fields); WARPS per thread block
// (16 warps per SM either way: 124-128 registers per thread)
// TRACE (cf_trace_sim through this kernel): the call holds one simulation, lane 0 of warp 0; it
// writes every request's system arrival and final departure, the warp's lanes the request types
template <int VMAX, int CMAX, bool HAS_DELAY, bool T8, int WARPS, bool TRACE = false, bool PW = false>
__global__ void __launch_bounds__(WARPS * 32, 16 / WARPS)
cf_sim32_kernel(const __grid_constant__ KParams prm) {
  static_assert(!PW || CMAX <= 6, "the materialised stream holds 32-byte records (C <= 6)");
  using SL = SmemLayout32<VMAX, CMAX, WARPS, PW>;
  constexpr int kW = StageRec32<VMAX>::kWords;
  extern __shared__ __align__(16) uint8_t smem[];
  const uint32_t smem_sa = (uint32_t)__cvta_generic_to_shared(smem);
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint32_t trial = prm.trial_base + blockIdx.x % prm.k_launch;
  const CtaDesc cta = prm.ctas[blockIdx.x / prm.k_launch];
  const uint32_t variant = prm.variant_lo + cta.variant;

  uint4* tiles = reinterpret_cast<uint4*>(smem + SL::tiles);
  uint64_t* totals = reinterpret_cast<uint64_t*>(smem + SL::totals);
  uint32_t* cnt_s = reinterpret_cast<uint32_t*>(smem + SL::cnt) + (PW ? warp * 8 : 0);
  uint32_t* l32_s = reinterpret_cast<uint32_t*>(smem + SL::l32);
  uint2* inc_s = reinterpret_cast<uint2*>(smem + SL::inc);
  uint4* wbuf = reinterpret_cast<uint4*>(smem + SL::wbuf) + warp * 32 * kW;
  // shared addresses of this lane's state records (stage s at + s*512) and of its heap column
  const uint32_t st_sa = smem_sa + SL::state + (uint32_t)warp * VMAX * 512u + (uint32_t)lane * 16u;

  if (PW ? lane < 8 : tid < 8) cnt_s[PW ? lane : tid] = 0;
  if (tid < 8) {
    const int64_t L = prm.L_us[tid];
    // L >= 2^32-1 is held as 2^32-1: exact while the sojourn fits 32 bits; a longer sojourn that
    // misses this bound sends the lane to the 64-bit kernel (see the a8 test below)
    l32_s[tid] = (uint32_t)(L < 0 ? 0 : (L > 0xffffffffll ? 0xffffffffll : L));
    const uint32_t one = (L < 0) ? 0u : (1u << (8 * (tid & 3)));  // L < 0: never a hit
    inc_s[tid] = make_uint2(tid < 4 ? one : 0u, tid < 4 ? 0u : one);
  }

  // ---- per-lane simulation setup -------------------------------------------------------------
  const bool warp_active = warp < (int)cta.n_warps;
  WarpDesc wd;
  wd.heap_off32 = 0; wd.heap_rows32 = 0; wd.topo = 0;
  uint32_t period = 1, pr = 0, plan = 0, n_stages = 0;
  bool lane_live = false, skip = false, flagged = false;
  if (warp_active) {
    wd = prm.warps[cta.warp_begin + warp];
    n_stages = prm.topos[wd.topo].n_stages;
    lane_live = lane < (int)wd.n_lanes;
    const SimDesc sd = prm.sims[wd.sim_begin + (lane_live ? lane : 0)];  // idle lanes mirror lane 0
    pr = sd.pr;
    plan = sd.plan;
    const uint32_t rate = prm.rates[pr];
    if (rate < 1u || rate > 1000000000u) {
      if (prm.bisect_mode && rate == 0u) skip = true; else flagged = true;  // bad rate: the 64-bit kernel reports it
    } else {
      period = (1000000000u + rate / 2u) / rate;
    }
  }
  const bool wanted = warp_active && lane_live && !skip;
  const size_t slot = (size_t)pr * prm.K + trial;
  if (!__syncthreads_or(wanted)) {  // bisection: every bracket of this CTA has closed
    if (warp_active && lane_live) {
      for (uint32_t t = 0; t < 2 * prm.T; ++t) prm.out_counts[slot * prm.T * 2 + t] = 0u;
      if (prm.out_dep_sum) prm.out_dep_sum[slot] = 0ull;
      if (prm.out_makespan) prm.out_makespan[slot] = 0ll;
      prm.flags[slot] = 0;
    }
    return;
  }
  const uint32_t heap_sa = smem_sa + SL::heaps + wd.heap_off32 + (uint32_t)lane * 16u;
  if (warp_active) {
    // all replicas free at time 0: every key 0 (packed with its slot), +inf beyond node c-1
    for (uint32_t j = 0; j < wd.heap_rows32; ++j) sts128(heap_sa + j * 512u, make_uint4(0u, 1u, 2u, 3u));
    uint32_t row = 0;  // this lane's stages are laid out one after another
    for (uint32_t s = 0; s < (uint32_t)VMAX; ++s) {
      uint32_t nq = 0;
      if (s < n_stages) {
        const uint32_t c = prm.plan_c[plan * 8 + s];
        nq = heap_quads(c);
        if (nq) {
          const uint32_t j = nq - 1u;  // only the last quad can hold nodes >= c
          uint32_t v[4];
#pragma unroll
          for (uint32_t e = 0; e < 4; ++e) v[e] = (4u * j + 1u + e >= c) ? kInf32 : e;
          sts128(heap_sa + (row + j) * 512u, make_uint4(v[0], v[1], v[2], v[3]));
        }
      }
      const uint32_t hb = nq ? heap_sa + row * 512u : st_sa + s * 512u;
      sts128(st_sa + s * 512u, make_uint4(0u, 0u, 0u, hb | (nq << 18)));
      row += nq;
    }
  }
  TopoDesc topo;
  if (warp_active) topo = prm.topos[wd.topo];
  constexpr int kTypes = T8 ? 8 : 4;
  uint32_t hits[kTypes];
#pragma unroll
  for (int t = 0; t < kTypes; ++t) hits[t] = 0;
  uint64_t dep_sum = 0, cu_base = 0, tile_base = 0, last_cu = 0;
  uint64_t origin = 0;  // O: absolute time of offset 0 (microseconds)
  uint64_t makespan = 0;
  const uint64_t delay = (uint64_t)prm.edge_delay;

  const uint32_t n_tiles = (prm.N + kTile - 1) / kTile;
  // a warp whose lanes all skip (closed brackets) only helps producing the tiles
  const bool consume = __any_sync(kFull, wanted);
  __syncthreads();
  if (!PW) produce_tile<CMAX, WARPS>(prm, cta.variant, trial, variant, 0, tiles, totals, cnt_s, tid, warp, lane);
  if (!PW) __syncthreads();
  // PW: this warp's records [n] of (its variant, the block's trial), its ring and the two barriers
  const uint4* wsrc = nullptr;
  const uint32_t ring_sa = smem_sa + SL::tiles + (uint32_t)warp * 2048u;
  const uint32_t bar_sa = smem_sa + SL::totals + (uint32_t)warp * 16u;
  const uint32_t n_chunks = (prm.N + 31u) / 32u;
  uint32_t my_cnt = 0;  // PW: lane t counts the requests of type t
  auto fetch = [&](uint32_t g) {  // lane 0: chunk g -> ring slot g & 1
    const uint32_t bytes = min(32u, prm.N - g * 32u) * 32u;
    mbar_expect_tx(bar_sa + (g & 1u) * 8u, bytes);
    bulk_load(ring_sa + (g & 1u) * 1024u, wsrc + (size_t)g * 64u, bytes, bar_sa + (g & 1u) * 8u);
  };
  if (PW) {
    if (!consume) return;  // nothing below synchronises the block
    wsrc = prm.stream + (size_t)(wd.variant * prm.K + trial) * prm.N * 2;
    if (lane == 0) {
      mbar_init(bar_sa, 1u);
      mbar_init(bar_sa + 8u, 1u);
      asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      fetch(0u);
      if (n_chunks > 1u) fetch(1u);
    }
    __syncwarp();
  }

  // the origin moves forward by delta: every stage base goes to max(earliest free time, new origin)
  // and the stage's heap is re-keyed (keys below the new base are clamped to it: DESIGN.md 5.2)
  auto rebase_all = [&](uint64_t delta) {
    for (uint32_t s = 0; s < n_stages; ++s) {
      const uint32_t sa = st_sa + s * 512u;
      const uint4 st = lds128(sa);
      const uint64_t base = ((uint64_t)st.y << 32) | st.x;
      const uint64_t fmin = base + st.z;
      const uint64_t nb = fmin > delta ? fmin : delta;  // new base, still relative to the old origin
      const uint64_t shift = nb - base;                 // >= root key: the new root key is 0
      const uint64_t nbr = nb - delta;                  // ... relative to the new origin
      sts128(sa, make_uint4((uint32_t)nbr, (uint32_t)(nbr >> 32), 0u, st.w));
      const uint32_t sh4 = shift >= (1ull << 30) ? 0xfffffffcu : ((uint32_t)shift << 2);
      const uint32_t nq = st.w >> 18, ha = st.w & kHbMask;
      if (sh4 != 0u)
        for (uint32_t j = 0; j < nq; ++j) {
          uint4 q = lds128(ha + j * 512u);
          q.x = rebase_packed(q.x, sh4, 0u); q.y = rebase_packed(q.y, sh4, 1u);
          q.z = rebase_packed(q.z, sh4, 2u); q.w = rebase_packed(q.w, sh4, 3u);
          sts128(ha + j * 512u, q);
        }
    }
  };
  uint32_t flush_idx = 0;  // requests [flush_idx, current) are accumulated in dep relative to origin

  for (uint32_t tile_idx = 0; tile_idx < n_tiles; ++tile_idx) {
    if (!PW && tile_idx + 1 < n_tiles)
      produce_tile<CMAX, WARPS>(prm, cta.variant, trial, variant, tile_idx + 1, tiles, totals, cnt_s, tid, warp, lane);
    if (consume) {
      const uint32_t buf = tile_idx & 1u;
      const uint4* tb = tiles + buf * kTile * CompRec<CMAX>::kWords;
      const uint32_t n0 = tile_idx * kTile;
      // ---- tile prologue: move the origin to the arrival of the last request before the tile,
      //      every stage base to max(earliest free time, origin), and re-key the stage's heap
      const uint64_t acc0 = tile_base * (uint64_t)period + 32768ull;  // wraps only if R17 fails later
      // a3 constant of this lane: A_n - O = (C + d_n * period) >> 16 (C = the low 16 bits of acc0
      // while O is the tile origin; moving the origin forward by m microseconds subtracts m << 16)
      uint64_t C = acc0 & 0xffffull;
      if (tile_idx != 0) {
        const uint64_t o_new = acc0 >> 16;
        rebase_all(o_new - origin);
        origin = o_new;
      }
      uint32_t hlo = 0, hhi = 0;
      auto flush_hits = [&]() {
#pragma unroll
        for (int t = 0; t < 4; ++t) {
          hits[t] += (hlo >> (8 * t)) & 0xffu;
          if (T8) hits[T8 ? t + 4 : t] += (hhi >> (8 * t)) & 0xffu;
        }
        hlo = 0; hhi = 0;
      };
      uint64_t dep = 0, mk = 0;
#pragma unroll 1
      for (int ch = 0; ch < kChunks; ++ch) {
        const uint32_t nc0 = n0 + ch * 32;
        if (nc0 >= prm.N) break;
        const int n_here = (int)min(32u, prm.N - nc0);
        bool chunk_long = false;
        uint64_t chunk_work = 0;
        // ---- a4: component-level record -> list of visited stages for this warp's topology ----
        {
          const uint32_t g = tile_idx * kChunks + (uint32_t)ch;  // chunk index
          if (PW) mbar_wait(bar_sa + (g & 1u) * 8u, (g >> 1) & 1u);  // the chunk's bytes have landed
          const uint4* src = PW ? tiles + warp * 128 + (g & 1u) * 64 + lane * 2
                                : tb + (ch * 32 + lane) * CompRec<CMAX>::kWords;
          uint4 w0 = src[0], w1 = src[1];
          if (PW && lane >= n_here) w0 = w1 = make_uint4(0u, 0u, 0u, 0u);  // beyond N: the slot holds stale bytes
          int32_t svc[8];
          svc[0] = (int32_t)w0.z; svc[1] = (int32_t)w0.w; svc[2] = (int32_t)w1.x;
          svc[3] = (int32_t)w1.y; svc[4] = (int32_t)w1.z; svc[5] = (int32_t)w1.w;
          svc[6] = 0; svc[7] = 0;
          uint32_t route_u = 0;
          if (CMAX > 6) { const uint4 w2 = src[2]; svc[6] = (int32_t)w2.x; svc[7] = (int32_t)w2.y; route_u = w2.z; }
          const uint32_t t = w0.y >> 24;
          const uint32_t rmask = CMAX > 6 ? route_stages(prm, wd.topo, t, route_u) : 0xffu;  // R26
          if (PW) {
            for (uint32_t tt = 0; tt < prm.T; ++tt) {
              const uint32_t b = __ballot_sync(kFull, lane < n_here && t == tt);
              if ((uint32_t)lane == tt) my_cnt += __popc(b);
            }
            __syncwarp();  // every lane has read its record: the slot may be refilled
            if (lane == 0 && g + 2u < n_chunks) fetch(g + 2u);
          }
          if (TRACE && warp == 0 && lane < n_here && prm.tr_type) prm.tr_type[nc0 + lane] = (uint8_t)t;
          const uint64_t cu = (((uint64_t)(w0.y & 0x00ffffffu) << 32) | w0.x) + cu_base;  // absolute
          const uint64_t d64 = cu - tile_base;
          if (__any_sync(kFull, lane < n_here && (d64 >> 32) != 0)) flagged = true;  // tile too long
          last_cu = __shfl_sync(kFull, cu, n_here - 1);
          const uint32_t tm = prm.type_mask[t];
          const uint2 inc = inc_s[t];
          uint8_t* dst = reinterpret_cast<uint8_t*>(wbuf + lane * kW);
          *reinterpret_cast<uint4*>(dst) = make_uint4((uint32_t)d64, l32_s[t], inc.x, inc.y);
          *reinterpret_cast<uint2*>(dst + 16) = make_uint2(0xffffffffu, 0xffffffffu);  // no visits yet
          uint32_t nv = 0, work = 0;  // work: this request's services (the host caps the worst case at 2^30)
#pragma unroll
          for (int s = 0; s < VMAX; ++s) {
            const uint32_t sm = (s < (int)n_stages) ? topo.mask[s] : 0u;
            if ((sm & tm) && ((rmask >> s) & 1u)) {
              int32_t acc = 0;
#pragma unroll
              for (int i = 0; i < CMAX; ++i) acc += ((sm >> i) & 1u) ? svc[i] : 0;
              dst[16 + nv] = (uint8_t)s;
              *reinterpret_cast<int32_t*>(dst + 24 + 4 * nv) = acc;
              work += (uint32_t)acc;
              ++nv;
            }
          }
          if (lane >= n_here) work = 0;
          // services of the whole chunk (each request's share clamped to 2^26 so the sum fits 32 bits;
          // a longer one makes the chunk "long") plus every possible hop
          chunk_long = __any_sync(kFull, work >= (1u << 26));
          chunk_work = (uint64_t)__reduce_add_sync(kFull, min(work, 1u << 26)) + 32ull * 7ull * delay;
        }
        __syncwarp();
        // ---- the per-request loop: every lane runs its own simulation over the same 32 requests.
        // Loads are issued ahead of their use by hand (the shared-memory accesses are ordered asm):
        // the next record during the current request, the next visit's state record and the current
        // stage's top heap quad before the 64-bit max/add chain.
        const uint32_t wb_sa = smem_sa + SL::wbuf + (uint32_t)warp * 32u * kW * 16u;
        // one request: the record is in (w0..w3); the next record is loaded into (n0..n3).
        // Mode 0 (narrow): every time of this chunk provably fits 32 bits (see the bound below): x,
        // the free times and the SLO test are 32-bit. Mode 1: the running departure x is 64-bit.
        // Mode 2 (sparse arrivals): as mode 1, and a lane whose arrival is 2^29 us or more past its
        // origin first moves its origin to that arrival (a private, exact rebase), so that keys and
        // arrival offsets stay small however long the gaps are.
        uint32_t kmax = 0, mk32 = 0;
        auto request = [&](auto mode_tag, const uint4& w0, const uint4& w1, const uint4& w2, const uint4& w3,
                           uint4& n0w, uint4& n1w, uint4& n2w, uint4& n3w, int r) {
          constexpr int MODE = decltype(mode_tag)::value;
          constexpr bool NARROW = MODE == 0;
          using X = typename std::conditional<NARROW, uint32_t, uint64_t>::type;
          uint32_t sid = w1.x & 0xffu;
          uint4 st;
          if (sid != 0xffu) st = lds128(st_sa + sid * 512u);
          {  // next record (the buffer has 32 records; reading one past the chunk's last is harmless)
            const uint32_t na = wb_sa + (uint32_t)min(r + 1, 31) * (kW * 16u);
            n0w = lds128(na); n1w = lds128(na + 16u);
            if (kW > 2) n2w = lds128(na + 32u);
            if (kW > 3) n3w = lds128(na + 48u);
          }
          // a3: A - O = (C + d * period) >> 16
          uint64_t a64 = mad_wide_u32(w0.x, period, C) >> 16;
          if (MODE == 2 && a64 >= (1ull << 29)) {
            const uint32_t idx = nc0 + (uint32_t)r;  // requests [flush_idx, idx) are in dep
            dep_sum += dep + (uint64_t)(idx - flush_idx) * origin;
            flush_idx = idx;
            dep = 0;
            if (origin + mk > makespan) makespan = origin + mk;
            mk = mk > a64 ? mk - a64 : 0;
            rebase_all(a64);
            origin += a64;
            C -= a64 << 16;
            a64 = 0;
            // the state record of the first visit was loaded before the rebase: reload it
            if ((w1.x & 0xffu) != 0xffu) st = lds128(st_sa + (w1.x & 0xffu) * 512u);
          }
          const uint32_t a = (uint32_t)a64;
          X x = a;
#pragma unroll
          for (int j = 0; j < VMAX; ++j) {
            if (sid == 0xffu) break;  // warp-uniform: all lanes see the same request
            const uint32_t S = j == 0 ? w1.z : j == 1 ? w1.w : j == 2 ? w2.x : j == 3 ? w2.y
                             : j == 4 ? w2.z : j == 5 ? w2.w : j == 6 ? w3.x : w3.y;
            const uint32_t sa = st_sa + sid * 512u;
            const uint4 cur = st;
            const uint32_t nq512 = (cur.w >> 9) & ~0x1ffu, hb = cur.w & kHbMask;  // nq * 512
            const uint4 q = lds128v(hb);  // top quad of this stage's heap (the state record if nq == 0)
            if (j + 1 < VMAX) {          // state record of the next visit
              sid = __byte_perm(j + 1 < 4 ? w1.x : w1.y, 0u, 0x4440u + ((j + 1) & 3));  // one PRMT
              uint4 nxt;  // left undefined after the last visit: no copy of the old record is kept
              if (sid != 0xffu) nxt = lds128(st_sa + sid * 512u);
              st = nxt;
            } else {
              sid = 0xffu;
            }
            uint32_t key;
            if (NARROW) {
              const uint32_t f = cur.x + cur.z;  // earliest free time of the stage (base_hi == 0)
              if (HAS_DELAY && j > 0) x += (X)delay;
              x = max((uint32_t)x, f) + S;       // a5/a6: start at max(arrival, earliest free)
              key = (uint32_t)x - cur.x;
              kmax = max(kmax, key);             // window check after the chunk
            } else {
              const uint64_t base = ((uint64_t)cur.y << 32) | cur.x;
              const uint64_t f = base + cur.z;
              if (HAS_DELAY && j > 0) x += (X)delay;
              x = (X)(((uint64_t)x > f ? (uint64_t)x : f) + S);
              const uint64_t key64 = (uint64_t)x - base;
              if (key64 >= (uint64_t)kKeyLimit) flagged = true;
              key = (uint32_t)key64;
            }
            if (nq512) key = heap4_replace_min(hb, nq512, key, q);
            sts32(sa + 8u, key);
          }
          if (TRACE && tid == 0) {  // lane 0 of warp 0 is the traced simulation
            const uint32_t n = nc0 + (uint32_t)r;
            if (prm.tr_arrival) prm.tr_arrival[n] = (int64_t)(origin + a);
            if (prm.tr_departure) prm.tr_departure[n] = (int64_t)(origin + (uint64_t)x);
          }
          // a8
          if (NARROW) {
            if ((uint32_t)x - a <= w0.y) { hlo += w0.z; if (T8) hhi += w0.w; }  // sojourn < 2^32 here
            dep = mad_wide_u32((uint32_t)x, 1u, dep);
            mk32 = max(mk32, (uint32_t)x);
          } else {
            const uint64_t soj = (uint64_t)x - a;
            if (soj <= (uint64_t)w0.y) { hlo += w0.z; if (T8) hhi += w0.w; }
            else if (w0.y == 0xffffffffu) flagged = true;  // L_t >= 2^32-1 was clamped: the 64-bit kernel decides
            dep += (uint64_t)x;
            mk = (uint64_t)x > mk ? (uint64_t)x : mk;
          }
        };
        // Bound for the chunk: every departure is at most M + (all services and hops of the chunk),
        // M = max(latest departure so far, last arrival of the chunk), both relative to the origin
        // (induction over x = max(arrival, F) + S; every free time is some earlier departure).
        const uint64_t a_last = mad_wide_u32((uint32_t)(last_cu - tile_base), period, C) >> 16;
        uint64_t seen = makespan > origin ? makespan - origin : 0;
        if (mk > seen) seen = mk;
        if (a_last > seen) seen = a_last;
        const bool sparse = __any_sync(kFull, a_last >= (1ull << 29));
        const bool narrow = __all_sync(kFull, !chunk_long && seen + chunk_work < 0xffffffffull);
        uint4 a0 = lds128(wb_sa), a1 = lds128(wb_sa + 16u);
        uint4 a2 = make_uint4(0, 0, 0, 0), a3 = make_uint4(0, 0, 0, 0);
        if (kW > 2) a2 = lds128(wb_sa + 32u);
        if (kW > 3) a3 = lds128(wb_sa + 48u);
        uint4 b0, b1, b2 = make_uint4(0, 0, 0, 0), b3 = make_uint4(0, 0, 0, 0);
        int r = 0;
        if (sparse) {
          const std::integral_constant<int, 2> tag;
#pragma unroll 1
          for (; r < n_here; ++r) {
            request(tag, a0, a1, a2, a3, b0, b1, b2, b3, r);
            a0 = b0; a1 = b1; a2 = b2; a3 = b3;
          }
        } else if (narrow) {
          const std::integral_constant<int, 0> tag;
#pragma unroll 1
          for (; r + 1 < n_here; r += 2) {  // two requests per trip: the record registers ping-pong
            request(tag, a0, a1, a2, a3, b0, b1, b2, b3, r);
            request(tag, b0, b1, b2, b3, a0, a1, a2, a3, r + 1);
          }
          if (r < n_here) request(tag, a0, a1, a2, a3, b0, b1, b2, b3, r);
          if (kmax >= kKeyLimit) flagged = true;
          if (mk32 > mk) mk = mk32;
        } else {
          const std::integral_constant<int, 1> tag;
#pragma unroll 1
          for (; r + 1 < n_here; r += 2) {
            request(tag, a0, a1, a2, a3, b0, b1, b2, b3, r);
            request(tag, b0, b1, b2, b3, a0, a1, a2, a3, r + 1);
          }
          if (r < n_here) request(tag, a0, a1, a2, a3, b0, b1, b2, b3, r);
        }
        __syncwarp();
        if (!PW) cu_base += totals[buf * kChunks + ch];
        if ((ch & 3) == 3) flush_hits();  // a byte field holds at most 128 hits
      }
      // ---- tile epilogue: absolute outputs, window checks
      const uint32_t idx_end = min(n0 + (uint32_t)kTile, prm.N);
      dep_sum += dep + (uint64_t)(idx_end - flush_idx) * origin;
      flush_idx = idx_end;
      makespan = max(makespan, origin + mk);
      tile_base = last_cu;
      flush_hits();
    }
    if (!PW) __syncthreads();
  }
  if (PW) {  // the warp's type counts -> its row of cnt_s
    if (lane < 8) cnt_s[lane] = my_cnt;
    __syncwarp();
  }

  // ---- outputs ---------------------------------------------------------------------------------
  if (warp_active && lane_live) {
    if (!skip && !flagged) {  // DESIGN.md R17: the 64-bit kernel zeroes the outputs and raises the status
      const uint64_t hi = __umul64hi(last_cu, (uint64_t)period);
      const uint64_t lo = last_cu * (uint64_t)period;
      if (hi != 0 || lo >= (1ull << 62) - 32768ull) flagged = true;
    }
    const bool redo = flagged && !skip;
    prm.flags[slot] = redo ? 1 : 0;
    if (redo) {
      atomicAdd(reinterpret_cast<uint32_t*>(prm.status) + 1, 1u);
    } else {
      uint32_t* oc = prm.out_counts + slot * prm.T * 2;
      for (uint32_t t = 0; t < prm.T; ++t) {
        oc[2 * t + 0] = skip ? 0u : cnt_s[t];
        oc[2 * t + 1] = skip ? 0u : hits[t < (uint32_t)kTypes ? t : 0];
      }
      if (prm.out_dep_sum) prm.out_dep_sum[slot] = skip ? 0ull : dep_sum;
      if (prm.out_makespan) prm.out_makespan[slot] = skip ? 0ll : (int64_t)makespan;
    }
  }
}

}  // namespace cfk
