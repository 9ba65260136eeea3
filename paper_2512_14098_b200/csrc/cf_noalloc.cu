// cf_noalloc.cu -- cf_pareto_select_static: Pareto pruning + policy (Algorithm 2 l.12, 16-18,
// PAPER.md:251-259; R23) for callers that cannot provide device scratch because they cannot
// allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
//
// The scratch of this variant lives in ONE file-scope device array of a fixed, modest size that every
// GPU which loads the library holds until the process exits:
//     kStaticMaxPlans = 65 536 plans  ->  (32 + 65 536) x 8 B = 512.25 KiB per device.
// scratch[0]      = max over live plans of (sum of goodput + 1)   (must start at 0: cleared per call)
// scratch[32 + p] = sum of plan p's goodput vector                (written before it is read)
// The entry point calls no cudaMalloc / cudaFree / allocating library routine: three kernel launches
// and, once per device, cudaGetSymbolAddress. All calls on a device SHARE the array and it keeps the
// last call's contents: two calls that overlap on the GPU (different streams, or graph branches that
// may run concurrently) race on it -- keep them on one stream or order them with events.
//
// In host code the NAME of a __device__ array is a host-side stand-in, not a device address, so the
// host side below never passes `g_pareto_scratch` to a kernel: it asks the runtime for the device
// address (cudaGetSymbolAddress, with the target device current, once per device) and passes that.
// This file shares no kernel with cf_api.cu's cf_pareto_select: that path is unchanged.
#include <cstdint>
#include <cstdio>
#include <mutex>

#include <cuda_runtime.h>

#include "../../include/cf.h"

static constexpr uint32_t kStaticMaxPlans = CF_PARETO_STATIC_MAX_PLANS;
static constexpr uint32_t kSumBase = 32;  // scratch[32 + p]: 256-byte aligned start of the per-plan sums
static constexpr int kMaxDevices = 64;

static __device__ __align__(256) unsigned long long g_pareto_scratch[kSumBase + kStaticMaxPlans];

namespace {

std::mutex g_addr_mutex;
unsigned long long* g_scratch_addr[kMaxDevices] = {nullptr};  // device address of the array, per device

// device address of this device's copy of the array; `dev` is the CURRENT device
cudaError_t scratch_address(int dev, unsigned long long** out) {
  std::lock_guard<std::mutex> lk(g_addr_mutex);
  if (!g_scratch_addr[dev]) {
    void* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&p, g_pareto_scratch);
    if (e != cudaSuccess) return e;
    g_scratch_addr[dev] = static_cast<unsigned long long*>(p);
  }
  *out = g_scratch_addr[dev];
  return cudaSuccess;
}

__global__ void pareto_static_init_kernel(unsigned long long* scratch, uint32_t* out_best, uint32_t* out_n) {
  scratch[0] = 0ull;  // the array keeps the last call's maximum
  if (out_best) *out_best = 0xffffffffu;
  if (out_n) *out_n = 0u;
}

// one thread per plan p; candidate dominators q staged through shared memory 256 at a time (R23:
// strict dominance, only live plans dominate). Also leaves sum_t G_p[t] in scratch[32 + p].
template <int T>
__global__ void __launch_bounds__(256)
pareto_static_dom_kernel(const uint32_t* __restrict__ G, uint32_t P, const uint8_t* __restrict__ alive,
                         uint8_t* out_pruned, uint32_t* out_n, unsigned long long* scratch) {
  __shared__ uint32_t gq[256 * T];
  __shared__ uint8_t lq[256];
  const uint32_t p = blockIdx.x * 256 + threadIdx.x;
  uint32_t gp[T];
  const bool live = p < P && (!alive || alive[p]);
  unsigned long long sum = 0;
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
    scratch[kSumBase + p] = sum;
    if (live) atomicMax(scratch, sum + 1ull);
  }
  const uint32_t surv = __syncthreads_count(live && !dominated);
  if (threadIdx.x == 0 && surv && out_n) atomicAdd(out_n, surv);
}

// default policy: the live plan with the largest sum of goodput, lowest index on ties
__global__ void __launch_bounds__(256)
pareto_static_best_kernel(uint32_t P, const uint8_t* __restrict__ alive, const unsigned long long* scratch,
                          uint32_t* out_best) {
  const uint32_t p = blockIdx.x * 256 + threadIdx.x;
  if (p >= P || (alive && !alive[p])) return;
  if (scratch[kSumBase + p] + 1ull == scratch[0]) atomicMin(out_best, p);
}

template <int T>
void launch_dom(const uint32_t* G, uint32_t P, const uint8_t* alive, uint8_t* out_pruned, uint32_t* out_n,
                unsigned long long* scratch, cudaStream_t st) {
  pareto_static_dom_kernel<T><<<(P + 255) / 256, 256, 0, st>>>(G, P, alive, out_pruned, out_n, scratch);
}

}  // namespace

extern "C" {

uint32_t cf_pareto_static_max_plans(void) { return kStaticMaxPlans; }

int32_t cf_pareto_select_static(const uint32_t* goodput_mrps, uint32_t n_plans, uint32_t n_types,
                                const uint8_t* alive, uint8_t* out_pruned, uint32_t* out_best,
                                uint32_t* out_n_survivors, void* stream) {
  if (!goodput_mrps || !out_pruned || n_plans < 1 || n_types < 1 || n_types > 8) return CF_ERR_ARG;
  if (n_plans > kStaticMaxPlans) {
    std::fprintf(stderr, "libcf_b200: cf_pareto_select_static: %u plans exceed the static scratch (at most %u); "
                         "use cf_pareto_select with a caller-provided workspace\n", n_plans, kStaticMaxPlans);
    return CF_ERR_RANGE;
  }
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e == cudaSuccess && (dev < 0 || dev >= kMaxDevices)) e = cudaErrorInvalidDevice;
  unsigned long long* scratch = nullptr;
  if (e == cudaSuccess) e = scratch_address(dev, &scratch);
  if (e != cudaSuccess) {
    std::fprintf(stderr, "libcf_b200: CUDA error: %s\n", cudaGetErrorString(e));
    return CF_ERR_CUDA;
  }
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  pareto_static_init_kernel<<<1, 1, 0, st>>>(scratch, out_best, out_n_survivors);
  switch (n_types) {
    case 1: launch_dom<1>(goodput_mrps, n_plans, alive, out_pruned, out_n_survivors, scratch, st); break;
    case 2: launch_dom<2>(goodput_mrps, n_plans, alive, out_pruned, out_n_survivors, scratch, st); break;
    case 3: launch_dom<3>(goodput_mrps, n_plans, alive, out_pruned, out_n_survivors, scratch, st); break;
    case 4: launch_dom<4>(goodput_mrps, n_plans, alive, out_pruned, out_n_survivors, scratch, st); break;
    case 5: launch_dom<5>(goodput_mrps, n_plans, alive, out_pruned, out_n_survivors, scratch, st); break;
    case 6: launch_dom<6>(goodput_mrps, n_plans, alive, out_pruned, out_n_survivors, scratch, st); break;
    case 7: launch_dom<7>(goodput_mrps, n_plans, alive, out_pruned, out_n_survivors, scratch, st); break;
    default: launch_dom<8>(goodput_mrps, n_plans, alive, out_pruned, out_n_survivors, scratch, st); break;
  }
  if (out_best)
    pareto_static_best_kernel<<<(n_plans + 255) / 256, 256, 0, st>>>(n_plans, alive, scratch, out_best);
  e = cudaGetLastError();
  if (e != cudaSuccess) {
    std::fprintf(stderr, "libcf_b200: CUDA error: %s\n", cudaGetErrorString(e));
    return CF_ERR_CUDA;
  }
  return CF_OK;
}

}  // extern "C"
