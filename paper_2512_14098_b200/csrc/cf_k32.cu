// cf_k32.cu -- instantiations and launches of the 32-bit fast kernel (cf_rel32.cuh) for ONE
// (VMAX, CMAX) pair: build.py compiles this file once per pair with -DCF_VMAX=.. -DCF_CMAX=..
#include "cf_launch.h"
#include "cf_rel32.cuh"

#ifndef CF_VMAX
#error "compile with -DCF_VMAX=<2|4|6|8> -DCF_CMAX=<6|8>"
#endif

#define CF_CAT2(a, b, c, d) a##b##c##d
#define CF_CAT(a, b, c, d) CF_CAT2(a, b, c, d)
#define CF_K32_LAUNCH CF_CAT(launch_k32_v, CF_VMAX, c, CF_CMAX)
#define CF_K32_REGS CF_CAT(regs_k32_v, CF_VMAX, c, CF_CMAX)

namespace cfk {
namespace {

constexpr uint32_t kMaxSmem = 227u * 1024u;

template <bool HAS_DELAY, bool T8, int W>
cudaError_t launch_one(const KParams& kp, const LaunchCfg& lc, cudaStream_t st) {
  auto kern = cf_sim32_kernel<CF_VMAX, CF_CMAX, HAS_DELAY, T8, W>;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kMaxSmem);
  if (e != cudaSuccess) return e;
  kern<<<lc.blocks, W * 32, lc.smem_bytes, st>>>(kp);
  return cudaGetLastError();
}

// cf_trace_sim: one simulation; the delay / 8-type variant covers every call (delay 0 adds 0)
cudaError_t launch_trace(const KParams& kp, const LaunchCfg& lc, cudaStream_t st) {
  auto kern = cf_sim32_kernel<CF_VMAX, CF_CMAX, true, true, 4, true>;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kMaxSmem);
  if (e != cudaSuccess) return e;
  kern<<<lc.blocks, 4 * 32, lc.smem_bytes, st>>>(kp);
  return cudaGetLastError();
}

// materialised stream: per-warp chunk rings, blocks of 4 warps
#if CF_CMAX <= 6
template <bool HAS_DELAY, bool T8>
cudaError_t launch_pw(const KParams& kp, const LaunchCfg& lc, cudaStream_t st) {
  auto kern = cf_sim32_kernel<CF_VMAX, CF_CMAX, HAS_DELAY, T8, 4, false, true>;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kMaxSmem);
  if (e != cudaSuccess) return e;
  kern<<<lc.blocks, 4 * 32, lc.smem_bytes, st>>>(kp);
  return cudaGetLastError();
}
#endif

template <int W>
cudaError_t launch_w(const KParams& kp, const LaunchCfg& lc, cudaStream_t st) {
  const bool d = kp.edge_delay != 0, t8 = kp.T > 4;
  if (d) return t8 ? launch_one<true, true, W>(kp, lc, st) : launch_one<true, false, W>(kp, lc, st);
  return t8 ? launch_one<false, true, W>(kp, lc, st) : launch_one<false, false, W>(kp, lc, st);
}

}  // namespace

cudaError_t CF_K32_LAUNCH(const KParams& kp, const LaunchCfg& lc, cudaStream_t st) {
  if (kp.tr_arrival || kp.tr_departure || kp.tr_type) return lc.warps_per_cta == 4 ? launch_trace(kp, lc, st) : cudaErrorInvalidConfiguration;
  if (kp.stream) {
#if CF_CMAX <= 6
    if (lc.warps_per_cta != 4) return cudaErrorInvalidConfiguration;
    const bool d = kp.edge_delay != 0, t8 = kp.T > 4;
    if (d) return t8 ? launch_pw<true, true>(kp, lc, st) : launch_pw<true, false>(kp, lc, st);
    return t8 ? launch_pw<false, true>(kp, lc, st) : launch_pw<false, false>(kp, lc, st);
#else
    return cudaErrorInvalidConfiguration;
#endif
  }
  return lc.warps_per_cta == 4 ? launch_w<4>(kp, lc, st) : launch_w<8>(kp, lc, st);
}

int CF_K32_REGS() {
  static int regs = [] {
    cudaFuncAttributes a;
    if (cudaFuncGetAttributes(&a, cf_sim32_kernel<CF_VMAX, CF_CMAX, false, true, 8>) != cudaSuccess) {
      cudaGetLastError();
      return 128;  // __launch_bounds__ cap of this build; used when no device is present
    }
    return a.numRegs;
  }();
  return regs;
}

}  // namespace cfk
