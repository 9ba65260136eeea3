// cf_k64.cu -- instantiations and launches of the 64-bit simulation kernel (cf_device.cuh).
#include "cf_launch.h"

namespace cfk {
namespace {

constexpr uint32_t kMaxSmem = 227u * 1024u;

template <int VMAX, int CMAX, bool HAS_DELAY, int W, bool HAS_CPU = false, bool JOIN = false>
cudaError_t launch_one(const KParams& kp, const LaunchCfg& lc, cudaStream_t st) {
  auto kern = cf_sim_kernel<VMAX, CMAX, HAS_DELAY, W, HAS_CPU, JOIN>;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kMaxSmem);
  if (e != cudaSuccess) return e;
  kern<<<lc.blocks, W * 32, lc.smem_bytes, st>>>(kp, 0u);
  return cudaGetLastError();
}

template <int VMAX, int CMAX>
cudaError_t launch_v(const KParams& kp, const LaunchCfg& lc, cudaStream_t st) {
  const bool d = kp.edge_delay != 0;
  if (kp.join) {  // fork-join routing (R25): the CPU variant covers graphs without CPU tables (times of 0)
    if (lc.warps_per_cta == 4) return launch_one<VMAX, CMAX, true, 4, true, true>(kp, lc, st);
    return launch_one<VMAX, CMAX, true, 8, true, true>(kp, lc, st);
  }
  if (kp.has_cpu) {  // CPU-GPU overlap (R24): the delay variant covers delay 0 as well
    if (lc.warps_per_cta == 4) return launch_one<VMAX, CMAX, true, 4, true>(kp, lc, st);
    return launch_one<VMAX, CMAX, true, 8, true>(kp, lc, st);
  }
  if (lc.warps_per_cta == 4)
    return d ? launch_one<VMAX, CMAX, true, 4>(kp, lc, st) : launch_one<VMAX, CMAX, false, 4>(kp, lc, st);
  return d ? launch_one<VMAX, CMAX, true, 8>(kp, lc, st) : launch_one<VMAX, CMAX, false, 8>(kp, lc, st);
}

template <int VMAX, int CMAX>
int regs_of() {
  static int regs = [] {
    cudaFuncAttributes a;
    if (cudaFuncGetAttributes(&a, cf_sim_kernel<VMAX, CMAX, false, 8>) != cudaSuccess) {
      cudaGetLastError();
      return VMAX <= 2 ? 64 : 128;  // ptxas figures of this build; used when no device is present
    }
    return a.numRegs;
  }();
  return regs;
}

}  // namespace

cudaError_t launch_k64(int vmax, int cmax, const KParams& kp, const LaunchCfg& lc, cudaStream_t st) {
  if (cmax == 8) return launch_v<8, 8>(kp, lc, st);
  if (vmax == 2) return launch_v<2, 6>(kp, lc, st);
  if (vmax == 6) return launch_v<6, 6>(kp, lc, st);
  return launch_v<8, 6>(kp, lc, st);
}

int regs_k64(int vmax, int cmax) {
  if (cmax == 8) return regs_of<8, 8>();
  if (vmax == 2) return regs_of<2, 6>();
  if (vmax == 6) return regs_of<6, 6>();
  return regs_of<8, 6>();
}

}  // namespace cfk
