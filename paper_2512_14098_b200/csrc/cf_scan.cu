// cf_scan.cu -- instantiations and launches of the max-plus scan kernel (cf_scan.cuh).
#include "cf_launch.h"
#include "cf_scan.cuh"

namespace cfk {

cudaError_t launch_scan_k(int cmax, const KParams& kp, uint32_t blocks, uint32_t R, uint32_t n_sims,
                          cudaStream_t st) {
  const uint32_t* pv = kp.stream ? kp.plan_var : nullptr;
  if (cmax == 8)
    cf_scan_kernel<8><<<blocks, kScanWarps * 32, 0, st>>>(kp, kp.plan_topo, pv, R, n_sims);
  else
    cf_scan_kernel<6><<<blocks, kScanWarps * 32, 0, st>>>(kp, kp.plan_topo, pv, R, n_sims);
  return cudaGetLastError();
}

}  // namespace cfk
