// cf_fcfs.cu -- instantiations and launches of the arrival-order kernels (cf_fcfs.cuh).
#include "cf_launch.h"
#include "cf_fcfs.cuh"

namespace cfk {

namespace {
template <int CMAX, bool HAS_CPU>
cudaError_t launch_cpl(int cpl, const KParams& kp, const FcfsParams& fp, cudaStream_t st) {
  const uint32_t blocks = (fp.n_slots + kFcfsWarps - 1) / kFcfsWarps;
  const dim3 b(kFcfsWarps * 32);
  switch (cpl) {
    case 1: cf_fcfs_kernel<CMAX, HAS_CPU, 1><<<blocks, b, 0, st>>>(kp, fp); break;
    case 2: cf_fcfs_kernel<CMAX, HAS_CPU, 2><<<blocks, b, 0, st>>>(kp, fp); break;
    case 4: cf_fcfs_kernel<CMAX, HAS_CPU, 4><<<blocks, b, 0, st>>>(kp, fp); break;
    case 8: cf_fcfs_kernel<CMAX, HAS_CPU, 8><<<blocks, b, 0, st>>>(kp, fp); break;
    default: return cudaErrorInvalidValue;
  }
  return cudaGetLastError();
}
}  // namespace

cudaError_t launch_fcfs_k(int cmax, bool has_cpu, int cpl, const KParams& kp, const FcfsParams& fp, cudaStream_t st) {
  if (fp.n_slots == 0) return cudaErrorInvalidValue;
  if (cmax == 8) return has_cpu ? launch_cpl<8, true>(cpl, kp, fp, st) : launch_cpl<8, false>(cpl, kp, fp, st);
  return has_cpu ? launch_cpl<6, true>(cpl, kp, fp, st) : launch_cpl<6, false>(cpl, kp, fp, st);
}

cudaError_t launch_fcfs_records_k(int cmax, bool has_cpu, const KParams& kp, const FcfsParams& fp, cudaStream_t st) {
  const uint64_t warps = (uint64_t)kp.k_launch * fp.n_seg;
  if (warps == 0 || warps > 0x7fffffffull) return cudaErrorInvalidValue;
  const uint32_t blocks = (uint32_t)((warps + kFcfsWarps - 1) / kFcfsWarps);
  const dim3 b(kFcfsWarps * 32);
  cf_fcfs_totals_kernel<<<blocks, b, 0, st>>>(kp, fp);
  if (cmax == 8) {
    if (has_cpu) cf_fcfs_records_kernel<8, true><<<blocks, b, 0, st>>>(kp, fp);
    else cf_fcfs_records_kernel<8, false><<<blocks, b, 0, st>>>(kp, fp);
  } else {
    if (has_cpu) cf_fcfs_records_kernel<6, true><<<blocks, b, 0, st>>>(kp, fp);
    else cf_fcfs_records_kernel<6, false><<<blocks, b, 0, st>>>(kp, fp);
  }
  return cudaGetLastError();
}

}  // namespace cfk
