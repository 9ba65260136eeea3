// cf_fcfs.cu -- instantiations and launches of the arrival-order kernels (cf_fcfs.cuh).
#include <algorithm>

#include "cf_launch.h"
#include "cf_fcfs.cuh"

namespace cfk {

namespace {
template <int CMAX, bool HAS_CPU>
cudaError_t launch_cpl(int cpl, const KParams& kp, const FcfsParams& fp, cudaStream_t st) {
  // one wave: no more warps than the device holds at once (a simulation in flight is a warp with a
  // scratch slot; the call's simulations take turns on them, so a second, thin wave would only add a tail)
  void (*kern)(KParams, FcfsParams) = nullptr;
  switch (cpl) {
    case 1: kern = cf_fcfs_kernel<CMAX, HAS_CPU, 1>; break;
    case 2: kern = cf_fcfs_kernel<CMAX, HAS_CPU, 2>; break;
    case 4: kern = cf_fcfs_kernel<CMAX, HAS_CPU, 4>; break;
    case 8: kern = cf_fcfs_kernel<CMAX, HAS_CPU, 8>; break;
    default: return cudaErrorInvalidValue;
  }
  int dev = 0, sms = 0, per_sm = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, kFcfsWarps * 32, 0);
  if (e != cudaSuccess) return e;
  FcfsParams f = fp;
  f.n_slots = std::min<uint32_t>(fp.n_slots, (uint32_t)std::max(1, sms * per_sm) * kFcfsWarps);
  const uint32_t blocks = (f.n_slots + kFcfsWarps - 1) / kFcfsWarps;
  kern<<<blocks, kFcfsWarps * 32, 0, st>>>(kp, f);
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
