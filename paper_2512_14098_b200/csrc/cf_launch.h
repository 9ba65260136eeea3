// cf_launch.h -- launch entry points of the simulation kernels. Every kernel family is its own
// translation unit (they are compiled in parallel by build.py); cf_api.cu only sees these prototypes.
#pragma once
#include "cf_device.cuh"

namespace cfk {

struct LaunchCfg {
  uint32_t blocks;      // 1-D grid: block b = (schedule block b / k_launch, trial b % k_launch)
  uint32_t smem_bytes;  // dynamic shared memory
  int warps_per_cta;    // 4 or 8
};

// 64-bit kernel (cf_k64.cu): vmax in {2, 6, 8}, cmax in {6, 8}
cudaError_t launch_k64(int vmax, int cmax, const KParams& kp, const LaunchCfg& lc, cudaStream_t st);
int regs_k64(int vmax, int cmax);

// 32-bit fast kernel: cf_k32.cu is compiled once per (VMAX, CMAX) with -DCF_VMAX= -DCF_CMAX=
#define CF_K32_DECL(V, C)                                                                      \
  cudaError_t launch_k32_v##V##c##C(const KParams& kp, const LaunchCfg& lc, cudaStream_t st); \
  int regs_k32_v##V##c##C();
CF_K32_DECL(2, 6)
CF_K32_DECL(4, 6)
CF_K32_DECL(6, 6)
CF_K32_DECL(8, 6)
CF_K32_DECL(8, 8)
#undef CF_K32_DECL

// max-plus scan kernel (cf_scan.cu): cmax in {6, 8}
cudaError_t launch_scan_k(int cmax, const KParams& kp, uint32_t blocks, uint32_t R, uint32_t n_sims,
                          cudaStream_t st);

// arrival-order kernel (cf_fcfs.cu): cmax in {6, 8}, cpl = free-time elements per lane in {1, 2, 4, 8}
cudaError_t launch_fcfs_k(int cmax, bool has_cpu, int cpl, const KParams& kp, const FcfsParams& fp, cudaStream_t st);
// ... and the two launches that draw the request records of the call's kp.k_launch trials
cudaError_t launch_fcfs_records_k(int cmax, bool has_cpu, const KParams& kp, const FcfsParams& fp, cudaStream_t st);

}  // namespace cfk
