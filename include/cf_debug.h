/*
 * cf_debug.h -- test, tuning and bench hooks of libcf_b200.so. NOT part of the product ABI (cf.h):
 * nothing here is needed to evaluate plans. The hooks select among code paths that all return
 * bit-identical results (tests run every path against the CPU oracle), or report bookkeeping.
 *
 * There are no process-wide knobs: a choice is made per call through a cf_options argument of the
 * *_opt twins of the cf.h entry points (opt == NULL: defaults, i.e. exactly the cf.h call).
 */
#ifndef CF_DEBUG_H
#define CF_DEBUG_H

#include "cf.h"

#ifdef __cplusplus
extern "C" {
#endif

enum {
  CF_KERNEL_AUTO = 0,   /* 32-bit fast kernel + 64-bit fixup pass, or the max-plus scan kernel for
                           one-replica calls with <= 8192 simulations           */
  CF_KERNEL_WIDE64 = 1, /* the 64-bit thread-per-simulation kernel only (cf_device.cuh)             */
  CF_KERNEL_FAST32 = 2, /* as AUTO but never the scan kernel; cf_trace_sim_opt traces the fast kernel */
  CF_KERNEL_SCAN = 3    /* the max-plus scan kernel; CF_ERR_ARG unless every stage has one replica
                           and the call has <= 8192 simulations                                      */
};

typedef struct {
  uint32_t kernel_mode;    /* CF_KERNEL_*                                                            */
  uint32_t bisect_depth;   /* bisection steps simulated per pass (speculative decision tree of
                              2^depth - 1 rates per plan): 0 = chosen from P*K, 1..4  */
  uint32_t bisect_predict; /* 0 = default (on where the pass would otherwise be over-subscribed),
                              1 = always simulate the full tree, 2 = always predict  */
  uint32_t reserved[5];    /* must be 0                                                              */
} cf_options;

int32_t cf_eval_plans_opt(const cf_options* opt, const cf_graph* g, const cf_plans* pl,
                          const uint32_t* rate_mrps, uint32_t R, const cf_slo* slo, uint64_t seed,
                          uint32_t variant, uint32_t* out_counts, uint64_t* out_dep_sum,
                          int64_t* out_makespan, void* workspace, size_t workspace_bytes, void* stream);
int32_t cf_eval_plans_stream_opt(const cf_options* opt, const cf_graph* g, const cf_plans* pl,
                                 const uint32_t* rate_mrps, uint32_t R, const cf_slo* slo,
                                 const void* stream_records, uint32_t n_variants,
                                 const uint32_t* plan_variant, uint32_t* out_counts,
                                 uint64_t* out_dep_sum, int64_t* out_makespan, void* workspace,
                                 size_t workspace_bytes, void* stream);
int32_t cf_goodput_bisect_opt(const cf_options* opt, const cf_graph* g, const cf_plans* pl,
                              const uint32_t* rate_hi_mrps, uint32_t n_steps, const cf_slo* slo,
                              uint64_t seed, uint32_t variant, uint32_t* out_rate_mrps,
                              uint32_t* out_goodput_mrps, uint32_t* out_counts, void* workspace,
                              size_t workspace_bytes, void* stream);
int32_t cf_goodput_bisect_stream_opt(const cf_options* opt, const cf_graph* g, const cf_plans* pl,
                                     const uint32_t* rate_hi_mrps, uint32_t n_steps, const cf_slo* slo,
                                     const void* stream_records, uint32_t n_variants,
                                     const uint32_t* plan_variant, uint32_t* out_rate_mrps,
                                     uint32_t* out_goodput_mrps, uint32_t* out_counts,
                                     void* workspace, size_t workspace_bytes, void* stream);
/* kernel_mode CF_KERNEL_AUTO / WIDE64: the 64-bit kernel; FAST32: the fast kernel (then its fixup
 * pass); SCAN: the scan kernel (the traced plan must have one replica at every stage). */
int32_t cf_trace_sim_opt(const cf_options* opt, const cf_graph* g, const cf_plans* pl, uint32_t plan,
                         uint32_t rate_mrps, uint32_t trial, uint64_t seed, uint32_t variant,
                         int64_t* out_arrival, int64_t* out_departure, uint8_t* out_type,
                         void* workspace, size_t workspace_bytes, void* stream);

/* Bookkeeping for bench.py's `gpu_launches`: kernels enqueued by the last compute call made on the
 * calling host thread (a thread-local statistic; nothing in the library reads it). */
uint32_t cf_last_launch_count(void);

/* Micro-benchmark used by bench.py for the ALU roofline denominator: runs `iters` rounds of an
 * unrolled, independent 32-bit integer instruction mix on every SM and writes the number of
 * lane-operations executed to *out_ops (host). mix: 0 = IADD3/LOP3 only (ALU pipe), 1 = IMAD only
 * (FMA pipe), 2 = alternating. Returns the elapsed milliseconds * 1000 (microseconds) in
 * *out_usec (host), measured with CUDA events on `stream`. Synchronises. */
int32_t cf_bench_int32_peak(uint32_t mix, uint32_t iters, uint64_t* out_ops, uint64_t* out_usec,
                            void* stream);

#ifdef __cplusplus
}
#endif
#endif
