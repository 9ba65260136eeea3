#!/usr/bin/env python
"""bench.py -- request-stage simulation updates/s of the plan-evaluation hot path on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1] [--impl ours|reference]

A "step" is one pass of the whole hot path over one BASELINE.json
config: every (plan, rate, trial) simulation of the config through the C ABI (cf_eval_plans, or the
materialised stream + cf_goodput_bisect_stream for config 4). Default workload: configs[1].
Prints ONE JSON line.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2512_14098_b200 import workloads as W  # noqa: E402

METRIC = "request-stage sim updates/s"
UNIT = "updates/s"

# Algorithmic INT32 lane-operations of the method: per request
# (arrival scaling, type decode, SLO test, checksum, makespan), per visited stage (visit test, 64-bit
# max + add) and per heap level the Kiefer-Wolfowitz replace-min has to descend (two 64-bit loads,
# two 64-bit compares, select, store, index arithmetic).
OPS_PER_REQUEST = 18
OPS_PER_UPDATE = 7
OPS_PER_HEAP_LEVEL = 11

# dram__bytes_read.sum + dram__bytes_write.sum of the simulation kernel, per launch at full size,
# from the ncu captures in profiles/r01_ncu_full_s31_cfg2s_cfg1.txt (config 1) and
# profiles/r01_ncu_metrics_cfg2_fullsize_s31.csv (config 2) (the outputs stay in the 126 MB L2
# past the end of the launch, so almost nothing is written back in time; what is read is the
# schedule, the tables and cold-cache instruction fetch, and varies by a few hundred KB per capture)
NCU_TRAFFIC_BYTES = {1: 657_152, 2: 1_164_032}


def make_workload(cfg: int, scale: float = 1.0):
    if cfg == 0:
        return [W.config0_mm1(m) for m in W.CONFIG0_SERVICE_MEANS_US]
    if cfg == 1:
        return [W.config1_mllm(n_req=max(1, int(100_000 * scale)))]
    if cfg == 2:
        return [W.config2_omni(n_req=max(1, int((1 << 17) * scale)))]
    if cfg == 3:
        return [W.config3_multireplica(n_req=max(1, int((1 << 16) * scale)))]
    if cfg == 4:
        return [W.config4_sweep(n_req=max(1, int((1 << 18) * scale)))]
    raise SystemExit(f"unknown config {cfg}")


def workload_name(cfg: int) -> str:
    return ["cfg0 M/M/1 sanity (8 calls)", "cfg1 MLLM 2-stage Encoder->LLM, 512 plans x 16 rates x 8 trials x 100k req",
            "cfg2 Omni 6-comp, 4096 plans x 16 rates x 8 trials x 2^17 req",
            "cfg3 multi-replica stress, 16384 plans x 8 rates x 4 trials x 2^16 req, Gamma CV=3",
            "cfg4 coarse-to-fine sweep, 4096 plans x 32-step bisection x 8 trials x 2^18 req, stream in HBM"][cfg]


class ClockSampler:
    """nvidia-smi clocks/throttle reasons during the timed region (B200_PROFILING.md recipe)."""

    def __init__(self, index: int):
        self.rows = []
        self.proc = None
        self.index = index

    def start(self):
        q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, reasons, power = [], [], set(), []
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); power.append(float(r[2]))
            except (ValueError, IndexError):
                continue
            names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
            for nm, v in zip(names, r[4:8]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None,
                "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(power) if power else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def oracle_sample(w, budget_s: float, n_threads: int):
    """The oracle, as it stands, on a bounded sample of the workload: whole plans (all their rates
    and trials) taken at a stride until ~budget_s seconds of wall time are spent. Returns
    (updates, seconds, description)."""
    from oracle import cf_oracle as orc
    P = w.plans.n_plans
    order = np.random.default_rng(0).permutation(P)
    done_updates, spent, n_done = 0, 0.0, 0
    batch = max(1, n_threads // 2)
    if w.rate_mrps is None:  # bisection config: sample = eval at 2 rates around 0.6/0.9 of the bound
        rates_all = W.rate_grid(W.flow_bound_mrps(w.graph, w.plans), [0.6, 0.9])
    else:
        rates_all = w.rate_mrps
    while spent < budget_s and n_done < P:
        idx = order[n_done:n_done + batch]
        t0 = time.perf_counter()
        o = orc.eval_plans(w.graph, w.plans.subset(idx), rates_all[idx], w.slo, w.seed, n_threads=n_threads)
        dt = time.perf_counter() - t0
        spent += dt
        done_updates += W.count_updates(w.graph, w.plans.subset(idx), o["counts"])
        n_done += len(idx)
        if n_done == batch and dt < budget_s / 40:
            batch = min(P, batch * 4)
    desc = (f"{n_done} of {P} plans (random order, seed 0), all {rates_all.shape[1]} rates x "
            f"{w.graph.n_trials} trials x {w.graph.n_req} requests each")
    return done_updates, spent, desc


def run_reference(args):
    """--impl reference: the CPU oracle timed on this box's host cores (tier contract)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    cores = os.cpu_count() or 1
    ws = make_workload(args.config, args.scale)
    budget = max(2.0, min(30.0, 150.0 / max(1, args.steps + args.warmup)))
    for _ in range(args.warmup):
        oracle_sample(ws[0], min(1.0, budget), cores)
    tot_u, tot_t, desc = 0, 0.0, ""
    for _ in range(args.steps):
        for w in ws:
            u, t, desc = oracle_sample(w, budget / len(ws), cores)
            tot_u += u
            tot_t += t
    value = tot_u / tot_t
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1000.0 * tot_t / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "int64",
            "data": "synthetic", "config": {"workload": workload_name(args.config), "sample": desc},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=1)
    ap.add_argument("--scale", type=float, default=1.0, help="scale n_req (debug only; 1.0 = BASELINE size)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist
    from paper_2512_14098_b200 import binding as cf

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl")
    dev = torch.device("cuda", local_rank)
    stream = torch.cuda.current_stream()

    ws = make_workload(args.config, args.scale)
    # weak scaling: every rank evaluates the whole config on its own Philox variant (independent
    # candidate-set replicas); no data-path collective
    variant = rank

    # ---- device-resident inputs, outputs, workspaces (allocated once, outside the timed region)
    calls = []
    for w in ws:
        c = {"w": w}
        if w.rate_mrps is not None:
            P, R = w.rate_mrps.shape
            c["rates_host"] = torch.from_numpy(w.rate_mrps.view(np.int32).copy()).pin_memory()
            c["rates"] = c["rates_host"].to(dev)
            K, T = w.graph.n_trials, w.graph.n_types
            c["counts"] = torch.empty((P, R, K, T, 2), dtype=torch.int32, device=dev)
            c["dep"] = torch.empty((P, R, K), dtype=torch.int64, device=dev)
            c["mk"] = torch.empty((P, R, K), dtype=torch.int64, device=dev)
            c["ws"] = cf.alloc_workspace(w.graph, w.plans, R)
            c["h_counts"] = torch.empty(c["counts"].shape, dtype=torch.int32).pin_memory()
            c["h_dep"] = torch.empty(c["dep"].shape, dtype=torch.int64).pin_memory()
            c["h_mk"] = torch.empty(c["mk"].shape, dtype=torch.int64).pin_memory()
        else:
            c["hi_host"] = torch.from_numpy(w.rate_hi_mrps.view(np.int32).copy()).pin_memory()
            c["hi"] = c["hi_host"].to(dev)
            c["ws"] = cf.alloc_workspace(w.graph, w.plans, 1)
            c["stream_records"] = cf.cf_materialize_stream(w.graph, w.seed, variant * w.n_variants, w.n_variants)
            # the a10 producer, timed once on its own (outside the step): records written per second
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            cf.cf_materialize_stream(w.graph, w.seed, variant * w.n_variants, w.n_variants, out=c["stream_records"])
            e1.record(stream)
            torch.cuda.synchronize()
            c["materialize_ms"] = e0.elapsed_time(e1)
        calls.append(c)

    launches = [0]

    def step(host_io: bool):
        """One pass of the hot path over the config. host_io: inputs start in pinned host memory and
        results are read back to the host (the e2e leg)."""
        out = []
        for c in calls:
            w = c["w"]
            if w.rate_mrps is not None:
                rates = c["rates"]
                if host_io:
                    rates = c["rates_host"].to(dev, non_blocking=True)
                r = cf.cf_eval_plans(w.graph, w.plans, rates, w.slo, w.seed, variant, out_counts=c["counts"],
                                     out_dep_sum=c["dep"], out_makespan=c["mk"], workspace=c["ws"], stream=stream)
                launches[0] += cf.cf_last_launch_count()
                if host_io:
                    c["h_counts"].copy_(c["counts"], non_blocking=True)
                    c["h_dep"].copy_(c["dep"], non_blocking=True)
                    c["h_mk"].copy_(c["mk"], non_blocking=True)
                out.append(r)
            else:
                hi = c["hi"]
                if host_io:
                    hi = c["hi_host"].to(dev, non_blocking=True)
                r = cf.cf_goodput_bisect(w.graph, w.plans, hi, w.n_steps, w.slo, w.seed,
                                         workspace=c["ws"], stream=stream, stream_records=c["stream_records"],
                                         n_variants=w.n_variants, plan_variant=w.plan_variant)
                launches[0] += cf.cf_last_launch_count()
                if host_io:
                    c["h_rate"] = r["rate_mrps"].cpu()
                    c["h_good"] = r["goodput_mrps"].cpu()
                c["bisect"] = r
                out.append(r)
        return out

    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)  # > 126 MB L2

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    for _ in range(args.warmup):
        step(False)
    barrier()

    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    # ---- device-timed region: K steps, CUDA events on the launching stream, L2 flushed between
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    launches[0] = 0
    barrier()
    for i in range(args.steps):
        flush.fill_(i & 0xFF)
        ev[i][0].record(stream)
        step(False)
        ev[i][1].record(stream)
    barrier()
    dev_ms = sum(a.elapsed_time(b) for a, b in ev)
    gpu_launches = launches[0]
    clocks = sampler.stop() if rank == 0 else None

    # ---- e2e: the same steps through the public API with host buffers, copies inside the region
    barrier()
    t0 = time.perf_counter()
    for i in range(args.steps):
        step(True)
        torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    barrier()

    # ---- exact update count of one step (outside the timed region)
    updates = 0
    heap_levels = 0
    requests = 0
    wide = 0
    h2d = d2h = 0
    for c in calls:
        w = c["w"]
        wide += cf.cf_workspace_wide_count(c["ws"])
        if w.rate_mrps is not None:
            cnts = cf.to_numpy_u32(c["counts"])
            updates += W.count_updates(w.graph, w.plans, cnts)
            heap_levels += W.count_heap_levels(w.graph, w.plans, cnts)
            requests += int(np.prod(w.rate_mrps.shape)) * w.graph.n_trials * w.graph.n_req
            h2d += c["rates_host"].numel() * 4
            d2h += c["h_counts"].numel() * 4 + c["h_dep"].numel() * 8 + c["h_mk"].numel() * 8
        else:
            # bisection: only the probes ON the bisection path count (the library reports how many
            # each plan had; closed brackets are no-ops, speculative tree nodes are overhead). The
            # type counts of a (variant, trial) do not depend on the rate (common random numbers,
            # R4), so one probe of plan p does count_updates(type counts of its stream) updates.
            P = w.plans.n_plans
            probes = cf.cf_bisect_probes(c["ws"], P).astype(np.int64)
            ones = np.ones((P, 1), dtype=np.uint32)
            c1 = cf.cf_eval_plans(w.graph, w.plans, np.maximum(w.rate_hi_mrps.reshape(P, 1) // 4, 1) * ones, w.slo,
                                  w.seed, stream_records=c["stream_records"], n_variants=w.n_variants,
                                  plan_variant=w.plan_variant, aux=False)
            cnts = cf.to_numpy_u32(c1["counts"])  # [P,1,K,T,2]
            updates += int((probes * W.count_updates(w.graph, w.plans, cnts, per_plan=True)).sum())
            heap_levels += int((probes * W.count_heap_levels(w.graph, w.plans, cnts, per_plan=True)).sum())
            requests += int(probes.sum()) * w.graph.n_trials * w.graph.n_req
            c["probes_total"] = int(probes.sum())
            h2d += c["hi_host"].numel() * 4
            d2h += P * 4 + P * w.graph.n_types * 4

    t_dev = torch.tensor([dev_ms / 1000.0, e2e_s], dtype=torch.float64, device=dev)
    u_all = torch.tensor([float(updates)], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(t_dev, op=dist.ReduceOp.MAX)
        dist.all_reduce(u_all, op=dist.ReduceOp.SUM)
    dev_s, e2e_s = float(t_dev[0]), float(t_dev[1])
    total_updates = float(u_all[0])
    value = total_updates * args.steps / dev_s
    e2e_value = total_updates * args.steps / e2e_s

    if rank == 0:
        # ---- ALU roofline: peak derived from unit counts x clock, measured beside it
        peaks = {}
        try:
            for mix, nm in ((0, "alu_pipe"), (1, "fma_pipe"), (2, "both_pipes")):
                ops, usec = cf.cf_bench_int32_peak(mix, 4000)
                peaks[nm] = ops / (usec * 1e-6) / 1e12
        except Exception as e:  # noqa: BLE001
            peaks["error"] = str(e)
        sm_count = torch.cuda.get_device_properties(dev).multi_processor_count
        sm_mhz = (clocks or {}).get("sm_max_mhz") or 1965.0
        peak_tops = sm_count * 4 * 32 * sm_mhz * 1e6 / 1e12  # 4 schedulers x 32 lanes x 1 inst/clk
        step_s = dev_ms / 1000.0 / args.steps
        alg_ops = OPS_PER_REQUEST * requests + OPS_PER_UPDATE * updates + OPS_PER_HEAP_LEVEL * heap_levels
        achieved = alg_ops / step_s / 1e12
        alu = {"bound": "alu", "achieved": achieved, "peak": peak_tops, "unit": "Tlane-op/s",
               "frac": achieved / peak_tops,
               "traffic": NCU_TRAFFIC_BYTES.get(args.config) if args.scale == 1.0 else None,
               "traffic_unit": "bytes per launch (ncu dram read+write, profiles/)",
               "frac_of_measured_alu_pipe_peak": (achieved / peaks["alu_pipe"]) if "alu_pipe" in peaks else None,
               "peak_source": f"derived: {sm_count} SMs x 4 schedulers x 32 lanes x {sm_mhz:.0f} MHz",
               "measured_int32_peaks_tops": peaks,
               "ops_model": {"per_request": OPS_PER_REQUEST, "per_update": OPS_PER_UPDATE,
                             "per_heap_level": OPS_PER_HEAP_LEVEL, "requests": requests, "updates": updates,
                             "heap_levels": heap_levels}}
        if args.config == 4:
            # materialised variant: algorithmic bytes = one 32-byte record per request per simulation
            # on the bisection path; peak = measured HBM copy bandwidth
            try:
                peak_gbs = float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"])
                peak_src = "MEASURED_PEAKS.json hbm_gbs (measured)"
            except (OSError, KeyError, ValueError):
                peak_gbs, peak_src = 6650.0, "fallback 6.65 TB/s (B200_PROFILING.md)"
            gbs = 32.0 * requests / step_s / 1e9
            roofline = {"bound": "hbm", "achieved": gbs, "peak": peak_gbs, "unit": "GB/s", "frac": gbs / peak_gbs,
                        "traffic": None, "peak_source": peak_src,
                        "note": "a thread block reads each record once for all its simulations, so DRAM traffic "
                                "is far below the algorithmic bytes; the kernel is latency/ALU-bound: see alu",
                        "alu": alu}
        else:
            roofline = alu
        cpu = None
        if not args.no_cpu_baseline:
            cores = os.cpu_count() or 1
            u, t, desc = oracle_sample(ws[0], 12.0, cores)
            cpu = {"value": u / t, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc}
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": 1000.0 * dev_s / args.steps, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "int64", "data": "synthetic",
                "config": {"workload": workload_name(args.config), "scale": args.scale,
                           "updates_per_step": total_updates, "l2": "flushed between timed steps (256 MiB fill)",
                           "stream_materialise": next(({"ms": c["materialize_ms"], "GB/s": c["stream_records"].numel() / c["materialize_ms"] / 1e6}
                                                       for c in calls if "materialize_ms" in c), None),
                           "wide_fixups": wide, "bisect_probes": sum(c.get("probes_total", 0) for c in calls),
                           "parallelism": f"replicas x{world} (one Philox variant per rank)"},
                "clocks": clocks,
                "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h},
                "gpu_launches": gpu_launches, "roofline": roofline, "cpu_baseline": cpu}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
