#!/usr/bin/env python
"""bench.py -- request-stage simulation updates/s of the plan-evaluation hot path on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference]

A "step" is one pass of the whole hot path over one BASELINE.json
config through the C ABI: cf_eval_plans for configs 0-3, cf_goodput_bisect_stream on the
materialised stream for config 4. With no --config the line's headline is configs[4] at full size
(the largest single-GPU config) and `config.per_config` carries configs[2] and [3] at full size,
each with its own value, ms_per_step, roofline, e2e and wide_fixups: the three configs north_star's
roofline target names. --config C measures that one config only.
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

# Algorithmic INT32 lane-operations of the method (derived instruction by instruction in DESIGN.md
# section 6 "Roofline accounting"; the annotated SASS of the request loop is
# profiles/r02_sass_request_loop.md): per request, per visited stage, and per comparison level the
# Kiefer-Wolfowitz replace-min descends on a binary heap of c free times (floor(log2 c) levels).
OPS_PER_REQUEST = 12
OPS_PER_UPDATE = 5
OPS_PER_HEAP_LEVEL = 7

# Per-launch hardware counters of the simulation kernel at FULL size, copied from the ncu captures
# under profiles/ (NOT measured by the run that prints them; the file is named beside the numbers):
# dram = dram__bytes_read.sum + dram__bytes_write.sum, inst = smsp__inst_executed.sum (warp
# instructions), per step of the config.
NCU_FULL_SIZE = {}
try:
    with open(os.path.join(ROOT, "profiles", "r02_ncu_counters.json")) as _f:
        NCU_FULL_SIZE = {int(k): v for k, v in json.load(_f).items() if k.isdigit()}
except (OSError, ValueError):
    pass

# The oracle's bounded samples: a FIXED set of whole plans (the first n of a seed-0 permutation),
# the same in this arm's cpu_baseline and in --impl reference. (all-core plans, one-core plans)
ORACLE_SAMPLE_PLANS = {0: (1, 1), 1: (48, 6), 2: (16, 2), 3: (128, 16), 4: (64, 8)}


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


# --------------------------------------------------------------------------------------------
# the oracle leg (cpu_baseline and --impl reference): oracle/ as it stands, on the host cores
# --------------------------------------------------------------------------------------------
def oracle_sample_plans(w, cfg: int, one_core: bool):
    """The fixed sample: the first n plans of a seed-0 permutation of the config's plans."""
    P = w.plans.n_plans
    n = ORACLE_SAMPLE_PLANS[cfg][1 if one_core else 0]
    return np.sort(np.random.default_rng(0).permutation(P)[:min(n, P)])


def oracle_sample_rates(w):
    if w.rate_mrps is None:  # bisection config: the sample evaluates 2 rates at 0.6 / 0.9 of the flow bound
        return W.rate_grid(W.flow_bound_mrps(w.graph, w.plans), [0.6, 0.9])
    return w.rate_mrps


def oracle_sample(w, cfg: int, n_threads: int, one_core: bool = False):
    """Times oracle.eval_plans on the fixed sample of whole plans (all their rates and trials).
    Returns dict(updates, seconds, idx, rates, out, sample)."""
    from oracle import cf_oracle as orc
    idx = oracle_sample_plans(w, cfg, one_core)
    rates = oracle_sample_rates(w)[idx]
    variant = 0
    t0 = time.perf_counter()
    if w.plan_variant is not None:  # materialised config: plan p reads stream variant plan_variant[p]
        outs = {}
        for v in np.unique(w.plan_variant[idx]):
            sel = np.nonzero(w.plan_variant[idx] == v)[0]
            outs[int(v)] = (sel, orc.eval_plans(w.graph, w.plans.subset(idx[sel]), rates[sel], w.slo, w.seed,
                                                int(v), n_threads=n_threads))
        dt = time.perf_counter() - t0
        K, T = w.graph.n_trials, w.graph.n_types
        out = {"counts": np.zeros((len(idx), rates.shape[1], K, T, 2), np.uint32),
               "dep_sum": np.zeros((len(idx), rates.shape[1], K), np.uint64),
               "makespan": np.zeros((len(idx), rates.shape[1], K), np.int64)}
        for sel, o in outs.values():
            for key in out:
                out[key][sel] = o[key]
    else:
        out = orc.eval_plans(w.graph, w.plans.subset(idx), rates, w.slo, w.seed, variant, n_threads=n_threads)
        dt = time.perf_counter() - t0
    updates = W.count_updates(w.graph, w.plans.subset(idx), out["counts"])
    sample = (f"{len(idx)} of {w.plans.n_plans} plans (first {len(idx)} of a seed-0 permutation), "
              f"{rates.shape[1]} rates x {w.graph.n_trials} trials x {w.graph.n_req} requests each")
    return dict(updates=updates, seconds=dt, idx=idx, rates=rates, out=out, sample=sample)


def cpu_baseline_record(ws, cfg: int, cores: int):
    """cpu_baseline of a config: the oracle on all cores and on one core."""
    tot_u = tot_t = 0.0
    one_u = one_t = 0.0
    samples, one_samples, alls = [], [], []
    for w in ws:
        a = oracle_sample(w, cfg, cores)
        o = oracle_sample(w, cfg, 1, one_core=True)
        tot_u += a["updates"]; tot_t += a["seconds"]; samples.append(a["sample"]); alls.append(a)
        one_u += o["updates"]; one_t += o["seconds"]; one_samples.append(o["sample"])
    rec = {"value": tot_u / tot_t, "unit": UNIT, "cores": cores, "kind": "oracle",
           "sample": samples[0] + (f" (x{len(ws)} calls)" if len(ws) > 1 else ""), "seconds": tot_t,
           "one_core": {"value": one_u / one_t, "unit": UNIT, "cores": 1, "seconds": one_t,
                        "sample": one_samples[0] + (f" (x{len(ws)} calls)" if len(ws) > 1 else "")}}
    return rec, alls


def default_config(args) -> int:
    return 4 if args.config is None else args.config


def run_reference(args):
    """--impl reference: the CPU oracle timed on this box's host cores (tier contract). Each step is
    the same fixed sample of the headline workload that the GPU arm's cpu_baseline uses."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    cores = os.cpu_count() or 1
    cfg = default_config(args)
    ws = make_workload(cfg, args.scale)
    for _ in range(min(args.warmup, 1)):  # one warm-up pass is enough to page the library and inputs in
        for w in ws:
            oracle_sample(w, cfg, cores)
    tot_u, tot_t, desc = 0, 0.0, ""
    for _ in range(args.steps):
        for w in ws:
            a = oracle_sample(w, cfg, cores)
            tot_u += a["updates"]; tot_t += a["seconds"]; desc = a["sample"]
    value = tot_u / tot_t
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1000.0 * tot_t / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "int64",
            "data": "synthetic", "config": {"workload": workload_name(cfg), "scale": args.scale},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


# --------------------------------------------------------------------------------------------
# the GPU leg
# --------------------------------------------------------------------------------------------
class Measurement:
    """Device buffers of one config and its timed legs. Everything goes through the Python binding
    of the C ABI (argument marshalling only)."""

    def __init__(self, cfg, scale, rank, dev, stream, torch, cf):
        self.cfg, self.scale, self.torch, self.cf, self.dev, self.stream = cfg, scale, torch, cf, dev, stream
        self.ws = make_workload(cfg, scale)
        # weak scaling: every rank evaluates the whole config on its own Philox variant (independent
        # candidate-set replicas); no data-path collective
        self.variant = rank
        self.calls = []
        self.launches = 0
        for w in self.ws:
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
                c["stream_records"] = cf.cf_materialize_stream(w.graph, w.seed, self.variant * w.n_variants, w.n_variants)
                # the a10 producer, timed once on its own (outside the step): records written per second
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                cf.cf_materialize_stream(w.graph, w.seed, self.variant * w.n_variants, w.n_variants,
                                         out=c["stream_records"])
                e1.record(stream)
                torch.cuda.synchronize()
                c["materialize_ms"] = e0.elapsed_time(e1)
            self.calls.append(c)

    def step(self, host_io: bool):
        """One pass of the hot path over the config. host_io: inputs start in pinned host memory and
        results are read back to the host (the e2e leg)."""
        cf, dev = self.cf, self.dev
        for c in self.calls:
            w = c["w"]
            if w.rate_mrps is not None:
                rates = c["rates"]
                if host_io:
                    rates = c["rates_host"].to(dev, non_blocking=True)
                cf.cf_eval_plans(w.graph, w.plans, rates, w.slo, w.seed, self.variant, out_counts=c["counts"],
                                 out_dep_sum=c["dep"], out_makespan=c["mk"], workspace=c["ws"], stream=self.stream)
                self.launches += cf.cf_last_launch_count()
                if host_io:
                    c["h_counts"].copy_(c["counts"], non_blocking=True)
                    c["h_dep"].copy_(c["dep"], non_blocking=True)
                    c["h_mk"].copy_(c["mk"], non_blocking=True)
            else:
                hi = c["hi"]
                if host_io:
                    hi = c["hi_host"].to(dev, non_blocking=True)
                r = cf.cf_goodput_bisect(w.graph, w.plans, hi, w.n_steps, w.slo, w.seed,
                                         workspace=c["ws"], stream=self.stream, stream_records=c["stream_records"],
                                         n_variants=w.n_variants, plan_variant=w.plan_variant)
                self.launches += cf.cf_last_launch_count()
                if host_io:
                    c["h_rate"] = r["rate_mrps"].cpu()
                    c["h_good"] = r["goodput_mrps"].cpu()
                c["bisect"] = r

    def count_work(self):
        """Exact update / request / heap-level counts of one step (outside the timed region)."""
        cf = self.cf
        updates = heap_levels = requests = wide = h2d = d2h = probes_total = 0
        for c in self.calls:
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
                probes_total += int(probes.sum())
                h2d += c["hi_host"].numel() * 4
                d2h += P * 4 + P * w.graph.n_types * 4
        return dict(updates=updates, heap_levels=heap_levels, requests=requests, wide=wide, h2d=h2d, d2h=d2h,
                    probes=probes_total)

    def parity_check(self, alls):
        """The GPU outputs of this run against the oracle on exactly the simulations the cpu_baseline
        leg ran. Returns (checked simulations, exact)."""
        cf = self.cf
        checked, exact = 0, True
        for c, a in zip(self.calls, alls):
            w, idx, o = c["w"], a["idx"], a["out"]
            if w.rate_mrps is not None:
                got = dict(counts=cf.to_numpy_u32(c["counts"])[idx], dep_sum=cf.to_numpy_u64(c["dep"])[idx],
                           makespan=c["mk"].cpu().numpy()[idx])
            else:  # the sample's two rates per plan, evaluated on the same materialised stream
                r = cf.cf_eval_plans(w.graph, w.plans.subset(idx), a["rates"], w.slo, w.seed,
                                     stream_records=c["stream_records"], n_variants=w.n_variants,
                                     plan_variant=w.plan_variant[idx])
                got = dict(counts=cf.to_numpy_u32(r["counts"]), dep_sum=cf.to_numpy_u64(r["dep_sum"]),
                           makespan=r["makespan"].cpu().numpy())
            for key in ("counts", "dep_sum", "makespan"):
                exact = exact and bool(np.array_equal(got[key], o[key]))
            checked += int(np.prod(o["dep_sum"].shape))
        return checked, exact


def measure(cfg, args, rank, world, dev, stream, torch, dist, cf, local_rank, with_cpu):
    """Times one config: K device-timed steps (CUDA events, L2 flushed between steps), the e2e leg,
    exact work counts, roofline objects, cpu_baseline + parity. Returns the record (rank 0) or None."""
    m = Measurement(cfg, args.scale, rank, dev, stream, torch, cf)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)  # > 126 MB L2

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    for _ in range(args.warmup):
        m.step(False)
    barrier()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    m.launches = 0
    barrier()
    for i in range(args.steps):
        flush.fill_(i & 0xFF)
        ev[i][0].record(stream)
        m.step(False)
        ev[i][1].record(stream)
    barrier()
    dev_ms = sum(a.elapsed_time(b) for a, b in ev)
    gpu_launches = m.launches
    clocks = sampler.stop() if rank == 0 else None

    # e2e: the same steps through the public API with host buffers, copies inside the timed region
    e2e_steps = max(1, min(args.steps, args.e2e_steps))
    barrier()
    t0 = time.perf_counter()
    for i in range(e2e_steps):
        m.step(True)
        torch.cuda.synchronize()
    e2e_s = (time.perf_counter() - t0) * args.steps / e2e_steps  # scaled to K steps
    barrier()

    work = m.count_work()
    t_dev = torch.tensor([dev_ms / 1000.0, e2e_s], dtype=torch.float64, device=dev)
    u_all = torch.tensor([float(work["updates"])], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(t_dev, op=dist.ReduceOp.MAX)
        dist.all_reduce(u_all, op=dist.ReduceOp.SUM)
    dev_s, e2e_s = float(t_dev[0]), float(t_dev[1])
    total_updates = float(u_all[0])
    if rank != 0:
        return None
    value = total_updates * args.steps / dev_s
    step_s = dev_ms / 1000.0 / args.steps

    # ---- ALU roofline: peak derived from unit counts x clock
    sm_count = torch.cuda.get_device_properties(dev).multi_processor_count
    sm_mhz = (clocks or {}).get("sm_max_mhz") or 1965.0
    peak_tops = sm_count * 4 * 32 * sm_mhz * 1e6 / 1e12  # 4 schedulers x 32 lanes x 1 inst/clk
    requests, updates, heap_levels = work["requests"], work["updates"], work["heap_levels"]
    alg_ops = OPS_PER_REQUEST * requests + OPS_PER_UPDATE * updates + OPS_PER_HEAP_LEVEL * heap_levels
    achieved = alg_ops / step_s / 1e12
    ncu = NCU_FULL_SIZE.get(cfg) if args.scale == 1.0 else None
    roofline = {"bound": "alu", "achieved": achieved, "peak": peak_tops, "unit": "Tlane-op/s",
                "frac": achieved / peak_tops,
                "achieved_is": "algorithmic lane-ops of the method (ops_model) / measured step time",
                "peak_source": f"derived: {sm_count} SMs x 4 schedulers x 32 lanes x {sm_mhz:.0f} MHz (INT32 issue)",
                "traffic": ncu["dram_bytes"] if ncu else None,
                "traffic_source": (ncu["source"] + " (ncu capture of an earlier run, not this run)") if ncu else None,
                # executed warp instructions x 32 lanes of the committed ncu capture / this run's time / peak
                "issue_slot_util": (ncu["warp_inst"] * 32.0 / step_s / 1e12 / peak_tops) if ncu else None,
                "ncu_issue_active_pct": ncu.get("issue_active_pct") if ncu else None,
                "warp_inst_per_request": (ncu["warp_inst"] * 32.0 / requests) if ncu and requests else None,
                "ops_model": {"per_request": OPS_PER_REQUEST, "per_update": OPS_PER_UPDATE,
                              "per_heap_level": OPS_PER_HEAP_LEVEL, "requests": requests, "updates": updates,
                              "heap_levels": heap_levels}}
    if cfg == 4:
        # materialised variant (north_star 4): algorithmic bytes = one 32-byte record per request per
        # simulation on the bisection path against the measured HBM copy bandwidth.
        # A warp reads a record once for its 32 simulations, so the DRAM traffic (ncu) is far below
        # that figure and the kernel is bound by INT32 issue: the alu object above is the bound.
        try:
            peak_gbs = float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"])
            peak_src = "MEASURED_PEAKS.json hbm_gbs (measured)"
        except (OSError, KeyError, ValueError):
            peak_gbs, peak_src = 6650.0, "fallback 6.65 TB/s (B200_PROFILING.md)"
        gbs = 32.0 * requests / step_s / 1e9
        dram = ncu["dram_bytes"] if ncu else None
        roofline["hbm"] = {"bound": "hbm", "achieved": gbs, "peak": peak_gbs, "unit": "GB/s", "frac": gbs / peak_gbs,
                           "achieved_is": "algorithmic bytes (32 B x on-path requests x simulations) / step time",
                           "peak_source": peak_src, "traffic": dram,
                           "dram_gbs": (dram / step_s / 1e9) if dram else None,
                           "dram_frac_of_peak": (dram / step_s / 1e9 / peak_gbs) if dram else None,
                           "read_amplification": (dram / (32.0 * requests)) if dram else None}
    rec = {"value": value, "ms_per_step": 1000.0 * dev_s / args.steps, "updates_per_step": total_updates,
           "e2e": {"value": total_updates * args.steps / e2e_s, "unit": UNIT, "h2d_bytes_per_step": work["h2d"],
                   "d2h_bytes_per_step": work["d2h"], "steps_timed": e2e_steps},
           "gpu_launches": gpu_launches, "wide_fixups": work["wide"], "bisect_probes": work["probes"],
           "roofline": roofline, "clocks": clocks, "workload": workload_name(cfg),
           "stream_materialise": next(({"ms": c["materialize_ms"], "GB/s": c["stream_records"].numel() / c["materialize_ms"] / 1e6}
                                       for c in m.calls if "materialize_ms" in c), None)}
    if with_cpu:
        cores = os.cpu_count() or 1
        cpu, alls = cpu_baseline_record(m.ws, cfg, cores)
        checked, exact = m.parity_check(alls)
        rec["cpu_baseline"] = cpu
        rec["parity"] = {"checked_sims": checked, "exact": exact,
                         "what": "counts, departure checksum, makespan of the cpu_baseline sample, GPU vs oracle"}
    del m, flush
    torch.cuda.empty_cache()
    return rec


def measure_phases(torch, cf, stream, n_plans=1_000_000):
    """Sub-record: the cheap phases of Algorithm 2 (flow bound -> Monte-Carlo latency -> Pareto prune
    of the non-redundant plans) on a 10^6-plan candidate set, chained on the device; milliseconds per
    call through the C ABI (host descriptors in, device arrays out), best of 3."""
    w = W.config_phase_sweep(n_plans)
    g, pl, slo = w.graph, w.plans, w.slo

    def timed(fn):
        best, out = None, None
        for _ in range(3):
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            out = fn()
            e1.record(stream)
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1)
            best = ms if best is None else min(best, ms)
        return out, best

    f, ms_flow = timed(lambda: cf.cf_flow_bound(g, pl, 4, 5))
    mc, ms_mc = timed(lambda: cf.cf_mc_latency(g, pl, f["rate_mrps"], slo, w.seed, want_counts=False))
    alive = (1 - f["redundant"]).to(torch.uint8)
    pr, ms_par = timed(lambda: cf.cf_pareto_select(mc["goodput_mrps"], alive))
    P = pl.n_plans
    return {"plans": P, "graph": "configs[2] Omni graph, 32 KEEP/MERGE patterns, sum c <= 64",
            "flow_bound_ms": ms_flow, "mc_latency_ms": ms_mc, "pareto_select_ms": ms_par,
            "mc_requests_sampled": g.n_req * g.n_trials, "non_redundant": int(alive.sum()),
            "pareto_survivors": int(cf.to_numpy_u32(pr["n_survivors"])[0]),
            "plans_per_s_flow_plus_mc": P / ((ms_flow + ms_mc) * 1e-3),
            "paper_context": "Table 6 (PAPER.md:480-481): flow 3.48 s on 483.41 M plans, Monte Carlo 34.23 s on 1.95 M "
                             "plans, planner host CPU not stated"}


def measure_fidelity(torch, cf, stream):
    """Sub-record: the simulator fidelity variants, milliseconds through the C
    ABI (best of 3) and updates/s. Arrival-order service (cf_graph.order_mode = 1, R27) on
    configs[1] at full size next to the index-order run of the same call, with the largest per-type
    attainment difference between the two disciplines over all (plan, rate); CPU-GPU overlap (R24),
    fork-join (R25) and routed plans (R26). Parity of the variants with the oracle:
    tests/test_gpu_{fcfs,overlap,forkjoin,routing}.py."""
    w = W.config1_mllm()
    g, pl = w.graph, w.plans
    out = {"workload": workload_name(1)}
    for mode, name in ((0, "index_order"), (1, "arrival_order")):
        g.order_mode = mode
        ws = cf.alloc_workspace(g, pl, w.rate_mrps.shape[1])
        best = None
        for _ in range(3):
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            res = cf.cf_eval_plans(g, pl, w.rate_mrps, w.slo, w.seed, workspace=ws, stream=stream)
            e1.record(stream)
            torch.cuda.synchronize()
            best = e0.elapsed_time(e1) if best is None else min(best, e0.elapsed_time(e1))
        counts = cf.to_numpy_u32(res["counts"])
        upd = int(W.count_updates(g, pl, counts))
        out[name] = {"ms": best, "updates_per_s": upd / (best * 1e-3), "workspace_gib": ws.numel() / 2**30}
        if mode == 1:
            out["attainment_shift_vs_index_order"] = float(np.abs(
                counts[..., 1].sum(axis=2) / np.maximum(counts[..., 0].sum(axis=2), 1) - out.pop("_att0")).max())
        else:
            out["_att0"] = counts[..., 1].sum(axis=2) / np.maximum(counts[..., 0].sum(axis=2), 1)
        del ws
    g.order_mode = 0

    def timed(graph, plans, rates, slo, seed):
        ws2 = cf.alloc_workspace(graph, plans, rates.shape[1])
        best2, res2 = None, None
        for _ in range(3):
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            res2 = cf.cf_eval_plans(graph, plans, rates, slo, seed, workspace=ws2, stream=stream)
            e1.record(stream)
            torch.cuda.synchronize()
            best2 = e0.elapsed_time(e1) if best2 is None else min(best2, e0.elapsed_time(e1))
        upd2 = int(W.count_updates(graph, plans, cf.to_numpy_u32(res2["counts"])))
        return {"ms": best2, "updates_per_s": upd2 / (best2 * 1e-3)}

    # CPU-GPU overlap (R24): configs[1] with a CPU pre-processing table (exponential, 10 ms) on the encoder
    w = W.config1_mllm()
    w.graph.tabs = list(w.graph.tabs) + [W.exponential_qtab(10_000.0)]
    cpu = np.full(w.graph.n_comp * w.graph.n_types, 0xFFFF, np.uint16)
    cpu[0:w.graph.n_types] = len(w.graph.tabs) - 1
    w.graph.cpu_tab = cpu
    out["cpu_gpu_overlap"] = dict(timed(w.graph, w.plans, w.rate_mrps, w.slo, w.seed), workload=workload_name(1), kernel="64-bit, HAS_CPU")
    # fork-join (R25): configs[4]'s graph (up to three encoders in parallel), 512 plans x 4 rates x 8 trials x 2^15
    w = W.config4_sweep(n_req=1 << 15, vectors_per_pattern=16, n_variants=1)
    rates = W.rate_grid(W.flow_bound_mrps(w.graph, w.plans), [0.5, 0.7, 0.9, 1.1])
    base = timed(w.graph, w.plans, rates, w.slo, w.seed)
    w.graph.join_mode = 1
    out["fork_join"] = dict(timed(w.graph, w.plans, rates, w.slo, w.seed), path_mode_ms=base["ms"], kernel="64-bit, JOIN",
                            workload="configs[4] graph, 512 plans x 4 rates x 8 trials x 2^15 requests")
    # routing (R26): configs[1]'s graph, per plan the disaggregated path AND a colocated node, split 50/50 per type
    w = W.config1_mllm()
    P = 256
    c = w.plans.stage_c[256:512, :2].astype(np.int64)   # the disaggregated plans' (e, l)
    pl = W.make_plans([[(0b01, int(e)), (0b10, max(1, int(l) // 2)), (0b11, max(1, (int(l) + 1) // 2))] for e, l in c], max_stages=3)
    rm = np.tile(np.array([[0b011, 0b100], [0b011, 0b100]], np.uint8), (P, 1, 1))
    rc = np.tile(np.array([[1 << 31, 0xFFFFFFFF], [1 << 31, 0xFFFFFFFF]], np.uint32), (P, 1, 1))
    routed = W.Plans(pl.n_stages, pl.stage_mask, pl.stage_c, 2, rm, rc)
    fb = cf.cf_flow_bound(w.graph, routed)
    rr = W.rate_grid(cf.to_numpy_u32(fb["bound_mrps"]).astype(np.float64), np.arange(0.40, 1.16, 0.05))
    out["routing"] = dict(timed(w.graph, routed, rr, w.slo, w.seed), kernel="fast kernel, route draw in the 3-word record",
                          workload="configs[1] graph, 256 plans with two routes per type x 16 rates x 8 trials x 100k requests")
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=None,
                    help="one config 0..4; default: configs[4] headline + configs[2], [3] in config.per_config")
    ap.add_argument("--scale", type=float, default=1.0, help="scale n_req (debug only; 1.0 = BASELINE size)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--e2e-steps", type=int, default=5, help="steps of the e2e leg (at most --steps)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        print("bench.py: note: fewer than 3 warm-up steps", file=sys.stderr)
    if args.impl == "reference":
        return run_reference(args)

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.gpus != world:
        raise SystemExit(f"bench.py: --gpus {args.gpus} needs {args.gpus} ranks: launch with `python -m torch.distributed.run "
                         f"--nnodes=1 --nproc-per-node {args.gpus} --master-addr 127.0.0.1 bench.py --gpus {args.gpus} ...` "
                         f"(WORLD_SIZE is {world})")
    import torch
    import torch.distributed as dist
    from paper_2512_14098_b200 import binding as cf

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl")
    dev = torch.device("cuda", local_rank)
    stream = torch.cuda.current_stream()

    head_cfg = default_config(args)
    with_cpu = (not args.no_cpu_baseline) and rank == 0
    head = measure(head_cfg, args, rank, world, dev, stream, torch, dist, cf, local_rank, with_cpu)
    per = {}
    if args.config is None:
        for c in (2, 3):
            per[c] = measure(c, args, rank, world, dev, stream, torch, dist, cf, local_rank, with_cpu)

    if rank == 0:
        peaks = {}
        try:
            for mix, nm in ((0, "alu_pipe"), (1, "fma_pipe"), (2, "both_pipes")):
                ops, usec = cf.cf_bench_int32_peak(mix, 4000)
                peaks[nm] = ops / (usec * 1e-6) / 1e12
        except Exception as e:  # noqa: BLE001
            peaks["error"] = str(e)
        head["roofline"]["measured_int32_peaks_tops"] = peaks
        config = {"workload": head["workload"], "scale": args.scale, "updates_per_step": head["updates_per_step"],
                  "l2": "flushed between timed steps (256 MiB fill)", "stream_materialise": head["stream_materialise"],
                  "wide_fixups": head["wide_fixups"], "bisect_probes": head["bisect_probes"],
                  "parallelism": f"replicas x{world} (one Philox variant per rank)"}
        if args.config is None and world == 1:
            try:
                config["phases"] = measure_phases(torch, cf, stream)
            except Exception as e:  # noqa: BLE001
                config["phases"] = {"error": str(e)}
            try:
                config["fidelity"] = measure_fidelity(torch, cf, stream)
            except Exception as e:  # noqa: BLE001
                config["fidelity"] = {"error": str(e)}
        if per:
            config["per_config"] = {f"cfg{c}": {k: v for k, v in r.items() if k != "stream_materialise"}
                                    for c, r in per.items()}
        line = {"metric": METRIC, "value": head["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": head["ms_per_step"], "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "int64", "data": "synthetic",
                "config": config, "clocks": head["clocks"], "e2e": head["e2e"],
                "gpu_launches": head["gpu_launches"] + sum(r["gpu_launches"] for r in per.values()),
                "roofline": head["roofline"], "cpu_baseline": head.get("cpu_baseline"), "parity": head.get("parity")}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
