"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, bit for bit.

All arithmetic is integer, so the bar is exact equality of SLO-hit counts, departure checksums,
makespans, traced departures, stream records, bisected rates and goodput (north_star)."""
import os

import numpy as np
import pytest

from paper_2512_14098_b200 import workloads as W

pytestmark = pytest.mark.gpu

NT = os.cpu_count() or 1


@pytest.fixture(scope="module")
def cf():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_2512_14098_b200 import binding
    return binding


def check_eval(cf, orc, w, graph=None, plans=None, rates=None, variant=0, **kw):
    g = graph or w.graph
    pl = plans or w.plans
    rates = w.rate_mrps if rates is None else rates
    got = cf.cf_eval_plans(g, pl, rates, w.slo, w.seed, variant, **kw)
    status = cf.cf_workspace_status(got["workspace"])
    want = orc.eval_plans(g, pl, rates, w.slo, w.seed, variant, n_threads=NT)
    assert status == want["rc"]
    np.testing.assert_array_equal(cf.to_numpy_u32(got["counts"]), want["counts"])
    np.testing.assert_array_equal(cf.to_numpy_u64(got["dep_sum"]), want["dep_sum"])
    np.testing.assert_array_equal(got["makespan"].cpu().numpy(), want["makespan"])
    return got, want


# ---------------------------------------------------------------------------------------------
# the five configs at reduced sizes (several tiles + ragged tail), every sim compared
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("mean_us", W.CONFIG0_SERVICE_MEANS_US)
def test_cfg0_mm1_full_size(cf, orc, mean_us):
    w = W.config0_mm1(mean_us)  # full BASELINE size: 10,000 requests x 4 trials x 8 rates
    check_eval(cf, orc, w)
    b = cf.cf_goodput_bisect(w.graph, w.plans, w.rate_hi_mrps, w.n_steps, w.slo, w.seed)
    bo = orc.goodput_bisect(w.graph, w.plans, w.rate_hi_mrps, w.n_steps, w.slo, w.seed, n_threads=NT)
    np.testing.assert_array_equal(cf.to_numpy_u32(b["rate_mrps"]), bo["rate_mrps"])
    np.testing.assert_array_equal(cf.to_numpy_u32(b["goodput_mrps"]), bo["goodput_mrps"])
    np.testing.assert_array_equal(cf.to_numpy_u32(b["counts"]), bo["counts"])


def test_cfg1_reduced(cf, orc):
    w = W.config1_mllm(n_req=3000, n_trials=2, n_rates=4)  # all 512 plans, c up to 39
    check_eval(cf, orc, w)


def test_cfg2_reduced(cf, orc):
    w = W.config2_omni(n_req=2100, n_trials=2, n_rates=3, vectors_per_pattern=4)  # 32 topologies
    check_eval(cf, orc, w)


def test_cfg3_reduced(cf, orc):
    w = W.config3_multireplica(n_req=1500, n_trials=2, n_rates=3, plans_per_topology=40)
    check_eval(cf, orc, w)


def test_cfg4_reduced_stream_and_bisect(cf, orc):
    w = W.config4_sweep(n_req=1300, n_trials=2, n_steps=10, vectors_per_pattern=4, n_variants=3)
    g, pl = w.graph, w.plans
    w.plan_variant = ((np.arange(pl.n_plans) // 5) % 3).astype(np.uint32)
    # materialised records == oracle records
    rec = cf.cf_materialize_stream(g, w.seed, 0, w.n_variants)
    want = orc.materialize_stream(g, w.seed, 0, w.n_variants)
    np.testing.assert_array_equal(rec.cpu().numpy().reshape(-1), want.view(np.uint8).reshape(-1))
    # stream evaluation == in-register evaluation == oracle, variant by variant
    rates = W.rate_grid(W.flow_bound_mrps(g, pl), [0.6, 0.9])
    got = cf.cf_eval_plans(g, pl, rates, w.slo, w.seed, stream_records=rec, n_variants=w.n_variants,
                           plan_variant=w.plan_variant)
    for v in range(w.n_variants):
        idx = np.nonzero(w.plan_variant == v)[0]
        o = orc.eval_plans(g, pl.subset(idx), rates[idx], w.slo, w.seed, v, n_threads=NT)
        np.testing.assert_array_equal(cf.to_numpy_u32(got["counts"])[idx], o["counts"])
        np.testing.assert_array_equal(cf.to_numpy_u64(got["dep_sum"])[idx], o["dep_sum"])
        reg = cf.cf_eval_plans(g, pl.subset(idx), rates[idx], w.slo, w.seed, v)
        np.testing.assert_array_equal(cf.to_numpy_u32(reg["counts"]), o["counts"])
    # default mapping p % n_variants
    got = cf.cf_eval_plans(g, pl, rates, w.slo, w.seed, stream_records=rec, n_variants=w.n_variants)
    for v in range(w.n_variants):
        idx = np.nonzero(np.arange(pl.n_plans) % w.n_variants == v)[0]
        o = orc.eval_plans(g, pl.subset(idx), rates[idx], w.slo, w.seed, v, n_threads=NT)
        np.testing.assert_array_equal(cf.to_numpy_u32(got["counts"])[idx], o["counts"])
    # device-side bisection on the stream
    b = cf.cf_goodput_bisect(g, pl, w.rate_hi_mrps, w.n_steps, w.slo, w.seed, stream_records=rec,
                             n_variants=w.n_variants, plan_variant=w.plan_variant)
    for v in range(w.n_variants):
        idx = np.nonzero(w.plan_variant == v)[0]
        bo = orc.goodput_bisect(g, pl.subset(idx), w.rate_hi_mrps[idx], w.n_steps, w.slo, w.seed, v,
                                n_threads=NT)
        np.testing.assert_array_equal(cf.to_numpy_u32(b["rate_mrps"])[idx], bo["rate_mrps"])
        np.testing.assert_array_equal(cf.to_numpy_u32(b["goodput_mrps"])[idx], bo["goodput_mrps"])
        np.testing.assert_array_equal(cf.to_numpy_u32(b["counts"])[idx], bo["counts"])
    assert (cf.to_numpy_u32(b["rate_mrps"]) > 0).any()


# ---------------------------------------------------------------------------------------------
# traces, edge cases
# ---------------------------------------------------------------------------------------------
def check_trace(cf, orc, g, pl, p, rate, k, seed, variant, modes):
    o = orc.trace_sim(g, pl, p, rate, k, seed, variant=variant)
    for mode in modes:
        cf.cf_debug_kernel_mode(mode)
        try:
            t = cf.cf_trace_sim(g, pl, p, rate, k, seed, variant=variant)
        finally:
            cf.cf_debug_kernel_mode(0)
        assert t["status"] == o["rc"] == 0
        np.testing.assert_array_equal(t["arrival"].cpu().numpy(), o["arrival"], err_msg=f"mode {mode}")
        np.testing.assert_array_equal(t["departure"].cpu().numpy(), o["departure"], err_msg=f"mode {mode}")
        np.testing.assert_array_equal(t["type"].cpu().numpy(), o["type"], err_msg=f"mode {mode}")
        if mode == cf.CF_KERNEL_FAST32:
            assert t["wide"] == 0  # the departures came from the fast kernel, not from its fixup pass
    return o


def test_trace_matches_oracle(cf, orc):
    """Per-request arrivals, departures and types of the 64-bit kernel, the fast kernel (the one
    that does the benchmarked work) and -- for one-replica plans -- the max-plus scan kernel."""
    w = W.config2_omni(n_req=777, n_trials=3, n_rates=2, vectors_per_pattern=2, n_patterns=8)
    w.graph.edge_delay_us = 10_000
    both = (cf.CF_KERNEL_AUTO, cf.CF_KERNEL_WIDE64, cf.CF_KERNEL_FAST32)
    for p in (0, 3, 7, 15):
        for k in (0, 2):
            check_trace(cf, orc, w.graph, w.plans, p, int(w.rate_mrps[p, 1]), k, w.seed, 5, both)
    # overloaded (waits grow without bound: the 64-bit request body and mid-chunk mode changes) and
    # sparse arrivals (1 and 40 mrps: hours between requests, per-request origin moves)
    w = W.config3_multireplica(n_req=2500, n_trials=2, n_rates=2, plans_per_topology=6)
    R_p = W.flow_bound_mrps(w.graph, w.plans)
    for p in (1, 8, 13, 22):
        o = check_trace(cf, orc, w.graph, w.plans, p, int(3.0 * R_p[p]), 1, w.seed, 0, both)
        assert (o["departure"] - o["arrival"]).max() > 10 * (o["departure"] - o["arrival"])[:20].max()
        for rate in (1, 40):
            check_trace(cf, orc, w.graph, w.plans, p, rate, 0, w.seed, 2, both)
    # long overload: departures beyond 2^32 us while the keys stay in the window
    g = W.Graph(1, 1, 9000, 1, [1], W.mix_thresholds([1.0]), [0], [W.lognormal_qtab(1_000_000.0, 0.3)],
                W.exponential_qtab(65536.0), np.zeros((0, 2)))
    o = check_trace(cf, orc, g, W.make_plans([[(1, 2)], [(1, 1)]]), 0, 6000, 0, 11, 0, both)
    assert o["departure"].max() > 1 << 32
    # one replica at every stage: all four paths, the scan kernel included
    w = W.config2_omni(n_req=1000, n_trials=2, n_rates=2, vectors_per_pattern=1, n_patterns=32)
    w.plans = W.Plans(w.plans.n_stages, w.plans.stage_mask, np.ones_like(w.plans.stage_c))
    w.graph.edge_delay_us = 333
    R_p = W.flow_bound_mrps(w.graph, w.plans)
    for p in (0, 9, 31):
        for rate in (1, int(0.8 * R_p[p]), int(2.5 * R_p[p])):
            check_trace(cf, orc, w.graph, w.plans, p, max(rate, 1), 1, w.seed, 7, both + (cf.CF_KERNEL_SCAN,))
    # the scan kernel refuses a plan with more than one replica
    w2 = W.config1_mllm(n_req=100, n_trials=1, n_rates=1, llm_max=4, e_steps=2)
    cf.cf_debug_kernel_mode(cf.CF_KERNEL_SCAN)
    try:
        assert cf.cf_trace_sim(w2.graph, w2.plans, 3, 1000, 0, 1, check=False)["rc"] == cf.CF_ERR_ARG
    finally:
        cf.cf_debug_kernel_mode(0)


@pytest.mark.parametrize("L,B", [(1, 10), (1, 0), (4, 3), (32, 2), (8, 16), (20, 0), (16, 6)])
def test_quantile_table_shapes(cf, orc, L, B):
    """The device table lookup at every (levels, log2_cells) shape the oracle's geometric pin covers
    (tests/test_oracle_draws.py), through cf_eval_plans (both kernels), the materialised stream and
    the max-plus scan kernel: service AND arrival tables of that shape, random monotone entries."""
    rng = np.random.default_rng(L * 100 + B)
    n = (L << B) + 1
    tabs = [W.QTab(L, B, np.sort(rng.integers(0, 40_000, n)).astype(np.int32)),
            W.QTab(L, B, np.sort(rng.integers(0, 300_000, n)).astype(np.int32))]
    arr = W.QTab(L, B, np.sort(rng.integers(0, 4 * 65536, n)).astype(np.int32))
    g = W.Graph(2, 2, 1100, 2, [0b10, 0b11], W.mix_thresholds([0.6, 0.4]), [0, 0, 1, 1], tabs, arr, [[0, 1]],
                edge_delay_us=77)
    pl = W.make_plans([[(0b11, 3)], [(0b01, 1), (0b10, 2)], [(0b01, 2), (0b10, 7)], [(0b11, 1)]], max_stages=2)
    rates = np.maximum(W.rate_grid(W.flow_bound_mrps(g, pl), [0.5, 0.9, 1.3]), 1)
    w = W.Workload("shapes", g, pl, W.Slo([400_000, 600_000], [9, 9], [10, 10]), seed=L * 1000 + B, rate_mrps=rates)
    want = orc.eval_plans(g, pl, rates, w.slo, w.seed, 4, n_threads=NT)
    for mode in (0, 1):
        cf.cf_debug_kernel_mode(mode)
        try:
            got = cf.cf_eval_plans(g, pl, rates, w.slo, w.seed, 4)
        finally:
            cf.cf_debug_kernel_mode(0)
        np.testing.assert_array_equal(cf.to_numpy_u32(got["counts"]), want["counts"])
        np.testing.assert_array_equal(cf.to_numpy_u64(got["dep_sum"]), want["dep_sum"])
        np.testing.assert_array_equal(got["makespan"].cpu().numpy(), want["makespan"])
    rec = cf.cf_materialize_stream(g, w.seed, 4, 2)
    np.testing.assert_array_equal(rec.cpu().numpy().reshape(-1),
                                  orc.materialize_stream(g, w.seed, 4, 2).view(np.uint8).reshape(-1))
    got = cf.cf_eval_plans(g, pl, rates, w.slo, w.seed, stream_records=rec, n_variants=2,
                           plan_variant=np.zeros(4, np.uint32))
    np.testing.assert_array_equal(cf.to_numpy_u32(got["counts"]), want["counts"])
    # one replica everywhere: the scan kernel draws with the same lookup
    pl1 = W.Plans(pl.n_stages, pl.stage_mask, np.ones_like(pl.stage_c))
    want1 = orc.eval_plans(g, pl1, rates, w.slo, w.seed, 4, n_threads=NT)
    got1 = cf.cf_eval_plans(g, pl1, rates, w.slo, w.seed, 4)
    np.testing.assert_array_equal(cf.to_numpy_u32(got1["counts"]), want1["counts"])
    np.testing.assert_array_equal(cf.to_numpy_u64(got1["dep_sum"]), want1["dep_sum"])


def test_edge_delay_and_variant(cf, orc):
    w = W.config2_omni(n_req=900, n_trials=2, n_rates=2, vectors_per_pattern=2, n_patterns=32)
    w.graph.edge_delay_us = 10_000
    check_eval(cf, orc, w, variant=9)
    w1 = W.config1_mllm(n_req=700, n_trials=2, n_rates=2, llm_max=6, e_steps=3)
    w1.graph.edge_delay_us = 123
    check_eval(cf, orc, w1, variant=1)


@pytest.mark.parametrize("n_req", [1, 31, 32, 33, 127, 128, 129, 257])
def test_ragged_request_counts(cf, orc, n_req):
    w = W.config1_mllm(n_req=n_req, n_trials=3, n_rates=2, llm_max=5, e_steps=2)
    check_eval(cf, orc, w)


def test_eight_components_eight_stages(cf, orc):
    # C = 8, T = 8, plans with up to 8 stages: the wide-record template
    rng = np.random.default_rng(5)
    C = T = 8
    tabs = [W.lognormal_qtab(float(rng.integers(5_000, 60_000)), 0.5) for _ in range(C)]
    masks = [int(m) | 1 << int(rng.integers(0, C)) for m in rng.integers(0, 256, T)]
    masks[3] = 0  # a type with an empty route (R14)
    frac = rng.dirichlet(np.ones(T))
    svc_tab = np.repeat(np.arange(C, dtype=np.uint16), T)
    edges = [[i, i + 1] for i in range(C - 1)]
    g = W.Graph(C, T, 1000, 2, masks, W.mix_thresholds(frac), svc_tab, tabs,
                W.gamma_qtab(0.5, 65536.0), edges, edge_delay_us=250)
    plan_list = []
    for _ in range(40):
        cuts = sorted(rng.choice(np.arange(1, C), size=int(rng.integers(0, C)), replace=False).tolist())
        bounds = [0] + cuts + [C]
        plan_list.append([(sum(1 << i for i in range(a, b)), int(rng.integers(1, 9)))
                          for a, b in zip(bounds, bounds[1:])])
    pl = W.make_plans(plan_list, max_stages=8)
    rates = W.rate_grid(W.flow_bound_mrps(g, pl), [0.5, 0.9, 1.3])
    slo = W.Slo(rng.integers(50_000, 400_000, T), [9] * T, [10] * T)
    w = W.Workload("c8", g, pl, slo, seed=99, rate_mrps=rates)
    assert orc.validate(g, pl) == 0
    got, want = check_eval(cf, orc, w)
    assert want["counts"][..., 3, 0].sum() > 0
    np.testing.assert_array_equal(want["counts"][..., 3, 0], want["counts"][..., 3, 1])


def test_large_replica_counts(cf, orc):
    # c far above N (never queues) and c = 59, 64, 200 (deep heaps)
    tab = W.lognormal_qtab(50_000.0, 0.6)
    g = W.Graph(1, 1, 600, 2, [1], W.mix_thresholds([1.0]), [0], [tab], W.exponential_qtab(65536.0),
                np.zeros((0, 2)))
    pl = W.make_plans([[(1, c)] for c in (1, 2, 3, 59, 64, 200, 700)])
    rates = W.rate_grid(W.flow_bound_mrps(g, pl), [0.7, 1.5])
    w = W.Workload("bigc", g, pl, W.Slo([80_000], [9], [10]), seed=6, rate_mrps=rates)
    check_eval(cf, orc, w)


def test_out_of_range_rates_zeroed_and_flagged(cf, orc):
    w = W.config1_mllm(n_req=200, n_trials=2, n_rates=3, llm_max=4, e_steps=2)
    rates = w.rate_mrps.copy()
    rates[1, 2] = 0
    rates[2, 0] = 1_000_000_001
    got, want = check_eval(cf, orc, w, rates=rates)
    assert want["rc"] == orc.ORC_ERR_RANGE
    assert (cf.to_numpy_u32(got["counts"])[1, 2] == 0).all()
    # arrival horizon beyond 2^62 us (R17)
    g = W.Graph(1, 1, 1 << 12, 1, [1], W.mix_thresholds([1.0]), [0], [W.constant_qtab(5)],
                W.constant_qtab(2**31 - 1), np.zeros((0, 2)))
    pl = W.make_plans([[(1, 1)]])
    w2 = W.Workload("horizon", g, pl, W.Slo([10], [9], [10]), seed=0,
                    rate_mrps=np.array([[1, 1000, 1_000_000_000]], dtype=np.uint32))
    got, want = check_eval(cf, orc, w2)
    assert want["sim_status"].reshape(-1).tolist() == [orc.ORC_ERR_RANGE, orc.ORC_ERR_RANGE, 0]


def test_bisect_parity_and_degenerate_brackets(cf, orc):
    w = W.config1_mllm(n_req=1500, n_trials=3, n_rates=2, llm_max=8, e_steps=3)
    R_p = W.flow_bound_mrps(w.graph, w.plans)
    hi = np.ceil(1.5 * R_p).astype(np.uint32)
    hi[0], hi[1], hi[2] = 0, 1, 2
    for steps in (1, 5, 20):
        b = cf.cf_goodput_bisect(w.graph, w.plans, hi, steps, w.slo, w.seed)
        assert cf.cf_workspace_status(b["workspace"]) == 0
        bo = orc.goodput_bisect(w.graph, w.plans, hi, steps, w.slo, w.seed, n_threads=NT)
        np.testing.assert_array_equal(cf.to_numpy_u32(b["rate_mrps"]), bo["rate_mrps"])
        np.testing.assert_array_equal(cf.to_numpy_u32(b["goodput_mrps"]), bo["goodput_mrps"])
        np.testing.assert_array_equal(cf.to_numpy_u32(b["counts"]), bo["counts"])


def test_bisect_out_of_range_probe_is_infeasible_r18(cf, orc):
    # the hand-worked R18 case of tests/test_oracle_invariants.py, on the device
    from test_oracle_invariants import R18_HI, R18_RATE, r18_case
    g, pl1, slo = r18_case()
    pl2 = W.make_plans([[(1, 2)]] * 4)  # two replicas: the thread-per-simulation kernels + fixup pass
    for pl, depth in ((pl1, 0), (pl1, 1), (pl1, 3), (pl2, 0), (pl2, 2)):
        cf.cf_debug_bisect_depth(depth)
        try:
            b = cf.cf_goodput_bisect(g, pl, R18_HI, 20, slo, 0)
        finally:
            cf.cf_debug_bisect_depth(0)
        assert cf.cf_workspace_status(b["workspace"]) == cf.CF_ERR_RANGE
        np.testing.assert_array_equal(cf.to_numpy_u32(b["rate_mrps"]), R18_RATE)
        np.testing.assert_array_equal(cf.to_numpy_u32(b["goodput_mrps"])[:, 0], R18_RATE)
        c = cf.to_numpy_u32(b["counts"])
        assert (c[:2] == 0).all() and (c[2:] == 1 << 12).all()


def test_host_errors_on_gpu(cf):
    w = W.config1_mllm(n_req=100, n_trials=1, n_rates=1, llm_max=2, e_steps=1)
    bad = W.make_plans([[(0b10, 1), (0b01, 1)]])
    r = cf.cf_eval_plans(w.graph, bad, [[1000]], w.slo, 0, check=False)
    assert r["rc"] == cf.CF_ERR_PLAN
    with pytest.raises(cf.CfError):
        cf.cf_eval_plans(w.graph, bad, [[1000]], w.slo, 0)


# ---------------------------------------------------------------------------------------------
# full BASELINE sizes in the bench's launch configuration: sampled simulations vs the oracle
# ---------------------------------------------------------------------------------------------
def sampled_full_size(cf, orc, w, n_samples, seed):
    got = cf.cf_eval_plans(w.graph, w.plans, w.rate_mrps, w.slo, w.seed)
    assert cf.cf_workspace_status(got["workspace"]) == 0
    counts = cf.to_numpy_u32(got["counts"])
    dep = cf.to_numpy_u64(got["dep_sum"])
    mk = got["makespan"].cpu().numpy()
    rng = np.random.default_rng(seed)
    P, R = w.rate_mrps.shape
    ps = rng.integers(0, P, n_samples)
    rs = rng.integers(0, R, n_samples)
    o = orc.eval_plans(w.graph, w.plans.subset(ps), w.rate_mrps[ps, rs].reshape(-1, 1), w.slo, w.seed,
                       n_threads=NT)
    np.testing.assert_array_equal(counts[ps, rs], o["counts"][:, 0])
    np.testing.assert_array_equal(dep[ps, rs], o["dep_sum"][:, 0])
    np.testing.assert_array_equal(mk[ps, rs], o["makespan"][:, 0])
    # properties that hold at any size
    c = counts.astype(np.int64)
    assert (c[..., 0].sum(-1) == w.graph.n_req).all()
    assert (c[..., 1] <= c[..., 0]).all()
    assert (c[..., 0] == c[0, 0][None, None, ..., 0]).all()  # CRN: type counts independent of plan
    return counts


def test_cfg1_full_size_sampled(cf, orc):
    w = W.config1_mllm()
    counts = sampled_full_size(cf, orc, w, 64, 1)
    # R16: colocated plans with equal l+e are duplicates and must agree exactly (same rates)
    pl = w.plans
    seen = {}
    for p in range(256):
        key = (int(pl.stage_c[p, 0]), tuple(w.rate_mrps[p]))
        if key in seen:
            np.testing.assert_array_equal(counts[p], counts[seen[key]])
        seen[key] = p


def test_cfg2_full_size_sampled(cf, orc):
    sampled_full_size(cf, orc, W.config2_omni(), 64, 2)


def test_cfg3_full_size_sampled(cf, orc):
    sampled_full_size(cf, orc, W.config3_multireplica(), 64, 3)


def test_cfg4_full_size_sampled(cf, orc):
    """configs[4] exactly as bench.py runs it (4 GiB materialised stream, 32-step device-side
    bisection, speculative passes, fixup pass): sampled plans against the oracle's bisection."""
    w = W.config4_sweep()
    rec = cf.cf_materialize_stream(w.graph, w.seed, 0, w.n_variants)
    b = cf.cf_goodput_bisect(w.graph, w.plans, w.rate_hi_mrps, w.n_steps, w.slo, w.seed, stream_records=rec,
                             n_variants=w.n_variants, plan_variant=w.plan_variant)
    assert cf.cf_workspace_status(b["workspace"]) == 0
    rate = cf.to_numpy_u32(b["rate_mrps"])
    good = cf.to_numpy_u32(b["goodput_mrps"])
    counts = cf.to_numpy_u32(b["counts"])
    probes = cf.cf_bisect_probes(b["workspace"], w.plans.n_plans)
    rng = np.random.default_rng(4)
    for p in rng.integers(0, w.plans.n_plans, 16):
        idx = np.array([p])
        bo = orc.goodput_bisect(w.graph, w.plans.subset(idx), w.rate_hi_mrps[idx], w.n_steps, w.slo, w.seed,
                                int(w.plan_variant[p]), n_threads=NT)
        np.testing.assert_array_equal(rate[idx], bo["rate_mrps"])
        np.testing.assert_array_equal(good[idx], bo["goodput_mrps"])
        np.testing.assert_array_equal(counts[idx], bo["counts"])
    # properties that hold at any size
    assert (rate < w.rate_hi_mrps).all() and (rate > 0).any()
    assert (probes <= w.n_steps).all() and (probes >= 1).all()
    c = counts.astype(np.int64)
    feasible = rate > 0
    assert (c[feasible][..., 0].sum(-1) == w.graph.n_req).all()
    assert (c[~feasible] == 0).all()
    att_ok = c[feasible][..., 1].sum(1) * 10 >= 9 * c[feasible][..., 0].sum(1)  # pooled 90 % per type
    assert att_ok.all()


def test_prepared_call_cache_and_streams(cf, orc):
    """Repeated calls reuse the pinned schedule / descriptor blob (cf.h "Conventions"); any change of a
    descriptor byte must miss the cache. More distinct calls than the cache holds (eviction while
    earlier uploads may be in flight), on a side stream, then cf_cache_clear."""
    import torch
    side = torch.cuda.Stream()
    w = W.config1_mllm(n_req=400, n_trials=2, n_rates=2, llm_max=6, e_steps=2)
    wants = {}
    for rep in range(2):
        for seed in range(20):  # 20 distinct descriptor sets > 16 cache entries
            got = cf.cf_eval_plans(w.graph, w.plans, w.rate_mrps, w.slo, seed, stream=side if seed % 2 else None)
            if seed not in wants:
                wants[seed] = orc.eval_plans(w.graph, w.plans, w.rate_mrps, w.slo, seed, n_threads=NT)
            (side if seed % 2 else torch.cuda.current_stream()).synchronize()
            np.testing.assert_array_equal(cf.to_numpy_u32(got["counts"]), wants[seed]["counts"])
            np.testing.assert_array_equal(cf.to_numpy_u64(got["dep_sum"]), wants[seed]["dep_sum"])
    # same descriptors, different device inputs (rates): a hit that must still see the new rates
    r2 = (w.rate_mrps * 3 // 4).astype(np.uint32)
    got = cf.cf_eval_plans(w.graph, w.plans, r2, w.slo, 19)
    np.testing.assert_array_equal(cf.to_numpy_u32(got["counts"]),
                                  orc.eval_plans(w.graph, w.plans, r2, w.slo, 19, n_threads=NT)["counts"])
    # one table entry, one replica count, one target changed: each a miss with the right answer
    w2 = W.config1_mllm(n_req=400, n_trials=2, n_rates=2, llm_max=6, e_steps=2)
    w2.graph.tabs[0].q[100] += 1
    check_eval(cf, orc, w2)
    w2.plans.stage_c[3, 0] += 1
    check_eval(cf, orc, w2)
    w2.slo = W.Slo([1_500_000, 3_000_000], [9, 9], [10, 10])
    check_eval(cf, orc, w2)
    hi = np.full(w.plans.n_plans, 30_000, np.uint32)
    for steps, num in ((6, 9), (6, 8), (7, 9), (6, 9)):
        slo = W.Slo(w.slo.L_us, [num, num], [10, 10])
        b = cf.cf_goodput_bisect(w.graph, w.plans, hi, steps, slo, w.seed, stream=side)
        side.synchronize()
        bo = orc.goodput_bisect(w.graph, w.plans, hi, steps, slo, w.seed, n_threads=NT)
        np.testing.assert_array_equal(cf.to_numpy_u32(b["rate_mrps"]), bo["rate_mrps"])
        np.testing.assert_array_equal(cf.to_numpy_u32(b["counts"]), bo["counts"])
    cf.cf_cache_clear()
    check_eval(cf, orc, w)
