"""GPU parity of the CPU-GPU overlap rule (R24):
graphs with CPU pre-processing tables run on the 64-bit kernel; counts, checksums, makespans, traces,
bisected rates and the Monte-Carlo estimate against the oracle, bit for bit."""
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


def test_closed_forms_on_the_device(cf, orc):
    from test_oracle_overlap import dd1
    G, Cc = 400_000, 300_000
    for gap, c in ((65536, 1), (32768, 1), (16384, 1), (16384, 3)):
        g, pl = dd1(gap, Cc, G, 300, c=c)
        t = cf.cf_trace_sim(g, pl, 0, 1000, 0, 0)
        o = orc.trace_sim(g, pl, 0, 1000, 0, seed=0)
        np.testing.assert_array_equal(t["departure"].cpu().numpy(), o["departure"])
        np.testing.assert_array_equal(t["arrival"].cpu().numpy(), o["arrival"])
    g, pl = dd1(32768, Cc, G, 300)  # busy stretches of 3 requests: CPU paid once per stretch
    t = cf.cf_trace_sim(g, pl, 0, 1000, 0, 0)
    A, D = t["arrival"].cpu().numpy(), t["departure"].cpu().numpy()
    n = np.arange(300)
    np.testing.assert_array_equal(D, A[n - n % 3] + Cc + (n % 3 + 1) * G)


def omni_overlap(n_req, n_trials, n_rates, **kw):
    """configs[2] with CPU pre-processing on the three encoders (image decode, video decode, audio resampling)."""
    w = W.config2_omni(n_req=n_req, n_trials=n_trials, n_rates=n_rates, **kw)
    g = w.graph
    g.tabs = g.tabs + [W.lognormal_qtab(25_000.0, 0.5), W.lognormal_qtab(220_000.0, 0.6), W.exponential_qtab(8_000.0)]
    cpu = np.full(6 * 4, 0xFFFF, np.uint16)
    for i in range(3):
        cpu[i * 4:(i + 1) * 4] = 6 + i
    g.cpu_tab = cpu
    return w


def test_eval_trace_bisect_parity(cf, orc):
    from test_oracle_overlap import overlap_graph
    w = omni_overlap(1900, 2, 3, vectors_per_pattern=3)
    w.graph.edge_delay_us = 6_000
    w.rate_mrps = np.maximum(W.rate_grid(W.flow_bound_mrps(w.graph, w.plans), [0.05, 0.8, 1.3]), 1)
    assert orc.validate(w.graph, w.plans) == 0
    want = orc.eval_plans(w.graph, w.plans, w.rate_mrps, w.slo, w.seed, 2, n_threads=NT)
    base = W.config2_omni(n_req=1900, n_trials=2, n_rates=3, vectors_per_pattern=3)
    base.graph.edge_delay_us = 6_000
    plain = orc.eval_plans(base.graph, base.plans, w.rate_mrps, w.slo, w.seed, 2, n_threads=NT)
    assert (want["dep_sum"] != plain["dep_sum"]).any()  # the CPU time matters
    for mode in (cf.CF_KERNEL_AUTO, cf.CF_KERNEL_WIDE64, cf.CF_KERNEL_FAST32):  # every mode lands on the 64-bit kernel
        cf.cf_debug_kernel_mode(mode)
        try:
            got = cf.cf_eval_plans(w.graph, w.plans, w.rate_mrps, w.slo, w.seed, 2)
            assert cf.cf_workspace_wide_count(got["workspace"]) == 0
        finally:
            cf.cf_debug_kernel_mode(0)
        np.testing.assert_array_equal(cf.to_numpy_u32(got["counts"]), want["counts"])
        np.testing.assert_array_equal(cf.to_numpy_u64(got["dep_sum"]), want["dep_sum"])
        np.testing.assert_array_equal(got["makespan"].cpu().numpy(), want["makespan"])
    for p in (0, 17, 95):
        rate = int(w.rate_mrps[p, 2])
        t = cf.cf_trace_sim(w.graph, w.plans, p, rate, 1, w.seed, variant=2)
        o = orc.trace_sim(w.graph, w.plans, p, rate, 1, w.seed, variant=2)
        np.testing.assert_array_equal(t["departure"].cpu().numpy(), o["departure"])
    # one replica everywhere: still the thread-per-simulation kernel (the idle/busy rule is not max-plus linear)
    pl1 = W.Plans(w.plans.n_stages, w.plans.stage_mask, np.ones_like(w.plans.stage_c))
    r1 = np.maximum(W.rate_grid(W.flow_bound_mrps(w.graph, pl1), [0.5, 1.2]), 1)
    got = cf.cf_eval_plans(w.graph, pl1, r1, w.slo, w.seed)
    o1 = orc.eval_plans(w.graph, pl1, r1, w.slo, w.seed, n_threads=NT)
    np.testing.assert_array_equal(cf.to_numpy_u32(got["counts"]), o1["counts"])
    np.testing.assert_array_equal(cf.to_numpy_u64(got["dep_sum"]), o1["dep_sum"])
    cf.cf_debug_kernel_mode(cf.CF_KERNEL_SCAN)
    try:
        assert cf.cf_eval_plans(w.graph, pl1, r1, w.slo, w.seed, check=False)["rc"] == cf.CF_ERR_ARG
    finally:
        cf.cf_debug_kernel_mode(0)
    # bisection and the Monte-Carlo estimate
    hi = orc.flow_bound(w.graph, w.plans, 3, 2)["rate_mrps"]
    b = cf.cf_goodput_bisect(w.graph, w.plans, hi, 9, w.slo, w.seed)
    bo = orc.goodput_bisect(w.graph, w.plans, hi, 9, w.slo, w.seed, n_threads=NT)
    np.testing.assert_array_equal(cf.to_numpy_u32(b["rate_mrps"]), bo["rate_mrps"])
    np.testing.assert_array_equal(cf.to_numpy_u32(b["counts"]), bo["counts"])
    slo = W.Slo([150_000, 4_000_000, 450_000, 4_200_000], [9] * 4, [10] * 4)
    m = cf.cf_mc_latency(w.graph, w.plans, hi, slo, w.seed, 3)
    mo = orc.mc_latency(w.graph, w.plans, hi, slo, w.seed, 3)
    np.testing.assert_array_equal(cf.to_numpy_u32(m["counts"]), mo["counts"])
    np.testing.assert_array_equal(cf.to_numpy_u32(m["goodput_mrps"]), mo["goodput_mrps"])
    # 3 components incl. one on each Philox CPU block boundary is covered by the 8-component case below
    g3 = overlap_graph(n_req=900, n_trials=2)
    pl3 = W.make_plans([[(0b001, 2), (0b010, 1), (0b100, 3)], [(0b011, 2), (0b100, 2)], [(0b111, 4)]], max_stages=3)
    r3 = np.maximum(W.rate_grid(W.flow_bound_mrps(g3, pl3), [0.3, 0.9, 1.4]), 1)
    s3 = W.Slo([400_000, 500_000, 600_000], [9] * 3, [10] * 3)
    got = cf.cf_eval_plans(g3, pl3, r3, s3, 8, 1)
    o3 = orc.eval_plans(g3, pl3, r3, s3, 8, 1, n_threads=NT)
    np.testing.assert_array_equal(cf.to_numpy_u32(got["counts"]), o3["counts"])
    np.testing.assert_array_equal(cf.to_numpy_u64(got["dep_sum"]), o3["dep_sum"])


def test_eight_components_and_refusals(cf, orc):
    rng = np.random.default_rng(9)
    C = T = 8
    tabs = [W.lognormal_qtab(float(rng.integers(5_000, 60_000)), 0.5) for _ in range(C)] + \
           [W.exponential_qtab(float(rng.integers(2_000, 30_000))) for _ in range(4)]
    masks = [int(m) | 1 << int(rng.integers(0, C)) for m in rng.integers(0, 256, T)]
    cpu = np.full(C * T, 0xFFFF, np.uint16)
    for i in (0, 3, 4, 7):  # both Philox CPU blocks (components 0..3 and 4..7)
        cpu[i * T:(i + 1) * T] = 8 + [0, 3, 4, 7].index(i)
    g = W.Graph(C, T, 1000, 2, masks, W.mix_thresholds(rng.dirichlet(np.ones(T))), np.repeat(np.arange(C, dtype=np.uint16), T),
                tabs, W.gamma_qtab(0.5, 65536.0), [[i, i + 1] for i in range(C - 1)], edge_delay_us=250, cpu_tab=cpu)
    plan_list = []
    for _ in range(30):
        cuts = sorted(rng.choice(np.arange(1, C), size=int(rng.integers(0, C)), replace=False).tolist())
        bounds = [0] + cuts + [C]
        plan_list.append([(sum(1 << i for i in range(a, b)), int(rng.integers(1, 9))) for a, b in zip(bounds, bounds[1:])])
    pl = W.make_plans(plan_list, max_stages=8)
    rates = np.maximum(W.rate_grid(W.flow_bound_mrps(g, pl), [0.5, 0.9, 1.3]), 1)
    slo = W.Slo(rng.integers(50_000, 400_000, T), [9] * T, [10] * T)
    got = cf.cf_eval_plans(g, pl, rates, slo, 99)
    want = orc.eval_plans(g, pl, rates, slo, 99, n_threads=NT)
    np.testing.assert_array_equal(cf.to_numpy_u32(got["counts"]), want["counts"])
    np.testing.assert_array_equal(cf.to_numpy_u64(got["dep_sum"]), want["dep_sum"])
    np.testing.assert_array_equal(got["makespan"].cpu().numpy(), want["makespan"])
    # a materialised stream has no room for CPU times
    w = omni_overlap(100, 1, 1, vectors_per_pattern=1, n_patterns=2)
    import torch
    rec = torch.zeros((1, 1, 100, 32), dtype=torch.uint8, device="cuda")
    assert cf.cf_eval_plans(w.graph, w.plans, [[1000]] * 2, w.slo, 0, stream_records=rec, check=False)["rc"] == cf.CF_ERR_ARG
    with pytest.raises(cf.CfError):
        cf.cf_materialize_stream(w.graph, 0, 0, 1)
