"""GPU parity of the cheap phases around the simulation (cf_flow_bound, cf_mc_latency,
cf_pareto_select; SURVEY.md 8(f) NEXT-1..3) against the oracle's plain statements, bit for bit,
and of the whole coarse-to-fine funnel chained on the device (Algorithm 2)."""
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


def u32(cf, t):
    return cf.to_numpy_u32(t)


def check_flow(cf, orc, g, pl, num=1, den=1):
    f = cf.cf_flow_bound(g, pl, num, den)
    o = orc.flow_bound(g, pl, num, den)
    assert o["rc"] == 0
    np.testing.assert_array_equal(u32(cf, f["rate_mrps"]), o["rate_mrps"])
    np.testing.assert_array_equal(u32(cf, f["bound_mrps"]), o["bound_mrps"])
    np.testing.assert_array_equal(f["bottleneck"].cpu().numpy(), o["bottleneck"])
    np.testing.assert_array_equal(f["redundant"].cpu().numpy(), o["redundant"])
    return f, o


def test_flow_bound_hand_worked_and_configs(cf, orc):
    from test_oracle_phases import HAND_BOUND, HAND_PLANS, hand_graph
    f, _ = check_flow(cf, orc, hand_graph(), W.make_plans(HAND_PLANS, max_stages=3), 3, 2)
    np.testing.assert_array_equal(u32(cf, f["bound_mrps"]), HAND_BOUND)
    for w in (W.config1_mllm(n_req=10, n_trials=1, n_rates=1), W.config2_omni(n_req=10, n_trials=1, n_rates=1),
              W.config3_multireplica(n_req=10, n_trials=1, n_rates=1, plans_per_topology=300), W.config4_sweep(n_req=10, n_trials=1)):
        _, o = check_flow(cf, orc, w.graph, w.plans, 3, 2)
        assert 0 < o["redundant"].sum() < w.plans.n_plans
    g0 = W.Graph(1, 1, 8, 1, [0], W.mix_thresholds([1.0]), [0], [W.constant_qtab(5)], W.exponential_qtab(65536.0),
                 np.zeros((0, 2)))
    check_flow(cf, orc, g0, W.make_plans([[(1, 1)], [(1, 2)]]))


@pytest.mark.parametrize("L,B", [(1, 10), (1, 0), (4, 3), (32, 2), (8, 16), (20, 0)])
def test_flow_bound_table_shapes(cf, orc, L, B):
    rng = np.random.default_rng(L * 100 + B)
    n = (L << B) + 1
    tabs = [W.QTab(L, B, np.sort(rng.integers(0, 2**30, n)).astype(np.int32)),
            W.QTab(L, B, np.sort(rng.integers(0, 50_000, n)).astype(np.int32))]
    g = W.Graph(2, 2, 16, 1, [0b10, 0b11], W.mix_thresholds([0.6, 0.4]), [0, 0, 1, 1], tabs, W.exponential_qtab(65536.0),
                [[0, 1]])
    pl = W.make_plans([[(0b11, 3)], [(0b01, 1), (0b10, 2)], [(0b01, 2), (0b10, 65535)], [(0b11, 1)]], max_stages=2)
    check_flow(cf, orc, g, pl, 7, 5)


def test_mc_latency_parity(cf, orc):
    w = W.config2_omni(n_req=1100, n_trials=3, n_rates=1, vectors_per_pattern=2, n_patterns=32)
    slo = W.Slo([150_000, 4_000_000, 350_000, 4_200_000], [9] * 4, [10] * 4)
    for delay, variant in ((0, 0), (10_000, 4)):
        w.graph.edge_delay_us = delay
        rate = orc.flow_bound(w.graph, w.plans, 4, 5)["rate_mrps"]
        o = orc.mc_latency(w.graph, w.plans, rate, slo, w.seed, variant)
        m = cf.cf_mc_latency(w.graph, w.plans, rate, slo, w.seed, variant)
        np.testing.assert_array_equal(u32(cf, m["counts"]), o["counts"])
        np.testing.assert_array_equal(u32(cf, m["goodput_mrps"]), o["goodput_mrps"])
    # 8 components / 8 types / up to 8 stages, negative and huge targets, the largest rate
    rng = np.random.default_rng(5)
    C = T = 8
    tabs = [W.lognormal_qtab(float(rng.integers(5_000, 60_000)), 0.5) for _ in range(C)]
    masks = [int(m) | 1 << int(rng.integers(0, C)) for m in rng.integers(0, 256, T)]
    masks[3] = 0
    g = W.Graph(C, T, 777, 2, masks, W.mix_thresholds(rng.dirichlet(np.ones(T))), np.repeat(np.arange(C, dtype=np.uint16), T),
                tabs, W.gamma_qtab(0.5, 65536.0), [[i, i + 1] for i in range(C - 1)], edge_delay_us=2_500)
    plan_list = []
    for _ in range(40):
        cuts = sorted(rng.choice(np.arange(1, C), size=int(rng.integers(0, C)), replace=False).tolist())
        bounds = [0] + cuts + [C]
        plan_list.append([(sum(1 << i for i in range(a, b)), int(rng.integers(1, 9))) for a, b in zip(bounds, bounds[1:])])
    pl = W.make_plans(plan_list, max_stages=8)
    slo = W.Slo([60_000, -1, 1 << 40, 0, 90_000, 120_000, 30_000, 200_000], [9] * T, [10] * T)
    rate = rng.integers(1, 2**32 - 1, pl.n_plans).astype(np.uint32)
    rate[0] = 2**32 - 1
    o = orc.mc_latency(g, pl, rate, slo, 99, 1)
    m = cf.cf_mc_latency(g, pl, rate, slo, 99, 1)
    np.testing.assert_array_equal(u32(cf, m["counts"]), o["counts"])
    np.testing.assert_array_equal(u32(cf, m["goodput_mrps"]), o["goodput_mrps"])


def test_pareto_parity(cf, orc):
    from test_oracle_phases import test_pareto_hand_worked  # noqa: F401  (the hand-worked cases, on the device)
    for G, alive, pruned, best, ns in (([[5, 5], [6, 4], [5, 4]], None, [0, 0, 1], 0, 2),
                                       ([[3, 3], [3, 3], [2, 9]], None, [0, 0, 0], 2, 3),
                                       ([[5, 5], [6, 6], [1, 7]], [1, 0, 1], [0, 1, 0], 0, 2),
                                       ([[0, 0]], [0], [1], 0xFFFFFFFF, 0)):
        r = cf.cf_pareto_select(G, alive)
        assert r["pruned"].cpu().numpy().tolist() == pruned
        assert int(u32(cf, r["best"])[0]) == best and int(u32(cf, r["n_survivors"])[0]) == ns
    rng = np.random.default_rng(3)
    for P, T, hi in ((1, 1, 5), (17, 3, 4), (255, 8, 3), (256, 2, 50), (257, 5, 6), (3000, 4, 12), (5000, 8, 2**32 - 1)):
        G = rng.integers(0, hi, (P, T), dtype=np.uint64).astype(np.uint32)
        for alive in (None, (rng.integers(0, 4, P) > 0).astype(np.uint8)):
            o = orc.pareto_select(G, alive)
            r = cf.cf_pareto_select(G, alive)
            np.testing.assert_array_equal(r["pruned"].cpu().numpy(), o["pruned"])
            assert int(u32(cf, r["best"])[0]) == o["best"]
            assert int(u32(cf, r["n_survivors"])[0]) == o["n_survivors"]


def test_coarse_to_fine_funnel_on_the_device(cf, orc):
    """Algorithm 2 end to end without a host pass between the phases: flow bound -> alpha R_d ->
    Monte-Carlo goodput -> Pareto prune (redundant plans out) -> rate bisection of the survivors'
    bracket [0, 1.5 R_d) -> Pareto prune + policy. Every intermediate equals the oracle's."""
    import torch
    w = W.config2_omni(n_req=1500, n_trials=2, n_rates=1, vectors_per_pattern=3, n_patterns=32)
    g, pl, slo = w.graph, w.plans, w.slo
    f = cf.cf_flow_bound(g, pl, 4, 5)                      # alpha = 0.8 (Table 5)
    fo = orc.flow_bound(g, pl, 4, 5)
    mc = cf.cf_mc_latency(g, pl, f["rate_mrps"], slo, w.seed, want_counts=False)
    mo = orc.mc_latency(g, pl, fo["rate_mrps"], slo, w.seed)
    np.testing.assert_array_equal(u32(cf, mc["goodput_mrps"]), mo["goodput_mrps"])
    alive = (1 - f["redundant"]).to(torch.uint8)           # Algorithm 2 l.5
    p1 = cf.cf_pareto_select(mc["goodput_mrps"], alive)    # l.12
    p1o = orc.pareto_select(mo["goodput_mrps"], 1 - fo["redundant"])
    np.testing.assert_array_equal(p1["pruned"].cpu().numpy(), p1o["pruned"])
    hi = cf.cf_flow_bound(g, pl, 3, 2)["rate_mrps"]        # the bisection bracket, straight from the device
    b = cf.cf_goodput_bisect(g, pl, hi, 14, slo, w.seed)   # l.13-15 (here on every plan; the verdicts select)
    bo = orc.goodput_bisect(g, pl, orc.flow_bound(g, pl, 3, 2)["rate_mrps"], 14, slo, w.seed, n_threads=NT)
    np.testing.assert_array_equal(u32(cf, b["goodput_mrps"]), bo["goodput_mrps"])
    p2 = cf.cf_pareto_select(b["goodput_mrps"], (1 - p1["pruned"]).to(torch.uint8))  # l.16-17
    p2o = orc.pareto_select(bo["goodput_mrps"], 1 - p1o["pruned"])
    np.testing.assert_array_equal(p2["pruned"].cpu().numpy(), p2o["pruned"])
    assert int(u32(cf, p2["best"])[0]) == p2o["best"] != 0xFFFFFFFF
    assert 0 < p2o["n_survivors"] <= p1o["n_survivors"] < pl.n_plans
