"""GPU parity of arrival-order service (cf_graph.order_mode = 1; R27; SURVEY.md 8(f) NEXT-4
"true stage-arrival-order FCFS"): the warp-per-simulation kernel of cf_fcfs.cuh against the oracle's
order_mode = 1, bit for bit -- counts, checksums, makespans, traces, bisected rates; with routes,
CPU-GPU overlap, every free-time vector width, ragged sizes, more simulations than warps in flight."""
import os

import numpy as np
import pytest

from paper_2512_14098_b200 import workloads as W
from test_oracle_fcfs import omni_like
from test_oracle_overlap import overlap_graph
from test_oracle_routing import mllm, two_path_plans

pytestmark = pytest.mark.gpu

NT = os.cpu_count() or 1


@pytest.fixture(scope="module")
def cf():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_2512_14098_b200 import binding
    return binding


def check(cf, orc, g, pl, rates, slo, seed, variant=0, workspace=None):
    assert g.order_mode == 1
    want = orc.eval_plans(g, pl, rates, slo, seed, variant, n_threads=NT)
    got = cf.cf_eval_plans(g, pl, rates, slo, seed, variant, workspace=workspace)
    assert cf.cf_workspace_status(got["workspace"]) == want["rc"] == 0
    np.testing.assert_array_equal(cf.to_numpy_u32(got["counts"]), want["counts"])
    np.testing.assert_array_equal(cf.to_numpy_u64(got["dep_sum"]), want["dep_sum"])
    np.testing.assert_array_equal(got["makespan"].cpu().numpy(), want["makespan"])
    return want


def test_hand_worked_example_on_the_device(cf):
    rows = [[int(v) for v in l.split()] for l in open(os.path.join(os.path.dirname(__file__), "golden", "fcfs_overtake.txt"))
            if l.strip() and not l.startswith("#")]
    g = W.Graph(2, 2, 8, 1, [0b11, 0b10], W.mix_thresholds([0.5, 0.5]), [0, 0, 1, 1],
                [W.constant_qtab(900_000), W.constant_qtab(400_000)], W.constant_qtab(65536), [[0, 1]], order_mode=1)
    pl = W.make_plans([[(0b01, 2), (0b10, 1)]])
    t = cf.cf_trace_sim(g, pl, 0, 10_000, 0, 3)
    assert t["type"].cpu().numpy().tolist() == [r[1] for r in rows]
    assert t["arrival"].cpu().numpy().tolist() == [r[2] for r in rows]
    assert t["departure"].cpu().numpy().tolist() == [r[4] for r in rows]
    g.order_mode = 0
    t = cf.cf_trace_sim(g, pl, 0, 10_000, 0, 3)
    assert t["departure"].cpu().numpy().tolist() == [r[3] for r in rows]


@pytest.mark.parametrize("n_req", [1, 31, 33, 1000, 4097])
def test_parity_ragged_sizes(cf, orc, n_req):
    g = omni_like(n_req, n_trials=2)
    pl = W.make_plans([[(0b0011, 2), (0b0100, 3), (0b1000, 2)], [(0b0001, 1), (0b0010, 1), (0b0100, 5), (0b1000, 1)],
                       [(0b0111, 4), (0b1000, 2)], [(0b1111, 6)]])
    rates = np.maximum(W.rate_grid(W.flow_bound_mrps(g, pl), [0.4, 0.9, 1.2]), 1)
    slo = W.Slo([500_000, 600_000, 900_000, 1_000_000], [9] * 4, [10] * 4)
    for delay in (0, 6_000):
        g.edge_delay_us = delay
        check(cf, orc, g, pl, rates, slo, 5, variant=1)


def test_parity_config_shapes_traces_and_bisection(cf, orc):
    w = W.config2_omni(n_req=3000, n_trials=2, n_rates=3, vectors_per_pattern=2)   # 64 plans, 6 components, Sum c <= 64
    g, pl = w.graph, w.plans
    g.order_mode = 1
    a = check(cf, orc, g, pl, w.rate_mrps, w.slo, w.seed)
    g.order_mode = 0
    b = orc.eval_plans(g, pl, w.rate_mrps, w.slo, w.seed, n_threads=NT)
    g.order_mode = 1
    assert (a["dep_sum"] != b["dep_sum"]).any()       # the discipline matters on plans whose types skip stages
    for p in (0, 17, 63):
        t = cf.cf_trace_sim(g, pl, p, int(w.rate_mrps[p, 2]), 1, w.seed)
        o = orc.trace_sim(g, pl, p, int(w.rate_mrps[p, 2]), 1, w.seed)
        np.testing.assert_array_equal(t["arrival"].cpu().numpy(), o["arrival"])
        np.testing.assert_array_equal(t["departure"].cpu().numpy(), o["departure"])
        np.testing.assert_array_equal(t["type"].cpu().numpy(), o["type"])
    hi = np.ceil(1.5 * W.flow_bound_mrps(g, pl)).astype(np.uint32)
    bb = cf.cf_goodput_bisect(g, pl, hi, 12, w.slo, w.seed)
    bo = orc.goodput_bisect(g, pl, hi, 12, w.slo, w.seed, n_threads=NT)
    np.testing.assert_array_equal(cf.to_numpy_u32(bb["rate_mrps"]), bo["rate_mrps"])
    np.testing.assert_array_equal(cf.to_numpy_u32(bb["goodput_mrps"]), bo["goodput_mrps"])
    np.testing.assert_array_equal(cf.to_numpy_u32(bb["counts"]), bo["counts"])
    # config 3's shape: bursty arrivals (Gamma, CV = 3), replica counts up to 32
    w = W.config3_multireplica(n_req=2000, n_trials=2, n_rates=3, plans_per_topology=12)
    w.graph.order_mode = 1
    check(cf, orc, w.graph, w.plans, w.rate_mrps, w.slo, w.seed)


@pytest.mark.parametrize("c_big", [33, 64, 100, 256])
def test_wide_free_time_vectors(cf, orc, c_big):
    g = omni_like(1500, n_trials=1)
    pl = W.make_plans([[(0b0011, c_big), (0b0100, 2), (0b1000, 3)], [(0b0011, 1), (0b0100, c_big), (0b1000, c_big - 1)]])
    R = W.flow_bound_mrps(g, pl)
    rates = np.maximum(W.rate_grid(R, [0.7, 1.1]), 1)
    slo = W.Slo([500_000, 600_000, 900_000, 1_000_000], [9] * 4, [10] * 4)
    check(cf, orc, g, pl, rates, slo, 21)
    # saturate the wide stage: a service far above the gap fills all its replicas
    g2 = W.Graph(1, 1, 2500, 1, [1], W.mix_thresholds([1.0]), [0], [W.exponential_qtab(2_000_000.0)],
                 W.exponential_qtab(65536.0), np.zeros((0, 2)), order_mode=1)
    pl2 = W.make_plans([[(1, c_big)]])
    r2 = np.maximum(W.rate_grid(W.flow_bound_mrps(g2, pl2), [0.9, 1.3]), 1)
    check(cf, orc, g2, pl2, r2, W.Slo([4_000_000], [9], [10]), 8)


def test_routes_overlap_and_wide_graph(cf, orc):
    # R26: routes (the 3-word record carries the route draw)
    g = mllm(2500, n_trials=2)
    g.order_mode = 1
    pl = two_path_plans([(2, 3, 2), (1, 6, 1), (3, 2, 4)], 0.6, 0.4)
    rates = np.array([[3_000, 9_000], [4_000, 12_000], [5_000, 15_000]], np.uint32)
    slo = W.Slo([2_000_000, 3_000_000], [9, 9], [10, 10])
    check(cf, orc, g, pl, rates, slo, 13)
    # R24: the idle/busy rule
    g = overlap_graph(n_req=2200, n_trials=2)
    g.order_mode = 1
    pl = W.make_plans([[(0b001, 2), (0b010, 1), (0b100, 3)], [(0b011, 2), (0b100, 2)], [(0b111, 4)]])
    rates = np.maximum(W.rate_grid(W.flow_bound_mrps(g, pl), [0.5, 0.9, 1.2]), 1)
    check(cf, orc, g, pl, rates, W.Slo([300_000, 400_000, 500_000], [9] * 3, [10] * 3), 11)
    t = cf.cf_trace_sim(g, pl, 0, int(rates[0, 1]), 1, 11)
    o = orc.trace_sim(g, pl, 0, int(rates[0, 1]), 1, 11)
    np.testing.assert_array_equal(t["departure"].cpu().numpy(), o["departure"])
    # eight components, eight types, eight stages
    rng = np.random.default_rng(4)
    C = T = 8
    tabs = [W.lognormal_qtab(float(rng.integers(5_000, 60_000)), 0.5) for _ in range(C)]
    masks = [int(m) | 1 << int(rng.integers(0, C)) for m in rng.integers(0, 256, T)]
    g = W.Graph(C, T, 1300, 2, masks, W.mix_thresholds(rng.dirichlet(np.ones(T))), np.repeat(np.arange(C, dtype=np.uint16), T),
                tabs, W.gamma_qtab(0.5, 65536.0), [[i, i + 1] for i in range(C - 1)], edge_delay_us=2_000, order_mode=1)
    plan_list = []
    for _ in range(20):
        cuts = sorted(rng.choice(np.arange(1, C), size=int(rng.integers(0, C)), replace=False).tolist())
        bounds = [0] + cuts + [C]
        plan_list.append([(sum(1 << i for i in range(a, b)), int(rng.integers(1, 9))) for a, b in zip(bounds, bounds[1:])])
    pl = W.make_plans(plan_list, max_stages=8)
    rates = np.maximum(W.rate_grid(W.flow_bound_mrps(g, pl), [0.5, 0.9, 1.3]), 1)
    check(cf, orc, g, pl, rates, W.Slo(rng.integers(50_000, 400_000, T), [9] * T, [10] * T), 77)


def test_forkjoin_under_arrival_order(cf, orc):
    """R25 + R27: predecessor stages gate a request's arrival at a stage; service in order of readiness."""
    w = W.config4_sweep(n_req=1700, n_trials=2, vectors_per_pattern=3, n_variants=1)   # 8 types, up to 3 parallel encoders
    g, pl = w.graph, w.plans
    g.join_mode, g.order_mode = 1, 1
    rates = np.maximum(W.rate_grid(W.flow_bound_mrps(g, pl), [0.05, 0.8, 1.3]), 1)
    for delay in (0, 9_000):
        g.edge_delay_us = delay
        a = check(cf, orc, g, pl, rates, w.slo, w.seed, 2)
    g.order_mode = 0
    b = orc.eval_plans(g, pl, rates, w.slo, w.seed, 2, n_threads=NT)
    g.order_mode = 1
    assert (a["dep_sum"] != b["dep_sum"]).any()
    for p in (0, 40, 95):
        t = cf.cf_trace_sim(g, pl, p, int(rates[p, 1]), 1, w.seed, variant=2)
        o = orc.trace_sim(g, pl, p, int(rates[p, 1]), 1, w.seed, variant=2)
        np.testing.assert_array_equal(t["departure"].cpu().numpy(), o["departure"])
    hi = orc.flow_bound(g, pl, 3, 2)["rate_mrps"]
    bb = cf.cf_goodput_bisect(g, pl, hi, 9, w.slo, w.seed)
    bo = orc.goodput_bisect(g, pl, hi, 9, w.slo, w.seed, n_threads=NT)
    np.testing.assert_array_equal(cf.to_numpy_u32(bb["rate_mrps"]), bo["rate_mrps"])
    np.testing.assert_array_equal(cf.to_numpy_u32(bb["counts"]), bo["counts"])
    # with CPU-GPU overlap on the encoders on top (R24 + R25 + R27)
    g.tabs = g.tabs + [W.lognormal_qtab(25_000.0, 0.5), W.lognormal_qtab(220_000.0, 0.6), W.exponential_qtab(8_000.0)]
    cpu = np.full(6 * 8, 0xFFFF, np.uint16)
    for i in range(3):
        cpu[i * 8:(i + 1) * 8] = 6 + i
    g.cpu_tab = cpu
    check(cf, orc, g, pl, rates, w.slo, w.seed, 1)
    # an 8-component DAG with two fan-ins, 8 stages
    rng = np.random.default_rng(4)
    C = T = 8
    tabs = [W.lognormal_qtab(float(rng.integers(5_000, 60_000)), 0.5) for _ in range(C)]
    masks = [int(m) | 1 << int(rng.integers(0, C)) for m in rng.integers(0, 256, T)]
    edges = [[0, 3], [1, 3], [2, 3], [3, 4], [3, 5], [4, 6], [5, 6], [6, 7]]
    g = W.Graph(C, T, 1000, 2, masks, W.mix_thresholds(rng.dirichlet(np.ones(T))), np.repeat(np.arange(C, dtype=np.uint16), T),
                tabs, W.gamma_qtab(0.5, 65536.0), edges, edge_delay_us=2_000, join_mode=1, order_mode=1)
    plan_list = []
    for _ in range(30):
        cuts = sorted(rng.choice(np.arange(1, C), size=int(rng.integers(0, C)), replace=False).tolist())
        bounds = [0] + cuts + [C]
        plan_list.append([(sum(1 << i for i in range(a, b)), int(rng.integers(1, 9))) for a, b in zip(bounds, bounds[1:])])
    pl = W.make_plans(plan_list, max_stages=8)
    rates = np.maximum(W.rate_grid(W.flow_bound_mrps(g, pl), [0.5, 0.9, 1.3]), 1)
    check(cf, orc, g, pl, rates, W.Slo(rng.integers(50_000, 400_000, T), [9] * T, [10] * T), 77)


def test_more_simulations_than_warps_in_flight_and_edge_cases(cf, orc):
    import torch
    g = omni_like(300, n_trials=12)
    pl = W.make_plans(([[(0b0011, 2), (0b0100, 3), (0b1000, 2)]] * 3 + [[(0b0111, 4), (0b1000, 2)]] * 2) * 10)
    rates = np.maximum(W.rate_grid(W.flow_bound_mrps(g, pl), [0.3, 0.5, 0.7, 0.9, 1.1, 1.3]), 1)
    slo = W.Slo([500_000, 600_000, 900_000, 1_000_000], [9] * 4, [10] * 4)
    # 3 600 simulations; cf_workspace_bytes holds the scratch of 3 552 in flight, so some warps run two
    want = check(cf, orc, g, pl, rates, slo, 9)
    np.testing.assert_array_equal(want["counts"][0], want["counts"][1])       # duplicate plans (R4)
    # an out-of-range rate zeroes that simulation and raises the sticky status; the others are unaffected
    bad = rates.copy()
    bad[1, 2] = 0
    got = cf.cf_eval_plans(g, pl, bad, slo, 9, check=False)
    assert cf.cf_workspace_status(got["workspace"]) == cf.CF_ERR_RANGE
    c = cf.to_numpy_u32(got["counts"])
    assert (c[1, 2] == 0).all()
    np.testing.assert_array_equal(c[0], want["counts"][0])
    # refusals: materialised stream, too many replicas, unknown mode
    w = W.config4_sweep(n_req=100, n_trials=1, vectors_per_pattern=1, n_patterns=2, n_variants=1)
    w.graph.order_mode = 1
    rec = torch.zeros((1, 1, 100, 32), dtype=torch.uint8, device="cuda")
    assert cf.cf_eval_plans(w.graph, w.plans, [[1000]] * 2, w.slo, 0, stream_records=rec, check=False)["rc"] == cf.CF_ERR_ARG
    big = W.make_plans([[(0b0111, 257), (0b1000, 2)]])
    assert cf.cf_eval_plans(g, big, [[1000]], slo, 9, check=False)["rc"] == cf.CF_ERR_RANGE
    g.order_mode = 2
    assert cf.cf_eval_plans(g, pl, rates, slo, 9, check=False)["rc"] == cf.CF_ERR_ARG
