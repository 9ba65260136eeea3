"""GPU parity of the fork-join routing mode (R25): graphs with
join_mode = 1 run on the JOIN variant of the 64-bit kernel; everything against the oracle, bit for bit."""
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


def check(cf, orc, g, pl, rates, slo, seed, variant=0):
    want = orc.eval_plans(g, pl, rates, slo, seed, variant, n_threads=NT)
    got = cf.cf_eval_plans(g, pl, rates, slo, seed, variant)
    assert cf.cf_workspace_status(got["workspace"]) == want["rc"] == 0
    np.testing.assert_array_equal(cf.to_numpy_u32(got["counts"]), want["counts"])
    np.testing.assert_array_equal(cf.to_numpy_u64(got["dep_sum"]), want["dep_sum"])
    np.testing.assert_array_equal(got["makespan"].cpu().numpy(), want["makespan"])
    return want


def test_forkjoin_parity(cf, orc):
    w = W.config4_sweep(n_req=1700, n_trials=2, vectors_per_pattern=3, n_variants=1)  # 8 types, up to 3 parallel encoders
    g, pl = w.graph, w.plans
    g.join_mode = 1
    rates = np.maximum(W.rate_grid(W.flow_bound_mrps(g, pl), [0.05, 0.8, 1.3]), 1)
    for delay in (0, 9_000):
        g.edge_delay_us = delay
        a = check(cf, orc, g, pl, rates, w.slo, w.seed, 2)
    g.join_mode = 0
    b = orc.eval_plans(g, pl, rates, w.slo, w.seed, 2, n_threads=NT)
    g.join_mode = 1
    assert (a["dep_sum"] != b["dep_sum"]).any()  # parallel encoders finish earlier than queued one after another
    for p in (0, 40, 95):
        t = cf.cf_trace_sim(g, pl, p, int(rates[p, 1]), 1, w.seed, variant=2)
        o = orc.trace_sim(g, pl, p, int(rates[p, 1]), 1, w.seed, variant=2)
        np.testing.assert_array_equal(t["arrival"].cpu().numpy(), o["arrival"])
        np.testing.assert_array_equal(t["departure"].cpu().numpy(), o["departure"])
    hi = orc.flow_bound(g, pl, 3, 2)["rate_mrps"]
    bb = cf.cf_goodput_bisect(g, pl, hi, 9, w.slo, w.seed)
    bo = orc.goodput_bisect(g, pl, hi, 9, w.slo, w.seed, n_threads=NT)
    np.testing.assert_array_equal(cf.to_numpy_u32(bb["rate_mrps"]), bo["rate_mrps"])
    np.testing.assert_array_equal(cf.to_numpy_u32(bb["counts"]), bo["counts"])
    # one replica everywhere still runs the thread-per-simulation kernel; the scan kernel refuses
    pl1 = W.Plans(pl.n_stages, pl.stage_mask, np.ones_like(pl.stage_c))
    r1 = np.maximum(W.rate_grid(W.flow_bound_mrps(g, pl1), [0.6, 1.2]), 1)
    check(cf, orc, g, pl1, r1, w.slo, w.seed)
    # with CPU-GPU overlap on the encoders on top (R24 + R25)
    g.tabs = g.tabs + [W.lognormal_qtab(25_000.0, 0.5), W.lognormal_qtab(220_000.0, 0.6), W.exponential_qtab(8_000.0)]
    cpu = np.full(6 * 8, 0xFFFF, np.uint16)
    for i in range(3):
        cpu[i * 8:(i + 1) * 8] = 6 + i
    g.cpu_tab = cpu
    check(cf, orc, g, pl, rates, w.slo, w.seed, 1)


def test_forkjoin_monte_carlo_latency(cf, orc):
    """Phase 2 under fork-join (R25): the critical path of every sampled request, per plan."""
    w = W.config4_sweep(n_req=4000, n_trials=3, vectors_per_pattern=2, n_variants=1)
    g, pl = w.graph, w.plans
    g.join_mode = 1
    g.edge_delay_us = 9_000
    slo = W.Slo([150_000, 200_000, 180_000, 260_000, 3_600_000, 3_700_000, 3_650_000, 3_800_000], [9] * 8, [10] * 8)
    rate = orc.flow_bound(g, pl, 4, 5)["rate_mrps"]
    o = orc.mc_latency(g, pl, rate, slo, w.seed, 2)
    m = cf.cf_mc_latency(g, pl, rate, slo, w.seed, 2)
    assert o["rc"] == 0
    np.testing.assert_array_equal(cf.to_numpy_u32(m["counts"]), o["counts"])
    np.testing.assert_array_equal(cf.to_numpy_u32(m["goodput_mrps"]), o["goodput_mrps"])
    g.join_mode = 0
    seq = orc.mc_latency(g, pl, rate, slo, w.seed, 2)
    assert (seq["counts"][..., 1] <= o["counts"][..., 1]).all() and seq["counts"][..., 1].sum() < o["counts"][..., 1].sum()
    g.join_mode = 1
    # an 8-component DAG with two fan-ins, 8 types, CPU times on three components
    rng = np.random.default_rng(5)
    C = T = 8
    tabs = [W.lognormal_qtab(float(rng.integers(5_000, 60_000)), 0.5) for _ in range(C)] + [W.exponential_qtab(9_000.0)]
    masks = [int(mm) | 1 << int(rng.integers(0, C)) for mm in rng.integers(0, 256, T)]
    edges = [[0, 3], [1, 3], [2, 3], [3, 4], [3, 5], [4, 6], [5, 6], [6, 7]]
    cpu = np.full(C * T, 0xFFFF, np.uint16)
    cpu[:3 * T] = C
    g = W.Graph(C, T, 2500, 2, masks, W.mix_thresholds(rng.dirichlet(np.ones(T))), np.repeat(np.arange(C, dtype=np.uint16), T),
                tabs, W.gamma_qtab(0.5, 65536.0), edges, edge_delay_us=2_000, join_mode=1, cpu_tab=cpu)
    plan_list = []
    for _ in range(30):
        cuts = sorted(rng.choice(np.arange(1, C), size=int(rng.integers(0, C)), replace=False).tolist())
        bounds = [0] + cuts + [C]
        plan_list.append([(sum(1 << i for i in range(a, b)), int(rng.integers(1, 9))) for a, b in zip(bounds, bounds[1:])])
    pl = W.make_plans(plan_list, max_stages=8)
    slo = W.Slo(rng.integers(50_000, 300_000, T), [9] * T, [10] * T)
    rate = rng.integers(1, 2**31, 30).astype(np.uint32)
    o = orc.mc_latency(g, pl, rate, slo, 77, 1)
    m = cf.cf_mc_latency(g, pl, rate, slo, 77, 1)
    np.testing.assert_array_equal(cf.to_numpy_u32(m["counts"]), o["counts"])
    np.testing.assert_array_equal(cf.to_numpy_u32(m["goodput_mrps"]), o["goodput_mrps"])
    assert 0 < o["counts"][..., 1].sum() < o["counts"][..., 0].sum()


def test_forkjoin_wide_graph_and_refusals(cf, orc):
    import torch
    rng = np.random.default_rng(4)
    C = T = 8
    tabs = [W.lognormal_qtab(float(rng.integers(5_000, 60_000)), 0.5) for _ in range(C)]
    masks = [int(m) | 1 << int(rng.integers(0, C)) for m in rng.integers(0, 256, T)]
    # a DAG with two fan-ins: 0,1,2 -> 3; 3 -> 4,5; 4,5 -> 6; 6 -> 7
    edges = [[0, 3], [1, 3], [2, 3], [3, 4], [3, 5], [4, 6], [5, 6], [6, 7]]
    g = W.Graph(C, T, 1000, 2, masks, W.mix_thresholds(rng.dirichlet(np.ones(T))), np.repeat(np.arange(C, dtype=np.uint16), T),
                tabs, W.gamma_qtab(0.5, 65536.0), edges, edge_delay_us=2_000, join_mode=1)
    plan_list = []
    for _ in range(30):
        cuts = sorted(rng.choice(np.arange(1, C), size=int(rng.integers(0, C)), replace=False).tolist())
        bounds = [0] + cuts + [C]
        plan_list.append([(sum(1 << i for i in range(a, b)), int(rng.integers(1, 9))) for a, b in zip(bounds, bounds[1:])])
    pl = W.make_plans(plan_list, max_stages=8)
    assert orc.validate(g, pl) == 0
    rates = np.maximum(W.rate_grid(W.flow_bound_mrps(g, pl), [0.5, 0.9, 1.3]), 1)
    slo = W.Slo(rng.integers(50_000, 400_000, T), [9] * T, [10] * T)
    check(cf, orc, g, pl, rates, slo, 77)
    w = W.config4_sweep(n_req=100, n_trials=1, vectors_per_pattern=1, n_patterns=2, n_variants=1)
    w.graph.join_mode = 1
    rec = torch.zeros((1, 1, 100, 32), dtype=torch.uint8, device="cuda")
    assert cf.cf_eval_plans(w.graph, w.plans, [[1000]] * 2, w.slo, 0, stream_records=rec, check=False)["rc"] == cf.CF_ERR_ARG
    w.graph.join_mode = 2
    assert cf.cf_eval_plans(w.graph, w.plans, [[1000]] * 2, w.slo, 0, check=False)["rc"] == cf.CF_ERR_ARG
