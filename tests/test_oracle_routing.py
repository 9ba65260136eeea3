"""Pins of routing between alternative paths ("routing probabilities ... between
alternative parallel paths in the logical plan"; R26): degenerate tables reduce to plain
plans, 8-request inputs against the independent simulators of tests/refsim.py with the route drawn in
pure Python, route frequencies, a hand-worked flow bound, validation."""
import numpy as np
import pytest

import refsim
from paper_2512_14098_b200 import workloads as W


def mllm(n_req, n_trials=1, delay=4_000, constant=False):
    tabs = [W.constant_qtab(30_000), W.constant_qtab(400_000)] if constant else \
           [W.lognormal_qtab(30_000.0, 0.4), W.lognormal_qtab(400_000.0, 0.6)]
    return W.Graph(2, 2, n_req, n_trials, [0b10, 0b11], W.mix_thresholds([0.75, 0.25]), [0, 0, 1, 1], tabs,
                   W.exponential_qtab(65536.0), [[0, 1]], edge_delay_us=delay)


def two_path_plans(cs, p_disagg_text, p_disagg_image):
    """Stages s0 = {E}, s1 = {LLM} (the disaggregated path) and s2 = {E, LLM} (the colocated node); route 0 =
    disaggregated, route 1 = colocated; one plan per replica vector in cs."""
    P = len(cs)
    pl = W.make_plans([[(0b01, c[0]), (0b10, c[1]), (0b11, c[2])] for c in cs], max_stages=3)
    rm = np.tile(np.array([[0b011, 0b100], [0b011, 0b100]], np.uint8), (P, 1, 1))
    q = lambda x: min(int(round(x * 2**32)), 2**32 - 1)
    rc = np.tile(np.array([[q(p_disagg_text), 0xFFFFFFFF], [q(p_disagg_image), 0xFFFFFFFF]], np.uint32), (P, 1, 1))
    return W.Plans(pl.n_stages, pl.stage_mask, pl.stage_c, 2, rm, rc)


def test_degenerate_tables_reduce_to_plain_plans(orc):
    g = mllm(1500, 2)
    cs = [(1, 3, 2), (2, 5, 4)]
    rates = np.array([[3000, 9000], [6000, 15000]], np.uint32)
    slo = W.Slo([2_000_000, 3_000_000], [9, 9], [10, 10])
    plain_d = W.make_plans([[(0b01, c[0]), (0b10, c[1])] for c in cs], max_stages=3)
    plain_c = W.make_plans([[(0b11, c[2])] for c in cs], max_stages=3)
    for pd, plain in ((1.0, plain_d), (0.0, plain_c)):
        routed = two_path_plans(cs, pd, pd)
        if pd == 1.0:  # probability 1 is not representable in Q32: make the disaggregated route the catch-all
            routed.route_mask[:, :, 1] = 0b011
        assert orc.validate(g, routed) == 0
        a = orc.eval_plans(g, routed, rates, slo, 5, 1)
        b = orc.eval_plans(g, plain, rates, slo, 5, 1)
        for key in ("counts", "dep_sum", "makespan"):
            np.testing.assert_array_equal(a[key], b[key])
    # one route holding every stage == no routing table at all
    w = W.config2_omni(n_req=400, n_trials=2, n_rates=2, vectors_per_pattern=1, n_patterns=8)
    P, T = w.plans.n_plans, 4
    one = W.Plans(w.plans.n_stages, w.plans.stage_mask, w.plans.stage_c, 1, np.full((P, T, 1), 0xFF, np.uint8),
                  np.zeros((P, T, 1), np.uint32))
    a = orc.eval_plans(w.graph, one, w.rate_mrps, w.slo, w.seed)
    b = orc.eval_plans(w.graph, w.plans, w.rate_mrps, w.slo, w.seed)
    np.testing.assert_array_equal(a["dep_sum"], b["dep_sum"])
    np.testing.assert_array_equal(a["counts"], b["counts"])


def routes_by_hand(g, pl, p, seed, variant, trial, types, svc):
    """The route of every request from Philox block 0, word 2 (restated in pure Python) and its (stage, S) list."""
    key = (seed & refsim.MASK, (seed >> 32) & refsim.MASK)
    out, chosen = [], []
    for n, t in enumerate(types):
        u = refsim.philox4x32_10((n, trial, 0, variant), key)[2]
        MR = pl.max_routes
        r = next((rr for rr in range(MR) if u < int(pl.route_cum[p, t, rr])), MR - 1)
        chosen.append(r)
        rm, tm = int(pl.route_mask[p, t, r]), int(g.type_mask[t])
        route = []
        for s in range(int(pl.n_stages[p])):
            m = int(pl.stage_mask[p, s]) & tm
            if m and (rm >> s) & 1:
                route.append((s, sum(svc[n][i] for i in range(g.n_comp) if (m >> i) & 1)))
        out.append(route)
    return out, chosen


@pytest.mark.parametrize("seed", range(5))
def test_eight_requests_against_independent_simulators(orc, seed):
    g = mllm(8)
    rng = np.random.default_rng(seed)
    for c_hi in (1, 3):
        cs = [tuple(int(x) for x in rng.integers(1, c_hi + 1, 3))]
        pl = two_path_plans(cs, float(rng.uniform(0.2, 0.8)), float(rng.uniform(0.2, 0.8)))
        for rate in (2_000, 12_000):
            A, types, svc = refsim.gen_requests(g, 90 + seed, 2, 0, rate)
            routes, chosen = routes_by_hand(g, pl, 0, 90 + seed, 2, 0, types, svc)
            t = orc.trace_sim(g, pl, 0, rate, 0, seed=90 + seed, variant=2)
            assert t["departure"].tolist() == refsim.per_server_sim(A, routes, list(cs[0]), g.edge_delay_us)
            if c_hi == 1:
                assert t["departure"].tolist() == refsim.event_sim(A, routes, list(cs[0]), g.edge_delay_us)


def test_route_frequencies_and_monotone_effect(orc):
    # 20 000 requests: the share that took the colocated route, read off the departures of an
    # unlimited-replica plan (colocated: no hop, disaggregated image requests pay one delay)
    g = mllm(20_000, 1, delay=1_000_000, constant=True)   # a 1 s hop makes the two routes unmistakable
    pl = two_path_plans([(20_000, 20_000, 20_000)], 0.5, 0.3)
    t = orc.trace_sim(g, pl, 0, 1000, 0, seed=3)
    soj = t["departure"] - t["arrival"]
    img = t["type"] == 1
    assert set(np.unique(soj[img])) == {430_000, 1_430_000} and set(np.unique(soj[~img])) == {400_000}
    frac = (soj[img] == 1_430_000).mean()
    assert abs(frac - 0.3) < 4 * np.sqrt(0.3 * 0.7 / img.sum())


def test_flow_bound_with_routing_hand_worked(orc):
    # E 30 ms, LLM 400 ms; text 75 %, image 25 %; every type takes either path with probability 1/2:
    # demands s0 = .25*.5*30 000 = 3 750, s1 = (.75*.5 + .25*.5)*400 000 = 200 000,
    # s2 = .75*.5*400 000 + .25*.5*430 000 = 203 750 us per arriving request
    g = mllm(16, constant=True)
    pl = two_path_plans([(1, 4, 2), (1, 4, 50), (1, 3, 2)], 0.5, 0.5)
    f = orc.flow_bound(g, pl)
    assert f["rc"] == 0
    assert f["bound_mrps"].tolist() == [2 * 10**9 // 203_750, 4 * 10**9 // 200_000, 2 * 10**9 // 203_750]
    assert f["bottleneck"].tolist() == [2, 1, 2]
    assert f["redundant"].tolist() == [1, 1, 1]  # plan 0: s1 sustains 9 815 with 3 executors (15 000); plan 2: with 2 (10 000)
    pl = two_path_plans([(1, 2, 2)], 0.5, 0.5)   # s1 with one executor fewer: 5 000 < 9 815; s2: 4 907 < 9 815
    assert orc.flow_bound(g, pl)["redundant"].tolist() == [0]


def test_monte_carlo_latency_with_routes(orc):
    # constant services (E 30 ms, LLM 400 ms) and a 1 s hop: a text request always takes 400 ms, an image
    # request 430 ms on the colocated node and 1 430 ms on the disaggregated path; with L = 1 s the image
    # hits are exactly the requests that drew the colocated route
    g = mllm(4000, 2, delay=1_000_000, constant=True)
    pl = two_path_plans([(1, 1, 1), (5, 5, 5)], 0.5, 0.3)
    slo = W.Slo([1_000_000, 1_000_000], [9, 9], [10, 10])
    mc = orc.mc_latency(g, pl, [1000, 2000], slo, 3)
    assert mc["rc"] == 0
    for k in range(2):
        t = orc.trace_sim(g, two_path_plans([(4000, 4000, 4000)], 0.5, 0.3), 0, 1000, k, seed=3)
        img = t["type"] == 1
        colocated = (t["departure"] - t["arrival"])[img] == 430_000
        for p in range(2):   # replica counts do not matter to phase 2
            assert mc["counts"][p, k, :, 0].tolist() == [int((~img).sum()), int(img.sum())]
            assert mc["counts"][p, k, :, 1].tolist() == [int((~img).sum()), int(colocated.sum())]
    # random tables: phase 2 == the simulation with unlimited replicas, route draws included
    g = mllm(900, 2, delay=30_000)
    pl = two_path_plans([(2, 3, 2), (1, 1, 4)], 0.6, 0.4)
    slo = W.Slo([450_000, 520_000], [9, 9], [10, 10])
    big = W.Plans(pl.n_stages, pl.stage_mask, np.full_like(pl.stage_c, 900), pl.max_routes, pl.route_mask, pl.route_cum)
    sim = orc.eval_plans(g, big, np.array([[7_000], [9_000]], np.uint32), slo, 5, 1, n_threads=4)
    mc = orc.mc_latency(g, pl, [7_000, 9_000], slo, 5, 1)
    np.testing.assert_array_equal(mc["counts"], sim["counts"][:, 0])
    h = mc["counts"][..., 1].astype(np.int64).sum(1)
    np.testing.assert_array_equal(mc["goodput_mrps"], np.array([[7_000], [9_000]]) * h // 1800)
    assert 0 < h.sum() < 2 * 1800


def test_validation(orc):
    g = mllm(16)
    pl = two_path_plans([(1, 1, 1)], 0.5, 0.5)
    assert orc.validate(g, pl) == 0
    bad = two_path_plans([(1, 1, 1)], 0.5, 0.5)
    bad.route_mask[0, 1, 0] = 0b010      # image requests on the disaggregated path would skip the encoder
    assert orc.validate(g, bad) == orc.ORC_ERR_PLAN
    bad = two_path_plans([(1, 1, 1)], 0.5, 0.5)
    bad.route_mask[0, 0, 1] = 0b110      # text requests would be served by the LLM twice
    assert orc.validate(g, bad) == orc.ORC_ERR_PLAN
    bad = two_path_plans([(1, 1, 1)], 0.5, 0.5)
    bad.route_cum[0, 0] = [9, 3]
    assert orc.validate(g, bad) == orc.ORC_ERR_PLAN
    bad = two_path_plans([(1, 1, 1)], 0.5, 0.5)
    bad.max_routes = 5
    assert orc.validate(g, bad) == orc.ORC_ERR_ARG
    plain = W.make_plans([[(0b01, 1), (0b10, 1), (0b11, 1)]])  # overlapping masks need a routing table
    assert orc.validate(g, plain) == orc.ORC_ERR_PLAN
