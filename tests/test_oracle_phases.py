"""Pins of the oracle's phase-1 / phase-2 / selection functions (oracle/cf_oracle_phases.cpp;
SURVEY.md 8(f) NEXT-1..3) against things other than themselves: hand-worked examples, closed forms,
exact rational arithmetic, brute force on tiny inputs, the independent pure-Python request generator
of tests/refsim.py, and the identity "Monte Carlo latency = simulation with unlimited replicas"
("queuing not modeled")."""
from fractions import Fraction

import numpy as np
import pytest

import refsim
from paper_2512_14098_b200 import workloads as W


# ------------------------------------------------------------------------------------------
# table means (R21)
# ------------------------------------------------------------------------------------------
def exact_mean(tab) -> Fraction:
    """Sum over cells of P(cell) x (q_i + q_{i+1}) / 2 in exact rationals, from the table's
    geometric definition (level k covers [1-2^-k, 1-2^-(k+1)), the last level the rest)."""
    L, B = tab.levels, tab.log2_cells
    total = Fraction(0)
    for k in range(L):
        level_p = Fraction(1, 2 ** (k + 1)) if k < L - 1 else Fraction(1, 2 ** (L - 1))
        for m in range(1 << B):
            i = (k << B) + m
            total += level_p / (1 << B) * Fraction(int(tab.q[i]) + int(tab.q[i + 1]), 2)
    return total


@pytest.mark.parametrize("L,B", [(16, 6), (1, 10), (1, 0), (4, 3), (32, 2), (8, 16), (20, 0)])
def test_table_mean_is_the_exact_cell_average(orc, L, B):
    rng = np.random.default_rng(L * 100 + B)
    q = np.sort(rng.integers(0, 2**31 - 1, (L << B) + 1)).astype(np.int32)
    tab = W.QTab(L, B, q)
    want = exact_mean(tab) * 65536
    assert orc.qtab_mean_q16(tab) == want.numerator // want.denominator  # floor of the exact value


def test_table_mean_special_cases(orc):
    assert orc.qtab_mean_q16(W.constant_qtab(12345)) == 12345 * 65536
    assert orc.qtab_mean_q16(W.QTab(1, 0, np.array([10, 31], np.int32))) == (10 + 31) * 32768
    tab = W.exponential_qtab(1_000_000.0)  # against the harness's float moments and the exponential's mean
    assert abs(orc.qtab_mean_q16(tab) / 65536 / W.qtab_moments(tab)[0] - 1) < 1e-9
    assert abs(orc.qtab_mean_q16(tab) / 65536 / 1e6 - 1) < 2e-4


# ------------------------------------------------------------------------------------------
# phase 1: flow bound, bottleneck, redundant capacity
# ------------------------------------------------------------------------------------------
def hand_graph():
    """E -> LLM with constant services E = 30 ms, LLM = 400 ms; text 75 % {LLM}, image+text 25 %
    {E, LLM}; a third component nobody uses. Demands per arriving request: E 0.25 x 30 000 =
    7 500 us, LLM 400 000 us, colocated {E,LLM} 0.75 x 400 000 + 0.25 x 430 000 = 407 500 us."""
    tabs = [W.constant_qtab(30_000), W.constant_qtab(400_000), W.constant_qtab(77)]
    return W.Graph(3, 2, 64, 2, [0b010, 0b011], W.mix_thresholds([0.75, 0.25]), [0, 0, 1, 1, 2, 2], tabs,
                   W.exponential_qtab(65536.0), [[0, 1]])


HAND_PLANS = [
    [(0b011, 4)],                          # A colocated, 4 executors: R = 4e9 / 407 500 = 9815.95 -> 9815
    [(0b001, 1), (0b010, 4)],              # B E: 1e9/7 500 = 133 333; LLM: 4e9/400 000 = 10 000 -> LLM
    [(0b001, 3), (0b010, 4)],              # C as B, but E keeps 266 666 >= 10 000 with 2 executors: redundant
    [(0b001, 1), (0b010, 60)],             # D LLM 150 000, E 133 333 -> E; LLM with 59: 147 500 >= 133 333: redundant
    [(0b001, 1), (0b010, 4), (0b100, 1)],  # E a node without demand, one executor: not redundant
    [(0b001, 1), (0b010, 4), (0b100, 2)],  # F the same node with two executors: redundant
]
HAND_BOUND = [9815, 10_000, 10_000, 133_333, 10_000, 10_000]
HAND_BOTTLENECK = [0, 1, 1, 0, 1, 1]
HAND_REDUNDANT = [0, 0, 1, 1, 0, 1]


def test_flow_bound_hand_worked(orc):
    g = hand_graph()
    assert int(g.type_thresh[0]) == 3 * 2**30  # the 75 % split is exact in Q32
    pl = W.make_plans(HAND_PLANS, max_stages=3)
    f = orc.flow_bound(g, pl, 3, 2)
    assert f["rc"] == 0
    np.testing.assert_array_equal(f["bound_mrps"], HAND_BOUND)
    np.testing.assert_array_equal(f["bottleneck"], HAND_BOTTLENECK)
    np.testing.assert_array_equal(f["redundant"], HAND_REDUNDANT)
    np.testing.assert_array_equal(f["rate_mrps"], [b * 3 // 2 for b in HAND_BOUND])  # alpha R_d
    # no demand anywhere: capped at the largest valid rate, no bottleneck
    g0 = W.Graph(1, 1, 8, 1, [0], W.mix_thresholds([1.0]), [0], [W.constant_qtab(5)], W.exponential_qtab(65536.0),
                 np.zeros((0, 2)))
    f0 = orc.flow_bound(g0, W.make_plans([[(1, 1)], [(1, 2)]]))
    assert f0["bound_mrps"].tolist() == [10**9, 10**9] and f0["bottleneck"].tolist() == [255, 255]
    assert f0["redundant"].tolist() == [0, 1]


def test_flow_bound_matches_the_float_formula(orc):
    # R_p = min_s c_s / sum_t pi_t E[S_{s,t}] as the harness computes it in float64
    for w in (W.config1_mllm(n_req=10, n_trials=1, n_rates=1),
              W.config2_omni(n_req=10, n_trials=1, n_rates=1, vectors_per_pattern=8),
              W.config4_sweep(n_req=10, n_trials=1, vectors_per_pattern=4)):
        f = orc.flow_bound(w.graph, w.plans)
        R = W.flow_bound_mrps(w.graph, w.plans)
        assert np.abs(f["bound_mrps"].astype(np.float64) - R).max() < 1.0 + 1e-6 * R.max()  # floor + Q16/Q32 rounding
        # the bottleneck is the stage with the smallest capacity / demand ratio; redundancy by its definition
        for p in range(0, w.plans.n_plans, 7):
            caps = []
            for s in range(int(w.plans.n_stages[p])):
                one = W.make_plans([[(int(w.plans.stage_mask[p, s]), 1)] +
                                    [(int(w.plans.stage_mask[p, j]), 1000) for j in range(int(w.plans.n_stages[p])) if j != s]])
                # capacity of stage s alone, per executor, from the float formula on a plan where s is the bottleneck
                caps.append(W.flow_bound_mrps(w.graph, one)[0] * int(w.plans.stage_c[p, s]))
            assert int(f["bottleneck"][p]) == int(np.argmin(caps))
            c = w.plans.stage_c[p, :len(caps)].astype(np.float64)
            slack = [(c[s] - 1) / c[s] * caps[s] >= min(caps) * (1 + 1e-9) for s in range(len(caps)) if c[s] >= 2]
            tight = [(c[s] - 1) / c[s] * caps[s] <= min(caps) * (1 - 1e-9) for s in range(len(caps)) if c[s] >= 2]
            if any(slack):
                assert f["redundant"][p] == 1
            if all(tight):
                assert f["redundant"][p] == 0


# ------------------------------------------------------------------------------------------
# phase 2: Monte-Carlo latency
# ------------------------------------------------------------------------------------------
def test_mc_equals_simulation_with_unlimited_replicas(orc):
    # "queuing not modeled": with at least N replicas at every stage nobody ever waits, so the
    # request-level simulator's sojourn is the accumulated latency, at any rate
    w = W.config2_omni(n_req=700, n_trials=2, n_rates=2, vectors_per_pattern=1, n_patterns=32)
    w.graph.edge_delay_us = 10_000
    big = W.Plans(w.plans.n_stages, w.plans.stage_mask, np.full_like(w.plans.stage_c, 700))
    slo = W.Slo([150_000, 4_000_000, 350_000, 4_200_000], [9] * 4, [10] * 4)
    sim = orc.eval_plans(w.graph, big, w.rate_mrps * 3, slo, w.seed, 5, n_threads=8)
    rate = w.rate_mrps[:, 0]
    mc = orc.mc_latency(w.graph, w.plans, rate, slo, w.seed, 5)
    assert mc["rc"] == 0
    np.testing.assert_array_equal(mc["counts"], sim["counts"][:, 0])
    np.testing.assert_array_equal(mc["counts"], sim["counts"][:, 1])
    h = mc["counts"][..., 1].astype(np.int64).sum(1)  # pooled over trials: [P, T]
    assert 0 < h.sum() < 700 * 2 * w.plans.n_plans    # some requests miss, some hit
    np.testing.assert_array_equal(mc["goodput_mrps"], rate[:, None].astype(np.int64) * h // (700 * 2))
    # the hop count matters: a disaggregated plan pays the delay per edge, the colocated one does not
    assert len({tuple(c) for c in mc["counts"][..., 1].reshape(w.plans.n_plans, -1)}) > 1


def test_mc_eight_requests_by_hand(orc):
    # 8 requests drawn by the independent pure-Python generator; latency = sum of the services on the
    # request's path + one delay per hop between visited stages, straight from the sentence in PAPER.md:278
    w = W.config2_omni(n_req=8, n_trials=1, n_rates=1, vectors_per_pattern=1, n_patterns=32)
    g = w.graph
    g.edge_delay_us = 25_000
    for p in (0, 5, 31):
        for variant in (0, 3):
            _, types, svc = refsim.gen_requests(g, w.seed, variant, 0, rate_mrps=1000)
            L = [120_000, 3_500_000, 300_000, 3_700_000]
            cnt, hits = [0] * 4, [0] * 4
            for n in range(8):
                route = [s for s in range(int(w.plans.n_stages[p])) if int(w.plans.stage_mask[p, s]) & int(g.type_mask[types[n]])]
                lat = sum(svc[n].values()) + 25_000 * (len(route) - 1 if route else 0)
                cnt[types[n]] += 1
                hits[types[n]] += lat <= L[types[n]]
            mc = orc.mc_latency(g, w.plans.subset([p]), [7777], W.Slo(L, [9] * 4, [10] * 4), w.seed, variant)
            assert mc["counts"][0, 0, :, 0].tolist() == cnt and mc["counts"][0, 0, :, 1].tolist() == hits
            assert mc["goodput_mrps"][0].tolist() == [7777 * h // 8 for h in hits]


# ------------------------------------------------------------------------------------------
# Pareto pruning and the default policy
# ------------------------------------------------------------------------------------------
def test_pareto_hand_worked(orc):
    # plan 2 is dominated by plan 0 (5>=5, 5>4) and by plan 1 (6>5, 4>=4); 0 and 1 do not dominate each other
    r = orc.pareto_select([[5, 5], [6, 4], [5, 4]])
    assert r["pruned"].tolist() == [0, 0, 1] and r["n_survivors"] == 2 and r["best"] == 0  # sums 10, 10, 9: lowest index
    r = orc.pareto_select([[3, 3], [3, 3], [2, 9]])     # equal vectors do not prune each other (R23)
    assert r["pruned"].tolist() == [0, 0, 0] and r["best"] == 2
    r = orc.pareto_select([[5, 5], [6, 6], [1, 7]], alive=[1, 0, 1])  # a dead plan dominates nobody and cannot win
    assert r["pruned"].tolist() == [0, 1, 0] and r["best"] == 0 and r["n_survivors"] == 2
    r = orc.pareto_select([[0, 0]], alive=[0])
    assert r["pruned"].tolist() == [1] and r["best"] == 0xFFFFFFFF and r["n_survivors"] == 0


def test_pareto_brute_force(orc):
    rng = np.random.default_rng(12)
    for _ in range(60):
        P, T = int(rng.integers(1, 17)), int(rng.integers(1, 9))
        G = rng.integers(0, 6, (P, T)).astype(np.uint32)  # small values: many ties and duplicates
        alive = rng.integers(0, 4, P) > 0 if rng.random() < 0.5 else None
        live = np.ones(P, bool) if alive is None else alive
        ge = (G[None, :, :] >= G[:, None, :]).all(-1)      # [p, q]: q >= p everywhere
        gt = (G[None, :, :] > G[:, None, :]).any(-1)
        dominated = (ge & gt & live[None, :]).any(1)
        r = orc.pareto_select(G, None if alive is None else alive.astype(np.uint8))
        np.testing.assert_array_equal(r["pruned"].astype(bool), dominated | ~live)
        assert r["n_survivors"] == int((~dominated & live).sum())
        if live.any():
            sums = np.where(live, G.astype(np.int64).sum(1), -1)
            assert r["best"] == int(np.argmax(sums))       # first index of the maximum
            assert not r["pruned"][r["best"]]               # the policy's choice is never Pareto-suboptimal
