"""Invariants, metamorphic properties, bisection and argument validation of the oracle (CPU)."""
import math
import os

import numpy as np
import pytest

import refsim
from paper_2512_14098_b200 import workloads as W

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def small_cfg1(**kw):
    return W.config1_mllm(n_req=kw.pop("n_req", 3000), n_trials=kw.pop("n_trials", 2),
                          n_rates=kw.pop("n_rates", 4), llm_max=kw.pop("llm_max", 4),
                          e_steps=kw.pop("e_steps", 3))


def test_counts_invariants_and_crn_monotonicity(orc):
    w = small_cfg1()
    r = orc.eval_plans(w.graph, w.plans, w.rate_mrps, w.slo, w.seed)
    assert r["rc"] == 0
    c = r["counts"].astype(np.int64)
    assert (c[..., 0].sum(-1) == w.graph.n_req).all()       # sum_t cnt_t = N
    assert (c[..., 1] <= c[..., 0]).all()                   # hits <= cnt
    # R4 common random numbers: type counts do not depend on plan or rate
    assert (c[..., 0] == c[0, 0][None, None, ..., 0]).all()
    # rates ascend along axis 1 -> hits non-increasing (sojourns monotone in the period)
    assert (np.diff(w.rate_mrps.astype(np.int64), axis=1) >= 0).all()
    assert (np.diff(c[..., 1], axis=1) <= 0).all()
    assert (np.diff(r["makespan"], axis=1) <= 0).all()      # higher rate -> earlier last arrival


def test_duplicate_plans_identical_outputs(orc):
    # R16: colocated plans with equal l+e are duplicates on purpose
    w = small_cfg1()
    pl = w.plans
    key = {}
    dup = 0
    rates = np.tile(np.array([[30_000, 60_000]], dtype=np.uint32), (pl.n_plans, 1))
    r = orc.eval_plans(w.graph, pl, rates, w.slo, w.seed)
    for p in range(pl.n_plans):
        sig = (int(pl.n_stages[p]), tuple(pl.stage_mask[p]), tuple(pl.stage_c[p]))
        if sig in key:
            q = key[sig]
            dup += 1
            assert (r["counts"][p] == r["counts"][q]).all()
            assert (r["dep_sum"][p] == r["dep_sum"][q]).all()
        key[sig] = p
    assert dup > 0


def test_sojourn_lower_bound_and_stage_monotonicity(orc):
    w = W.config2_omni(n_req=400, n_trials=2, n_rates=2, vectors_per_pattern=2, n_patterns=8)
    g = w.graph
    g.edge_delay_us = 10_000
    for p in range(0, w.plans.n_plans, 3):
        for k in range(2):
            rate = int(w.rate_mrps[p, 1])
            tr = orc.trace_sim(g, w.plans, p, rate, k, seed=w.seed)
            A, types, svc = refsim.gen_requests(g, w.seed, 0, k, rate)
            routes = refsim.stage_services(g, w.plans, p, types, svc)
            lb = np.array([a + sum(s for _, s in rt) + 10_000 * max(len(rt) - 1, 0)
                           for a, rt in zip(A, routes)])
            assert (tr["departure"] >= lb).all()
            # R14: a type with an empty route departs on arrival (none here: every type uses L_th)
            assert all(len(rt) > 0 for rt in routes)


def test_infinite_replicas_is_phase2_monte_carlo(orc):
    # no queueing -> latency = accumulated processing latencies
    w = W.config2_omni(n_req=300, n_trials=1, n_rates=1, vectors_per_pattern=1, n_patterns=4)
    pl = W.Plans(w.plans.n_stages, w.plans.stage_mask, np.where(w.plans.stage_c > 0, 300, 0))
    for p in range(pl.n_plans):
        tr = orc.trace_sim(w.graph, pl, p, 5000, 0, seed=9)
        A, types, svc = refsim.gen_requests(w.graph, 9, 0, 0, 5000)
        want = [a + sum(s.values()) for a, s in zip(A, svc)]
        assert tr["departure"].tolist() == want


def test_empty_route_type(orc):
    # R14: type 1 uses no component -> D = A, always a hit
    tabs = [W.exponential_qtab(5000.0)]
    g = W.Graph(1, 2, 200, 1, [1, 0], W.mix_thresholds([0.5, 0.5]), [0, 0], tabs,
                W.exponential_qtab(65536.0), np.zeros((0, 2)))
    pl = W.make_plans([[(1, 1)]])
    slo = W.Slo([10_000, 0], [9, 9], [10, 10])
    r = orc.eval_plans(g, pl, [[150_000]], slo, seed=1)
    c = r["counts"][0, 0, 0]
    assert c[1, 0] == c[1, 1] > 0
    tr = orc.trace_sim(g, pl, 0, 150_000, 0, seed=1)
    m = tr["type"] == 1
    assert (tr["departure"][m] == tr["arrival"][m]).all()


def test_theorem_a1_scale_invariance(orc):
    # scaling a type's times and its deadline by the same factor leaves its
    # attainment unchanged. Exact here: table entries, period and SLO scaled by the integer 3
    # (gaps are Q16 multiples of the period, so arrivals scale exactly when rounding is avoided).
    base = W.lognormal_qtab(8000.0, 0.6)
    gap = W.constant_qtab(65536)
    for scale in (1, 3):
        tab = W.QTab(base.levels, base.log2_cells, base.q * scale)
        g = W.Graph(1, 1, 2000, 1, [1], W.mix_thresholds([1.0]), [0], [tab], gap, np.zeros((0, 2)))
        pl = W.make_plans([[(1, 1)]])
        period = 9000 * scale
        rate = 10**9 // period
        assert (10**9 + rate // 2) // rate == period
        slo = W.Slo([30_000 * scale], [9], [10])
        r = orc.eval_plans(g, pl, [[rate]], slo, seed=5)
        if scale == 1:
            ref = r["counts"].copy()
        else:
            # the lerp floor is applied after scaling, so allow a handful of boundary flips
            assert abs(int(r["counts"][0, 0, 0, 0, 1]) - int(ref[0, 0, 0, 0, 1])) <= 2


def test_checksum_and_makespan_match_trace(orc):
    w = small_cfg1(n_req=500)
    r = orc.eval_plans(w.graph, w.plans, w.rate_mrps, w.slo, w.seed)
    for p in (0, 5, w.plans.n_plans - 1):
        for k in range(2):
            tr = orc.trace_sim(w.graph, w.plans, p, int(w.rate_mrps[p, 2]), k, seed=w.seed)
            assert int(r["dep_sum"][p, 2, k]) == int(tr["departure"].astype(np.uint64).sum())
            assert int(r["makespan"][p, 2, k]) == int(tr["departure"].max())


# ------------------------------------------------------------------------------------------
# bisection
# ------------------------------------------------------------------------------------------
def test_bisect_equals_linear_scan_on_small_grid(orc):
    w = W.config0_mm1(20_000, n_req=4000, n_trials=3)
    g, pl, slo = w.graph, w.plans, w.slo
    hi = 64
    # pooled predicate evaluated by brute force on every integer rate below hi (in mrps*1000 units
    # the grid would be huge; use a coarse model: scale by making hi small and services large)
    tab = W.exponential_qtab(20_000_000.0)  # 20 s service -> rates of a few dozen mrps matter
    g.tabs = [tab]
    slo = W.Slo([100_000_000], [9], [10])
    feas = []
    for rate in range(1, hi):
        r = orc.eval_plans(g, pl, [[rate]], slo, seed=0)
        c = r["counts"][0, 0].astype(np.int64).sum(0)  # pooled over trials: [T][2]
        feas.append(bool(c[0, 1] * 10 >= 9 * c[0, 0]))
    # CRN makes feasibility monotone (R4)
    assert feas == sorted(feas, reverse=True)
    best = max([0] + [rate for rate, f in zip(range(1, hi), feas) if f])
    for steps in (1, 3, 6, 10):
        b = orc.goodput_bisect(g, pl, [hi], steps, slo, seed=0)
        lo, h = 0, hi
        for _ in range(steps):
            mid = lo + (h - lo) // 2
            if mid == lo:
                continue
            if feas[mid - 1]:
                lo = mid
            else:
                h = mid
        assert int(b["rate_mrps"][0]) == lo
        if steps >= 6:
            assert lo == best
    # goodput = floor(rate* x pooled hits / (N K)) and counts are those at rate*
    r = orc.eval_plans(g, pl, [[best]], slo, seed=0)
    assert (b["counts"][0] == r["counts"][0, 0]).all()
    hits = int(r["counts"][0, 0, :, 0, 1].astype(np.int64).sum())
    assert int(b["goodput_mrps"][0, 0]) == best * hits // (g.n_req * g.n_trials)


def test_bisect_zero_and_closed_bracket(orc):
    w = W.config0_mm1(20_000, n_req=500, n_trials=2)
    b = orc.goodput_bisect(w.graph, w.plans, [1], 8, w.slo, seed=0)  # hi=1 -> mid == lo always
    assert int(b["rate_mrps"][0]) == 0 and (b["goodput_mrps"] == 0).all() and (b["counts"] == 0).all()
    b = orc.goodput_bisect(w.graph, w.plans, [0], 8, w.slo, seed=0)
    assert int(b["rate_mrps"][0]) == 0


def r18_case():
    """Constant gaps of 2^31-1 Q16 units, N = 2^12: CU_N = 2^43 - 2^12, so the R17 horizon
    CU_N * period + 2^15 < 2^62 holds iff period <= 524288, i.e. iff rate >= 1908 mrps
    (round(1e9/1908) = 524109, round(1e9/1907) = 524384). Service 5 us <= L = 10 us and hours
    between arrivals: every in-range probe is feasible with every request a hit."""
    g = W.Graph(1, 1, 1 << 12, 2, [1], W.mix_thresholds([1.0]), [0], [W.constant_qtab(5)],
                W.constant_qtab(2**31 - 1), np.zeros((0, 2)))
    return g, W.make_plans([[(1, 1)]] * 4), W.Slo([10], [9], [10])


# bracket hi -> rate* worked by hand from the rule "an out-of-range probe is infeasible" (R18):
#  3000: mids 1500, 750, ... all out of range                      -> 0
#  3814: mid 1907 out of range -> hi = 1907, then as above          -> 0
#  3816: mid 1908 in range, feasible -> lo = 1908; 2862, 3339, ... -> 3815
#  4000: mid 2000 feasible; 3000, 3500, ...                         -> 3999
R18_HI = np.array([3000, 3814, 3816, 4000], dtype=np.uint32)
R18_RATE = np.array([0, 0, 3815, 3999], dtype=np.uint32)


def test_bisect_out_of_range_probe_is_infeasible_r18(orc):
    g, pl, slo = r18_case()
    assert (10**9 + 1908 // 2) // 1908 == 524109 and (10**9 + 1907 // 2) // 1907 == 524384
    cu_n = (1 << 12) * (2**31 - 1)
    assert cu_n * 524288 + 32768 < 1 << 62 <= cu_n * 524289 + 32768
    b = orc.goodput_bisect(g, pl, R18_HI, 20, slo, seed=0)
    assert b["rc"] == orc.ORC_ERR_RANGE                       # the sticky status is still raised
    np.testing.assert_array_equal(b["rate_mrps"], R18_RATE)
    np.testing.assert_array_equal(b["goodput_mrps"][:, 0], R18_RATE)  # every request a hit: rate* x 1
    assert (b["counts"][:2] == 0).all() and (b["counts"][2:] == 1 << 12).all()
    # a bracket that never probes out of range raises nothing
    b = orc.goodput_bisect(g, pl.subset([3]), R18_HI[3:], 20, slo, seed=0)
    assert b["rc"] == 0 and int(b["rate_mrps"][0]) == 3999


@pytest.mark.parametrize("s_ms,lam", [(5.0, 176.97), (20.0, 26.97)])
def test_bisect_mm1_closed_form(orc, s_ms, lam):
    # lambda* = 1/s - ln(10)/L; statistical, a few percent
    assert abs(1000.0 / s_ms - math.log(10) / 0.1 - lam) < 6e-3
    w = W.config0_mm1(int(s_ms * 1000), n_req=1 << 18, n_trials=4)
    b = orc.goodput_bisect(w.graph, w.plans, w.rate_hi_mrps, 24, w.slo, seed=0)
    got = int(b["rate_mrps"][0]) / 1000.0
    assert abs(got / lam - 1.0) < 0.04, got


# ------------------------------------------------------------------------------------------
# validation / error behaviour
# ------------------------------------------------------------------------------------------
def test_validation_errors(orc):
    w = small_cfg1(n_req=100)
    g, pl = w.graph, w.plans
    assert orc.validate(g, pl) == orc.ORC_OK
    bad = W.Plans(pl.n_stages.copy(), pl.stage_mask.copy(), pl.stage_c.copy())
    bad.stage_c[3, 0] = 0
    assert orc.validate(g, bad) == orc.ORC_ERR_PLAN
    bad = W.make_plans([[(0b01, 1), (0b11, 1)]])          # overlap
    assert orc.validate(g, bad) == orc.ORC_ERR_PLAN
    bad = W.make_plans([[(0b01, 1)]])                     # LLM (used) has no stage
    assert orc.validate(g, bad) == orc.ORC_ERR_PLAN
    bad = W.make_plans([[(0b10, 1), (0b01, 1)]])          # order violates E -> LLM
    assert orc.validate(g, bad) == orc.ORC_ERR_PLAN
    tq = g.tabs[0].q.copy()
    tq[10] = tq[9] - 1
    g2 = W.Graph(g.n_comp, g.n_types, g.n_req, g.n_trials, g.type_mask, g.type_thresh, g.svc_tab,
                 [W.QTab(16, 6, tq), g.tabs[1]], g.arr_tab, g.edges)
    assert orc.validate(g2, pl) == orc.ORC_ERR_TABLE
    g3 = W.Graph(g.n_comp, g.n_types, 0, g.n_trials, g.type_mask, g.type_thresh, g.svc_tab, g.tabs,
                 g.arr_tab, g.edges)
    assert orc.validate(g3, pl) == orc.ORC_ERR_ARG
    big = W.constant_qtab(2**31 - 1)
    g4 = W.Graph(g.n_comp, g.n_types, g.n_req, g.n_trials, g.type_mask, g.type_thresh, g.svc_tab,
                 [big, big], g.arr_tab, g.edges)
    assert orc.validate(g4, pl) == orc.ORC_ERR_RANGE      # summed service would overflow int32


def test_out_of_range_sims_are_zeroed(orc):
    w = small_cfg1(n_req=100)
    rates = w.rate_mrps.copy()
    rates[1, 2] = 0
    rates[2, 0] = 1_000_000_001
    r = orc.eval_plans(w.graph, w.plans, rates, w.slo, w.seed)
    assert r["rc"] == orc.ORC_ERR_RANGE
    assert (r["sim_status"][1, 2] == orc.ORC_ERR_RANGE).all() and (r["counts"][1, 2] == 0).all()
    assert (r["sim_status"][2, 0] == orc.ORC_ERR_RANGE).all() and (r["dep_sum"][2, 0] == 0).all()
    assert (r["sim_status"][0] == 0).all() and r["counts"][0].sum() > 0
    # arrival horizon: huge gaps x huge period exceeds 2^62 us (R17)
    g = W.Graph(1, 1, 1 << 12, 1, [1], W.mix_thresholds([1.0]), [0], [W.constant_qtab(5)],
                W.constant_qtab(2**31 - 1), np.zeros((0, 2)))
    pl = W.make_plans([[(1, 1)]])
    slo = W.Slo([10], [9], [10])
    r = orc.eval_plans(g, pl, [[1, 1000]], slo, seed=0)
    # rate 1 mrps: period 1e9; CU_N = 2^12*(2^31-1) ~ 2^43; product ~ 2^73 -> out of range
    assert r["sim_status"][0, 0, 0] == orc.ORC_ERR_RANGE and (r["counts"][0, 0] == 0).all()
    # rate 1000 mrps: period 1e6 ~ 2^20: product ~ 2^63 > 2^62 -> also out of range
    assert r["sim_status"][0, 1, 0] == orc.ORC_ERR_RANGE
    r = orc.eval_plans(g, pl, [[1_000_000_000]], slo, seed=0)  # period 1: fine
    assert r["rc"] == 0 and r["counts"][0, 0, 0, 0, 0] == 1 << 12
