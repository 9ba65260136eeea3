"""Pins for the oracle's recursions: brute force on tiny inputs, exact D/D/c cases, and queueing
closed forms (M/M/1, Pollaczek-Khinchine, Erlang-C). All CPU, no GPU."""
import math
import os

import numpy as np
import pytest

import refsim
from paper_2512_14098_b200 import workloads as W

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def golden(kind):
    rows = []
    for line in open(os.path.join(GOLDEN, "queueing_closed_forms.txt")):
        p = line.split()
        if p and p[0] == kind:
            rows.append([float(x) for x in p[1:]])
    return rows


# ------------------------------------------------------------------------------------------
# helpers
# ------------------------------------------------------------------------------------------
def single_stage(service_tab, arr_tab, c, n_req, n_trials=1):
    g = W.Graph(1, 1, n_req, n_trials, [1], W.mix_thresholds([1.0]), [0], [service_tab], arr_tab,
                np.zeros((0, 2)))
    return g, W.make_plans([[(1, c)]])


def small_omni(n_req, n_trials=1, edge_delay=0, arr=None):
    w = W.config2_omni(n_req=n_req, n_trials=n_trials, n_rates=1, vectors_per_pattern=1,
                       n_patterns=1)
    g = w.graph
    g.edge_delay_us = edge_delay
    if arr is not None:
        g.arr_tab = arr
    return g


NO_SLO = W.Slo([0] * 8, [1] * 8, [1] * 8)


# ------------------------------------------------------------------------------------------
# brute force on 8-request inputs
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("rate", [20_000, 150_000, 400_000])
def test_lindley_vs_n2_closed_form(orc, rate):
    g, pl = single_stage(W.exponential_qtab(5000.0), W.exponential_qtab(65536.0), 1, 8, 3)
    for k in range(3):
        tr = orc.trace_sim(g, pl, 0, rate, k, seed=11)
        A, types, svc = refsim.gen_requests(g, 11, 0, k, rate)
        S = [s[0] for s in svc]
        assert tr["arrival"].tolist() == A
        assert tr["departure"].tolist() == refsim.lindley_bruteforce(A, S)


@pytest.mark.parametrize("c", [1, 2, 3, 5, 8, 9])
@pytest.mark.parametrize("rate", [100_000, 900_000])
def test_kiefer_wolfowitz_vs_event_sim_single_stage(orc, c, rate):
    g, pl = single_stage(W.lognormal_qtab(20_000.0, 0.8), W.gamma_qtab(1 / 9.0, 65536.0), c, 8, 4)
    for k in range(4):
        tr = orc.trace_sim(g, pl, 0, rate, k, seed=5, variant=2)
        A, types, svc = refsim.gen_requests(g, 5, 2, k, rate)
        routes = refsim.stage_services(g, pl, 0, types, svc)
        assert tr["departure"].tolist() == refsim.event_sim(A, routes, [c])


def test_tandem_vs_last_passage(orc):
    # 3-stage c=1 tandem, every request visits every stage: single type using comps 0,1,2
    tabs = [W.exponential_qtab(4000.0), W.lognormal_qtab(6000.0, 0.7), W.exponential_qtab(5000.0)]
    g = W.Graph(3, 1, 8, 3, [0b111], W.mix_thresholds([1.0]), [0, 1, 2], tabs,
                W.exponential_qtab(65536.0), [[0, 1], [1, 2]])
    pl = W.make_plans([[(1, 1), (2, 1), (4, 1)]])
    for k in range(3):
        for rate in (50_000, 250_000):
            tr = orc.trace_sim(g, pl, 0, rate, k, seed=3)
            A, types, svc = refsim.gen_requests(g, 3, 0, k, rate)
            S = [[svc[n][s] for n in range(8)] for s in range(3)]
            want = refsim.tandem_last_passage(A, S)
            assert tr["departure"].tolist() == want
            routes = refsim.stage_services(g, pl, 0, types, svc)
            assert refsim.event_sim(A, routes, [1, 1, 1]) == want  # FCFS == index order here


def _omni_plans(rng, c_of_stage):
    pats = W.merge_patterns(6, W.OMNI_EDGES)
    plan_list = []
    for pat in (0b00000, 0b00111, 0b10000, 0b11111, 0b01010):
        for _ in range(3):
            plan_list.append([(m, c_of_stage(m, rng)) for m in pats[pat]])
    return W.make_plans(plan_list, max_stages=6)


@pytest.mark.parametrize("edge_delay", [0, 10_000])
def test_multistage_skipping_types_c1_vs_ticket_event_sim(orc, edge_delay):
    # Omni graph, 4 types that skip stages, merged and disaggregated topologies, every c = 1:
    # index-order service (R2) == a causal event simulation with per-stage ticket queues.
    g = small_omni(n_req=12, n_trials=3, edge_delay=edge_delay)
    pl = _omni_plans(np.random.default_rng(9), lambda m, rng: 1)
    assert orc.validate(g, pl) == 0
    for p in range(0, pl.n_plans, 3):
        for k in range(3):
            for rate in (300, 3000):  # light and heavily overloaded (talker ~3 s)
                tr = orc.trace_sim(g, pl, p, rate, k, seed=21)
                A, types, svc = refsim.gen_requests(g, 21, 0, k, rate)
                assert tr["type"].tolist() == types
                routes = refsim.stage_services(g, pl, p, types, svc)
                c = [int(x) for x in pl.stage_c[p, :pl.n_stages[p]]]
                assert tr["departure"].tolist() == refsim.event_sim(A, routes, c, edge_delay), (p, k, rate)


@pytest.mark.parametrize("edge_delay", [0, 10_000])
def test_multistage_monotone_c_gt1_vs_event_sim(orc, edge_delay):
    # Fully disaggregated Omni plan with c > 1 exactly at the stages whose visitors all arrive in
    # index order (E_vid, E_aud: straight from system arrival; L_ta: all visitors come from the
    # c = 1 thinker): there the recursion coincides with causal FCFS, so the event simulator pins it.
    g = small_omni(n_req=14, n_trials=3, edge_delay=edge_delay)
    stages = W.merge_patterns(6, W.OMNI_EDGES)[0]
    names = {1 << i: nm for i, nm in enumerate(W.OMNI_COMPS)}
    for cvec in ({"E_vid": 2, "E_aud": 3, "L_ta": 2}, {"E_vid": 3, "L_ta": 4}, {"L_ta": 3}):
        pl = W.make_plans([[(m, cvec.get(names[m], 1)) for m in stages]], max_stages=6)
        for k in range(3):
            for rate in (300, 2000):
                tr = orc.trace_sim(g, pl, 0, rate, k, seed=33)
                A, types, svc = refsim.gen_requests(g, 33, 0, k, rate)
                routes = refsim.stage_services(g, pl, 0, types, svc)
                c = [int(x) for x in pl.stage_c[0, :pl.n_stages[0]]]
                assert tr["departure"].tolist() == refsim.event_sim(A, routes, c, edge_delay)


def test_single_type_tandem_c_gt1_vs_event_sim(orc):
    # one type visiting three stages; c > 1 first (monotone system arrivals) or last (fed by c = 1)
    tabs = [W.exponential_qtab(9000.0), W.lognormal_qtab(6000.0, 0.7), W.exponential_qtab(8000.0)]
    g = W.Graph(3, 1, 10, 3, [0b111], W.mix_thresholds([1.0]), [0, 1, 2], tabs,
                W.exponential_qtab(65536.0), [[0, 1], [1, 2]], edge_delay_us=500)
    for cs in ([3, 1, 1], [1, 1, 2], [2, 1, 1]):
        pl = W.make_plans([[(1, cs[0]), (2, cs[1]), (4, cs[2])]])
        for k in range(3):
            tr = orc.trace_sim(g, pl, 0, 400_000, k, seed=4)
            A, types, svc = refsim.gen_requests(g, 4, 0, k, 400_000)
            routes = refsim.stage_services(g, pl, 0, types, svc)
            assert tr["departure"].tolist() == refsim.event_sim(A, routes, cs, 500)


@pytest.mark.parametrize("edge_delay", [0, 10_000])
def test_multistage_general_vs_per_server_restatement(orc, edge_delay):
    # c > 1 anywhere with skipping types: stage arrivals are not index-monotone, the recursion is a
    # model choice (R2), pinned by an explicit per-server (unsorted, argmin) restatement.
    g = small_omni(n_req=40, n_trials=2, edge_delay=edge_delay)
    pl = _omni_plans(np.random.default_rng(9), lambda m, rng: int(rng.integers(1, 5)))
    differs_from_ticket_order = 0
    for p in range(pl.n_plans):
        for k in range(2):
            for rate in (300, 3000):
                tr = orc.trace_sim(g, pl, p, rate, k, seed=21)
                A, types, svc = refsim.gen_requests(g, 21, 0, k, rate)
                routes = refsim.stage_services(g, pl, p, types, svc)
                c = [int(x) for x in pl.stage_c[p, :pl.n_stages[p]]]
                assert tr["departure"].tolist() == refsim.per_server_sim(A, routes, c, edge_delay)
                differs_from_ticket_order += tr["departure"].tolist() != refsim.event_sim(A, routes, c, edge_delay)
    assert differs_from_ticket_order > 0  # documents that R2 is a genuine modelling choice for c > 1


# ------------------------------------------------------------------------------------------
# exact integer special cases
# ------------------------------------------------------------------------------------------
def test_dd1_exact(orc):
    gap = W.constant_qtab(65536)  # exactly one period between arrivals
    g, pl = single_stage(W.constant_qtab(7000), gap, 1, 50)
    # rho < 1: period 10000 > S: D_n = A_n + S
    tr = orc.trace_sim(g, pl, 0, 100_000, 0, seed=0)
    assert tr["arrival"].tolist() == [10_000 * (n + 1) for n in range(50)]
    assert (tr["departure"] - tr["arrival"]).tolist() == [7000] * 50
    # rho > 1: period 5000 < S: D_n = A_0 + (n+1) S
    tr = orc.trace_sim(g, pl, 0, 200_000, 0, seed=0)
    assert tr["departure"].tolist() == [5000 + 7000 * (n + 1) for n in range(50)]
    # all-zero gaps: D_n = prefix sum of S
    g0, pl0 = single_stage(W.constant_qtab(7000), W.constant_qtab(0), 1, 50)
    tr = orc.trace_sim(g0, pl0, 0, 100_000, 0, seed=0)
    assert tr["departure"].tolist() == [7000 * (n + 1) for n in range(50)]


@pytest.mark.parametrize("c", [2, 3, 7])
def test_ddc_exact(orc, c):
    gap = W.constant_qtab(65536)
    S, period = 7000, 1000
    g, pl = single_stage(W.constant_qtab(S), gap, c, 60)
    tr = orc.trace_sim(g, pl, 0, 1_000_000, 0, seed=0)  # period 1000 us
    A = [period * (n + 1) for n in range(60)]
    if c * period >= S:  # no waiting
        want = [a + S for a in A]
    else:  # round-robin over c servers, each busy back to back
        want = []
        for n in range(60):
            start = A[n] if n < c else max(A[n], want[n - c])
            want.append(start + S)
    assert tr["departure"].tolist() == want


def test_c_equals_one_is_lindley_and_c_ge_n_is_no_wait(orc):
    svc, arr = W.lognormal_qtab(30_000.0, 0.6), W.exponential_qtab(65536.0)
    g, pl = single_stage(svc, arr, 1, 300)
    tr1 = orc.trace_sim(g, pl, 0, 40_000, 0, seed=8)
    A, _, s = refsim.gen_requests(g, 8, 0, 0, 40_000)
    S = [x[0] for x in s]
    d, want = 0, []
    for a, sv in zip(A, S):
        d = max(a, d) + sv
        want.append(d)
    assert tr1["departure"].tolist() == want
    g, pl = single_stage(svc, arr, 300, 300)
    tr = orc.trace_sim(g, pl, 0, 40_000, 0, seed=8)
    assert (tr["departure"] - tr["arrival"]).tolist() == S


# ------------------------------------------------------------------------------------------
# closed forms (statistical, N = 2^20 x 4 trials; bounds >= 4 sigma per SURVEY.md 8(c))
# ------------------------------------------------------------------------------------------
BIG_N, BIG_K = 1 << 20, 4


def mean_sojourn_and_attainment(orc, g, pl, rate, L_us):
    slo = W.Slo([L_us], [9], [10])
    soj = []
    for k in range(g.n_trials):
        tr = orc.trace_sim(g, pl, 0, rate, k, seed=1234)
        soj.append((tr["departure"] - tr["arrival"]).astype(np.float64))
    soj = np.concatenate(soj)
    r = orc.eval_plans(g, pl, [[rate]], slo, seed=1234)
    att = r["counts"][0, 0, :, 0, 1].sum() / r["counts"][0, 0, :, 0, 0].sum()
    assert abs(att - (soj <= L_us).mean()) < 1e-12  # counters agree with the trace
    return soj.mean(), att


def effective(g, rate):
    """(lambda per us, E[S], E[S^2]) actually realised by the integer model."""
    period = (10**9 + rate // 2) // rate
    gap_mean = W.qtab_moments(g.arr_tab)[0] / 65536.0 * period
    m1, m2 = W.qtab_moments(g.tabs[0])
    return 1.0 / gap_mean, m1, m2


def test_mm1_closed_form_golden_is_consistent():
    for s_ms, rho, mean_ms, att in golden("mm1"):
        assert abs(s_ms / (1 - rho) - mean_ms) < 1e-9
        assert abs(1 - math.exp(-(1 - rho) * 100.0 / s_ms) - att) < 1e-4
    for c, a, val in golden("erlang_c"):
        assert abs(refsim.erlang_c(int(c), a) - val) < 2e-6
    for s_ms, lam in golden("mm1_bisect"):
        assert abs(1000.0 / s_ms - math.log(10) / 0.1 - lam) < 6e-3


@pytest.mark.parametrize("s_ms,rho,mean_ms,att", golden("mm1"))
def test_mm1_mean_sojourn_and_attainment(orc, s_ms, rho, mean_ms, att):
    g, pl = single_stage(W.exponential_qtab(s_ms * 1000.0), W.exponential_qtab(65536.0), 1, BIG_N,
                         BIG_K)
    rate = int(round(rho / (s_ms * 1000.0) * 1e9))
    mean, a = mean_sojourn_and_attainment(orc, g, pl, rate, 100_000)
    tol = 0.03 if rho >= 0.8 else 0.01
    assert abs(mean / 1000.0 / mean_ms - 1.0) < tol
    assert abs(a - att) < (0.01 if rho >= 0.8 else 0.003)


@pytest.mark.parametrize("rho,wq_over_s", [(0.5, 0.5), (0.8, 2.0), (0.9, 4.5)])
def test_md1_pollaczek_khinchine(orc, rho, wq_over_s):
    s = 10_000
    g, pl = single_stage(W.constant_qtab(s), W.exponential_qtab(65536.0), 1, BIG_N, BIG_K)
    rate = int(round(rho / s * 1e9))
    mean, _ = mean_sojourn_and_attainment(orc, g, pl, rate, 100_000)
    wq = mean - s
    assert abs(rho * s / (2 * (1 - rho)) / s - wq_over_s) < 1e-12  # the textbook values
    assert abs(wq / s / wq_over_s - 1.0) < (0.05 if rho >= 0.9 else 0.025)


def test_mg1_pollaczek_khinchine_lognormal(orc):
    tab = W.lognormal_qtab(8_000.0, 0.6)
    g, pl = single_stage(tab, W.exponential_qtab(65536.0), 1, BIG_N, BIG_K)
    m1, m2 = W.qtab_moments(tab)
    rate = int(round(0.7 / m1 * 1e9))
    lam, m1, m2 = effective(g, rate)
    mean, _ = mean_sojourn_and_attainment(orc, g, pl, rate, 100_000)
    want = m1 + lam * m2 / (2 * (1 - lam * m1))
    assert abs(mean / want - 1.0) < 0.02


@pytest.mark.parametrize("c,rho", [(2, 0.8), (4, 0.8), (8, 0.8), (16, 0.8), (32, 0.8), (2, 0.5),
                                   (4, 0.5), (8, 0.5)])
def test_mmc_erlang_c_mean_wait(orc, c, rho):
    s = 20_000.0
    g, pl = single_stage(W.exponential_qtab(s), W.exponential_qtab(65536.0), c, BIG_N // 2, BIG_K)
    rate = int(round(rho * c / s * 1e9))
    lam, m1, _ = effective(g, rate)
    a = lam * m1
    mean, _ = mean_sojourn_and_attainment(orc, g, pl, rate, 100_000)
    wq = mean - m1
    want = refsim.erlang_c(c, a) * m1 / (c - a)
    # relative s.d. of the mean wait grows as the wait shrinks; 4-sigma-ish bounds
    tol = {0.8: 0.05, 0.5: 0.06}[rho] * (2.0 if c >= 16 else 1.0)
    assert abs(wq / want - 1.0) < tol, (wq, want)


def test_index_order_versus_arrival_order_fcfs_gap(orc):
    """DESIGN.md R2: index-order service equals textbook FCFS whenever stage arrivals are monotone in
    the request index, and departs from it when types skip stages. The gap is MEASURED here on a
    configs[1]-like disaggregated plan (text skips the encoder) against an arrival-order event
    simulator, and bounded: per-type attainment within 0.02, mean sojourn within 5 % at 70-95 % load."""
    g = W.Graph(2, 2, 3000, 1, [0b10, 0b11], W.mix_thresholds([0.7, 0.3]), [0, 0, 1, 1],
                [W.lognormal_qtab(30_000.0, 0.4), W.lognormal_qtab(400_000.0, 0.6)], W.exponential_qtab(65536.0), [[0, 1]])
    worst_att, worst_soj = 0.0, 0.0
    for (e, l) in ((1, 4), (2, 8)):
        pl = W.make_plans([[(0b01, e), (0b10, l)]])
        R = float(W.flow_bound_mrps(g, pl)[0])
        for alpha in (0.7, 0.85, 0.95):
            rate = int(alpha * R)
            A, types, svc = refsim.gen_requests(g, 21, 0, 0, rate)
            routes = refsim.stage_services(g, pl, 0, types, svc)
            d_idx = np.array(orc.trace_sim(g, pl, 0, rate, 0, seed=21)["departure"])
            assert d_idx.tolist() == refsim.per_server_sim(A, routes, [e, l])  # the oracle's own discipline, restated
            d_fcfs = np.array(refsim.fcfs_event_sim(A, routes, [e, l]))
            soj_i, soj_f = d_idx - np.array(A), d_fcfs - np.array(A)
            assert soj_f.sum() <= soj_i.sum()                                   # waiting for an absent request only adds delay
            worst_soj = max(worst_soj, soj_i.mean() / soj_f.mean() - 1.0)
            for t, L in ((0, 2_000_000), (1, 3_000_000)):
                sel = np.array(types) == t
                worst_att = max(worst_att, abs((soj_i[sel] <= L).mean() - (soj_f[sel] <= L).mean()))
    print(f"index-order vs arrival-order FCFS: worst attainment gap {worst_att:.4f}, worst mean-sojourn excess {worst_soj:.4f}")
    assert worst_att <= 0.02 and worst_soj <= 0.05
    # single-path tandem with one replica per stage: stage arrivals are monotone, the two disciplines coincide
    g1 = W.Graph(2, 1, 400, 1, [0b11], W.mix_thresholds([1.0]), [0, 1], [W.lognormal_qtab(30_000.0, 0.4), W.lognormal_qtab(50_000.0, 0.6)],
                 W.exponential_qtab(65536.0), [[0, 1]])
    pl1 = W.make_plans([[(0b01, 1), (0b10, 1)]])
    A, types, svc = refsim.gen_requests(g1, 3, 0, 0, 15_000)
    routes = refsim.stage_services(g1, pl1, 0, types, svc)
    assert refsim.fcfs_event_sim(A, routes, [1, 1]) == orc.trace_sim(g1, pl1, 0, 15_000, 0, seed=3)["departure"].tolist()
