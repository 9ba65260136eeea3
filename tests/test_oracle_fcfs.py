"""Pins of the oracle's arrival-order service mode (orc_graph.order_mode = 1; R27; SURVEY.md
8(f) NEXT-4 "true stage-arrival-order FCFS"): a hand-worked example (tests/golden/fcfs_overtake.txt),
an independent event-queue simulator on random inputs (tests/refsim.fcfs_event_sim: explicit event
heap and per-stage waiting queues, where the oracle sorts stage by stage), the cases in which the two
disciplines must coincide, textbook M/M/c behind a stage that reorders, invariants, validation."""
import os

import numpy as np
import pytest

import refsim
from paper_2512_14098_b200 import workloads as W
from test_oracle_overlap import NONE, gen_cpu, overlap_graph
from test_oracle_routing import mllm, routes_by_hand, two_path_plans

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "fcfs_overtake.txt")


def omni_like(n_req, n_trials=1, delay=6_000, order_mode=1):
    """Four components E_img, E_aud -> LLM -> VOC; four types, two of which skip stages."""
    tabs = [W.lognormal_qtab(30_000.0, 0.5), W.lognormal_qtab(20_000.0, 0.4), W.lognormal_qtab(110_000.0, 0.6),
            W.exponential_qtab(60_000.0)]
    masks = [0b0100, 0b0101, 0b1110, 0b1111]
    svc_tab = np.repeat(np.arange(4, dtype=np.uint16), 4)
    return W.Graph(4, 4, n_req, n_trials, masks, W.mix_thresholds([0.4, 0.2, 0.2, 0.2]), svc_tab, tabs,
                   W.exponential_qtab(65536.0), [[0, 2], [1, 2], [2, 3]], edge_delay_us=delay, order_mode=order_mode)


def test_hand_worked_overtaking_example(orc):
    rows = [[int(v) for v in l.split()] for l in open(GOLDEN) if l.strip() and not l.startswith("#")]
    g = W.Graph(2, 2, 8, 1, [0b11, 0b10], W.mix_thresholds([0.5, 0.5]), [0, 0, 1, 1],
                [W.constant_qtab(900_000), W.constant_qtab(400_000)], W.constant_qtab(65536), [[0, 1]])
    pl = W.make_plans([[(0b01, 2), (0b10, 1)]])
    t0 = orc.trace_sim(g, pl, 0, 10_000, 0, seed=3)
    g.order_mode = 1
    t1 = orc.trace_sim(g, pl, 0, 10_000, 0, seed=3)
    assert t0["type"].tolist() == [r[1] for r in rows] == t1["type"].tolist()
    assert t0["arrival"].tolist() == [r[2] for r in rows] == t1["arrival"].tolist()
    assert t0["departure"].tolist() == [r[3] for r in rows]   # index order (R2)
    assert t1["departure"].tolist() == [r[4] for r in rows]   # arrival order (R27)


@pytest.mark.parametrize("seed", range(6))
def test_against_event_queue_simulator(orc, seed):
    rng = np.random.default_rng(100 + seed)
    g = omni_like(int(rng.integers(40, 400)), delay=int(rng.choice([0, 6_000])))
    for _ in range(3):
        pats = [[0b0001, 0b0010, 0b0100, 0b1000], [0b0011, 0b0100, 0b1000], [0b0001, 0b0010, 0b1100], [0b0111, 0b1000]]
        stages = pats[int(rng.integers(len(pats)))]
        cs = [int(c) for c in rng.integers(1, 6, len(stages))]
        pl = W.make_plans([list(zip(stages, cs))])
        rate = int(rng.uniform(0.5, 1.3) * float(W.flow_bound_mrps(g, pl)[0]))
        A, types, svc = refsim.gen_requests(g, 7 + seed, 1, 0, rate)
        routes = refsim.stage_services(g, pl, 0, types, svc)
        t = orc.trace_sim(g, pl, 0, rate, 0, seed=7 + seed, variant=1)
        assert t["arrival"].tolist() == A
        assert t["departure"].tolist() == refsim.fcfs_event_sim(A, routes, cs, g.edge_delay_us)


def test_with_cpu_overlap_and_with_routes_against_event_queue_simulator(orc):
    # R24: the idle/busy rule inside arrival-order service
    g = overlap_graph(n_req=300)
    g.order_mode = 1
    pl = W.make_plans([[(0b001, 2), (0b010, 1), (0b100, 3)]])
    for rate in (4_000, 9_000, 20_000):
        A, types, svc = refsim.gen_requests(g, 11, 0, 0, rate)
        cpu = gen_cpu(g, 11, 0, 0, types)
        routes = []
        for n, t in enumerate(types):
            tm, r = int(g.type_mask[t]), []
            for s in range(3):
                m = int(pl.stage_mask[0, s]) & tm
                if m:
                    r.append((s, sum(svc[n][i] for i in range(3) if (m >> i) & 1), sum(cpu[n].get(i, 0) for i in range(3) if (m >> i) & 1)))
            routes.append(r)
        t = orc.trace_sim(g, pl, 0, rate, 0, seed=11)
        assert t["departure"].tolist() == refsim.fcfs_event_sim(A, routes, [2, 1, 3], g.edge_delay_us)
    # R26: routes drawn per request, arrival order on whatever stages the route holds
    g = mllm(250)
    g.order_mode = 1
    pl = two_path_plans([(2, 3, 2)], 0.6, 0.4)
    for rate in (3_000, 11_000):
        A, types, svc = refsim.gen_requests(g, 13, 0, 0, rate)
        routes, _ = routes_by_hand(g, pl, 0, 13, 0, 0, types, svc)
        t = orc.trace_sim(g, pl, 0, rate, 0, seed=13)
        assert t["departure"].tolist() == refsim.fcfs_event_sim(A, routes, [2, 3, 2], g.edge_delay_us)


def test_coincides_with_index_order_where_stage_arrivals_are_monotone(orc):
    slo = W.Slo([300_000], [9], [10])
    # one stage, any replica count: requests reach it in index order
    g = W.Graph(1, 1, 3000, 2, [1], W.mix_thresholds([1.0]), [0], [W.lognormal_qtab(50_000.0, 0.8)],
                W.exponential_qtab(65536.0), np.zeros((0, 2)))
    pl = W.make_plans([[(1, c)] for c in (1, 2, 7)])
    rates = np.array([[12_000, 19_000], [30_000, 39_000], [100_000, 135_000]], np.uint32)
    a = orc.eval_plans(g, pl, rates, slo, 4)
    g.order_mode = 1
    b = orc.eval_plans(g, pl, rates, slo, 4)
    for key in ("counts", "dep_sum", "makespan"):
        np.testing.assert_array_equal(a[key], b[key])
    # a single-path tandem with one replica per stage: departures of a stage are in service order
    g = W.Graph(3, 1, 2000, 1, [0b111], W.mix_thresholds([1.0]), [0, 1, 2],
                [W.lognormal_qtab(30_000.0, 0.4), W.exponential_qtab(45_000.0), W.lognormal_qtab(20_000.0, 0.9)],
                W.exponential_qtab(65536.0), [[0, 1], [1, 2]], edge_delay_us=3_000)
    pl = W.make_plans([[(1, 1), (2, 1), (4, 1)], [(3, 1), (4, 1)]])
    for rate in (9_000, 21_000):
        for p in (0, 1):
            a = orc.trace_sim(g, pl, p, rate, 0, seed=9)
            g.order_mode = 1
            b = orc.trace_sim(g, pl, p, rate, 0, seed=9)
            g.order_mode = 0
            np.testing.assert_array_equal(a["departure"], b["departure"])


def test_second_stage_is_a_textbook_mmc_queue(orc):
    # An infinite-server first stage with exponential service turns Poisson arrivals into Poisson
    # arrivals in a DIFFERENT order (M/G/inf output theorem); in arrival order the second stage is then
    # an M/M/c queue, Erlang C: W_q = C(c, a) * s / (c - a). Index order would make it wait for stragglers.
    N, c, s2, rho = 1 << 17, 4, 40_000.0, 0.8
    g = W.Graph(2, 1, N, 1, [0b11], W.mix_thresholds([1.0]), [0, 1], [W.exponential_qtab(200_000.0), W.exponential_qtab(s2)],
                W.exponential_qtab(65536.0), [[0, 1]], order_mode=1)
    pl = W.make_plans([[(0b01, 256), (0b10, c)]])   # 16 busy on average: 256 replicas never queue
    rate = int(rho * c / s2 * 1e9)
    t = orc.trace_sim(g, pl, 0, rate, 0, seed=2)
    soj = (t["departure"] - t["arrival"]).astype(np.float64)
    a = rho * c
    wq = refsim.erlang_c(c, a) * s2 / (c - a)
    expect = 200_000.0 + s2 + wq
    assert abs(soj.mean() / expect - 1.0) < 0.02
    g.order_mode = 0
    t0 = orc.trace_sim(g, pl, 0, rate, 0, seed=2)
    assert (t0["departure"] - t0["arrival"]).mean() > 1.3 * expect   # index order: head-of-line blocking behind stragglers


def test_invariants_and_bisection(orc):
    g = omni_like(1200, n_trials=2)
    w_plans = W.make_plans([[(0b0011, 2), (0b0100, 3), (0b1000, 2)], [(0b0011, 2), (0b0100, 3), (0b1000, 2)],
                            [(0b0001, 1), (0b0010, 1), (0b1100, 4)]])
    R = W.flow_bound_mrps(g, w_plans)
    rates = W.rate_grid(R, [0.5, 0.8, 1.1])
    slo = W.Slo([500_000, 600_000, 900_000, 1_000_000], [9] * 4, [10] * 4)
    out = orc.eval_plans(g, w_plans, rates, slo, 17)
    cnt = out["counts"]
    assert (cnt[..., 0].sum(axis=-1) == g.n_req).all() and (cnt[..., 1] <= cnt[..., 0]).all()
    np.testing.assert_array_equal(out["dep_sum"][0], out["dep_sum"][1])      # duplicate plans (R4)
    np.testing.assert_array_equal(cnt[0], cnt[1])
    for p in range(3):                                                     # the trace agrees with the counters
        t = orc.trace_sim(g, w_plans, p, int(rates[p, 1]), 1, seed=17)
        soj = t["departure"] - t["arrival"]
        assert int(t["departure"].astype(np.uint64).sum()) == int(out["dep_sum"][p, 1, 1])
        assert int(t["departure"].max()) == int(out["makespan"][p, 1, 1])
        for ty in range(4):
            sel = t["type"] == ty
            assert sel.sum() == cnt[p, 1, 1, ty, 0] and (soj[sel] <= slo.L_us[ty]).sum() == cnt[p, 1, 1, ty, 1]
        # sojourn >= the request's own services and hops
        A, types, svc = refsim.gen_requests(g, 17, 0, 1, int(rates[p, 1]))
        routes = refsim.stage_services(g, w_plans, p, types, svc)
        floor = np.array([sum(s for _, s in r) + max(0, len(r) - 1) * g.edge_delay_us for r in routes])
        assert (soj >= floor).all()
    # bisection runs on the same simulation: the returned rate is feasible, the one above is not
    hi = np.ceil(1.5 * R).astype(np.uint32)
    b = orc.goodput_bisect(g, w_plans, hi, 24, slo, 17)
    for p in (0, 2):
        r = int(b["rate_mrps"][p])
        assert 0 < r < hi[p]
        for rr, want in ((r, True), (r + 1, False)):
            o = orc.eval_plans(g, w_plans.subset(np.array([p])), np.array([[rr]], np.uint32), slo, 17)
            c = o["counts"][0, 0].sum(axis=0)
            assert all(c[t, 1] * 10 >= 9 * c[t, 0] for t in range(4)) == want


def forkjoin_fcfs_event_sim(A, tasks, stage_c, delay):
    """Event-driven fork-join with ARRIVAL-order service: tasks[n] = {stage: (S, [pred stages])}; a task
    becomes ready when all its predecessors are done (+ delay each) and joins its stage's waiting queue;
    an idle server takes the waiting task that became ready first (ties: lower request index)."""
    import heapq
    V = len(stage_c)
    idle = list(stage_c)
    queue = [[] for _ in range(V)]
    done = [dict() for _ in range(len(A))]
    ev = []                                   # (time, kind, n, s): 0 = task ready, 1 = service completion
    for n in range(len(A)):
        for s, (_, pr) in tasks[n].items():
            if not pr:
                heapq.heappush(ev, (A[n], 0, n, s))

    def dispatch(s, now):
        while queue[s] and idle[s] > 0:
            _, n = heapq.heappop(queue[s])
            idle[s] -= 1
            heapq.heappush(ev, (now + tasks[n][s][0], 1, n, s))

    while ev:
        now, kind, n, s = heapq.heappop(ev)
        if kind == 0:
            heapq.heappush(queue[s], (now, n))
        else:
            idle[s] += 1
            done[n][s] = now
            for s2, (_, pr) in tasks[n].items():
                if s in pr and all(q in done[n] for q in pr):
                    heapq.heappush(ev, (max(done[n][q] + delay for q in pr), 0, n, s2))
        dispatch(s, now)
    return [max(done[n].values(), default=A[n]) for n in range(len(A))]


@pytest.mark.parametrize("seed", range(4))
def test_forkjoin_under_arrival_order(orc, seed):
    """R25 + R27: a stage starts a request when its predecessor stages are done, and serves in the order in
    which requests become ready -- against an event simulator with task dependencies and waiting queues."""
    from test_oracle_forkjoin import omni, stage_preds
    rng = np.random.default_rng(300 + seed)
    w = omni(n_req=int(rng.integers(30, 160)), delay=int(rng.choice([0, 9_000])))
    g = w.graph
    g.order_mode = 1
    for p in rng.choice(w.plans.n_plans, 3, replace=False):
        p = int(p)
        V = int(w.plans.n_stages[p])
        cs = [int(c) for c in rng.integers(1, 4, V)]
        pl = W.make_plans([[(int(w.plans.stage_mask[p, s]), cs[s]) for s in range(V)]])
        rate = int(rng.uniform(0.6, 1.4) * float(W.flow_bound_mrps(g, pl)[0]))
        A, types, svc = refsim.gen_requests(g, 40 + seed, 1, 0, rate)
        tasks = []
        for n, t in enumerate(types):
            masks, pred = stage_preds(g, pl, 0, t)
            tasks.append({s: (sum(svc[n][i] for i in range(6) if (masks[s] >> i) & 1), pr) for s, pr in pred.items()})
        got = orc.trace_sim(g, pl, 0, rate, 0, seed=40 + seed, variant=1)
        assert got["departure"].tolist() == forkjoin_fcfs_event_sim(A, tasks, cs, g.edge_delay_us)
    # unlimited replicas: nobody waits, the service order is immaterial -- the critical path of the index-order run
    big = W.Plans(w.plans.n_stages, w.plans.stage_mask, np.full_like(w.plans.stage_c, g.n_req))
    a = orc.trace_sim(g, big, 5, 3000, 0, seed=1)
    g.order_mode = 0
    b = orc.trace_sim(g, big, 5, 3000, 0, seed=1)
    np.testing.assert_array_equal(a["departure"], b["departure"])
    # on a chain graph fork-join is the path mode, in arrival order too
    w1 = W.config1_mllm(n_req=700, n_trials=1, n_rates=2, llm_max=4, e_steps=3)
    w1.graph.edge_delay_us = 5_000
    w1.graph.order_mode = 1
    a = orc.eval_plans(w1.graph, w1.plans, w1.rate_mrps, w1.slo, w1.seed, n_threads=4)
    w1.graph.join_mode = 1
    b = orc.eval_plans(w1.graph, w1.plans, w1.rate_mrps, w1.slo, w1.seed, n_threads=4)
    for key in ("counts", "dep_sum", "makespan"):
        np.testing.assert_array_equal(a[key], b[key])


def test_validation(orc):
    g = omni_like(16)
    pl = W.make_plans([[(0b0011, 1), (0b0100, 1), (0b1000, 1)]])
    assert orc.validate(g, pl) == 0
    g.order_mode = 2
    assert orc.validate(g, pl) == orc.ORC_ERR_ARG
    g.order_mode, g.join_mode = 1, 1     # arrival order composes with fork-join
    assert orc.validate(g, pl) == 0
