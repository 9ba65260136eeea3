"""Pins of the CPU-GPU overlap rule of the simulator (R24): a request
that finds the executor idle pays CPU + GPU time, one that had to queue pays GPU time alone.
Closed forms on deterministic inputs, an independent event simulator with explicit per-server
busy state on 8-request inputs, and the no-queueing identity."""
import heapq

import numpy as np
import pytest

import refsim
from paper_2512_14098_b200 import workloads as W

NONE = 0xFFFF


def dd1(gap_q16, cpu_us, gpu_us, n_req, c=1):
    """One component, one type, constant gaps / CPU / GPU times."""
    tabs = [W.constant_qtab(gpu_us), W.constant_qtab(cpu_us)]
    g = W.Graph(1, 1, n_req, 1, [1], W.mix_thresholds([1.0]), [0], tabs, W.constant_qtab(gap_q16), np.zeros((0, 2)),
                cpu_tab=[1])
    return g, W.make_plans([[(1, c)]])


def test_dd1_closed_forms(orc):
    # rate 1000 mrps -> period 1e6 us; gap table 65536 Q16 = one period: arrivals A_n = (n+1) s
    G, Cc = 400_000, 300_000
    # (i) gap 1 s >= CPU + GPU: every request finds the executor idle
    g, pl = dd1(65536, Cc, G, 50)
    t = orc.trace_sim(g, pl, 0, 1000, 0, seed=0)
    np.testing.assert_array_equal(t["departure"], t["arrival"] + Cc + G)
    # (ii) GPU < gap < CPU + GPU: period 0.5 s. A busy stretch of m requests lasts while n (gap - GPU) < CPU,
    # i.e. m = ceil(CPU / (gap - GPU)) = 3: D = A_first + CPU + (j+1) GPU for its j-th request, then it restarts
    g, pl = dd1(32768, Cc, G, 60)
    t = orc.trace_sim(g, pl, 0, 1000, 0, seed=0)
    A, D = t["arrival"], t["departure"]
    gap = 500_000
    assert (np.diff(A) == gap).all()
    m = -(-Cc // (gap - G))
    assert m == 3
    for n in range(60):
        first = n - n % m
        assert D[n] == A[first] + Cc + (n % m + 1) * G
    # (iii) gap < GPU (overload): only the first request ever sees an idle executor
    g, pl = dd1(16384, Cc, G, 40)
    t = orc.trace_sim(g, pl, 0, 1000, 0, seed=0)
    np.testing.assert_array_equal(t["departure"], t["arrival"][0] + Cc + G * np.arange(1, 41))
    # (iv) no CPU table for the pair: the plain recursion
    g.cpu_tab = np.array([NONE], np.uint16)
    t0 = orc.trace_sim(g, pl, 0, 1000, 0, seed=0)
    np.testing.assert_array_equal(t0["departure"], t0["arrival"][0] + G * np.arange(1, 41))
    # (v) c = 3 replicas, gap 0.25 s, GPU 0.4 s, CPU 0.3 s: capacity 3/0.4 = 7.5 > 4 req/s offered;
    # replica r serves requests r, r+3, ...: it frees at A_n + 0.7 s, the next one arrives 0.75 s later -> always idle
    g, pl = dd1(16384, Cc, G, 30, c=3)
    t = orc.trace_sim(g, pl, 0, 1000, 0, seed=0)
    np.testing.assert_array_equal(t["departure"], t["arrival"] + Cc + G)


def overlap_graph(n_req=8, n_trials=1, delay=7_000):
    """E_img, E_aud -> LLM; both encoders have CPU pre-processing, the LLM has none; three types."""
    tabs = [W.lognormal_qtab(30_000.0, 0.4), W.lognormal_qtab(20_000.0, 0.4), W.lognormal_qtab(120_000.0, 0.5),
            W.exponential_qtab(25_000.0), W.lognormal_qtab(9_000.0, 0.3)]
    T = 3
    masks = [0b100, 0b101, 0b111]
    svc_tab = np.repeat(np.arange(3, dtype=np.uint16), T)
    cpu_tab = np.array([3, 3, 3, 4, 4, 4, NONE, NONE, NONE], np.uint16)
    return W.Graph(3, T, n_req, n_trials, masks, W.mix_thresholds([0.3, 0.4, 0.3]), svc_tab, tabs,
                   W.exponential_qtab(65536.0), [[0, 2], [1, 2]], edge_delay_us=delay, cpu_tab=cpu_tab)


def gen_cpu(graph, seed, variant, trial, types):
    """CPU draws restated from DESIGN.md R24: Philox block 3 + i/4, word i % 4 (pure Python)."""
    key = (seed & refsim.MASK, (seed >> 32) & refsim.MASK)
    out = []
    for n, t in enumerate(types):
        d = {}
        for i in range(graph.n_comp):
            tid = int(graph.cpu_tab[i * graph.n_types + t])
            if (int(graph.type_mask[t]) >> i) & 1 and tid != NONE:
                b = refsim.philox4x32_10((n, trial, 3 + i // 4, variant), key)
                tb = graph.tabs[tid]
                d[i] = refsim.qtab_sample(tb.levels, tb.log2_cells, tb.q, b[i % 4])
        out.append(d)
    return out


def event_sim_overlap(A, routes, stage_c, delay):
    """Discrete-event simulation with explicit servers. routes[n] = [(stage, gpu, cpu), ...]. Each
    stage hands its visitors to servers in index order (R2); the request takes the server that frees
    first; if that server is idle when the request reaches the stage the service is cpu + gpu,
    otherwise gpu (the CPU work was done while it queued)."""
    free = [[0] * c for c in stage_c]              # per-server time at which it becomes free
    next_ticket = [0] * len(stage_c)
    tickets = [[n for n in range(len(A)) if any(s == st for s, _, _ in routes[n])] for st in range(len(stage_c))]
    pos = [0] * len(A)
    dep = [None] * len(A)
    ev = []
    for n in range(len(A)):
        if routes[n]:
            heapq.heappush(ev, (A[n], n))
        else:
            dep[n] = A[n]
    waiting = [dict() for _ in stage_c]            # stage -> {request: time it reached the stage}
    while ev:
        tnow, n = heapq.heappop(ev)
        st, gpu, cpu = routes[n][pos[n]]
        waiting[st][n] = tnow
        while next_ticket[st] < len(tickets[st]) and tickets[st][next_ticket[st]] in waiting[st]:
            r = tickets[st][next_ticket[st]]
            at = waiting[st].pop(r)
            _, g_r, c_r = routes[r][pos[r]]
            k = min(range(stage_c[st]), key=lambda j: free[st][j])
            idle = free[st][k] <= at
            done = (at + c_r + g_r) if idle else (free[st][k] + g_r)
            free[st][k] = done
            next_ticket[st] += 1
            pos[r] += 1
            if pos[r] == len(routes[r]):
                dep[r] = done
            else:
                heapq.heappush(ev, (done + delay, r))
    return dep


@pytest.mark.parametrize("seed", range(6))
def test_eight_requests_against_event_simulator(orc, seed):
    g = overlap_graph()
    rng = np.random.default_rng(seed)
    plans = [[(0b001, int(rng.integers(1, 3))), (0b010, int(rng.integers(1, 3))), (0b100, int(rng.integers(1, 4)))],
             [(0b011, int(rng.integers(1, 3))), (0b100, int(rng.integers(1, 3)))],
             [(0b111, int(rng.integers(1, 4)))]]
    pl = W.make_plans(plans, max_stages=3)
    for p in range(3):
        for rate in (3_000, 20_000, 90_000):      # from mostly idle to overloaded
            A, types, svc = refsim.gen_requests(g, 40 + seed, 2, 0, rate)
            cpu = gen_cpu(g, 40 + seed, 2, 0, types)
            routes = []
            for n, t in enumerate(types):
                r = []
                for s in range(int(pl.n_stages[p])):
                    m = int(pl.stage_mask[p, s]) & int(g.type_mask[t])
                    if m:
                        comps = [i for i in range(3) if (m >> i) & 1]
                        r.append((s, sum(svc[n][i] for i in comps), sum(cpu[n].get(i, 0) for i in comps)))
                routes.append(r)
            want = event_sim_overlap(A, routes, [int(c) for c in pl.stage_c[p, :int(pl.n_stages[p])]], g.edge_delay_us)
            t = orc.trace_sim(g, pl, p, rate, 0, seed=40 + seed, variant=2)
            assert t["arrival"].tolist() == A
            assert t["departure"].tolist() == want, (p, rate)


def test_unlimited_replicas_pay_cpu_everywhere(orc):
    # nobody queues: every executor is idle at every arrival, so the sojourn is the Monte-Carlo latency
    # with CPU + GPU time on every component that has a CPU table
    g = overlap_graph(n_req=600, n_trials=2, delay=4_000)
    pl = W.make_plans([[(0b001, 600), (0b010, 600), (0b100, 600)], [(0b011, 600), (0b100, 600)], [(0b111, 600)]], max_stages=3)
    slo = W.Slo([150_000, 200_000, 230_000], [9] * 3, [10] * 3)
    sim = orc.eval_plans(g, pl, [[50_000]] * 3, slo, 5, 1, n_threads=4)
    mc = orc.mc_latency(g, pl, [50_000] * 3, slo, 5, 1)
    np.testing.assert_array_equal(sim["counts"][:, 0], mc["counts"])
    g0 = overlap_graph(n_req=600, n_trials=2, delay=4_000)
    g0.cpu_tab = None
    mc0 = orc.mc_latency(g0, pl, [50_000] * 3, slo, 5, 1)
    assert (mc0["counts"][..., 1] >= mc["counts"][..., 1]).all() and (mc0["counts"][..., 1] > mc["counts"][..., 1]).any()


def test_validation_and_stream(orc):
    g = overlap_graph()
    pl = W.make_plans([[(0b111, 1)]])
    assert orc.validate(g, pl) == 0
    g.cpu_tab[1] = 9                                  # (component 0, type 1): a used pair
    assert orc.validate(g, pl) == orc.ORC_ERR_ARG
    g = overlap_graph()
    g.tabs[3] = W.constant_qtab(2**31 - 1)            # CPU + GPU of a request would overflow int32 (R17)
    assert orc.validate(g, pl) == orc.ORC_ERR_RANGE
