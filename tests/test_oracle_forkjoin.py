"""Pins of the fork-join routing mode (R25): a request reaches
a stage when all its predecessor stages (DAG edges restricted to the request's own components) have
finished. Critical-path closed form with unlimited replicas, an event-driven simulator with task
dependencies and per-stage ticket queues for one-replica stages, a per-server restatement for
several replicas, and the identity with the path mode on chain graphs."""
import heapq

import numpy as np
import pytest

import refsim
from paper_2512_14098_b200 import workloads as W


def omni(n_req=8, n_trials=1, delay=9_000, join=1):
    """configs[4]'s graph: 3 encoders -> thinker -> talker -> vocoder, 8 types."""
    w = W.config4_sweep(n_req=n_req, n_trials=n_trials, vectors_per_pattern=1, n_patterns=32, n_variants=1)
    w.graph.edge_delay_us = delay
    w.graph.join_mode = join
    return w


def stage_preds(g, pl, p, t):
    """pred[s] = visited stages s' != s with a DAG edge from a component of the request on s' into one on s."""
    tm = int(g.type_mask[t])
    V = int(pl.n_stages[p])
    masks = [int(pl.stage_mask[p, s]) & tm for s in range(V)]
    pred = {}
    for s in range(V):
        if not masks[s]:
            continue
        pred[s] = [sp for sp in range(V) if sp != s and masks[sp] and
                   any((masks[sp] >> int(u)) & 1 and (masks[s] >> int(v)) & 1 for u, v in g.edges)]
    return masks, pred


def test_unlimited_replicas_critical_path(orc):
    # nobody waits: the sojourn is the longest path through the request's own DAG of stages,
    # services on the nodes and one transfer delay per edge -- by explicit path enumeration
    w = omni(n_req=60, n_trials=2)
    g = w.graph
    big = W.Plans(w.plans.n_stages, w.plans.stage_mask, np.full_like(w.plans.stage_c, 60))
    for p in (0, 5, 17, 31):
        for k in (0, 1):
            A, types, svc = refsim.gen_requests(g, w.seed, 3, k, 2000)
            t = orc.trace_sim(g, big, p, 2000, k, w.seed, variant=3)
            for n in range(60):
                masks, pred = stage_preds(g, big, p, types[n])
                S = {s: sum(svc[n][i] for i in range(6) if (masks[s] >> i) & 1) for s in pred}

                def longest(s):  # longest path ending with stage s
                    return S[s] + max([longest(sp) + g.edge_delay_us for sp in pred[s]], default=0)

                want = A[n] + max([longest(s) for s in pred], default=0)
                assert int(t["departure"][n]) == want, (p, k, n)
    # and the path mode differs on requests with several encoders (they queue one after another there)
    g.join_mode = 0
    t0 = orc.trace_sim(g, big, 0, 2000, 0, w.seed, variant=3)
    g.join_mode = 1
    t1 = orc.trace_sim(g, big, 0, 2000, 0, w.seed, variant=3)
    assert (t1["departure"] <= t0["departure"]).all() and (t1["departure"] < t0["departure"]).any()


def forkjoin_event_sim(A, tasks, stage_c, delay):
    """Event-driven: tasks[n] = {stage: (S, [pred stages])}. A task becomes ready when all its
    predecessors are done (+ delay each); every stage hands its visitors to its servers in request
    index order (a ticket queue, R2), the next ticket starting as soon as it is ready and a server is
    idle -- which for ONE server per stage is exactly the index-order recursion."""
    V = len(stage_c)
    tickets = [[n for n in range(len(A)) if s in tasks[n]] for s in range(V)]
    nxt, idle = [0] * V, list(stage_c)
    ready = [dict() for _ in range(V)]
    done = [dict() for _ in range(len(A))]
    ev, seq = [], 0

    def release(n, s, now):
        nonlocal seq
        heapq.heappush(ev, (now, seq, 0, n, s)); seq += 1

    for n in range(len(A)):
        for s, (_, pr) in tasks[n].items():
            if not pr:
                release(n, s, A[n])

    def dispatch(s, now):
        nonlocal seq
        while nxt[s] < len(tickets[s]) and idle[s] > 0 and tickets[s][nxt[s]] in ready[s]:
            n = tickets[s][nxt[s]]
            idle[s] -= 1
            nxt[s] += 1
            heapq.heappush(ev, (max(now, ready[s][n]) + tasks[n][s][0], seq, 1, n, s)); seq += 1

    while ev:
        now, _, kind, n, s = heapq.heappop(ev)
        if kind == 0:
            ready[s][n] = now
        else:
            idle[s] += 1
            done[n][s] = now
            for s2, (_, pr) in tasks[n].items():
                if s in pr and all(q in done[n] for q in pr):
                    release(n, s2, max(done[n][q] + delay for q in pr))
        dispatch(s, now)
    return [max(done[n].values(), default=A[n]) for n in range(len(A))]


def per_server_forkjoin(A, tasks, stage_c, delay):
    """Several replicas: requests in index order, each task bound to the replica that frees first
    (argmin scan over an unsorted list), start = max(ready time, that replica's free time)."""
    free = [[0] * c for c in stage_c]
    out = []
    for n in range(len(A)):
        done = {}
        for s in sorted(tasks[n]):
            S, pr = tasks[n][s]
            ready = max([done[q] + delay for q in pr], default=A[n])
            j = min(range(stage_c[s]), key=lambda i: free[s][i])
            done[s] = max(ready, free[s][j]) + S
            free[s][j] = done[s]
        out.append(max(done.values(), default=A[n]))
    return out


@pytest.mark.parametrize("seed", range(5))
def test_eight_requests_against_event_simulators(orc, seed):
    w = omni(n_req=8)
    g = w.graph
    rng = np.random.default_rng(seed)
    for p in rng.choice(32, 6, replace=False):
        V = int(w.plans.n_stages[p])
        for c_hi in (1, 3):
            c = rng.integers(1, c_hi + 1, V).astype(np.uint16)
            pl = W.Plans(w.plans.n_stages[[p]], w.plans.stage_mask[[p]], np.pad(c, (0, 6 - V))[None, :].astype(np.uint16) | (np.arange(6) >= V).astype(np.uint16))
            for rate in (3_000, 30_000):
                A, types, svc = refsim.gen_requests(g, 70 + seed, 1, 0, rate)
                tasks = []
                for n in range(8):
                    masks, pred = stage_preds(g, pl, 0, types[n])
                    tasks.append({s: (sum(svc[n][i] for i in range(6) if (masks[s] >> i) & 1), pred[s]) for s in pred})
                t = orc.trace_sim(g, pl, 0, rate, 0, seed=70 + seed, variant=1)
                cs = [int(x) for x in pl.stage_c[0, :V]]
                assert t["departure"].tolist() == per_server_forkjoin(A, tasks, cs, g.edge_delay_us)
                if c_hi == 1:
                    assert t["departure"].tolist() == forkjoin_event_sim(A, tasks, cs, g.edge_delay_us)


def test_chain_graphs_are_unaffected(orc):
    # on a chain (E -> LLM) every stage has one predecessor: fork-join == path, bit for bit
    w = W.config1_mllm(n_req=900, n_trials=2, n_rates=3, llm_max=6, e_steps=3)
    w.graph.edge_delay_us = 5_000
    a = orc.eval_plans(w.graph, w.plans, w.rate_mrps, w.slo, w.seed, n_threads=4)
    w.graph.join_mode = 1
    b = orc.eval_plans(w.graph, w.plans, w.rate_mrps, w.slo, w.seed, n_threads=4)
    for key in ("counts", "dep_sum", "makespan"):
        np.testing.assert_array_equal(a[key], b[key])
    # ... and so is the Monte-Carlo latency (a critical path with one branch is the sum)
    m1 = orc.mc_latency(w.graph, w.plans, w.rate_mrps[:, 0], w.slo, w.seed)
    w.graph.join_mode = 0
    m0 = orc.mc_latency(w.graph, w.plans, w.rate_mrps[:, 0], w.slo, w.seed)
    assert m1["rc"] == m0["rc"] == 0
    np.testing.assert_array_equal(m1["counts"], m0["counts"])


def test_monte_carlo_latency_is_the_critical_path(orc):
    # phase 2 under fork-join (R25): "queuing not modeled" -- the simulation with unlimited replicas at any
    # rate; the simulation's fork-join rule is pinned above by path enumeration and two event simulators
    w = W.config4_sweep(n_req=600, n_trials=2, vectors_per_pattern=1, n_variants=1)   # up to 3 parallel encoders
    g, pl = w.graph, w.plans
    g.join_mode = 1
    g.edge_delay_us = 9_000
    slo = W.Slo([150_000, 200_000, 180_000, 260_000, 3_600_000, 3_700_000, 3_650_000, 3_800_000], [9] * 8, [10] * 8)
    big = W.Plans(pl.n_stages, pl.stage_mask, np.full_like(pl.stage_c, 600))
    rate = np.full(pl.n_plans, 50_000, np.uint32)
    sim = orc.eval_plans(g, big, rate[:, None], slo, w.seed, 2, n_threads=8)
    mc = orc.mc_latency(g, pl, rate, slo, w.seed, 2)
    assert mc["rc"] == 0
    np.testing.assert_array_equal(mc["counts"], sim["counts"][:, 0])
    h = mc["counts"][..., 1].sum()
    assert 0 < h < mc["counts"][..., 0].sum()
    g.join_mode = 0                      # the path mode queues the encoders one after another: later
    seq = orc.mc_latency(g, pl, rate, slo, w.seed, 2)
    assert (seq["counts"][..., 1] <= mc["counts"][..., 1]).all() and seq["counts"][..., 1].sum() < h
