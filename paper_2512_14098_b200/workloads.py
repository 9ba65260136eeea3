"""Seeded synthetic workload generators (inputs only -- none of the method's arithmetic).

This module serves BOTH the CUDA path's tests/bench and the CPU oracle's tests: it builds the
integer inputs (quantile tables, type mixes, plan lists, rate grids, SLOs) of the five
BASELINE.json configs. It never draws a Philox number, samples a table or runs a recursion; those
live separately in `oracle/` and in `csrc/`. Recipes are stated in DESIGN.md ("Synthetic inputs").

The paper's own workloads (ServeGen, DiffusionDB: PAPER.md:344-415) are not available; these
synthetic inputs take only their *shape* (<= 8 request types over 6 components, service-time scales
in the ratios of Table 2; Poisson or bursty arrivals) and stand in for them.
"""
from __future__ import annotations

import dataclasses
from typing import List, Optional, Sequence, Tuple

import numpy as np

QTAB_LEVELS = 16
QTAB_LOG2_CELLS = 6


# --------------------------------------------------------------------------------------------
# containers (plain numpy; both bindings marshal from these)
# --------------------------------------------------------------------------------------------
@dataclasses.dataclass
class QTab:
    levels: int
    log2_cells: int
    q: np.ndarray  # int32 [levels * 2**log2_cells + 1]

    def __post_init__(self):
        self.q = np.ascontiguousarray(self.q, dtype=np.int32)
        assert self.q.size == (self.levels << self.log2_cells) + 1


@dataclasses.dataclass
class Graph:
    n_comp: int
    n_types: int
    n_req: int
    n_trials: int
    type_mask: np.ndarray    # uint8 [T]
    type_thresh: np.ndarray  # uint32 [T] cumulative Q32
    svc_tab: np.ndarray      # uint16 [C*T]
    tabs: List[QTab]
    arr_tab: QTab
    edges: np.ndarray        # uint8 [n_edges, 2]
    edge_delay_us: int = 0
    comp_names: Tuple[str, ...] = ()
    type_names: Tuple[str, ...] = ()
    type_frac: Optional[np.ndarray] = None  # float64 [T], the mix the thresholds were built from
    cpu_tab: Optional[np.ndarray] = None    # uint16 [C*T] CPU pre-processing table of (i, t), 0xffff = none (R24)
    join_mode: int = 0                      # 1: fork-join along the DAG edges instead of a path (R25)
    order_mode: int = 0                     # 1: stages serve in arrival order (textbook FCFS, R27) instead of index order (R2)

    def __post_init__(self):
        if self.cpu_tab is not None:
            self.cpu_tab = np.ascontiguousarray(self.cpu_tab, dtype=np.uint16)
        self.type_mask = np.ascontiguousarray(self.type_mask, dtype=np.uint8)
        self.type_thresh = np.ascontiguousarray(self.type_thresh, dtype=np.uint32)
        self.svc_tab = np.ascontiguousarray(self.svc_tab, dtype=np.uint16)
        self.edges = np.ascontiguousarray(self.edges, dtype=np.uint8).reshape(-1, 2)


@dataclasses.dataclass
class Plans:
    n_stages: np.ndarray    # uint8 [P]
    stage_mask: np.ndarray  # uint8 [P, max_stages]
    stage_c: np.ndarray     # uint16 [P, max_stages]
    max_routes: int = 0                        # R26: 0 = no routing, else 1..4 routes per (plan, type)
    route_mask: Optional[np.ndarray] = None    # uint8 [P, T, max_routes] bitmask over the plan's stages
    route_cum: Optional[np.ndarray] = None     # uint32 [P, T, max_routes] cumulative probability, Q32

    def __post_init__(self):
        if self.route_mask is not None:
            self.route_mask = np.ascontiguousarray(self.route_mask, dtype=np.uint8)
            self.route_cum = np.ascontiguousarray(self.route_cum, dtype=np.uint32)
        self.n_stages = np.ascontiguousarray(self.n_stages, dtype=np.uint8)
        self.stage_mask = np.ascontiguousarray(self.stage_mask, dtype=np.uint8)
        self.stage_c = np.ascontiguousarray(self.stage_c, dtype=np.uint16)
        assert self.stage_mask.shape == self.stage_c.shape
        assert self.stage_mask.shape[0] == self.n_stages.shape[0]

    @property
    def n_plans(self) -> int:
        return int(self.n_stages.shape[0])

    @property
    def max_stages(self) -> int:
        return int(self.stage_mask.shape[1])

    def subset(self, idx) -> "Plans":
        idx = np.asarray(idx)
        if self.route_mask is None:
            return Plans(self.n_stages[idx], self.stage_mask[idx], self.stage_c[idx])
        return Plans(self.n_stages[idx], self.stage_mask[idx], self.stage_c[idx], self.max_routes,
                     self.route_mask[idx], self.route_cum[idx])


@dataclasses.dataclass
class Slo:
    L_us: np.ndarray     # int64 [T]
    att_num: np.ndarray  # uint32 [T]
    att_den: np.ndarray  # uint32 [T]

    def __post_init__(self):
        self.L_us = np.ascontiguousarray(self.L_us, dtype=np.int64)
        self.att_num = np.ascontiguousarray(self.att_num, dtype=np.uint32)
        self.att_den = np.ascontiguousarray(self.att_den, dtype=np.uint32)


@dataclasses.dataclass
class Workload:
    """One config: everything a cf_eval_plans / cf_goodput_bisect call needs."""
    name: str
    graph: Graph
    plans: Plans
    slo: Slo
    seed: int
    rate_mrps: Optional[np.ndarray] = None     # uint32 [P, R]  (eval configs)
    rate_hi_mrps: Optional[np.ndarray] = None  # uint32 [P]     (bisection configs)
    n_steps: int = 0
    n_variants: int = 1                        # materialised-stream variants (config 4)
    plan_variant: Optional[np.ndarray] = None  # uint32 [P]
    variant: int = 0


# --------------------------------------------------------------------------------------------
# quantile tables (R3): built once on the host in float64, entries rounded to integers
# --------------------------------------------------------------------------------------------
def qtab_node_probabilities(levels: int = QTAB_LEVELS, log2_cells: int = QTAB_LOG2_CELLS):
    """Upper-tail probabilities sf = 1 - p of every table node (exact in float64)."""
    cells = 1 << log2_cells
    sf = []
    for k in range(levels):
        width = 2.0 ** -(k + 1) if k < levels - 1 else 2.0 ** -(levels - 1)
        left_sf = 2.0 ** -k  # 1 - (1 - 2^-k)
        for m in range(cells):
            sf.append(left_sf - m * (width / cells))
    last_cell = (2.0 ** -(levels - 1)) / cells
    sf.append(last_cell / 2.0)  # finite end node Q(1 - w/2)
    return np.asarray(sf, dtype=np.float64)


def build_qtab(isf, scale: float, levels: int = QTAB_LEVELS,
               log2_cells: int = QTAB_LOG2_CELLS) -> QTab:
    """isf: vectorised inverse survival function of the unit distribution; entries =
    round(isf(sf) * scale) as int32, forced non-decreasing."""
    sf = qtab_node_probabilities(levels, log2_cells)
    x = np.asarray(isf(sf), dtype=np.float64) * scale
    x[0] = max(x[0], 0.0)
    q = np.rint(x)
    assert np.all(np.isfinite(q)) and q.max() <= 2**31 - 1 and q.min() >= 0
    q = np.maximum.accumulate(q).astype(np.int32)
    return QTab(levels, log2_cells, q)


def exponential_qtab(mean: float, levels=QTAB_LEVELS, log2_cells=QTAB_LOG2_CELLS) -> QTab:
    return build_qtab(lambda sf: -np.log(sf), mean, levels, log2_cells)


def lognormal_qtab(median: float, sigma: float, levels=QTAB_LEVELS,
                   log2_cells=QTAB_LOG2_CELLS) -> QTab:
    from scipy.stats import norm
    return build_qtab(lambda sf: np.exp(sigma * norm.isf(sf)), median, levels, log2_cells)


def gamma_qtab(shape: float, mean: float, levels=QTAB_LEVELS, log2_cells=QTAB_LOG2_CELLS) -> QTab:
    from scipy.stats import gamma
    return build_qtab(lambda sf: gamma.isf(sf, shape, scale=1.0 / shape), mean, levels, log2_cells)


def constant_qtab(value: int, levels=QTAB_LEVELS, log2_cells=QTAB_LOG2_CELLS) -> QTab:
    return QTab(levels, log2_cells, np.full((levels << log2_cells) + 1, value, dtype=np.int32))


def qtab_cell_probabilities(tab: QTab) -> np.ndarray:
    cells = 1 << tab.log2_cells
    pr = []
    for k in range(tab.levels):
        width = 2.0 ** -(k + 1) if k < tab.levels - 1 else 2.0 ** -(tab.levels - 1)
        pr.extend([width / cells] * cells)
    return np.asarray(pr)


def qtab_moments(tab: QTab) -> Tuple[float, float]:
    """E[X], E[X^2] of the piecewise-uniform distribution the table induces (ignoring the <1-unit
    floor of the integer lerp). Used to place rate grids and by closed-form tests."""
    pr = qtab_cell_probabilities(tab)
    a = tab.q[:-1].astype(np.float64)
    b = tab.q[1:].astype(np.float64)
    m1 = float(np.sum(pr * (a + b) / 2.0))
    m2 = float(np.sum(pr * (a * a + a * b + b * b) / 3.0))
    return m1, m2


def mix_thresholds(frac: Sequence[float]) -> np.ndarray:
    c = np.cumsum(np.asarray(frac, dtype=np.float64))
    c = c / c[-1]
    th = np.minimum(np.rint(c * 2.0**32), 2.0**32 - 1).astype(np.uint64).astype(np.uint32)
    th[-1] = 0xFFFFFFFF
    return th


# --------------------------------------------------------------------------------------------
# plan helpers
# --------------------------------------------------------------------------------------------
def make_plans(plan_list: Sequence[Sequence[Tuple[int, int]]], max_stages: Optional[int] = None) -> Plans:
    """plan_list[p] = [(component_mask, c), ...] in stage order."""
    P = len(plan_list)
    ms = max_stages or max(len(p) for p in plan_list)
    n_stages = np.zeros(P, dtype=np.uint8)
    mask = np.zeros((P, ms), dtype=np.uint8)
    c = np.zeros((P, ms), dtype=np.uint16)
    for p, stages in enumerate(plan_list):
        n_stages[p] = len(stages)
        for s, (m, cc) in enumerate(stages):
            mask[p, s] = m
            c[p, s] = cc
    return Plans(n_stages, mask, c)


def topo_stage_order(n_comp: int, edges: np.ndarray, groups: Sequence[int]) -> List[int]:
    """Kahn's algorithm on the quotient graph of component groups (bitmasks); ties broken by the
    smallest member component index (R8). Returns the groups in stage order."""
    groups = list(groups)
    gid = {}
    for gi, m in enumerate(groups):
        for i in range(n_comp):
            if (m >> i) & 1:
                gid[i] = gi
    succ = {gi: set() for gi in range(len(groups))}
    indeg = {gi: 0 for gi in range(len(groups))}
    for u, v in np.asarray(edges).reshape(-1, 2):
        if int(u) in gid and int(v) in gid:
            a, b = gid[int(u)], gid[int(v)]
            if a != b and b not in succ[a]:
                succ[a].add(b)
                indeg[b] += 1
    lowest = lambda gi: min(i for i in range(n_comp) if (groups[gi] >> i) & 1)
    ready = sorted([gi for gi in indeg if indeg[gi] == 0], key=lowest)
    order = []
    while ready:
        gi = ready.pop(0)
        order.append(groups[gi])
        for b in sorted(succ[gi]):
            indeg[b] -= 1
            if indeg[b] == 0:
                ready.append(b)
        ready.sort(key=lowest)
    assert len(order) == len(groups), "merge pattern creates a cycle"
    return order


def merge_patterns(n_comp: int, edges: np.ndarray) -> List[List[int]]:
    """All KEEP/MERGE patterns over the edges (Algorithm 1 l.3): pattern bit e set
    => edge e is MERGEd (its endpoints colocated). Returns, per pattern, the ordered stage masks;
    patterns whose quotient graph is cyclic are skipped."""
    edges = np.asarray(edges).reshape(-1, 2)
    out = []
    for pat in range(1 << len(edges)):
        parent = list(range(n_comp))

        def find(a):
            while parent[a] != a:
                parent[a] = parent[parent[a]]
                a = parent[a]
            return a

        for e, (u, v) in enumerate(edges):
            if (pat >> e) & 1:
                parent[find(int(u))] = find(int(v))
        groups = {}
        for i in range(n_comp):
            groups[find(i)] = groups.get(find(i), 0) | (1 << i)
        try:
            out.append(topo_stage_order(n_comp, edges, sorted(groups.values())))
        except AssertionError:
            continue
    return out


def flow_bound_mrps(graph: Graph, plans: Plans) -> np.ndarray:
    """Phase-1 flow bound R_p in milli-requests/s, from the exact table means:
    R_p = min_s c_s / sum_t pi_t E[S_{s,t}]. Host-side harness arithmetic for placing rate grids
    only (the device never sees it)."""
    C, T = graph.n_comp, graph.n_types
    means = np.array([qtab_moments(t)[0] for t in graph.tabs])
    th = graph.type_thresh.astype(np.float64)
    th[-1] = 2.0**32
    frac = np.diff(np.concatenate([[0.0], th])) / 2.0**32
    comp_demand = np.zeros(C)  # expected service microseconds per arriving request, per component
    for i in range(C):
        for t in range(T):
            if (int(graph.type_mask[t]) >> i) & 1:
                comp_demand[i] += frac[t] * means[int(graph.svc_tab[i * T + t])]
    R = np.zeros(plans.n_plans)
    for p in range(plans.n_plans):
        best = np.inf
        for s in range(int(plans.n_stages[p])):
            m = int(plans.stage_mask[p, s])
            d = sum(comp_demand[i] for i in range(C) if (m >> i) & 1)
            if d > 0:
                best = min(best, float(plans.stage_c[p, s]) / d)
        R[p] = best * 1e9  # per microsecond -> milli-requests per second
    return R


def rate_grid(R_p: np.ndarray, alphas: Sequence[float]) -> np.ndarray:
    r = np.rint(np.outer(R_p, np.asarray(alphas, dtype=np.float64)))
    return np.clip(r, 1, 1e9).astype(np.uint32)


# --------------------------------------------------------------------------------------------
# the five BASELINE.json configs (each takes scale knobs so tests can run reduced versions)
# --------------------------------------------------------------------------------------------
def config0_mm1(service_mean_us: int = 5000, n_req: int = 10_000, n_trials: int = 4,
                rhos: Sequence[float] = (0.1, 0.2, 0.3, 0.4, 0.5, 0.6, 0.7, 0.8)) -> Workload:
    """M/M/1 sanity (BASELINE.json configs[0]): one call per service mean (8 means 5..40 ms step 5,
    x 8 utilisations = 64 candidates); P=1 one-stage c=1 plan, R=8 rates rho/mean; seed 0."""
    g = Graph(1, 1, n_req, n_trials, [1], mix_thresholds([1.0]), [0],
              [exponential_qtab(service_mean_us)], exponential_qtab(65536.0), np.zeros((0, 2)),
              comp_names=("server",), type_names=("req",), type_frac=np.array([1.0]))
    plans = make_plans([[(1, 1)]])
    rates = np.rint(np.asarray(rhos) / service_mean_us * 1e9).astype(np.uint32).reshape(1, -1)
    slo = Slo([100_000], [9], [10])
    return Workload(f"cfg0_mm1_{service_mean_us}us", g, plans, slo, seed=0, rate_mrps=rates,
                    rate_hi_mrps=np.array([int(1e9 / service_mean_us)], dtype=np.uint32), n_steps=24)


CONFIG0_SERVICE_MEANS_US = tuple(range(5000, 40001, 5000))


def config1_mllm(n_req: int = 100_000, n_trials: int = 8, n_rates: int = 16,
                 llm_max: int = 32, e_steps: int = 8) -> Workload:
    """MLLM-like Encoder->LLM (configs[1]); plan index p = mode*e_steps*llm_max + e_idx*llm_max +
    (l-1); colocated (mode 0, e = e_idx in 0..7): one stage {E,LLM} with c = l+e; disaggregated
    (mode 1, e = e_idx+1 in 1..8): stages [{E}, c=e], [{LLM}, c=l] (R16)."""
    tabs = [lognormal_qtab(30_000.0, 0.4), lognormal_qtab(400_000.0, 0.6)]
    frac = np.array([0.7, 0.3])
    g = Graph(2, 2, n_req, n_trials, [0b10, 0b11], mix_thresholds(frac), [0, 0, 1, 1], tabs,
              exponential_qtab(65536.0), [[0, 1]], comp_names=("E", "LLM"),
              type_names=("text", "image+text"), type_frac=frac)
    pl = []
    for e_idx in range(e_steps):
        for l in range(1, llm_max + 1):
            pl.append([(0b11, l + e_idx)])
    for e_idx in range(e_steps):
        for l in range(1, llm_max + 1):
            pl.append([(0b01, e_idx + 1), (0b10, l)])
    plans = make_plans(pl, max_stages=2)
    alphas = 0.40 + 0.05 * np.arange(n_rates)
    rates = rate_grid(flow_bound_mrps(g, plans), alphas)
    slo = Slo([2_000_000, 3_000_000], [9, 9], [10, 10])
    return Workload("cfg1_mllm", g, plans, slo, seed=1, rate_mrps=rates)


OMNI_COMPS = ("E_img", "E_vid", "E_aud", "L_th", "L_ta", "G_voc")
OMNI_EDGES = np.array([[0, 3], [1, 3], [2, 3], [3, 4], [4, 5]], dtype=np.uint8)


def _omni_tabs() -> List[QTab]:
    return [lognormal_qtab(30_000.0, 0.4), lognormal_qtab(150_000.0, 0.5),
            lognormal_qtab(20_000.0, 0.4), lognormal_qtab(100_000.0, 0.6),
            lognormal_qtab(3_000_000.0, 0.6), lognormal_qtab(200_000.0, 0.3)]


def _omni_graph4(n_req, n_trials, arr_tab) -> Graph:
    T = 4
    masks = [0b001000, 0b111000, 0b001010, 0b111100]
    frac = np.array([0.50, 0.20, 0.15, 0.15])
    svc_tab = np.repeat(np.arange(6, dtype=np.uint16), T)  # table id = component id
    return Graph(6, T, n_req, n_trials, masks, mix_thresholds(frac), svc_tab, _omni_tabs(), arr_tab,
                 OMNI_EDGES, comp_names=OMNI_COMPS,
                 type_names=("text-out", "audio-out", "video-in", "audio-in+audio-out"),
                 type_frac=frac)


def _replica_vectors(rng: np.random.Generator, n_stages: int, count: int, budget_max: int = 64):
    """`count` replica vectors with c_s >= 1 and sum c_s <= budget_max (Eq. (1)):
    budget uniform in [n_stages, budget_max], split by Dirichlet(1) weights, floor, +1 each."""
    out = np.ones((count, n_stages), dtype=np.int64)
    for j in range(count):
        budget = int(rng.integers(n_stages, budget_max + 1))
        w = rng.dirichlet(np.ones(n_stages))
        out[j] += np.floor(w * (budget - n_stages)).astype(np.int64)
    return out


def config2_omni(n_req: int = 1 << 17, n_trials: int = 8, n_rates: int = 16,
                 vectors_per_pattern: int = 128, n_patterns: int = 32) -> Workload:
    """Omni-like graph (configs[2]): 32 KEEP/MERGE patterns x 128 replica vectors = 4096 plans."""
    g = _omni_graph4(n_req, n_trials, exponential_qtab(65536.0))
    rng = np.random.default_rng(2)
    pats = merge_patterns(6, OMNI_EDGES)[:n_patterns]
    pl = []
    for stages in pats:
        for cv in _replica_vectors(rng, len(stages), vectors_per_pattern):
            pl.append([(m, int(c)) for m, c in zip(stages, cv)])
    plans = make_plans(pl, max_stages=6)
    alphas = 0.40 + 0.05 * np.arange(n_rates)
    rates = rate_grid(flow_bound_mrps(g, plans), alphas)
    slo = Slo([1_000_000, 10_000_000, 2_000_000, 10_000_000], [9] * 4, [10] * 4)
    return Workload("cfg2_omni", g, plans, slo, seed=2, rate_mrps=rates)


def config3_multireplica(n_req: int = 1 << 16, n_trials: int = 4, n_rates: int = 8,
                         plans_per_topology: int = 4096) -> Workload:
    """Multi-replica stress (configs[3]): Omni graph, 4 topologies (fully disaggregated, encoders
    merged into the thinker, talker+vocoder merged, both) x 4096 replica vectors with
    c_s in {1,2,4,8,16,32}; Gamma(shape 1/9) unit-mean arrivals (CV = 3)."""
    g = _omni_graph4(n_req, n_trials, gamma_qtab(1.0 / 9.0, 65536.0))
    rng = np.random.default_rng(3)
    pats = merge_patterns(6, OMNI_EDGES)
    chosen = [pats[0b00000], pats[0b00111], pats[0b10000], pats[0b10111]]
    pl = []
    for stages in chosen:
        cs = 1 << rng.integers(0, 6, size=(plans_per_topology, len(stages)))
        for cv in cs:
            pl.append([(m, int(c)) for m, c in zip(stages, cv)])
    plans = make_plans(pl, max_stages=6)
    alphas = 0.5 + 0.1 * np.arange(n_rates)
    rates = rate_grid(flow_bound_mrps(g, plans), alphas)
    slo = Slo([1_000_000, 10_000_000, 2_000_000, 10_000_000], [9] * 4, [10] * 4)
    return Workload("cfg3_multireplica", g, plans, slo, seed=3, rate_mrps=rates)


def config4_sweep(n_req: int = 1 << 18, n_trials: int = 8, n_steps: int = 32,
                  vectors_per_pattern: int = 128, n_patterns: int = 32,
                  n_variants: int = 64) -> Workload:
    """Full coarse-to-fine sweep (configs[4]): 6 components, 8 types = {I, I+V, I+A, I+V+A} x
    {text, audio} (the shape of PAPER.md:350), Dirichlet(1) mix, 4096 plans x 32-step bisection,
    materialised stream with n_variants variants; plan p reads variant (p // 64) % n_variants."""
    rng = np.random.default_rng(4)
    T = 8
    ins = [0b000001, 0b000011, 0b000101, 0b000111]
    masks = [m | 0b001000 for m in ins] + [m | 0b111000 for m in ins]
    frac = rng.dirichlet(np.ones(T))
    svc_tab = np.repeat(np.arange(6, dtype=np.uint16), T)
    names = tuple(f"{i}->{o}" for o in ("T", "A") for i in ("I", "I+V", "I+A", "I+V+A"))
    g = Graph(6, T, n_req, n_trials, masks, mix_thresholds(frac), svc_tab, _omni_tabs(),
              exponential_qtab(65536.0), OMNI_EDGES, comp_names=OMNI_COMPS, type_names=names,
              type_frac=frac)
    pats = merge_patterns(6, OMNI_EDGES)[:n_patterns]
    pl = []
    for stages in pats:
        for cv in _replica_vectors(rng, len(stages), vectors_per_pattern):
            pl.append([(m, int(c)) for m, c in zip(stages, cv)])
    plans = make_plans(pl, max_stages=6)
    hi = np.ceil(1.5 * flow_bound_mrps(g, plans)).clip(2, 1e9).astype(np.uint32)
    L = [2_000_000, 3_000_000, 3_000_000, 4_000_000] + [10_000_000] * 4
    slo = Slo(L, [9] * T, [10] * T)
    pv = ((np.arange(plans.n_plans) // 64) % n_variants).astype(np.uint32)
    return Workload("cfg4_sweep", g, plans, slo, seed=4, rate_hi_mrps=hi, n_steps=n_steps,
                    n_variants=n_variants, plan_variant=pv)


def config_phase_sweep(n_plans: int = 1_000_000, n_req: int = 1 << 17, n_trials: int = 8) -> Workload:
    """A large candidate set for the cheap phases (flow bound, Monte-Carlo latency, Pareto pruning):
    the Omni graph of configs[2], its 32 KEEP/MERGE patterns x n_plans/32 replica vectors with
    sum c <= 64 drawn as in _replica_vectors but vectorised (numpy default_rng(6)). The paper's
    funnel evaluates 1.95 M plans in its Monte-Carlo phase (Table 6)."""
    g = _omni_graph4(n_req, n_trials, exponential_qtab(65536.0))
    rng = np.random.default_rng(6)
    pats = merge_patterns(6, OMNI_EDGES)[:32]
    per = max(1, n_plans // len(pats))
    ns, masks, cs = [], [], []
    for stages in pats:
        V = len(stages)
        budget = rng.integers(V, 65, size=per)
        wts = rng.dirichlet(np.ones(V), size=per)
        c = 1 + np.floor(wts * (budget - V)[:, None]).astype(np.int64)
        m = np.zeros((per, 6), dtype=np.uint8)
        cc = np.zeros((per, 6), dtype=np.uint16)
        m[:, :V] = np.asarray(stages, dtype=np.uint8)[None, :]
        cc[:, :V] = c
        ns.append(np.full(per, V, dtype=np.uint8)); masks.append(m); cs.append(cc)
    plans = Plans(np.concatenate(ns), np.concatenate(masks), np.concatenate(cs))
    slo = Slo([1_000_000, 10_000_000, 2_000_000, 10_000_000], [9] * 4, [10] * 4)
    return Workload("phase_sweep", g, plans, slo, seed=6)


def count_updates(graph: Graph, plans: Plans, counts: np.ndarray, per_plan: bool = False):
    """Exact number of request-stage updates from out_counts [P][R][K][T][2]: sum over sims and
    types of cnt_t * (number of stages of plan p that type t visits)."""
    P = plans.n_plans
    nvis = np.zeros((P, graph.n_types), dtype=np.int64)
    for t in range(graph.n_types):
        tm = int(graph.type_mask[t])
        for s in range(plans.max_stages):
            valid = s < plans.n_stages.astype(np.int64)
            nvis[:, t] += ((plans.stage_mask[:, s].astype(np.int64) & tm) != 0) & valid
    c = np.asarray(counts).reshape(P, -1, graph.n_types, 2)[..., 0].astype(np.int64)
    if per_plan:
        return np.einsum("pst,pt->p", c, nvis)
    return int(np.einsum("pst,pt->", c, nvis))


def count_heap_levels(graph: Graph, plans: Plans, counts: np.ndarray, per_plan: bool = False):
    """Sum over all request-stage updates of floor(log2 c) of the visited stage: the comparison
    levels a replace-min on a c-entry binary heap descends at most (0 for c = 1, the plain Lindley
    recursion). Used by bench.py's algorithmic-operation model."""
    P = plans.n_plans
    lev = np.zeros((P, graph.n_types), dtype=np.int64)
    for t in range(graph.n_types):
        tm = int(graph.type_mask[t])
        for s in range(plans.max_stages):
            valid = s < plans.n_stages.astype(np.int64)
            visit = ((plans.stage_mask[:, s].astype(np.int64) & tm) != 0) & valid
            c = np.maximum(plans.stage_c[:, s].astype(np.int64), 1)
            lev[:, t] += visit * np.floor(np.log2(c)).astype(np.int64)
    c = np.asarray(counts).reshape(P, -1, graph.n_types, 2)[..., 0].astype(np.int64)
    if per_plan:
        return np.einsum("pst,pt->p", c, lev)
    return int(np.einsum("pst,pt->", c, lev))
