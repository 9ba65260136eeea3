"""Seeded random graphs, plans, tables and rates (from sparse to overloaded) through both kernels,
bit for bit against the CPU oracle: the cross-product of the fast kernel's paths (32-bit / 64-bit /
sparse-arrival request bodies, tile rebases, heap depths 0..3, edge delay, 1..8 types and stages)
that the hand-written cases do not enumerate."""
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
    yield binding
    binding.cf_debug_kernel_mode(0)
    binding.cf_debug_bisect_depth(0)


# The committed campaign: 128 eval cases and 24 bisections. CF_FUZZ_EXTRA=n appends n more eval seeds
# and n/4 more bisection seeds (same generator), for longer runs on a GPU box.
EXTRA = int(os.environ.get("CF_FUZZ_EXTRA", "0"))
EVAL_SEEDS = list(range(128)) + list(range(5000, 5000 + EXTRA))
BISECT_SEEDS = list(range(100, 124)) + list(range(9000, 9000 + EXTRA // 4))
SHAPES = [(16, 6), (16, 6), (8, 4), (20, 2), (4, 8), (1, 9), (32, 1)]


def random_case(seed):
    rng = np.random.default_rng(seed)
    C = int(rng.integers(1, 9))
    T = int(rng.integers(1, 9))
    N = int(rng.integers(1, 700))
    K = int(rng.integers(1, 4))
    scale = float(rng.choice([2_000.0, 50_000.0, 3_000_000.0]))  # service scale: ms .. seconds
    tabs = []
    for _ in range(C):
        kind = rng.integers(0, 3)
        m = scale * float(rng.uniform(0.2, 3.0))
        L, B = SHAPES[int(rng.integers(0, len(SHAPES)))] if seed >= 64 else (16, 6)  # seeds < 64: round 1's cases
        sigma = float(rng.uniform(0.2, 0.9))
        try:
            tabs.append(W.lognormal_qtab(m, sigma, L, B) if kind == 0 else
                        W.exponential_qtab(m, L, B) if kind == 1 else W.constant_qtab(int(m), L, B))
        except AssertionError:  # a 32-level tail beyond int32 microseconds: keep the shape, drop the tail
            tabs.append(W.constant_qtab(int(m), L, B))
    masks = [int(rng.integers(0, 1 << C)) for _ in range(T)]
    if rng.random() < 0.8:
        masks = [m | (1 << int(rng.integers(0, C))) for m in masks]  # mostly non-empty routes
    frac = rng.dirichlet(np.ones(T))
    svc_tab = np.repeat(np.arange(C, dtype=np.uint16), T)
    arr = W.exponential_qtab(65536.0) if rng.random() < 0.6 else W.gamma_qtab(1.0 / 9.0, 65536.0)
    edges = [[i, i + 1] for i in range(C - 1)]
    delay = int(rng.choice([0, 0, 137, 10_000]))
    g = W.Graph(C, T, N, K, masks, W.mix_thresholds(frac), svc_tab, tabs, arr, edges, edge_delay_us=delay)
    plan_list = []
    for _ in range(int(rng.integers(1, 24))):
        n_cut = int(rng.integers(0, C))
        cuts = sorted(rng.choice(np.arange(1, C), size=n_cut, replace=False).tolist()) if C > 1 else []
        bounds = [0] + cuts + [C]
        plan_list.append([(sum(1 << i for i in range(a, b)), int(rng.choice([1, 1, 2, 3, 5, 6, 9, 21, 22, 40])))
                          for a, b in zip(bounds, bounds[1:])])
    if rng.random() < 0.25:  # one replica everywhere: the call runs on the max-plus scan kernel
        plan_list = [[(m, 1) for m, _ in stages] for stages in plan_list]
    pl = W.make_plans(plan_list, max_stages=8)
    R_p = np.maximum(W.flow_bound_mrps(g, pl), 8)
    alphas = rng.choice([0.001, 0.02, 0.3, 0.7, 0.95, 1.1, 2.5], size=int(rng.integers(1, 5)), replace=False)
    rates = np.maximum(W.rate_grid(R_p, list(alphas)), 1).astype(np.uint32)
    if rng.random() < 0.3:
        rates[0, 0] = 1  # one milli-request per second
    L = (scale * rng.uniform(0.5, 30.0, T)).astype(np.int64)
    slo = W.Slo(L, [9] * T, [10] * T)
    return W.Workload(f"fuzz{seed}", g, pl, slo, seed=1000 + seed, rate_mrps=rates), R_p


@pytest.mark.parametrize("seed", EVAL_SEEDS)
def test_random_eval(cf, orc, seed):
    w, _ = random_case(seed)
    if orc.validate(w.graph, w.plans) != 0:
        assert seed >= 128  # none of the committed seeds
        pytest.skip("the generator drew services whose worst-case sum exceeds int32 (R17)")
    want = orc.eval_plans(w.graph, w.plans, w.rate_mrps, w.slo, w.seed, 3, n_threads=NT)
    for mode in (0, 1):
        cf.cf_debug_kernel_mode(mode)
        try:
            got = cf.cf_eval_plans(w.graph, w.plans, w.rate_mrps, w.slo, w.seed, 3)
            status = cf.cf_workspace_status(got["workspace"])
        finally:
            cf.cf_debug_kernel_mode(0)
        assert status == want["rc"]
        np.testing.assert_array_equal(cf.to_numpy_u32(got["counts"]), want["counts"])
        np.testing.assert_array_equal(cf.to_numpy_u64(got["dep_sum"]), want["dep_sum"])
        np.testing.assert_array_equal(got["makespan"].cpu().numpy(), want["makespan"])


STREAM_SEEDS = [sd for sd in range(200, 330)] + list(range(12000, 12000 + EXTRA // 2))


@pytest.mark.parametrize("seed", STREAM_SEEDS)
def test_random_stream_eval_and_bisect(cf, orc, seed):
    """The materialised-stream path (per-warp chunk rings of the fast kernel, per-warp loads of the
    64-bit kernel, blocks that mix stream variants) on random graphs with at most 6 components."""
    w, R_p = random_case(seed)
    g, pl = w.graph, w.plans
    if g.n_comp > 6:
        pytest.skip("the 32-byte stream record holds 6 components")
    if orc.validate(g, pl) != 0:
        pytest.skip("the generator drew services whose worst-case sum exceeds int32 (R17)")
    rng = np.random.default_rng(seed)
    n_var = int(rng.integers(1, 4))
    pv = rng.integers(0, n_var, pl.n_plans).astype(np.uint32)
    rec = cf.cf_materialize_stream(g, w.seed, 7, n_var)
    np.testing.assert_array_equal(rec.cpu().numpy().reshape(-1),
                                  orc.materialize_stream(g, w.seed, 7, n_var).view(np.uint8).reshape(-1))
    for mode in (0, 1):
        cf.cf_debug_kernel_mode(mode)
        try:
            got = cf.cf_eval_plans(g, pl, w.rate_mrps, w.slo, w.seed, stream_records=rec, n_variants=n_var, plan_variant=pv)
            status = cf.cf_workspace_status(got["workspace"])
        finally:
            cf.cf_debug_kernel_mode(0)
        rc = 0
        for v in range(n_var):
            idx = np.nonzero(pv == v)[0]
            if idx.size == 0:
                continue
            o = orc.eval_plans(g, pl.subset(idx), w.rate_mrps[idx], w.slo, w.seed, 7 + v, n_threads=NT)
            rc = rc or o["rc"]
            np.testing.assert_array_equal(cf.to_numpy_u32(got["counts"])[idx], o["counts"])
            np.testing.assert_array_equal(cf.to_numpy_u64(got["dep_sum"])[idx], o["dep_sum"])
            np.testing.assert_array_equal(got["makespan"].cpu().numpy()[idx], o["makespan"])
        assert status == rc
    if seed % 4 == 0:
        hi = np.minimum(np.ceil(1.5 * np.minimum(R_p, 1e9)), 1_000_000_000).astype(np.uint32)
        b = cf.cf_goodput_bisect(g, pl, hi, 9, w.slo, w.seed, stream_records=rec, n_variants=n_var, plan_variant=pv)
        for v in range(n_var):
            idx = np.nonzero(pv == v)[0]
            if idx.size == 0:
                continue
            bo = orc.goodput_bisect(g, pl.subset(idx), hi[idx], 9, w.slo, w.seed, 7 + v, n_threads=NT)
            np.testing.assert_array_equal(cf.to_numpy_u32(b["rate_mrps"])[idx], bo["rate_mrps"])
            np.testing.assert_array_equal(cf.to_numpy_u32(b["counts"])[idx], bo["counts"])


VARIANT_SEEDS = list(range(400, 448)) + list(range(15000, 15000 + EXTRA // 4))


@pytest.mark.parametrize("seed", VARIANT_SEEDS)
def test_random_fidelity_variants(cf, orc, seed):
    """CPU-GPU overlap (R24) and fork-join (R25), alone and together, on the random graphs (chain DAGs
    with a few extra forward edges so that stages really fork)."""
    w, _ = random_case(seed)
    g, pl = w.graph, w.plans
    rng = np.random.default_rng(seed + 1)
    C, T = g.n_comp, g.n_types
    if seed % 3 != 1:  # overlap: CPU tables for a random subset of the components
        g.tabs = g.tabs + [W.exponential_qtab(float(rng.uniform(500.0, 40_000.0))) for _ in range(2)]
        cpu = np.full(C * T, 0xFFFF, np.uint16)
        for i in range(C):
            if rng.random() < 0.5:
                cpu[i * T:(i + 1) * T] = C + int(rng.integers(0, 2))
        g.cpu_tab = cpu
    if seed % 3 != 0:  # fork-join: skip-edges i -> i+2 turn the chain into a DAG with parallel branches
        edges = [[i, i + 2] for i in range(C - 2)] + ([[0, 1]] if C > 1 and rng.random() < 0.5 else [])
        g.edges = np.asarray(edges, dtype=np.uint8).reshape(-1, 2)
        g.join_mode = 1
    if orc.validate(g, pl) != 0:
        assert seed >= 448  # none of the committed seeds
        pytest.skip("the generator drew services whose worst-case sum exceeds int32 (R17)")
    want = orc.eval_plans(g, pl, w.rate_mrps, w.slo, w.seed, 2, n_threads=NT)
    got = cf.cf_eval_plans(g, pl, w.rate_mrps, w.slo, w.seed, 2)
    assert cf.cf_workspace_status(got["workspace"]) == want["rc"]
    np.testing.assert_array_equal(cf.to_numpy_u32(got["counts"]), want["counts"])
    np.testing.assert_array_equal(cf.to_numpy_u64(got["dep_sum"]), want["dep_sum"])
    np.testing.assert_array_equal(got["makespan"].cpu().numpy(), want["makespan"])


FCFS_SEEDS = list(range(500, 564)) + list(range(18000, 18000 + EXTRA // 4))


@pytest.mark.parametrize("seed", FCFS_SEEDS)
def test_random_arrival_order(cf, orc, seed):
    """Arrival-order service (R27, cf_fcfs.cuh) on the random graphs: radix sorts of 0..5 passes, both
    bodies of the recursion (rates of 1 milli-request/s span more than 2^32 us per batch), replica
    counts up to 40 (two free-time elements per lane); a third with CPU-GPU overlap, a fifth with
    fork-join, a fourth bisected."""
    w, R_p = random_case(seed)
    g, pl = w.graph, w.plans
    g.order_mode = 1
    rng = np.random.default_rng(seed + 2)
    if seed % 3 == 0:
        C, T = g.n_comp, g.n_types
        g.tabs = g.tabs + [W.exponential_qtab(float(rng.uniform(500.0, 40_000.0))) for _ in range(2)]
        cpu = np.full(C * T, 0xFFFF, np.uint16)
        for i in range(C):
            if rng.random() < 0.5:
                cpu[i * T:(i + 1) * T] = C + int(rng.integers(0, 2))
        g.cpu_tab = cpu
    if seed % 5 == 1:  # fork-join on top (R25): skip-edges turn the chain into a DAG with parallel branches
        C = g.n_comp
        edges = [[i, i + 2] for i in range(C - 2)] + ([[0, 1]] if C > 1 and rng.random() < 0.5 else [])
        g.edges = np.asarray(edges, dtype=np.uint8).reshape(-1, 2)
        g.join_mode = 1
    if orc.validate(g, pl) != 0:
        assert seed >= 564  # none of the committed seeds
        pytest.skip("the generator drew services whose worst-case sum exceeds int32 (R17)")
    want = orc.eval_plans(g, pl, w.rate_mrps, w.slo, w.seed, 4, n_threads=NT)
    got = cf.cf_eval_plans(g, pl, w.rate_mrps, w.slo, w.seed, 4)
    assert cf.cf_workspace_status(got["workspace"]) == want["rc"]
    np.testing.assert_array_equal(cf.to_numpy_u32(got["counts"]), want["counts"])
    np.testing.assert_array_equal(cf.to_numpy_u64(got["dep_sum"]), want["dep_sum"])
    np.testing.assert_array_equal(got["makespan"].cpu().numpy(), want["makespan"])
    if seed % 4 == 0:
        hi = np.minimum(np.ceil(1.5 * np.minimum(R_p, 1e9)), 1_000_000_000).astype(np.uint32)
        b = cf.cf_goodput_bisect(g, pl, hi, 9, w.slo, w.seed)
        bo = orc.goodput_bisect(g, pl, hi, 9, w.slo, w.seed, n_threads=NT)
        np.testing.assert_array_equal(cf.to_numpy_u32(b["rate_mrps"]), bo["rate_mrps"])
        np.testing.assert_array_equal(cf.to_numpy_u32(b["counts"]), bo["counts"])


@pytest.mark.parametrize("seed", BISECT_SEEDS)
def test_random_bisect(cf, orc, seed):
    w, R_p = random_case(seed)
    if orc.validate(w.graph, w.plans) != 0:
        assert seed >= 124  # none of the committed seeds
        pytest.skip("the generator drew services whose worst-case sum exceeds int32 (R17)")
    hi = np.minimum(np.ceil(1.5 * np.minimum(R_p, 1e9)), 1_000_000_000).astype(np.uint32)
    steps = int(np.random.default_rng(seed).integers(1, 22))
    bo = orc.goodput_bisect(w.graph, w.plans, hi, steps, w.slo, w.seed, n_threads=NT)
    for depth in (0, 3):
        cf.cf_debug_bisect_depth(depth)
        try:
            b = cf.cf_goodput_bisect(w.graph, w.plans, hi, steps, w.slo, w.seed)
        finally:
            cf.cf_debug_bisect_depth(0)
        np.testing.assert_array_equal(cf.to_numpy_u32(b["rate_mrps"]), bo["rate_mrps"])
        np.testing.assert_array_equal(cf.to_numpy_u32(b["goodput_mrps"]), bo["goodput_mrps"])
        np.testing.assert_array_equal(cf.to_numpy_u32(b["counts"]), bo["counts"])
