"""GPU parity of the fast kernel's machinery: the 30-bit key window and its
64-bit fixup pass, the forced 64-bit mode, clamped / negative latency targets, and the speculative
bisection at every depth. Everything is compared bit for bit with the CPU oracle."""
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


def eval_both_modes(cf, orc, w, variant=0):
    """auto mode (fast kernel + fixup) and forced 64-bit mode against the oracle; returns the number
    of simulations the fixup pass had to redo in auto mode."""
    want = orc.eval_plans(w.graph, w.plans, w.rate_mrps, w.slo, w.seed, variant, n_threads=NT)
    wide = None
    for mode in (0, 1):
        cf.cf_debug_kernel_mode(mode)
        try:
            got = cf.cf_eval_plans(w.graph, w.plans, w.rate_mrps, w.slo, w.seed, variant)
            assert cf.cf_workspace_status(got["workspace"]) == want["rc"]
            n_wide = cf.cf_workspace_wide_count(got["workspace"])
        finally:
            cf.cf_debug_kernel_mode(0)
        np.testing.assert_array_equal(cf.to_numpy_u32(got["counts"]), want["counts"])
        np.testing.assert_array_equal(cf.to_numpy_u64(got["dep_sum"]), want["dep_sum"])
        np.testing.assert_array_equal(got["makespan"].cpu().numpy(), want["makespan"])
        if mode == 0:
            wide = n_wide
        else:
            assert n_wide == 0  # the 64-bit kernel alone never defers anything
    return wide


def test_both_kernels_on_the_configs(cf, orc):
    assert eval_both_modes(cf, orc, W.config1_mllm(n_req=1100, n_trials=2, n_rates=3)) == 0
    assert eval_both_modes(cf, orc, W.config2_omni(n_req=900, n_trials=2, n_rates=3, vectors_per_pattern=3)) == 0
    assert eval_both_modes(cf, orc, W.config3_multireplica(n_req=700, n_trials=2, n_rates=2,
                                                           plans_per_topology=24)) == 0


def one_stage(service_tab, arr_tab, n_req, cs, rates, L=(10_000_000,), n_trials=2, seed=11):
    g = W.Graph(1, 1, n_req, n_trials, [1], W.mix_thresholds([1.0]), [0], [service_tab], arr_tab,
                np.zeros((0, 2)))
    pl = W.make_plans([[(1, c)] for c in cs])
    r = np.tile(np.asarray(rates, dtype=np.uint32), (len(cs), 1))
    return W.Workload("one", g, pl, W.Slo(list(L), [9], [10]), seed=seed, rate_mrps=r)


def test_key_window_exit_goes_through_the_fixup_pass(cf, orc):
    # 1000 s services on mostly idle replicas: a request that arrives 74 s or more into a tile
    # gets a key >= 2^30 (free time - stage base); those lanes are redone by the 64-bit kernel.
    w = one_stage(W.constant_qtab(1_000_000_000), W.exponential_qtab(65536.0), 700, (1, 50, 200),
                  (1000, 500, 200_000))
    wide = eval_both_modes(cf, orc, w)
    assert wide > 0
    # a tile spanning more than 2^32 gap units
    w = one_stage(W.constant_qtab(700), W.constant_qtab(2**31 - 1), 300, (1, 2), (1_000_000, 1_000_000_000))
    assert eval_both_modes(cf, orc, w) > 0


def test_sparse_arrivals_stay_on_the_fast_path(cf, orc):
    # rates down to 1 milli-request/s: consecutive arrivals are up to hours apart, a tile of 128
    # requests spans far more than 2^31 us; lanes move their origin request by request instead
    w = one_stage(W.lognormal_qtab(50_000.0, 0.5), W.exponential_qtab(65536.0), 400, (1, 3), (1, 8, 5000))
    assert eval_both_modes(cf, orc, w) == 0
    # the same with long services on many replicas (a mix of busy and idle replicas at every arrival)
    w = one_stage(W.lognormal_qtab(5_000_000.0, 0.5), W.gamma_qtab(1.0 / 9.0, 65536.0), 900, (2, 7, 40),
                  (1, 3, 40, 700), L=(40_000_000,))
    assert eval_both_modes(cf, orc, w) == 0
    # multi-stage graph with an edge delay, rates from sparse to overloaded in one call
    w2 = W.config2_omni(n_req=500, n_trials=2, n_rates=2, vectors_per_pattern=2, n_patterns=32)
    w2.graph.edge_delay_us = 10_000
    w2.rate_mrps = np.tile(np.array([[1, 30, 900, 60_000]], dtype=np.uint32), (w2.plans.n_plans, 1))
    assert eval_both_modes(cf, orc, w2) == 0


def test_unbounded_waits_stay_on_the_fast_path(cf, orc):
    # 3x overload, 20 000 requests of 1 s: waits reach hours (far beyond 32 bits of microseconds),
    # yet the keys stay small because they are relative to the stage base
    w = one_stage(W.lognormal_qtab(1_000_000.0, 0.3), W.exponential_qtab(65536.0), 20_000, (1, 2, 5),
                  (3000, 6000, 15_000), n_trials=1)
    assert eval_both_modes(cf, orc, w) == 0
    got = cf.cf_eval_plans(w.graph, w.plans, w.rate_mrps, w.slo, w.seed)
    assert int(got["makespan"].max()) > 1 << 32


def test_services_too_long_for_the_fast_path(cf, orc):
    # worst-case service above 2^30 us: the host never admits the fast kernel
    w = one_stage(W.constant_qtab(1_200_000_000), W.exponential_qtab(65536.0), 300, (1, 4), (1, 1000))
    assert eval_both_modes(cf, orc, w) == 0


def test_negative_and_huge_latency_targets(cf, orc):
    w = W.config1_mllm(n_req=800, n_trials=2, n_rates=3, llm_max=6, e_steps=3)
    w.slo = W.Slo([-5, 1 << 40], [9, 9], [10, 10])
    eval_both_modes(cf, orc, w)
    want = orc.eval_plans(w.graph, w.plans, w.rate_mrps, w.slo, w.seed, n_threads=NT)
    assert (want["counts"][..., 0, 1] == 0).all()                             # L < 0: never a hit
    np.testing.assert_array_equal(want["counts"][..., 1, 1], want["counts"][..., 1, 0])  # always a hit
    w.slo = W.Slo([0, 2**31 - 1], [9, 9], [10, 10])
    eval_both_modes(cf, orc, w)


def test_latency_targets_beyond_32_bits_with_long_sojourns(cf, orc):
    # 3x overload, 20 000 requests of 1 s: sojourns grow past 2^31 and 2^32 us. Targets
    # between 2^31 and 2^32 must be exact inside the fast kernel; targets of 2^32 or more ("no
    # target") are held clamped there and the lanes whose sojourn passes the clamp are redone by
    # the 64-bit kernel. Hits must match the oracle either way.
    for L, expect_fixups in ((3_000_000_000, False), ((1 << 32) - 1, None), (1 << 40, True), (2**63 - 1, True)):
        w = one_stage(W.lognormal_qtab(1_000_000.0, 0.3), W.exponential_qtab(65536.0), 20_000, (1, 2, 5),
                      (3000, 6000, 15_000), L=(L,), n_trials=1)
        wide = eval_both_modes(cf, orc, w)
        want = orc.eval_plans(w.graph, w.plans, w.rate_mrps, w.slo, w.seed, n_threads=NT)
        hits = want["counts"][..., 0, 1]
        if L >= 1 << 40:
            np.testing.assert_array_equal(hits, want["counts"][..., 0, 0])  # every request is a hit
        else:
            assert (hits < want["counts"][..., 0, 0]).any() and (hits > 0).all()
        if expect_fixups is not None:
            assert (wide > 0) == expect_fixups


def test_speculative_bisection_depths(cf, orc):
    w = W.config2_omni(n_req=600, n_trials=2, n_rates=2, vectors_per_pattern=2, n_patterns=16)
    R_p = W.flow_bound_mrps(w.graph, w.plans)
    hi = np.ceil(1.5 * R_p).astype(np.uint32)
    hi[0], hi[1], hi[2], hi[3] = 0, 1, 2, 3
    slo = W.Slo(w.slo.L_us, [9] * w.graph.n_types, [10] * w.graph.n_types)
    for steps in (1, 3, 7, 18):
        bo = orc.goodput_bisect(w.graph, w.plans, hi, steps, slo, w.seed, n_threads=NT)
        for depth in (1, 2, 3, 4, 0):
            cf.cf_debug_bisect_depth(depth)
            try:
                b = cf.cf_goodput_bisect(w.graph, w.plans, hi, steps, slo, w.seed)
                probes = cf.cf_bisect_probes(b["workspace"], w.plans.n_plans)
            finally:
                cf.cf_debug_bisect_depth(0)
            np.testing.assert_array_equal(cf.to_numpy_u32(b["rate_mrps"]), bo["rate_mrps"])
            np.testing.assert_array_equal(cf.to_numpy_u32(b["goodput_mrps"]), bo["goodput_mrps"])
            np.testing.assert_array_equal(cf.to_numpy_u32(b["counts"]), bo["counts"])
            # real probes: none for an empty bracket, one for [0,2), never more than steps or log2(hi)+1
            assert probes[0] == 0 and probes[1] == 0 and probes[2] == 1
            assert (probes <= steps).all()
            assert (probes <= np.floor(np.log2(np.maximum(hi, 1))) + 1).all()


def test_bisection_with_window_exits(cf, orc):
    # probes far above capacity with long services leave the key window; the bisection result
    # must not notice
    w = one_stage(W.constant_qtab(900_000_000), W.exponential_qtab(65536.0), 500, (40, 100, 300),
                  (1000,), L=(1_000_000_000,), n_trials=2)
    hi = np.array([4000, 4000, 4000], dtype=np.uint32)
    bo = orc.goodput_bisect(w.graph, w.plans, hi, 9, w.slo, w.seed, n_threads=NT)
    for depth in (1, 3):
        cf.cf_debug_bisect_depth(depth)
        try:
            b = cf.cf_goodput_bisect(w.graph, w.plans, hi, 9, w.slo, w.seed)
        finally:
            cf.cf_debug_bisect_depth(0)
        np.testing.assert_array_equal(cf.to_numpy_u32(b["rate_mrps"]), bo["rate_mrps"])
        np.testing.assert_array_equal(cf.to_numpy_u32(b["goodput_mrps"]), bo["goodput_mrps"])
        np.testing.assert_array_equal(cf.to_numpy_u32(b["counts"]), bo["counts"])


# ---------------------------------------------------------------------------------------------
# calls whose plans have one replica at every stage run on the max-plus scan kernel (cf_scan.cuh)
# ---------------------------------------------------------------------------------------------
def all_c1(w):
    w.plans = W.Plans(w.plans.n_stages, w.plans.stage_mask, np.ones_like(w.plans.stage_c))
    return w


@pytest.mark.parametrize("n_req", [1, 31, 32, 33, 500, 1025])
def test_scan_kernel_multistage(cf, orc, n_req):
    w = all_c1(W.config2_omni(n_req=n_req, n_trials=3, n_rates=4, vectors_per_pattern=1))  # 32 topologies
    w.graph.edge_delay_us = 10_000
    w.rate_mrps = np.maximum(W.rate_grid(W.flow_bound_mrps(w.graph, w.plans), [0.01, 0.6, 0.95, 1.4]), 1)
    want = orc.eval_plans(w.graph, w.plans, w.rate_mrps, w.slo, w.seed, 2, n_threads=NT)
    got = cf.cf_eval_plans(w.graph, w.plans, w.rate_mrps, w.slo, w.seed, 2)
    assert cf.cf_workspace_status(got["workspace"]) == want["rc"] == 0
    np.testing.assert_array_equal(cf.to_numpy_u32(got["counts"]), want["counts"])
    np.testing.assert_array_equal(cf.to_numpy_u64(got["dep_sum"]), want["dep_sum"])
    np.testing.assert_array_equal(got["makespan"].cpu().numpy(), want["makespan"])
    # the thread-per-simulation kernels give the same answer on the same call
    cf.cf_debug_kernel_mode(1)
    try:
        ref = cf.cf_eval_plans(w.graph, w.plans, w.rate_mrps, w.slo, w.seed, 2)
    finally:
        cf.cf_debug_kernel_mode(0)
    np.testing.assert_array_equal(cf.to_numpy_u32(ref["counts"]), want["counts"])
    np.testing.assert_array_equal(cf.to_numpy_u64(ref["dep_sum"]), want["dep_sum"])


def test_scan_kernel_stream_bisect_and_ranges(cf, orc):
    w = all_c1(W.config4_sweep(n_req=900, n_trials=2, n_steps=12, vectors_per_pattern=2, n_variants=3))
    g, pl = w.graph, w.plans
    w.plan_variant = ((np.arange(pl.n_plans) // 3) % 3).astype(np.uint32)
    w.rate_hi_mrps = np.ceil(1.5 * W.flow_bound_mrps(g, pl)).astype(np.uint32)
    rec = cf.cf_materialize_stream(g, w.seed, 0, w.n_variants)
    rates = np.maximum(W.rate_grid(W.flow_bound_mrps(g, pl), [0.5, 1.2]), 1)
    got = cf.cf_eval_plans(g, pl, rates, w.slo, w.seed, stream_records=rec, n_variants=w.n_variants,
                           plan_variant=w.plan_variant)
    b = cf.cf_goodput_bisect(g, pl, w.rate_hi_mrps, w.n_steps, w.slo, w.seed, stream_records=rec,
                             n_variants=w.n_variants, plan_variant=w.plan_variant)
    for v in range(w.n_variants):
        idx = np.nonzero(w.plan_variant == v)[0]
        o = orc.eval_plans(g, pl.subset(idx), rates[idx], w.slo, w.seed, v, n_threads=NT)
        np.testing.assert_array_equal(cf.to_numpy_u32(got["counts"])[idx], o["counts"])
        np.testing.assert_array_equal(cf.to_numpy_u64(got["dep_sum"])[idx], o["dep_sum"])
        np.testing.assert_array_equal(got["makespan"].cpu().numpy()[idx], o["makespan"])
        bo = orc.goodput_bisect(g, pl.subset(idx), w.rate_hi_mrps[idx], w.n_steps, w.slo, w.seed, v, n_threads=NT)
        np.testing.assert_array_equal(cf.to_numpy_u32(b["rate_mrps"])[idx], bo["rate_mrps"])
        np.testing.assert_array_equal(cf.to_numpy_u32(b["goodput_mrps"])[idx], bo["goodput_mrps"])
        np.testing.assert_array_equal(cf.to_numpy_u32(b["counts"])[idx], bo["counts"])
    # out-of-range rates and the R17 horizon on the scan path
    w1 = one_stage(W.constant_qtab(5), W.constant_qtab(2**31 - 1), 1 << 12, (1,), (1, 1000, 1_000_000_000), n_trials=1)
    want = orc.eval_plans(w1.graph, w1.plans, w1.rate_mrps, w1.slo, w1.seed, n_threads=NT)
    got = cf.cf_eval_plans(w1.graph, w1.plans, w1.rate_mrps, w1.slo, w1.seed)
    assert cf.cf_workspace_status(got["workspace"]) == want["rc"] == orc.ORC_ERR_RANGE
    np.testing.assert_array_equal(cf.to_numpy_u32(got["counts"]), want["counts"])
    w1.rate_mrps[0, 1] = 0
    want = orc.eval_plans(w1.graph, w1.plans, w1.rate_mrps, w1.slo, w1.seed, n_threads=NT)
    got = cf.cf_eval_plans(w1.graph, w1.plans, w1.rate_mrps, w1.slo, w1.seed)
    np.testing.assert_array_equal(cf.to_numpy_u32(got["counts"]), want["counts"])
    np.testing.assert_array_equal(got["makespan"].cpu().numpy(), want["makespan"])
