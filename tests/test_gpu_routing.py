"""GPU parity of routing between alternative paths (R26; SURVEY.md 8(f)
NEXT-4): routed plans run on the fast kernel (the route draw rides in the 3-word request record) and
on the 64-bit kernel; eval, trace, bisection and the routed flow bound against the oracle, bit for bit."""
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


def both_modes(cf, orc, g, pl, rates, slo, seed, variant=0):
    want = orc.eval_plans(g, pl, rates, slo, seed, variant, n_threads=NT)
    assert want["rc"] == 0
    for mode in (cf.CF_KERNEL_AUTO, cf.CF_KERNEL_WIDE64):
        cf.cf_debug_kernel_mode(mode)
        try:
            got = cf.cf_eval_plans(g, pl, rates, slo, seed, variant)
            assert cf.cf_workspace_status(got["workspace"]) == 0
        finally:
            cf.cf_debug_kernel_mode(0)
        np.testing.assert_array_equal(cf.to_numpy_u32(got["counts"]), want["counts"])
        np.testing.assert_array_equal(cf.to_numpy_u64(got["dep_sum"]), want["dep_sum"])
        np.testing.assert_array_equal(got["makespan"].cpu().numpy(), want["makespan"])
    return want


def omni_routed(n_req, n_trials, rng, n_plans=48):
    """The Omni graph of configs[2] with, per plan, the disaggregated 6-stage path AND a node that
    colocates {E_vid, L_th} AND one that colocates {L_ta, G_voc}: video requests choose between the
    E_vid -> L_th path and the merged node, audio-out requests between L_ta -> G_voc and the merged
    node, with per-plan probabilities in steps of 0.1."""
    base = W.config2_omni(n_req=n_req, n_trials=n_trials, n_rates=1, vectors_per_pattern=1, n_patterns=1)
    g = base.graph
    # stages: 0 E_img, 1 E_vid, 2 E_aud, 3 {E_vid, L_th}, 4 L_th, 5 L_ta, 6 {L_ta, G_voc}, 7 G_voc
    masks = [0b000001, 0b000010, 0b000100, 0b001010, 0b001000, 0b010000, 0b110000, 0b100000]
    plans, rmask, rcum = [], [], []
    T = 4
    for _ in range(n_plans):
        plans.append([(m, int(rng.integers(1, 9))) for m in masks])
        pv, pa = rng.integers(0, 11, 2) / 10.0
        q = lambda x: min(int(round(float(x) * 2**32)), 2**32 - 1)
        # types: 0 text-out {L_th}; 1 audio-out {L_th, L_ta, G_voc}; 2 video-in {E_vid, L_th}; 3 audio-in+out {E_aud, L_th, L_ta, G_voc}
        rm = np.zeros((T, 4), np.uint8)
        rc = np.zeros((T, 4), np.uint32)
        rm[0] = [0b00010000] * 4                                         # L_th alone
        rc[0] = [0xFFFFFFFF] * 4
        rm[1] = [0b10110000, 0b01010000, 0b01010000, 0b01010000]         # L_th, then (L_ta -> G_voc) or the merged node
        rc[1] = [q(pa), 0xFFFFFFFF, 0xFFFFFFFF, 0xFFFFFFFF]
        rm[2] = [0b00010010, 0b00001000, 0b00001000, 0b00001000]         # (E_vid -> L_th) or the merged node
        rc[2] = [q(pv), 0xFFFFFFFF, 0xFFFFFFFF, 0xFFFFFFFF]
        rm[3] = [0b10110100, 0b01010100, 0b01010100, 0b01010100]
        rc[3] = [q(pa), 0xFFFFFFFF, 0xFFFFFFFF, 0xFFFFFFFF]
        rmask.append(rm); rcum.append(rc)
    pl = W.make_plans(plans, max_stages=8)
    pl = W.Plans(pl.n_stages, pl.stage_mask, pl.stage_c, 4, np.array(rmask), np.array(rcum))
    return g, pl, base.slo


def test_routed_plans_parity(cf, orc):
    from test_oracle_routing import mllm, two_path_plans
    g = mllm(2100, 2)
    cs = [(1, 3, 2), (2, 5, 4), (1, 1, 1), (3, 8, 2), (2, 2, 7)]
    for pt, pi in ((0.5, 0.5), (0.2, 0.9), (0.0, 1.0 - 2**-32)):
        pl = two_path_plans(cs, pt, pi)
        rates = np.maximum(W.rate_grid(W.flow_bound_mrps(g, W.make_plans([[(0b11, c[1] + c[2])] for c in cs])), [0.3, 0.8, 1.2]), 1)
        both_modes(cf, orc, g, pl, rates, W.Slo([2_000_000, 3_000_000], [9, 9], [10, 10]), 5, 1)
    rng = np.random.default_rng(8)
    g, pl, slo = omni_routed(1900, 2, rng)
    g.edge_delay_us = 7_000
    assert orc.validate(g, pl) == 0
    fo = orc.flow_bound(g, pl, 1, 1)
    f = cf.cf_flow_bound(g, pl, 1, 1)
    np.testing.assert_array_equal(cf.to_numpy_u32(f["bound_mrps"]), fo["bound_mrps"])
    np.testing.assert_array_equal(f["bottleneck"].cpu().numpy(), fo["bottleneck"])
    np.testing.assert_array_equal(f["redundant"].cpu().numpy(), fo["redundant"])
    rates = np.maximum((fo["bound_mrps"][:, None] * np.array([0.4, 0.9, 1.3])).astype(np.uint32), 1)
    both_modes(cf, orc, g, pl, rates, slo, 11, 3)
    for p in (0, 17, 40):
        t = cf.cf_trace_sim(g, pl, p, int(rates[p, 1]), 1, 11, variant=3)
        o = orc.trace_sim(g, pl, p, int(rates[p, 1]), 1, 11, variant=3)
        np.testing.assert_array_equal(t["departure"].cpu().numpy(), o["departure"])
        cf.cf_debug_kernel_mode(cf.CF_KERNEL_FAST32)
        try:
            t = cf.cf_trace_sim(g, pl, p, int(rates[p, 1]), 1, 11, variant=3)
        finally:
            cf.cf_debug_kernel_mode(0)
        np.testing.assert_array_equal(t["departure"].cpu().numpy(), o["departure"])
    hi = (fo["bound_mrps"].astype(np.uint64) * 3 // 2).astype(np.uint32)
    b = cf.cf_goodput_bisect(g, pl, hi, 10, slo, 11)
    bo = orc.goodput_bisect(g, pl, hi, 10, slo, 11, n_threads=NT)
    np.testing.assert_array_equal(cf.to_numpy_u32(b["rate_mrps"]), bo["rate_mrps"])
    np.testing.assert_array_equal(cf.to_numpy_u32(b["goodput_mrps"]), bo["goodput_mrps"])
    np.testing.assert_array_equal(cf.to_numpy_u32(b["counts"]), bo["counts"])
    # fork-join on top of routing (R25 + R26)
    g.join_mode = 1
    both_modes(cf, orc, g, pl, rates, slo, 11, 3)


def test_monte_carlo_latency_with_routes(cf, orc):
    """Phase 2 on routed plans (R26): the per-plan kernel over shared request records, against the oracle."""
    from test_oracle_routing import mllm, two_path_plans
    g = mllm(5000, 3, delay=30_000)
    rng = np.random.default_rng(8)
    cs = [tuple(int(x) for x in rng.integers(1, 9, 3)) for _ in range(40)]
    pl = two_path_plans(cs, 0.6, 0.4)
    pl.route_cum[:, :, 0] = rng.integers(0, 2**32, (40, 2), dtype=np.uint64).astype(np.uint32)   # a different split per plan
    slo = W.Slo([430_000, 520_000], [9, 9], [10, 10])
    rate = rng.integers(1, 2**32, 40, dtype=np.uint64).astype(np.uint32)
    for variant in (0, 6):
        o = orc.mc_latency(g, pl, rate, slo, 21, variant)
        m = cf.cf_mc_latency(g, pl, rate, slo, 21, variant)
        assert o["rc"] == 0
        np.testing.assert_array_equal(cf.to_numpy_u32(m["counts"]), o["counts"])
        np.testing.assert_array_equal(cf.to_numpy_u32(m["goodput_mrps"]), o["goodput_mrps"])
    assert len({tuple(c) for c in o["counts"][..., 1].reshape(40, -1)}) > 10     # the plans' splits matter
    # the 8-stage Omni plan set with two routed choices, fork-join on top, CPU-GPU overlap on top of that
    g2, pl2, slo2 = omni_routed(3000, 2, np.random.default_rng(8))
    g2.edge_delay_us = 7_000
    r1 = orc.flow_bound(g2, pl2, 4, 5)["rate_mrps"]
    for join in (0, 1):
        g2.join_mode = join
        o = orc.mc_latency(g2, pl2, r1, slo2, 11, 2)
        m = cf.cf_mc_latency(g2, pl2, r1, slo2, 11, 2)
        np.testing.assert_array_equal(cf.to_numpy_u32(m["counts"]), o["counts"])
        np.testing.assert_array_equal(cf.to_numpy_u32(m["goodput_mrps"]), o["goodput_mrps"])
    g2.tabs = g2.tabs + [W.exponential_qtab(12_000.0)]
    cpu = np.full(g2.n_comp * g2.n_types, 0xFFFF, np.uint16)
    cpu[:2 * g2.n_types] = len(g2.tabs) - 1
    g2.cpu_tab = cpu
    o = orc.mc_latency(g2, pl2, r1, slo2, 11, 2)
    m = cf.cf_mc_latency(g2, pl2, r1, slo2, 11, 2, want_counts=False)
    np.testing.assert_array_equal(cf.to_numpy_u32(m["goodput_mrps"]), o["goodput_mrps"])


def test_routing_refusals(cf, orc):
    import torch
    from test_oracle_routing import mllm, two_path_plans
    g = mllm(64)
    pl = two_path_plans([(1, 1, 1)], 0.5, 0.5)
    slo = W.Slo([1, 1], [9, 9], [10, 10])
    rec = torch.zeros((1, 1, 64, 32), dtype=torch.uint8, device="cuda")
    assert cf.cf_eval_plans(g, pl, [[1000]], slo, 0, stream_records=rec, check=False)["rc"] == cf.CF_ERR_ARG
    bad = two_path_plans([(1, 1, 1)], 0.5, 0.5)
    bad.route_mask[0, 1, 0] = 0b010
    assert cf.cf_eval_plans(g, bad, [[1000]], slo, 0, check=False)["rc"] == cf.CF_ERR_PLAN == orc.validate(g, bad)
    plain = W.make_plans([[(0b01, 1), (0b10, 1), (0b11, 1)]])
    assert cf.cf_eval_plans(g, plain, [[1000]], slo, 0, check=False)["rc"] == cf.CF_ERR_PLAN
