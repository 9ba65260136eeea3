"""CPU-side checks of the CUDA library: it loads, exports every symbol include/cf.h declares, and
its host logic (validation, workspace sizing) behaves as documented. No compute calls succeed
without a GPU: they must fail loudly (CF_ERR_CUDA), never fall back to a CPU path."""
import ctypes as C
import os
import re

import numpy as np
import pytest
import torch

from paper_2512_14098_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def cf():
    from paper_2512_14098_b200 import build
    build.build()
    from paper_2512_14098_b200 import binding
    return binding


def test_exports_every_declared_symbol(cf):
    lib = C.CDLL(cf.LIB_PATH)
    for header, exports in (("cf.h", cf.EXPORTS), ("cf_debug.h", cf.DEBUG_EXPORTS)):
        hdr = open(os.path.join(ROOT, "include", header)).read()
        hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
        declared = set(re.findall(r"\b(cf_[a-z0-9_]+)\s*\(", hdr))
        assert declared == set(exports), (header, declared ^ set(exports))
        for name in declared:
            assert hasattr(lib, name), name
    # the product header declares no test knob
    assert not [n for n in cf.EXPORTS if "debug" in n or "bench" in n or n.endswith("_opt")]


def test_strerror(cf):
    assert cf.strerror(0) == "ok"
    for code in range(-6, 0):
        assert cf.strerror(code) not in ("ok", "unknown status")
    assert cf.strerror(-99) == "unknown status"


FAKE = C.c_void_p(0x10000)  # never dereferenced: host validation returns before any CUDA call


def raw_eval(cf, graph, plans, slo, R=1, ws_bytes=1 << 30):
    m = cf.Marshalled(graph, plans, slo)
    return cf._lib.cf_eval_plans(C.byref(m.g), C.byref(m.pl), FAKE, C.c_uint32(R), C.byref(m.slo),
                                 C.c_uint64(0), C.c_uint32(0), FAKE, None, None, FAKE,
                                 C.c_size_t(ws_bytes), None)


def test_host_validation(cf):
    w = W.config1_mllm(n_req=100, n_trials=2, n_rates=1, llm_max=4, e_steps=2)
    g, pl, slo = w.graph, w.plans, w.slo
    bad = W.Plans(pl.n_stages.copy(), pl.stage_mask.copy(), pl.stage_c.copy())
    bad.stage_c[3, 0] = 0
    assert raw_eval(cf, g, bad, slo) == cf.CF_ERR_PLAN
    assert raw_eval(cf, g, W.make_plans([[(0b01, 1), (0b11, 1)]]), slo) == cf.CF_ERR_PLAN
    assert raw_eval(cf, g, W.make_plans([[(0b01, 1)]]), slo) == cf.CF_ERR_PLAN
    assert raw_eval(cf, g, W.make_plans([[(0b10, 1), (0b01, 1)]]), slo) == cf.CF_ERR_PLAN
    tq = g.tabs[0].q.copy()
    tq[10] = tq[9] - 1
    g2 = W.Graph(g.n_comp, g.n_types, g.n_req, g.n_trials, g.type_mask, g.type_thresh, g.svc_tab,
                 [W.QTab(16, 6, tq), g.tabs[1]], g.arr_tab, g.edges)
    assert raw_eval(cf, g2, pl, slo) == cf.CF_ERR_TABLE
    g3 = W.Graph(g.n_comp, g.n_types, 0, g.n_trials, g.type_mask, g.type_thresh, g.svc_tab, g.tabs,
                 g.arr_tab, g.edges)
    assert raw_eval(cf, g3, pl, slo) == cf.CF_ERR_ARG
    big = W.constant_qtab(2**31 - 1)
    g4 = W.Graph(g.n_comp, g.n_types, g.n_req, g.n_trials, g.type_mask, g.type_thresh, g.svc_tab,
                 [big, big], g.arr_tab, g.edges)
    assert raw_eval(cf, g4, pl, slo) == cf.CF_ERR_RANGE
    g5 = W.Graph(g.n_comp, g.n_types, g.n_req, g.n_trials, g.type_mask, g.type_thresh, g.svc_tab,
                 g.tabs, g.arr_tab, g.edges, edge_delay_us=-1)
    assert raw_eval(cf, g5, pl, slo) == cf.CF_ERR_RANGE
    assert raw_eval(cf, g, pl, slo, ws_bytes=16) == cf.CF_ERR_WORKSPACE
    # replica counts whose heaps cannot fit one SM's shared memory
    assert raw_eval(cf, g, W.make_plans([[(0b11, 5000)]]), slo) == cf.CF_ERR_RANGE


def test_library_and_oracle_validate_alike(cf, orc):
    w = W.config2_omni(n_req=50, n_trials=1, n_rates=1, vectors_per_pattern=2, n_patterns=8)
    assert orc.validate(w.graph, w.plans) == 0
    rng = np.random.default_rng(0)
    for _ in range(60):  # random corruptions of the plan table
        bad = W.Plans(w.plans.n_stages.copy(), w.plans.stage_mask.copy(), w.plans.stage_c.copy())
        p = int(rng.integers(0, bad.n_plans))
        s = int(rng.integers(0, bad.max_stages))
        which = int(rng.integers(0, 3))
        if which == 0:
            bad.stage_mask[p, s] = int(rng.integers(0, 64))
        elif which == 1:
            bad.stage_c[p, s] = int(rng.integers(0, 3))
        else:
            bad.n_stages[p] = int(rng.integers(0, 8))
        want = orc.validate(w.graph, bad)
        got = raw_eval(cf, w.graph, bad, w.slo)
        if want != 0:
            assert got == want
        else:
            assert got in (cf.CF_OK, cf.CF_ERR_CUDA)


def test_workspace_bytes(cf):
    w = W.config1_mllm(n_req=100, n_trials=2, n_rates=1, llm_max=4, e_steps=2)
    a = cf.cf_workspace_bytes(w.graph, w.plans, 1)
    b = cf.cf_workspace_bytes(w.graph, w.plans, 16)
    c = cf.cf_workspace_bytes(w.graph, w.plans, 64)
    # R below the bisection's 15 speculative rates per plan does not shrink the scratch any further
    assert 0 < a <= b < c < 1 << 26


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks behaviour WITHOUT a GPU")
def test_no_cpu_fallback(cf):
    w = W.config1_mllm(n_req=100, n_trials=2, n_rates=1, llm_max=4, e_steps=2)
    with pytest.raises(RuntimeError):
        cf.cf_eval_plans(w.graph, w.plans, w.rate_mrps, w.slo, 0)
    # even through the raw ABI with valid arguments the call fails loudly instead of computing
    assert raw_eval(cf, w.graph, w.plans, w.slo, ws_bytes=1 << 30) == cf.CF_ERR_CUDA


def test_update_and_heap_level_counts():
    """bench.py's exact work counters: hand-computed on a two-plan example, and per-plan sums."""
    import numpy as np
    # 2 components, 2 types: type 0 visits {0}, type 1 visits {0, 1}
    tab = W.constant_qtab(1000)
    g = W.Graph(2, 2, 10, 1, [0b01, 0b11], W.mix_thresholds([0.5, 0.5]), [0, 0, 0, 0], [tab], tab, [[0, 1]])
    pl = W.make_plans([[(0b11, 8)], [(0b01, 1), (0b10, 5)]])  # colocated c=8; disaggregated c=1, c=5
    counts = np.zeros((2, 1, 1, 2, 2), dtype=np.uint32)
    counts[..., 0, 0] = 6  # 6 requests of type 0
    counts[..., 1, 0] = 4  # 4 of type 1
    # plan 0: every request visits its single stage once; plan 1: type 0 one stage, type 1 two
    assert W.count_updates(g, pl, counts) == (6 + 4) + (6 + 2 * 4)
    # floor(log2 c): plan 0: 3 per update; plan 1: stage 0 -> 0, stage 1 (type 1 only) -> 2
    assert W.count_heap_levels(g, pl, counts) == 3 * 10 + 2 * 4
    np.testing.assert_array_equal(W.count_updates(g, pl, counts, per_plan=True), [10, 14])
    np.testing.assert_array_equal(W.count_heap_levels(g, pl, counts, per_plan=True), [30, 8])
