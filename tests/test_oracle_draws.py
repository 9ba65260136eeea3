"""Pins for the oracle's draw generation: Philox4x32-10 and the integer quantile-table sampler."""
import os

import numpy as np
import pytest

import refsim
from paper_2512_14098_b200 import workloads as W

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _kats():
    out = []
    for line in open(os.path.join(GOLDEN, "philox4x32_10_kat.txt")):
        if line.startswith("#") or not line.strip():
            continue
        w = [int(x, 16) for x in line.split()]
        out.append((w[0:4], w[4:6], w[6:10]))
    return out


def test_philox_known_answers(orc):
    kats = _kats()
    assert len(kats) == 3
    for ctr, key, want in kats:
        assert orc.philox4x32_10(ctr, key) == want
        assert refsim.philox4x32_10(ctr, key) == want  # the independent restatement is pinned too


def test_philox_counter_layout(orc):
    # values in this build's counter layout (n, trial, block, variant)
    cases = [((1, 0, 0, 0), (0, 0), "f8e4cca4 5cb200db b1a574eb 097eff67"),
             ((2, 0, 0, 0), (0, 0), "04faa329 51c732a6 241513ad 459135e4"),
             ((0, 0, 1, 0), (0, 0), "844515e1 f08d6eaa 0f19c053 83f875f0"),
             ((7, 3, 2, 0), (42, 0), "258fa63d c33e9995 c653dee9 60e70864")]
    for ctr, key, want in cases:
        want = [int(x, 16) for x in want.split()]
        assert orc.philox4x32_10(ctr, key) == want
        assert refsim.philox4x32_10(ctr, key) == want


def test_philox_matches_restatement_random(orc):
    rng = np.random.default_rng(0)
    for _ in range(200):
        ctr = rng.integers(0, 2**32, 4)
        key = rng.integers(0, 2**32, 2)
        assert orc.philox4x32_10(ctr, key) == refsim.philox4x32_10(ctr, key)


EDGE_WORDS = [0, 1, 0x7FFFFFFF, 0x80000000, 0xBFFFFFFF, 0xC0000000, 0xFFFF0000, 0xFFFF7FFF,
              0xFFFF8000, 0xFFFFFFFE, 0xFFFFFFFF]


@pytest.mark.parametrize("L,B", [(16, 6), (1, 10), (1, 0), (4, 3), (32, 2), (8, 16), (20, 0)])
def test_qtab_matches_geometric_definition(orc, L, B):
    rng = np.random.default_rng(L * 100 + B)
    n = (L << B) + 1
    q = np.sort(rng.integers(0, 2**31 - 1, n)).astype(np.int32)
    tab = W.QTab(L, B, q)
    us = EDGE_WORDS + [int(x) for x in rng.integers(0, 2**32, 300)]
    # words with many leading ones exercise the deep levels
    us += [(0xFFFFFFFF << s) & 0xFFFFFFFF | int(rng.integers(0, 1 << s)) if s else 0xFFFFFFFF
           for s in range(0, 32)]
    for u in us:
        assert orc.qtab_sample(tab, u) == refsim.qtab_sample(L, B, q, u), hex(u)


def test_qtab_constant_and_monotone(orc):
    tab = W.constant_qtab(12345)
    for u in EDGE_WORDS:
        assert orc.qtab_sample(tab, u) == 12345
    tab = W.exponential_qtab(65536.0)
    us = np.sort(np.random.default_rng(1).integers(0, 2**32, 5000)).tolist() + [0xFFFFFFFF]
    vals = [orc.qtab_sample(tab, int(u)) for u in us]
    assert all(b >= a for a, b in zip(vals, vals[1:]))
    assert vals[0] >= 0 and vals[-1] <= int(tab.q[-1])
    assert orc.qtab_sample(tab, 0) == int(tab.q[0])


def test_qtab_identity_quantile(orc):
    # Table whose nodes are the quantile abscissae themselves, scaled to 2^30: sample(u) ~ u >> 2.
    L, B = W.QTAB_LEVELS, W.QTAB_LOG2_CELLS
    sf = W.qtab_node_probabilities(L, B)
    q = np.rint((1.0 - sf) * 2.0**30).astype(np.int32)
    tab = W.QTab(L, B, q)
    rng = np.random.default_rng(2)
    for u in EDGE_WORDS[:-2] + [int(x) for x in rng.integers(0, 2**32, 2000)]:
        if u >= 0xFFFFFFFF - (1 << 10):
            continue  # inside the last cell the end node is Q(1 - w/2), not Q(1)
        assert abs(orc.qtab_sample(tab, u) - (u >> 2)) <= 1 << 7, hex(u)


def test_exponential_table_moments(orc):
    # the distribution induced by the table reproduces the exponential's first two moments
    tab = W.exponential_qtab(1_000_000.0)
    m1, m2 = W.qtab_moments(tab)
    assert abs(m1 / 1e6 - 1.0) < 2e-4
    assert abs(m2 / 2e12 - 1.0) < 2e-4
    # and sampling the oracle on a fine regular grid of u reproduces those moments
    us = (np.arange(1 << 16, dtype=np.uint64) << 16) + (1 << 15)
    x = np.array([orc.qtab_sample(tab, int(u)) for u in us], dtype=np.float64)
    assert abs(x.mean() / m1 - 1.0) < 5e-3
    assert abs((x * x).mean() / m2 - 1.0) < 3e-2


def test_materialized_records_match_restatement(orc):
    # stream records (cu, type, services) == the independent pure-Python derivation
    w = W.config2_omni(n_req=40, n_trials=2, n_rates=2, vectors_per_pattern=1, n_patterns=2)
    recs = orc.materialize_stream(w.graph, seed=77, variant_lo=3, n_variants=2)
    for vi in range(2):
        for k in range(2):
            A, types, svc = refsim.gen_requests(w.graph, 77, 3 + vi, k, rate_mrps=1000)
            # rate 1000 mrps -> period 1e6: A = (cu*1e6 + 32768) >> 16
            for n in range(40):
                head = int(recs[vi, k, n]["head"])
                cu, t = head & ((1 << 56) - 1), head >> 56
                assert t == types[n]
                assert (cu * 10**6 + 32768) >> 16 == A[n]
                for i in range(6):
                    assert int(recs[vi, k, n]["svc"][i]) == svc[n].get(i, 0)
