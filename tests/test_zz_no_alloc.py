"""cf_pareto_select_static: the entry point that allocates nothing (its scratch is a fixed array inside
the library, at most cf_pareto_static_max_plans() plans) against cf_pareto_select, the existing path
with a caller-provided workspace -- exact equality, as in every other parity test here -- on two calls
in a row that share the array (the second smaller, with another type count and an `alive` mask, so
stale contents of the first would show). Collected last on purpose (the file name): the suite runs
with pytest -x. Passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def cf():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_2512_14098_b200 import binding
    return binding


def goodput_vectors(rng, P, T):
    """Per-type goodput vectors with ties, duplicates and dominated plans (small value range)."""
    g = rng.integers(0, 40, (P, T)).astype(np.uint32) * 1000
    g[rng.integers(0, P, P // 8)] = g[rng.integers(0, P, P // 8)]     # duplicates: equal vectors do not prune each other
    return g


def run_both(cf, torch, g, alive):
    gp = torch.from_numpy(g.view(np.int32)).cuda()
    al = None if alive is None else torch.from_numpy(alive).cuda()
    P = g.shape[0]
    # every buffer of the static call exists before it: the call itself must not allocate
    pruned = torch.full((P,), 7, dtype=torch.uint8, device="cuda")
    best = torch.full((1,), 12345, dtype=torch.int32, device="cuda")
    ns = torch.full((1,), 999, dtype=torch.int32, device="cuda")
    torch.cuda.synchronize()
    before = torch.cuda.memory_allocated()
    rc = cf.cf_pareto_select_static(gp, al, pruned, best, ns)
    torch.cuda.synchronize()
    assert rc == cf.CF_OK and torch.cuda.memory_allocated() == before
    want = cf.cf_pareto_select(gp, al)
    torch.cuda.synchronize()
    np.testing.assert_array_equal(pruned.cpu().numpy(), want["pruned"].cpu().numpy())
    assert int(best.item()) == int(want["best"].item())
    assert int(ns.item()) == int(want["n_survivors"].item())
    return pruned.cpu().numpy(), cf.to_numpy_u32(best)[0], int(ns.item())


def test_static_scratch_matches_the_workspace_path_on_two_calls_in_a_row(cf, orc):
    import torch
    rng = np.random.default_rng(11)
    # call 1: large, 4 types, everything live
    g1 = goodput_vectors(rng, 20_000, 4)
    p1, b1, n1 = run_both(cf, torch, g1, None)
    o1 = orc.pareto_select(g1)
    np.testing.assert_array_equal(p1, o1["pruned"])
    assert (int(b1), n1) == (o1["best"], o1["n_survivors"])
    # call 2 right after it on the same array: smaller, 7 types, two thirds live, smaller sums than call 1
    g2 = goodput_vectors(rng, 3_001, 7) // 8
    alive = (rng.random(3_001) < 0.66).astype(np.uint8)
    p2, b2, n2 = run_both(cf, torch, g2, alive)
    o2 = orc.pareto_select(g2, alive)
    np.testing.assert_array_equal(p2, o2["pruned"])
    assert (int(b2), n2) == (o2["best"], o2["n_survivors"])
    # call 3: nothing live -> no best, no survivors (the maximum cell was cleared)
    p3, b3, n3 = run_both(cf, torch, g2, np.zeros(3_001, np.uint8))
    assert int(b3) == 0xFFFFFFFF and n3 == 0 and p3.all()
    # the largest size the array holds, one type
    P = cf.cf_pareto_static_max_plans()
    assert P == 65_536
    run_both(cf, torch, goodput_vectors(rng, P, 1), None)


def test_sizes_beyond_the_static_scratch_are_rejected(cf, capfd):
    import torch
    P = cf.cf_pareto_static_max_plans() + 1
    gp = torch.zeros((P, 2), dtype=torch.int32, device="cuda")
    pruned = torch.full((P,), 7, dtype=torch.uint8, device="cuda")
    rc = cf.cf_pareto_select_static(gp, None, pruned, None, None, check=False)
    torch.cuda.synchronize()
    assert rc == cf.CF_ERR_RANGE
    assert (pruned == 7).all()                      # nothing was enqueued
    assert "exceed the static scratch" in capfd.readouterr().err
    with pytest.raises(cf.CfError):
        cf.cf_pareto_select_static(gp, None, pruned, None, None)
    assert cf.cf_pareto_select_static(gp[:0], None, pruned, None, None, check=False) == cf.CF_ERR_ARG
