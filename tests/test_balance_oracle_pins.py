"""Pins of oracle/balance_oracle.py (CPU only): what the paper and the mathematics fix about the
dynamic-sampling repack + workload-balancing step."""
import os

import numpy as np
import pytest

from oracle import balance_oracle as BO

GOLD = os.path.join(os.path.dirname(__file__), "golden", "balance_example.txt")


def read_golden():
    d = {}
    for line in open(GOLD):
        if line.startswith("#") or not line.strip():
            continue
        k, *v = line.split()
        d[k] = v
    return d


def test_splitmix64_published_vector():
    g = read_golden()
    assert [BO.splitmix64(0, b) for b in range(3)] == [int(x, 16) for x in g["splitmix64_seed0"]]


def test_hand_worked_example():
    g = read_golden()
    ints = lambda k: [int(x) for x in g[k]]
    r = BO.balance_plan(ints("cu_seqlens"), ints("group_offsets"), ints("keep"), 0, 1, 2, 0, False)
    assert r["order"].tolist() == ints("order")
    assert r["cu_out"].tolist() == ints("cu_out")
    assert r["src_token"].tolist() == ints("src_token")


def lognormal_lengths(n, seed):
    r = np.random.default_rng(seed)
    return np.clip(np.rint(r.lognormal(6.5, 1.0, n)), 32, 16384).astype(np.int64)


def test_step3_is_numpy_stable_argsort():
    L = lognormal_lengths(500, 1) // 64 * 64          # many ties
    cu = np.concatenate([[0], np.cumsum(L)])
    r = BO.balance_plan(cu, None, None, 3, 2, 500, 0, False)
    w = 3 * L + 2 * L * L
    assert r["order"].tolist() == np.argsort(w, kind="stable").tolist()


def test_invariants_with_drop_and_shuffle():
    rng = np.random.default_rng(2)
    L = lognormal_lengths(256, 0)
    L[rng.integers(0, 256, 5)] = 0                    # empty samples
    cu = np.concatenate([[0], np.cumsum(L)])
    go = np.arange(0, 257, 16)
    keep = np.ones(16, np.uint8)
    keep[[3, 7, 11, 15]] = 0
    plain = BO.balance_plan(cu, go, keep, 0, 1, 24, 5, False)
    shuf = BO.balance_plan(cu, go, keep, 0, 1, 24, 5, True)
    kept = [i for i in range(256) if keep[i // 16]]
    for r in (plain, shuf):
        assert sorted(r["order"].tolist()) == kept and r["n_kept"] == 192
        assert r["n_tokens"] == int(L[kept].sum()) == r["cu_out"][-1]
        assert np.array_equal(np.diff(r["cu_out"]), L[r["order"]])
        # the token map is a bijection onto the kept samples' tokens, contiguous per sample
        exp = np.concatenate([np.arange(cu[i], cu[i + 1]) for i in r["order"]])
        assert np.array_equal(r["src_token"], exp)
    # unshuffled: workloads ascend through the whole order; buckets are 24,...,24 (8 of them)
    w = (L * L)[plain["order"]]
    assert np.all(np.diff(w) >= 0)
    assert [len(b) for b in plain["buckets"]] == [24] * 8
    # the shuffle permutes whole buckets and nothing else
    key = lambda bs: sorted(tuple(b) for b in bs)
    assert key(plain["buckets"]) == key(shuf["buckets"])
    assert plain["buckets"] != shuf["buckets"]


def test_short_last_bucket_moves_as_a_unit():
    L = np.arange(1, 12)                               # 11 samples, bucket 4 -> 4, 4, 3
    cu = np.concatenate([[0], np.cumsum(L)])
    for seed in range(8):
        r = BO.balance_plan(cu, None, None, 1, 0, 4, seed, True)
        sizes = [len(b) for b in r["buckets"]]
        assert sorted(sizes) == [3, 4, 4]
        assert [8, 9, 10] in r["buckets"]


def test_sorting_reduces_wasted_compute():
    """PAPER.md:203 asserts < 10 % waste without a formula.  Under the lock-step reading of
    DESIGN.md sec 11 the claim holds for the linear cost model on the cfg3 length recipe with 256
    buckets of 16 (3.3 %; 14 % with 64 buckets of 64) and sorting is what makes it hold (75 %
    unsorted); the quadratic model (19 %) is only required to improve."""
    L = lognormal_lengths(4096, 0)
    cu = np.concatenate([[0], np.cumsum(L)])
    sorted_plan = BO.balance_plan(cu, None, None, 1, 0, 16, 0, True)
    unsorted = [list(range(a, a + 16)) for a in range(0, 4096, 16)]
    w_sorted = BO.wasted_fraction(L, sorted_plan["buckets"], 1, 0)
    w_unsorted = BO.wasted_fraction(L, unsorted, 1, 0)
    assert w_sorted < 0.10 < w_unsorted
    assert BO.wasted_fraction(L, sorted_plan["buckets"], 0, 1) < BO.wasted_fraction(L, unsorted, 0, 1)


def test_wasted_fraction_hand_values():
    """By hand.  Lengths [1, 3] in one bucket, linear cost: both samples cost the maximum 3, so
    padded = 2*3 = 6 against 1 + 3 = 4 of useful work: waste = 1 - 4/6 = 1/3.  Quadratic cost:
    w = [1, 9], padded 18, useful 10: 1 - 10/18 = 4/9.  Two buckets [[0], [1]]: nothing is padded,
    waste 0.  Mixed model w = 2 L + L^2 = [3, 15]: 1 - 18/30 = 2/5.  Three samples [2, 2, 5] in
    buckets [[0, 1], [2]]: padded 2*2 + 5 = 9 = useful: 0; in one bucket: 1 - 9/15 = 2/5."""
    L = [1, 3]
    assert BO.wasted_fraction(L, [[0, 1]], 1, 0) == pytest.approx(1 / 3, abs=1e-15)
    assert BO.wasted_fraction(L, [[0, 1]], 0, 1) == pytest.approx(4 / 9, abs=1e-15)
    assert BO.wasted_fraction(L, [[0], [1]], 1, 0) == 0.0
    assert BO.wasted_fraction(L, [[0, 1]], 2, 1) == pytest.approx(2 / 5, abs=1e-15)
    assert BO.wasted_fraction([2, 2, 5], [[0, 1], [2]], 1, 0) == 0.0
    assert BO.wasted_fraction([2, 2, 5], [[0, 1, 2]], 1, 0) == pytest.approx(2 / 5, abs=1e-15)
    assert BO.wasted_fraction([], [], 1, 0) == 0.0
