"""GPU parity of the repack + workload-balancing step (NEXT-1): integer work, bit-exact against
oracle/balance_oracle.py on the same seeded inputs; the repack gathers are checked against plain
indexing."""
import numpy as np
import pytest
import torch

from oracle import balance_oracle as BO

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    assert torch.cuda.is_available()
    from paper_2507_22789_b200 import binding
    return binding


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def make_case(R, group, seed, p_drop=0.25, empties=3):
    r = np.random.default_rng(seed)
    L = np.clip(np.rint(r.lognormal(4.0, 1.0, R)), 1, 2000).astype(np.int64)
    if R > empties:
        L[r.integers(0, R, empties)] = 0
    cu = np.concatenate([[0], np.cumsum(L)]).astype(np.int32)
    go = np.arange(0, R + 1, group, dtype=np.int32)
    if go[-1] != R:
        go = np.append(go, R).astype(np.int32)
    keep = (r.random(len(go) - 1) >= p_drop).astype(np.uint8)
    return cu, go, keep


def check(B, cu, go, keep, w_lin, w_quad, bucket, seed, shuffle):
    exp = BO.balance_plan(cu, go, keep, w_lin, w_quad, bucket, seed, shuffle)
    got = B.gc_balance_plan(dev(cu), None if go is None else dev(go), None if keep is None else dev(keep),
                            w_lin, w_quad, bucket, seed, shuffle)
    torch.cuda.synchronize()
    n, nt = int(got["n_kept"].item()), int(got["n_tokens"].item())
    assert n == exp["n_kept"] and nt == exp["n_tokens"]
    R = len(cu) - 1
    order = got["order"].cpu().numpy()
    assert np.array_equal(order[:n], exp["order"])
    assert np.all(order[n:R] == -1)
    cu_out = got["cu_out"].cpu().numpy()
    assert np.array_equal(cu_out[:n + 1], exp["cu_out"])
    assert np.all(cu_out[n:] == nt)
    assert np.array_equal(got["src_token"].cpu().numpy()[:nt], exp["src_token"])
    return got, exp


@pytest.mark.parametrize("R,group,bucket", [(1, 1, 1), (7, 2, 2), (256, 16, 24), (1000, 8, 64),
                                            (5000, 16, 512), (4097, 1, 1)])
@pytest.mark.parametrize("shuffle", [False, True])
def test_balance_plan_bit_exact(B, R, group, bucket, shuffle):
    cu, go, keep = make_case(R, group, seed=R + bucket)
    check(B, cu, go, keep, 0, 1, bucket, 1234567 + R, shuffle)
    check(B, cu, go, keep, 5, 3, bucket, 99, shuffle)


def test_balance_plan_edge_cases(B):
    cu, go, keep = make_case(300, 4, seed=1)
    check(B, cu, go, np.zeros_like(keep), 0, 1, 16, 0, True)           # everything dropped
    check(B, cu, go, None, 0, 1, 16, 0, True)                           # keep == NULL
    check(B, cu, None, None, 1, 0, 1000, 0, True)                       # no groups, one bucket
    eq = np.arange(0, 64 * 10 + 1, 10).astype(np.int32)                 # all lengths equal: pure ties
    check(B, eq, None, None, 0, 1, 8, 3, False)
    check(B, eq, None, None, 0, 1, 8, 3, True)
    # the golden hand-worked example
    g = check(B, np.array([0, 5, 8, 8, 20, 21, 30, 33], np.int32), np.array([0, 2, 4, 6, 7], np.int32),
              np.array([1, 1, 0, 1], np.uint8), 0, 1, 2, 0, False)[0]
    assert g["order"].cpu().numpy()[:5].tolist() == [2, 1, 6, 0, 3]


def test_repack_gathers(B):
    """cfg3-style flow: drop constant groups, balance, repack H / targets / old log-probs."""
    cu, go, keep = make_case(512, 16, seed=7)
    T = int(cu[-1])
    got, exp = check(B, cu, go, keep, 0, 1, 32, 11, True)
    gen = torch.Generator(device="cuda").manual_seed(0)
    H = torch.randn(T, 264, device="cuda", generator=gen).to(torch.bfloat16)
    y = torch.randint(0, 1000, (T,), device="cuda", dtype=torch.int32, generator=gen)
    old = torch.randn(T, device="cuda", generator=gen)
    nt = exp["n_tokens"]
    Hs = B.gc_gather_rows(H, got["src_token"], got["n_tokens"], T)
    ys = B.gc_gather_1d(y, got["src_token"], got["n_tokens"], T)
    os_ = B.gc_gather_1d(old, got["src_token"], got["n_tokens"], T)
    idx = torch.from_numpy(exp["src_token"].astype(np.int64)).cuda()
    assert torch.equal(Hs[:nt], H[idx]) and torch.equal(ys[:nt], y[idx]) and torch.equal(os_[:nt], old[idx])
    pad_end = min((nt + 255) // 256 * 256, T)
    assert float(Hs[nt:pad_end].float().abs().sum()) == 0.0
