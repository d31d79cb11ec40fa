"""GPU parity of the verdict-token scoring (NEXT-3, gc_token_logprobs_multi): K candidate tokens per
row in one pass of the forward contraction, against the fp64 oracle applied per candidate column."""
import numpy as np
import pytest
import torch

import oracle as O
from paper_2507_22789_b200 import inputs as I

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    assert torch.cuda.is_available()
    from paper_2507_22789_b200 import binding
    return binding


def make(T, D, V, K, seed, tau=1.0):
    H, W = I.make_hw(T, D, V, "bf16", seed, "cuda")
    r = np.random.default_rng(seed)
    y = r.integers(0, V, (T, K)).astype(np.int32)
    y[r.random((T, K)) < 0.1] = -1                      # absent candidates
    if K > 1:
        y[::7, 1] = y[::7, 0]                           # duplicates within a row
    y[0, 0], y[T - 1, K - 1] = 0, V - 1                 # first and last vocab id
    return H, W, y, tau


@pytest.mark.parametrize("T,D,V,K,tau", [(300, 256, 2048 + 40, 3, 1.0), (257, 512, 4096 + 8, 8, 0.7),
                                         (64, 128, 1000, 1, 1.0), (700, 256, 256 * 9, 5, 1.3)])
def test_multi_matches_oracle_per_column(B, T, D, V, K, tau):
    H, W, y, _ = make(T, D, V, K, seed=T + K)
    logp, ent, lse = B.gc_token_logprobs_multi(H, W, torch.from_numpy(y).cuda(), tau)
    torch.cuda.synchronize()
    H64 = H.float().cpu().numpy().astype(np.float64)
    W64 = W.float().cpu().numpy().astype(np.float64)
    lp_any, en_o, ls_o = O.token_logprobs(H64, W64, np.zeros(T, np.int32), None, tau)
    assert np.abs(ent.cpu().numpy() - en_o).max() <= 2e-4
    assert np.abs(lse.cpu().numpy() - ls_o).max() <= 1e-4
    got = logp.cpu().numpy()
    for k in range(K):
        lp_o = O.token_logprobs(H64, W64, y[:, k], None, tau)[0]      # 0 where y < 0
        assert np.abs(got[:, k] - lp_o).max() <= 1e-4, k
        assert np.all(got[y[:, k] < 0, k] == 0.0)
    # K = 1 agrees with the single-target entry point bit for bit where the target is present
    if K == 1:
        lp1, _, _ = B.gc_token_logprobs(H, W, torch.from_numpy(y[:, 0].copy()).cuda(), None, tau)
        ok = y[:, 0] >= 0
        assert np.array_equal(lp1.cpu().numpy()[ok], got[ok, 0])


def test_multi_whole_vocab_sums_to_one(B):
    """All 8 tokens of an 8-token vocabulary as candidates: the probabilities sum to 1."""
    T, D, V = 130, 64, 8
    H, W = I.make_hw(T, D, V, "bf16", 3, "cuda")
    W = (W.float() * 40).to(torch.bfloat16)              # spread the logits
    y = np.tile(np.arange(V, dtype=np.int32), (T, 1))
    logp, ent, lse = B.gc_token_logprobs_multi(H, W, torch.from_numpy(y).cuda())
    p = torch.exp(logp.double()).sum(dim=1)
    assert float((p - 1).abs().max()) <= 1e-5
    # entropy = -sum p ln p over the whole vocabulary
    e = -(torch.exp(logp.double()) * logp.double()).sum(dim=1)
    assert float((e - ent.double()).abs().max()) <= 1e-4


def test_multi_out_of_range_and_errors(B):
    H, W, y, _ = make(64, 128, 512, 2, seed=5)
    y[3, 1] = 512                                        # id >= V: treated as absent
    logp, _, _ = B.gc_token_logprobs_multi(H, W, torch.from_numpy(y).cuda())
    assert float(logp[3, 1]) == 0.0
    with pytest.raises(B.GcoreError):
        B.gc_token_logprobs_multi(H, W, torch.zeros(64, 9, dtype=torch.int32, device="cuda"))
