"""GPU parity of the PPO critic path (NEXT-2) against oracle/critic_oracle.py (fp64) on the same
seeded inputs: value head, GAE, clipped value loss + gradient, value-head backward."""
import numpy as np
import pytest
import torch

from oracle import critic_oracle as CO

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    assert torch.cuda.is_available()
    from paper_2507_22789_b200 import binding
    return binding


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def layout(R, seed, max_len=300):
    r = np.random.default_rng(seed)
    L = r.integers(0, max_len, R)
    L = np.maximum(L, 1)
    if R > 3:
        L[r.integers(0, R, 2)] = 0
        L[1] = 1
        L[2] = 1000                                   # longer than many 32-token chunks
    cu = np.concatenate([[0], np.cumsum(L)]).astype(np.int32)
    T = int(cu[-1])
    mask = (r.random(T) < 0.75).astype(np.uint8)
    for a in cu[:-1][:R // 2]:                        # masked prompt prefixes
        mask[a:a + 7] = 0
    return cu, T, mask


@pytest.mark.parametrize("dtype", [torch.bfloat16, torch.float32])
@pytest.mark.parametrize("T,D", [(1, 8), (333, 264), (2000, 4096), (70, 2048 + 8), (40013, 520)])
def test_value_head_fwd_bwd(B, dtype, T, D):
    # (40013 rows: more 64-row tiles than the backward's 296 persistent row blocks -- each block walks
    # several tiles, as on bench.py's 524288-row stand-in)
    g = torch.Generator(device="cuda").manual_seed(T + D)
    H = torch.randn(T, D, device="cuda", generator=g).to(dtype)
    w = (torch.randn(D, device="cuda", generator=g) / D ** 0.5).to(dtype)
    v = B.gc_value_head_fwd(H, w, 0.3)
    H64, w64 = H.double().cpu().numpy(), w.double().cpu().numpy()
    v_o = CO.value_head(H64, w64, 0.3)
    assert np.abs(v.cpu().numpy() - v_o).max() <= 2e-5 * max(1.0, np.abs(v_o).max())
    gt = torch.randn(T, device="cuda", generator=g) / T
    dH, dw, db = B.gc_value_head_bwd(H, w, gt)
    dH_o, dw_o, db_o = CO.value_head_backward(H64, w64, gt.double().cpu().numpy())
    tol = 4e-3 if dtype == torch.bfloat16 else 1e-6   # dH is rounded to H's dtype
    assert np.abs(dH.double().cpu().numpy() - dH_o).max() <= tol * np.abs(dH_o).max() + 1e-12
    assert np.abs(dw.cpu().numpy() - dw_o).max() <= 1e-5 * np.abs(dw_o).max() + 1e-9
    assert abs(db.item() - db_o) <= 1e-6 + 1e-5 * abs(db_o)
    dH2, dw2, _ = B.gc_value_head_bwd(H, w, gt)
    assert torch.equal(dH, dH2) and torch.equal(dw, dw2)


@pytest.mark.parametrize("R,seed", [(1, 0), (9, 1), (200, 2)])
@pytest.mark.parametrize("use_mask", [False, True])
def test_gae_matches_oracle(B, R, seed, use_mask):
    cu, T, mask = layout(R, seed)
    if T == 0:
        pytest.skip("empty")
    r = np.random.default_rng(seed + 10)
    rew = (r.normal(size=T) * 0.1).astype(np.float32)
    rew[cu[1:][cu[1:] > 0] - 1] += 1.0                # sequence reward on the last token
    val = r.normal(size=T).astype(np.float32)
    m = mask if use_mask else None
    for gamma, lam in ((1.0, 0.95), (0.99, 0.0), (1.0, 1.0)):
        adv, ret = B.gc_gae(dev(rew), dev(val), None if m is None else dev(m), dev(cu), gamma, lam)
        adv_o, ret_o = CO.gae(rew, val, m, cu, gamma, lam)
        scale = max(1.0, np.abs(adv_o).max())
        assert np.abs(adv.cpu().numpy() - adv_o).max() <= 2e-5 * scale
        assert np.abs(ret.cpu().numpy() - ret_o).max() <= 2e-5 * scale
        if m is not None:
            assert np.all(adv.cpu().numpy()[m == 0] == 0)


@pytest.mark.parametrize("T", [1, 1000, 70001, 3_000_001])   # the last: count blocks stride the grid
def test_value_loss_and_grad(B, T):
    r = np.random.default_rng(T)
    v = r.normal(size=T).astype(np.float32)
    vo = (v + 0.3 * r.normal(size=T)).astype(np.float32)
    ret = r.normal(size=T).astype(np.float32)
    mask = (r.random(T) < 0.7).astype(np.uint8)
    for m in (None, mask, np.zeros(T, np.uint8)):
        out3, g = B.gc_value_loss(dev(v), dev(vo), dev(ret), None if m is None else dev(m), 0.2, 0.5)
        loss_o, cf_o, n_o = CO.value_loss(v, vo, ret, m, 0.2)
        o = out3.cpu().numpy()
        assert abs(o[0] - loss_o) <= 1e-6 + 1e-5 * abs(loss_o) and o[2] == n_o
        # the clip decision is taken in fp32 on the GPU and fp64 in the oracle: allow near-ties
        assert abs(o[1] - cf_o) <= 2.0 / max(n_o, 1)
        g_o = CO.value_loss_grad(v, vo, ret, m, 0.2, 0.5)
        e1, e2 = (v.astype(np.float64) - ret) ** 2, (np.clip(v, vo - 0.2, vo + 0.2).astype(np.float64) - ret) ** 2
        near = np.abs(e1 - e2) < 1e-5
        assert np.abs(g.cpu().numpy() - g_o)[~near].max(initial=0) <= 1e-6 * max(1.0, np.abs(g_o).max())


def test_ppo_flow_small(B):
    """values -> GAE -> policy loss with per-token advantages (one 'response' per token) + value
    loss -> value-head backward; every stage against the oracle fed the previous stage's oracle."""
    import oracle as O
    cu, T, mask = layout(12, 5, max_len=120)
    D = 256
    g = torch.Generator(device="cuda").manual_seed(1)
    H = torch.randn(T, D, device="cuda", generator=g).to(torch.bfloat16)
    w = (torch.randn(D, device="cuda", generator=g) / 16).to(torch.bfloat16)
    r = np.random.default_rng(6)
    rew = np.zeros(T, np.float32); rew[cu[1:][cu[1:] > 0] - 1] = r.random(int((cu[1:] > 0).sum())).astype(np.float32)
    v = B.gc_value_head_fwd(H, w)
    adv, ret = B.gc_gae(dev(rew), v, dev(mask), dev(cu), 1.0, 0.95)
    v_o = CO.value_head(H.double().cpu().numpy(), w.double().cpu().numpy(), 0.0)
    adv_o, ret_o = CO.gae(rew, v_o, mask, cu, 1.0, 0.95)
    assert np.abs(adv.cpu().numpy() - adv_o).max() <= 1e-4
    logp = -r.random(T).astype(np.float32)
    old = (logp + 0.05 * r.normal(size=T)).astype(np.float32)
    cu_tok = np.arange(T + 1, dtype=np.int32)
    y = np.zeros(T, np.int32)
    out5, gl = B.gc_grpo_token_loss(dev(logp), dev(old), None, dev(y), dev(mask), dev(cu_tok), adv,
                                    beta=0.0)
    exp = O.grpo_loss(logp.astype(np.float64), old, None, mask != 0, adv.cpu().numpy(), cu_tok, 0.2, 0.2, 0.0)
    assert abs(out5[0].item() - exp["loss"]) <= 1e-6 + 1e-5 * abs(exp["loss"])
