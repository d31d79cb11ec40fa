"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times.

The oracle cannot materialise [T,V] here, so (SURVEY.md sec 8(c) "parity protocol"):
  (iii) rows are independent: logp / entropy / lse and dH are checked on sampled rows (tile
        boundary rows, sequence ends, masked rows, random rows) that the oracle computes from
        H[t,:], W and the mask alone;
  (iv)  the loss scalars and g_t at full T: the oracle's grpo_loss / grpo_loss_grad_logp run on the
        GPU's fp32 logp (isolates the loss kernels; logp itself is verified in (iii));
  (v)   dW at full T: >= 64 sampled vocab rows (rows that occur as targets, rows that never do,
        the edges of 256-row tiles, of the 128-row CTA halves and of the 32-row store slabs, the
        last rows of V) recomputed in fp64 by oracle.lm_head_backward_wrows from H, W, y, the
        oracle's g_t and the GPU's lse -- the hybrid check of the survey, legitimate because lse is
        verified in (iii) -- compared per row (rel. Frobenius 5e-3) and per element; whole rows
        cover every D band of the dW schedule (n_band < D/256 at these sizes).  Plus properties
        that hold at any size: every column sum of dW is 0, <dH,H> = <dW,W>, unscored dH rows are
        0, and the north_star invariant loss = -sum(mA)/sum(m) when policy = old and beta = 0.
No oracle input or expected value is produced by the CUDA path except where (iv)/(v) say so
(GPU logp / lse fed to the oracle's formulas): old/ref are synthesised by tests.harness.synth_policy_logp
(plain torch, harness side).
"""
import gc

import numpy as np
import psutil
import pytest
import torch

import oracle as O
from paper_2507_22789_b200 import inputs as I
from tests.harness import DeviceBatch
from tests.helpers import ELEM_BF16, elem_excess

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    assert torch.cuda.is_available()
    from paper_2507_22789_b200 import binding
    return binding


def sample_rows(T, cu, mask, n_random, seed):
    r = np.random.default_rng(seed)
    rows = {0, 1, 127, 128, 129, 255, 256, 257, 511, 512, T - 257, T - 256, T - 129, T - 128, T - 2,
            T - 1}
    for c in cu[1:-1][:6]:
        rows.update({int(c) - 1, int(c)})
    rows.update(int(x) for x in r.integers(0, T, n_random))
    un = np.nonzero(mask == 0)[0]
    if len(un):
        rows.update(int(x) for x in r.choice(un, min(8, len(un)), replace=False))
    return np.array(sorted(x for x in rows if 0 <= x < T), dtype=np.int64)


def sample_vocab_rows(V, y_scored, n_random, seed):
    """Vocab rows of dW to check: edges of 256-row tiles (first, middle, last tiles), of the
    128-row halves a CTA pair splits a tile into, of the 32-row slabs one TMA store covers, the
    last rows of V, rows that occur as targets and rows that never do."""
    r = np.random.default_rng(seed + 99)
    nt = -(-V // 256)
    rows = set()
    for t in {0, 1, nt // 2, nt - 2, nt - 1}:
        for off in (0, 31, 32, 127, 128, 255):
            rows.add(t * 256 + off)
    rows.update({V - 1, V - 2, V - 33})
    seen = np.unique(y_scored)
    rows.update(int(x) for x in r.choice(seen, min(n_random, len(seen)), replace=False))
    never = np.setdiff1d(np.arange(V), seen)
    if len(never):
        rows.update(int(x) for x in r.choice(never, min(n_random, len(never)), replace=False))
    return np.array(sorted(x for x in rows if 0 <= x < V), dtype=np.int64)


def check_full(B, b, n_random=64, seed=0):
    w = b.w
    need = w.V * w.D * 8 * 2.5
    if psutil.virtual_memory().available < need:
        pytest.skip(f"host RAM too small for the fp64 widening of W ({need / 1e9:.0f} GB)")
    lay = b.lay
    T = b.T
    adv, keep = B.gc_grpo_advantages(b.rewards, b.go, 1e-6, False, False)
    adv_ref, _ = O.grpo_advantages(b.rewards.cpu().numpy(), lay.group_offsets, 1e-6)
    assert np.allclose(adv.cpu().numpy(), adv_ref.astype(np.float32), rtol=3e-7, atol=1e-9)

    if w.backward:
        f = B.gc_grpo_loss_fwd(b.H, b.W, b.y, b.mask, w.tau, b.cu, adv, b.old, b.ref, w.clip_lo,
                               w.clip_hi, w.beta)
        dH, dW = B.gc_grpo_loss_bwd(b.H, b.W, b.y, b.mask, w.tau, b.cu, adv, b.old, b.ref,
                                    f["logp"], f["lse"], w.clip_lo, w.clip_hi, w.beta,
                                    dH=b.dH, dW=b.dW)
        logp, ent, lse = f["logp"], f["entropy"], f["lse"]
    else:
        logp, ent, lse = B.gc_token_logprobs(b.H, b.W, b.y, b.mask, w.tau)
    torch.cuda.synchronize()

    S = sample_rows(T, lay.cu_seqlens, lay.mask, n_random, seed)
    St = torch.from_numpy(S).cuda()
    H64 = b.H[St].float().cpu().numpy().astype(np.float64)
    W64 = b.W.float().cpu().numpy().astype(np.float64)
    yS = b.y[St].cpu().numpy()
    mS = lay.mask[S]
    lp_o, en_o, ls_o = O.token_logprobs(H64, W64, yS, mS, w.tau)
    d_lp = np.abs(logp[St].cpu().numpy() - lp_o).max()
    d_en = np.abs(ent[St].cpu().numpy() - en_o).max()
    d_ls = np.abs(lse[St].cpu().numpy() - ls_o).max()
    print(f"{w.name}: {len(S)} sampled rows |dlogp|={d_lp:.2e} |dentropy|={d_en:.2e} |dlse|={d_ls:.2e}")
    assert d_lp <= 1e-4 and d_en <= 2e-4 and d_ls <= 1e-4
    scored_full = (lay.mask != 0) & (b.y.cpu().numpy() >= 0)
    zero_rows = torch.from_numpy(np.nonzero(~scored_full)[0]).cuda()
    assert float(logp[zero_rows].abs().sum()) == 0.0 and float(lse[zero_rows].abs().sum()) == 0.0
    if not w.backward:
        return

    # g_t at the sampled rows from the oracle's own logp (token-mean: depends on row t and sum m)
    old = b.old.cpu().numpy()
    ref = b.ref.cpu().numpy()
    logp_full = old.astype(np.float64).copy()
    logp_full[S] = lp_o
    g_full = O.grpo_loss_grad_logp(logp_full, old, ref, scored_full, adv_ref, lay.cu_seqlens,
                                   w.clip_lo, w.clip_hi, w.beta)
    dH_o, _ = O.lm_head_backward(H64, W64, yS, mS, w.tau, g_full[S])
    dH_g = dH[St].float().cpu().numpy()
    sc = (mS != 0) & (yS >= 0)
    rel = np.linalg.norm(dH_g[sc] - dH_o[sc]) / np.linalg.norm(dH_o[sc])
    print(f"{w.name}: relF(dH sampled rows)={rel:.2e}")
    assert rel <= 5e-3
    assert np.all(dH_g[~sc] == 0.0)
    assert elem_excess(dH_g[sc], dH_o[sc], **ELEM_BF16) <= 1.0, elem_excess(dH_g[sc], dH_o[sc], **ELEM_BF16)
    del W64
    gc.collect()

    # (iv) loss scalars and g_t at full T: the oracle's loss on the GPU's fp32 logp
    logp_gpu = logp.cpu().numpy()
    res = O.grpo_loss(logp_gpu, old, ref, scored_full, adv_ref, lay.cu_seqlens, w.clip_lo, w.clip_hi,
                      w.beta)
    o5 = f["out5"].cpu().numpy().astype(np.float64)
    print(f"{w.name}: loss gpu={o5[0]:.8e} oracle(on gpu logp)={res['loss']:.8e} "
          f"kl={o5[2]:.6e}/{res['kl_mean']:.6e} clip={o5[3]:.3e}/{res['clip_frac']:.3e}")
    assert o5[4] == res["n_scored"] == scored_full.sum()
    assert abs(o5[0] - res["loss"]) <= 1e-5 * max(abs(res["loss"]), 1e-3)
    assert abs(o5[1] - res["pg_loss"]) <= 1e-5 * max(abs(res["pg_loss"]), 1e-3)
    assert abs(o5[2] - res["kl_mean"]) <= 1e-5 * max(abs(res["kl_mean"]), 1e-3)
    assert abs(o5[3] - res["clip_frac"]) <= 2.0 / max(res["n_scored"], 1)
    g_o = O.grpo_loss_grad_logp(logp_gpu, old, ref, scored_full, adv_ref, lay.cu_seqlens,
                                w.clip_lo, w.clip_hi, w.beta)
    _, g_gpu = B.gc_grpo_token_loss(logp, b.old, b.ref, b.y, b.mask, b.cu, adv, w.clip_lo,
                                    w.clip_hi, w.beta)
    g_gpu = g_gpu.cpu().numpy().astype(np.float64)
    rho = np.exp(logp_gpu.astype(np.float64) - old)
    near = (np.abs(rho - (1 + w.clip_hi)) < 1e-5) | (np.abs(rho - (1 - w.clip_lo)) < 1e-5)
    assert np.all(g_gpu[~scored_full] == 0.0)
    assert np.allclose(g_gpu[~near], g_o[~near], rtol=2e-5, atol=2e-6 * np.abs(g_o).max())
    assert near.sum() < 1e-3 * T + 2

    # (v) sampled vocab rows of dW, in fp64 from H, W, y, the oracle's g and the GPU's lse
    Vs = sample_vocab_rows(w.V, b.y.cpu().numpy()[scored_full], 24, seed)
    Wr = b.W[torch.from_numpy(Vs).cuda()].float().cpu().numpy().astype(np.float64)
    lse_gpu = lse.cpu().numpy().astype(np.float64)
    y_np = b.y.cpu().numpy()
    dW_o = np.zeros((len(Vs), w.D))
    for a in range(0, T, 8192):
        e = min(T, a + 8192)
        if not scored_full[a:e].any():
            continue
        Hs = b.H[a:e].float().cpu().numpy().astype(np.float64)
        dW_o += O.lm_head_backward_wrows(Hs, Wr, Vs, y_np[a:e], lay.mask[a:e], w.tau, g_o[a:e],
                                         lse_gpu[a:e])
    dW_g = dW[torch.from_numpy(Vs).cuda()].cpu().numpy().astype(np.float64)
    row_rel = np.linalg.norm(dW_g - dW_o, axis=1) / np.maximum(np.linalg.norm(dW_o, axis=1), 1e-300)
    hit = np.isin(Vs, y_np[scored_full])
    exc = elem_excess(dW_g, dW_o, **ELEM_BF16)
    print(f"{w.name}: {len(Vs)} sampled dW rows ({hit.sum()} occur as targets): max row relF="
          f"{row_rel.max():.2e}, elem excess={exc:.2f}")
    assert hit.sum() >= 8 and (~hit).sum() >= 8
    assert row_rel.max() <= 5e-3
    assert exc <= 1.0
    del Wr, dW_o, dW_g
    gc.collect()
    # properties at full size
    assert float(dH[zero_rows].float().abs().sum()) == 0.0
    colsum = dW.sum(dim=0, dtype=torch.float64).abs().max().item()
    dw_scale = dW.abs().sum(dim=0, dtype=torch.float64).max().item()
    assert colsum <= 2e-3 * dw_scale, (colsum, dw_scale)         # bf16 dS rounding does not cancel exactly
    e1 = (dH.double() * b.H.double()).sum().item()
    e2 = sum((dW[a:a + 16384].double() * b.W[a:a + 16384].double()).sum().item()
             for a in range(0, w.V, 16384))
    print(f"{w.name}: <dH,H>={e1:.6e} <dW,W>={e2:.6e} colsum={colsum:.2e}/{dw_scale:.2e}")
    assert abs(e1 - e2) <= 2e-2 * max(abs(e1), abs(e2), 1e-4)
    # north_star invariant at full size: policy = old, beta = 0 -> loss = -sum(m A)/sum(m)
    out5, _ = B.gc_grpo_token_loss(logp, logp, None, b.y, b.mask, b.cu, adv, beta=0.0,
                                   want_grad=False)
    A_tok = adv_ref[O.token_to_response(lay.cu_seqlens, T)]
    expect = -(A_tok * scored_full).sum() / max(scored_full.sum(), 1)
    assert abs(out5[0].item() - expect) <= 1e-6 + 1e-5 * abs(expect)
    assert out5[4].item() == scored_full.sum()
    # reruns are bit-identical at full size too: which CTA pair computes a tile (dynamic schedule)
    # and the L2-side dW accumulation (one TMA reduce-add per element per chunk, stream-ordered)
    # must not enter the result
    dH1, dW1 = dH.clone(), dW.clone()
    f2 = B.gc_grpo_loss_fwd(b.H, b.W, b.y, b.mask, w.tau, b.cu, adv, b.old, b.ref, w.clip_lo,
                            w.clip_hi, w.beta)
    B.gc_grpo_loss_bwd(b.H, b.W, b.y, b.mask, w.tau, b.cu, adv, b.old, b.ref, f2["logp"], f2["lse"],
                       w.clip_lo, w.clip_hi, w.beta, dH=b.dH, dW=b.dW)
    assert torch.equal(f2["logp"], logp) and torch.equal(f2["entropy"], ent)
    assert torch.equal(b.dH, dH1) and torch.equal(b.dW, dW1)
    # bf16 dW output at full size (fp32 staging in the workspace, cast kernel striding its grid):
    # equals the fp32 dW rounded once, bit for bit
    if w.V * w.D <= 6e8:
        _, dW16 = B.gc_grpo_loss_bwd(b.H, b.W, b.y, b.mask, w.tau, b.cu, adv, b.old, b.ref, f2["logp"],
                                     f2["lse"], w.clip_lo, w.clip_hi, w.beta, dH=b.dH,
                                     dW_dtype=torch.bfloat16)
        assert dW16.dtype == torch.bfloat16 and torch.equal(dW16, dW1.to(torch.bfloat16))
        assert torch.equal(b.dH, dH1)
        del dW16


@pytest.mark.parametrize("cfg", [1, 2, 4])
def test_full_size_config(B, cfg):
    b = DeviceBatch(I.CONFIGS[cfg], seed=0, device=torch.device("cuda", 0))
    try:
        check_full(B, b)
    finally:
        del b
        gc.collect()
        torch.cuda.empty_cache()


def test_full_size_config3_dynamic_sampling(B):
    """cfg3: lognormal varlen batch; constant groups dropped before the advantage step, kept
    groups repacked; the mask-instead-of-repack route gives the same loss."""
    w = I.CONFIGS[3]
    dev = torch.device("cuda", 0)
    full = DeviceBatch(w, seed=0, device=dev)
    assert full.T == 281898                                      # DESIGN.md sec 4 / SURVEY appendix A
    adv_all, keep = B.gc_grpo_advantages(full.rewards, full.go, 1e-6, False, True)
    keep_np = keep.cpu().numpy()
    assert np.array_equal(keep_np, O.group_filter(full.rewards.cpu().numpy(), full.lay.group_offsets))
    assert keep_np.sum() == 12
    resp_idx, tok_idx, lay2 = I.drop_groups(full.lay, keep_np, w.group_size)
    ti = torch.from_numpy(tok_idx).to(dev)
    # route A: repack the kept groups
    kept = DeviceBatch.__new__(DeviceBatch)
    kept.w, kept.lay, kept.T = w, lay2, lay2.T
    kept.H, kept.W, kept.y = full.H[ti].contiguous(), full.W, full.y[ti].contiguous()
    kept.mask = None
    kept.rewards = full.rewards[torch.from_numpy(resp_idx).to(dev)].contiguous()
    kept.go = torch.from_numpy(lay2.group_offsets).to(dev)
    kept.cu = torch.from_numpy(lay2.cu_seqlens).to(dev)
    kept.old, kept.ref = full.old[ti].contiguous(), full.ref[ti].contiguous()
    kept.dH = torch.empty(lay2.T, w.D, dtype=torch.bfloat16, device=dev)
    kept.dW = torch.empty(w.V, w.D, dtype=torch.float32, device=dev)
    # route B first (cheap): same loss with the dropped groups masked instead of removed
    mask_np = np.zeros(full.T, np.uint8)
    mask_np[tok_idx] = 1
    fB = B.gc_grpo_loss_fwd(full.H, full.W, full.y, torch.from_numpy(mask_np).to(dev), w.tau,
                            full.cu, adv_all, full.old, full.ref, w.clip_lo, w.clip_hi, w.beta)
    lossB = fB["out5"].cpu().numpy()
    del full.dH, full.dW
    check_full(B, kept, n_random=48)
    advA, _ = B.gc_grpo_advantages(kept.rewards, kept.go, 1e-6, False, False)
    fA = B.gc_grpo_loss_fwd(kept.H, kept.W, kept.y, None, w.tau, kept.cu, advA, kept.old, kept.ref,
                            w.clip_lo, w.clip_hi, w.beta)
    lossA = fA["out5"].cpu().numpy()
    assert lossA[4] == lossB[4] == lay2.T
    assert np.allclose(lossA[:4], lossB[:4], rtol=1e-5, atol=1e-7)
    # a row's result does not depend on the packing (only the split-V combine order differs)
    assert float((fA["logp"] - fB["logp"][ti]).abs().max()) <= 2e-5


def test_host_training_step_at_full_size_matches_the_device_path(B):
    """gc_grpo_step_host at the size bench.py's e2e figure times (configs[2]: 32768 x 4096 x 128256,
    75 % scored): every output against the device-resident calls on the same inputs, which
    check_full verifies against the oracle.  The host path scores H band by band (its own split-V
    plans), so log-probs agree to rounding, not bit for bit; out5, dH [T, D] and dW [V, D] follow."""
    w = I.CONFIGS[2]
    dev = torch.device("cuda", 0)
    b = DeviceBatch(w, seed=0, device=dev)
    adv, _ = B.gc_grpo_advantages(b.rewards, b.go, 1e-6, False, False)
    f = B.gc_grpo_loss_fwd(b.H, b.W, b.y, b.mask, w.tau, b.cu, adv, b.old, b.ref, w.clip_lo, w.clip_hi,
                           w.beta)
    dH_d, dW_d = B.gc_grpo_loss_bwd(b.H, b.W, b.y, b.mask, w.tau, b.cu, adv, b.old, b.ref, f["logp"],
                                    f["lse"], w.clip_lo, w.clip_hi, w.beta, fwd_state=f["state"])
    pin = lambda t: t.cpu().pin_memory()
    dW_h = torch.full((w.V, w.D), 3.0, dtype=torch.float32, device=dev)
    lp_h = torch.empty(b.T, dtype=torch.float32).pin_memory()
    out5_h, dH_h = B.gc_grpo_step_host(pin(b.H), b.W, pin(b.y), pin(b.mask), w.tau, pin(b.cu),
                                       pin(b.rewards), pin(b.go), pin(b.old), pin(b.ref), dW_h,
                                       clip_lo=w.clip_lo, clip_hi=w.clip_hi, beta=w.beta,
                                       logp_host=lp_h)
    torch.cuda.synchronize()
    o_h, o_d = out5_h.numpy().astype(np.float64), f["out5"].cpu().numpy().astype(np.float64)
    assert o_h[4] == o_d[4] == b.n_scored
    assert np.allclose(o_h[:3], o_d[:3], rtol=2e-5, atol=1e-7)
    assert abs(o_h[3] - o_d[3]) <= 4.0 / b.n_scored          # a few near-ties of the clip bound
    assert float((lp_h.to(dev) - f["logp"]).abs().max()) <= 2e-5
    scored = (b.lay.mask != 0) & (b.y.cpu().numpy() >= 0)
    dH_h = dH_h.to(dev).float()
    assert float(dH_h[torch.from_numpy(~scored).to(dev)].abs().sum()) == 0.0
    rel = lambda a, r: float((a - r).norm() / r.norm())
    # near-ties of the clip bound (not de-tied against the banded log-probs) may flip a branch on a
    # handful of rows; everything else differs by bf16 rounding of dH at most
    row_err = (dH_h - dH_d.float()).norm(dim=1) / dH_d.float().norm(dim=1).clamp_min(1e-30)
    assert int((row_err > 1e-2).sum()) <= 4
    assert rel(dH_h, dH_d.float()) <= 2e-3
    assert rel(dW_h, dW_d) <= 2e-3
