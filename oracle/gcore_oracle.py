"""Plain, slow, fp64 CPU oracle of the RLHF scoring hot path.  TEST INFRASTRUCTURE.

What it is
----------
The stage-3 / stage-4 computation of the 4-stage RLHF workflow (sec 2.2:
"the policy and reference policy computes their reference log probabilities"; "The actor ...
trained on the batch ... and the loss function"), for the GRPO algorithm the paper names as
typical (sec 2.3), with the dynamic-sampling group filter of PAPER.md:150
(sec 3.2).  The paper prints no formula; the arithmetic is the one stated in
BASELINE.json:north_star and restated step by step in SURVEY.md sec 8(c) steps 1-9.  Each
function below cites the step it follows.  Readings of silent points are DESIGN.md sec 3.

Rules it obeys
--------------
* numpy float64 everywhere; inputs are widened exactly (bf16/fp32 values are exactly
  representable in fp64), so the oracle consumes the very operand values the GPU sees.
* No blocking, fusion or reordering: logits are materialised as a dense [T, V] matrix with one
  library matmul, softmax is the textbook max-shifted definition, the backward is the chain
  rule written out.  Use it only at sizes where [T, V] fp64 fits in host memory.
* It shares no code with ``paper_2507_22789_b200`` and never imports it.
* Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline / reference legs
  may import it.

Pins (tests/test_oracle_pins.py, run with ``-m "not gpu"``)
-----------------------------------------------------------
token_logprobs      brute-force python loops on tiny V; closed forms (H=0 -> -ln V / ln V);
                    hand-derived values for a 2x4 example (tests/golden/tiny_softmax.txt);
                    sum_v exp(logp_v)=1; shift / temperature / permutation invariances;
                    scipy.special.log_softmax and scipy.stats.entropy as library routines.
grpo_advantages     hand-derived values (tests/golden/advantages.txt); zero mean / unit std;
                    affine invariance; constant group -> 0.
grpo_loss           hand-derived per-token values (tests/golden/loss_tokens.txt);
                    logp=old & beta=0 -> -sum(mA)/sum(m); logp=ref -> kl=0; k3>=0.
grpo_loss_grad_logp central finite differences of grpo_loss; hand-derived values.
lm_head_backward    central finite differences of the whole forward; row sums of dz = 0;
                    column sums of dW = 0; <dH,H> = <dW,W>; textbook cross-entropy gradient
                    in the special case logp=old=ref.
lm_head_backward_wrows  equality with lm_head_backward's rows (all rows, target rows, never-
                    target rows, token slices summed); central finite differences w.r.t. W[v,d].
Nothing here is "parity unpinned".
"""
from __future__ import annotations

import numpy as np

AGG_TOKEN_MEAN = 0
AGG_SEQ_MEAN = 1


def _f64(x):
    return np.ascontiguousarray(np.asarray(x, dtype=np.float64))


def _scored(targets, mask):
    """A token is scored iff mask==1 (or mask is None) and target >= 0.  SURVEY 8(b) conventions."""
    targets = np.asarray(targets)
    s = targets >= 0
    if mask is not None:
        s = s & (np.asarray(mask) != 0)
    return s


# ----------------------------------------------------------------------------------------------
# step 1: z[t,v] = (sum_d H[t,d] W[v,d]) / tau          (north_star: "fused LM-head contraction
#         H.W^T over the vocabulary"; tau from BASELINE.json configs[4])
# ----------------------------------------------------------------------------------------------
def logits(H, W, tau=1.0):
    H = _f64(H)
    W = _f64(W)
    return (H @ W.T) / float(tau)


# ----------------------------------------------------------------------------------------------
# steps 2-3: lse[t] = M + ln sum_v exp(z-M), M = max_v z;  logp[t] = z[t,y_t] - lse[t];
#            entropy[t] = -sum_v p ln p, p = exp(z - lse)       (north_star: "online log-softmax,
#            then a gather of the sampled token's log-prob and the per-token entropy")
# Outputs at unscored rows are exactly 0 (reading 11).
# ----------------------------------------------------------------------------------------------
def token_logprobs(H, W, targets, mask=None, tau=1.0):
    z = logits(H, W, tau)
    T, V = z.shape
    targets = np.asarray(targets, dtype=np.int64)
    scored = _scored(targets, mask)
    M = z.max(axis=1)
    lse = M + np.log(np.exp(z - M[:, None]).sum(axis=1))
    logp_all = z - lse[:, None]
    p = np.exp(logp_all)
    entropy = -(p * logp_all).sum(axis=1)
    y = np.where(scored, targets, 0)
    logp = logp_all[np.arange(T), y]
    zero = np.zeros(T)
    return (np.where(scored, logp, zero), np.where(scored, entropy, zero),
            np.where(scored, lse, zero))


def token_logprobs_row(h, W64, y, tau=1.0):
    """Steps 1-3 for ONE token (rows are independent): returns (logp, entropy, lse).

    ``W64`` must already be float64 (so that a caller checking many sampled rows of a large
    batch widens W once).  Used for sampled-row parity at sizes where [T,V] does not fit.
    """
    z = (W64 @ _f64(h)) / float(tau)
    M = z.max()
    lse = M + np.log(np.exp(z - M).sum())
    lp = z - lse
    p = np.exp(lp)
    return float(lp[int(y)]), float(-(p * lp).sum()), float(lse)


# ----------------------------------------------------------------------------------------------
# step 4: keep[g] = 0 iff all rewards of group g are equal (exact compare)
#         (sec 3.2: "filter out prompts with the accuracy equal to 1 and 0")
# ----------------------------------------------------------------------------------------------
def group_filter(rewards, group_offsets):
    rewards = np.asarray(rewards)
    group_offsets = np.asarray(group_offsets, dtype=np.int64)
    G = len(group_offsets) - 1
    keep = np.zeros(G, dtype=np.uint8)
    for g in range(G):
        r = rewards[group_offsets[g]:group_offsets[g + 1]]
        keep[g] = 0 if (len(r) == 0 or np.all(r == r[0])) else 1
    return keep


# ----------------------------------------------------------------------------------------------
# step 5: A_i = (r_i - mu_g) / (sigma_g + eps), mu_g, sigma_g over the group's responses
#         (north_star: "GRPO group-normalised advantages").  Reading 2: population std by
#         default, sample std if unbiased_std.  Reading 3: a dropped group gets A = 0.
# ----------------------------------------------------------------------------------------------
def grpo_advantages(rewards, group_offsets, eps=1e-6, unbiased_std=False,
                    drop_constant_groups=False):
    r_all = _f64(rewards)
    group_offsets = np.asarray(group_offsets, dtype=np.int64)
    G = len(group_offsets) - 1
    adv = np.zeros_like(r_all)
    keep = group_filter(rewards, group_offsets)
    for g in range(G):
        a, b = int(group_offsets[g]), int(group_offsets[g + 1])
        n = b - a
        if n == 0:
            continue
        if drop_constant_groups and not keep[g]:
            adv[a:b] = 0.0
            continue
        r = r_all[a:b]
        mu = r.sum() / n
        ss = ((r - mu) ** 2).sum()
        if unbiased_std:
            sigma = np.sqrt(ss / (n - 1)) if n > 1 else 0.0
        else:
            sigma = np.sqrt(ss / n)
        adv[a:b] = (r - mu) / (sigma + eps)
    if not drop_constant_groups:
        keep = np.ones(G, dtype=np.uint8)
    return adv, keep


def token_to_response(cu_seqlens, T):
    """resp[t] = r with cu_seqlens[r] <= t < cu_seqlens[r+1]; -1 if no such r.  Brute force."""
    cu = np.asarray(cu_seqlens, dtype=np.int64)
    resp = np.full(T, -1, dtype=np.int64)
    for r in range(len(cu) - 1):
        resp[cu[r]:cu[r + 1]] = r
    return resp


def _token_weights(scored, resp, R, agg):
    """Per-token weight w_t with loss = sum_t w_t * l_t  (steps 7-8, reading 4).

    token-mean: w_t = m_t / max(sum m, 1).
    seq-mean:   w_t = m_t / (R_kept * max(sum_{t' in r} m_t', 1)), R_kept = #responses with a
                scored token (max(.,1)).
    """
    m = scored.astype(np.float64)
    if agg == AGG_TOKEN_MEAN:
        return m / max(m.sum(), 1.0)
    cnt = np.zeros(R)
    for t in range(len(m)):
        if scored[t] and resp[t] >= 0:
            cnt[resp[t]] += 1.0
    r_kept = max(float((cnt > 0).sum()), 1.0)
    w = np.zeros_like(m)
    for t in range(len(m)):
        if scored[t] and resp[t] >= 0:
            w[t] = 1.0 / (r_kept * max(cnt[resp[t]], 1.0))
    return w


# ----------------------------------------------------------------------------------------------
# steps 6-7: rho = exp(logp-old); s = min(rho A, clip(rho,1-eps_lo,1+eps_hi) A);
#            d = ref - logp; k3 = exp(d) - d - 1; l = -s + beta k3;
#            loss = sum_t m_t l_t / max(sum m, 1)
#            (north_star: "clipped-ratio policy loss with a k3 KL penalty against the reference")
# ----------------------------------------------------------------------------------------------
def _per_token(logp, old, ref, adv_t, clip_lo, clip_hi, beta):
    rho = np.exp(logp - old)
    clipped = np.clip(rho, 1.0 - clip_lo, 1.0 + clip_hi)
    s1 = rho * adv_t
    s2 = clipped * adv_t
    unclipped = s1 <= s2                 # ties count as unclipped (reading 7)
    s = np.minimum(s1, s2)
    if ref is None:
        d = np.zeros_like(logp)
    else:
        d = ref - logp
    k3 = np.exp(d) - d - 1.0
    return rho, s, unclipped, d, k3


def grpo_loss(logp, old_logp, ref_logp, scored, adv, cu_seqlens,
              clip_lo=0.2, clip_hi=0.2, beta=0.04, agg=AGG_TOKEN_MEAN):
    """Returns dict(loss, pg_loss, kl_mean, clip_frac, n_scored, per_token).

    ``scored`` is the boolean token selector (mask & target>=0).  pg_loss and kl_mean are
    aggregated with the same weights as loss, so loss = pg_loss + beta*kl_mean; clip_frac is
    the fraction of scored tokens on the clipped branch.
    """
    logp = _f64(logp)
    old = _f64(old_logp)
    ref = None if ref_logp is None else _f64(ref_logp)
    adv = _f64(adv)
    scored = np.asarray(scored, dtype=bool)
    T = len(logp)
    R = len(cu_seqlens) - 1
    resp = token_to_response(cu_seqlens, T)
    scored = scored & (resp >= 0)
    adv_t = np.where(resp >= 0, adv[np.maximum(resp, 0)], 0.0)
    rho, s, unclipped, d, k3 = _per_token(logp, old, ref, adv_t, clip_lo, clip_hi, beta)
    w = _token_weights(scored, resp, R, agg)
    l = -s + beta * k3
    n = float(scored.sum())
    return dict(
        loss=float((w * l).sum()),
        pg_loss=float((w * (-s)).sum()),
        kl_mean=float((w * k3).sum()),
        clip_frac=float((scored & ~unclipped).sum() / max(n, 1.0)),
        n_scored=n,
        per_token=np.where(scored, l, 0.0),
    )


# ----------------------------------------------------------------------------------------------
# step 8: g_t = d loss / d logp_t = grad_loss * w_t * (-u_t rho A + beta (1 - exp(d)))
# ----------------------------------------------------------------------------------------------
def grpo_loss_grad_logp(logp, old_logp, ref_logp, scored, adv, cu_seqlens,
                        clip_lo=0.2, clip_hi=0.2, beta=0.04, agg=AGG_TOKEN_MEAN,
                        grad_loss=1.0):
    logp = _f64(logp)
    old = _f64(old_logp)
    ref = None if ref_logp is None else _f64(ref_logp)
    adv = _f64(adv)
    scored = np.asarray(scored, dtype=bool)
    T = len(logp)
    R = len(cu_seqlens) - 1
    resp = token_to_response(cu_seqlens, T)
    scored = scored & (resp >= 0)
    adv_t = np.where(resp >= 0, adv[np.maximum(resp, 0)], 0.0)
    rho, s, unclipped, d, k3 = _per_token(logp, old, ref, adv_t, clip_lo, clip_hi, beta)
    w = _token_weights(scored, resp, R, agg)
    dl = -np.where(unclipped, rho * adv_t, 0.0) + beta * (1.0 - np.exp(d))
    return grad_loss * w * dl


# ----------------------------------------------------------------------------------------------
# step 9: dz[t,v] = g_t (1[v=y_t] - p[t,v]);  dH[t,:] = (1/tau) sum_v dz[t,v] W[v,:];
#         dW[v,:] = (1/tau) sum_t dz[t,v] H[t,:]      (north_star: "produce dH and dW")
# ----------------------------------------------------------------------------------------------
def lm_head_backward(H, W, targets, mask, tau, g):
    H = _f64(H)
    W = _f64(W)
    g = _f64(g)
    z = (H @ W.T) / float(tau)
    T, V = z.shape
    targets = np.asarray(targets, dtype=np.int64)
    scored = _scored(targets, mask)
    M = z.max(axis=1, keepdims=True)
    lse = M + np.log(np.exp(z - M).sum(axis=1, keepdims=True))
    p = np.exp(z - lse)
    onehot = np.zeros_like(z)
    rows = np.nonzero(scored)[0]
    onehot[rows, targets[rows]] = 1.0
    gs = np.where(scored, g, 0.0)
    dz = gs[:, None] * (onehot - p)
    dH = (dz @ W) / float(tau)
    dW = (dz.T @ H) / float(tau)
    return dH, dW


def lm_head_backward_row(h, W64, y, tau, g_t):
    """dH[t,:] for ONE token (step 9 restricted to a row); W64 already float64."""
    z = (W64 @ _f64(h)) / float(tau)
    M = z.max()
    lse = M + np.log(np.exp(z - M).sum())
    p = np.exp(z - lse)
    dz = -g_t * p
    dz[int(y)] += g_t
    return (dz @ W64) / float(tau)


def lm_head_backward_wrows(H, W_rows, vocab_ids, targets, mask, tau, g, lse):
    """dW[v,:] for the vocab rows v in ``vocab_ids`` only (step 9 restricted to rows of dW):
        dW[v,:] = (1/tau) sum_t g_t (1[v = y_t] - exp(z[t,v] - lse[t])) H[t,:].
    A vocab row needs only the column z[:,v] = H W[v,:]^T / tau and the per-token lse, so this is
    the dense backward's definition with the other columns left out -- no other change.
    ``W_rows`` = W[vocab_ids] ([n, D]); ``lse`` [T] is the log-sum-exp over the FULL vocabulary
    (from token_logprobs, or -- in the hybrid full-size check of SURVEY.md sec 8(c) protocol (v) --
    the GPU's lse, itself verified on sampled rows).  dW is a sum over tokens, so a caller may
    sum this function over token slices.  Pinned against lm_head_backward's rows and by finite
    differences (tests/test_oracle_pins.py)."""
    H = _f64(H)
    Wr = _f64(W_rows)
    g = _f64(g)
    lse = _f64(lse)
    vocab_ids = np.asarray(vocab_ids, dtype=np.int64)
    targets = np.asarray(targets, dtype=np.int64)
    scored = _scored(targets, mask)
    z = (H @ Wr.T) / float(tau)                      # [T, n] columns of the logits
    p = np.exp(z - lse[:, None])
    onehot = (targets[:, None] == vocab_ids[None, :]) & scored[:, None]
    gs = np.where(scored, g, 0.0)
    dz = gs[:, None] * (onehot.astype(np.float64) - p)
    dz[~scored] = 0.0                                # lse is 0 at unscored rows: p is garbage there
    return (dz.T @ H) / float(tau)


def grpo_forward_backward(H, W, targets, mask, tau, cu_seqlens, adv, old_logp, ref_logp,
                          clip_lo=0.2, clip_hi=0.2, beta=0.04, agg=AGG_TOKEN_MEAN,
                          grad_loss=1.0, need_grads=True):
    """Steps 1-9 chained: the whole hot path after the advantages.  Returns a dict."""
    logp, entropy, lse = token_logprobs(H, W, targets, mask, tau)
    scored = _scored(targets, mask)
    out = grpo_loss(logp, old_logp, ref_logp, scored, adv, cu_seqlens,
                    clip_lo, clip_hi, beta, agg)
    out.update(logp=logp, entropy=entropy, lse=lse)
    if need_grads:
        g = grpo_loss_grad_logp(logp, old_logp, ref_logp, scored, adv, cu_seqlens,
                                clip_lo, clip_hi, beta, agg, grad_loss)
        dH, dW = lm_head_backward(H, W, targets, mask, tau, g)
        out.update(g=g, dH=dH, dW=dW)
    return out
