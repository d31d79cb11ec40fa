"""Pins for oracle/gcore_oracle.py against what the mathematics fixes (CPU only).

Each pin is chosen so that a plausible mistake (dropped term, wrong sign/index, transposed
operand, wrong ddof, wrong clip branch) fails at least one test.  No value here comes from the
CUDA path.  Citations: SURVEY.md sec 8(c) pins table; BASELINE.json:north_star invariants.
"""
import math

import numpy as np
import pytest
import scipy.special
import scipy.stats

import oracle as O


def rng(seed=0):
    return np.random.default_rng(seed)


# ------------------------------------------------------------------ steps 1-3: log-probs
def brute_logprobs(H, W, y, tau):
    """Pure-python loops, the definition written out with math.exp/log (tiny inputs only)."""
    T, D = len(H), len(H[0])
    V = len(W)
    out = []
    for t in range(T):
        z = [sum(H[t][d] * W[v][d] for d in range(D)) / tau for v in range(V)]
        Z = sum(math.exp(a) for a in z)
        p = [math.exp(a) / Z for a in z]
        ent = -sum(q * math.log(q) for q in p)
        out.append((math.log(p[y[t]]), ent, math.log(Z)))
    return np.array(out)


def test_tiny_worked_example(golden):
    g = golden("tiny_softmax.txt")
    H = [[1, 0], [0, 2]]
    W = [[1, 0], [0, 1], [-1, 0], [0, -1]]
    y = [0, 1]
    lp, en, ls = O.token_logprobs(H, W, y, None, 1.0)
    assert np.allclose(ls, [g["tau1.lse0"][0], g["tau1.lse1"][0]], atol=1e-11)
    assert np.allclose(lp, [g["tau1.logp0"][0], g["tau1.logp1"][0]], atol=1e-11)
    assert np.allclose(en, [g["tau1.entropy0"][0], g["tau1.entropy1"][0]], atol=1e-11)
    lp, en, ls = O.token_logprobs(H, W, y, None, 0.5)
    assert np.allclose(lp, [g["tau05.logp0"][0], g["tau05.logp1"][0]], atol=1e-11)
    assert np.allclose(en, [g["tau05.entropy0"][0], g["tau05.entropy1"][0]], atol=1e-11)
    # the closed forms themselves
    assert abs(ls_closed(1) - g["tau1.lse0"][0]) < 1e-11
    assert abs(ls_closed(2) - g["tau1.lse1"][0]) < 1e-11


def ls_closed(a):
    return math.log(math.exp(a) + 2 + math.exp(-a))


@pytest.mark.parametrize("tau", [1.0, 0.7, 2.5])
def test_brute_force_small(tau):
    r = rng(1)
    T, D, V = 6, 3, 7          # all different: a transposed operand cannot type-check
    H = r.normal(size=(T, D))
    W = r.normal(size=(V, D))
    y = r.integers(0, V, T)
    lp, en, ls = O.token_logprobs(H, W, y, None, tau)
    b = brute_logprobs(H.tolist(), W.tolist(), y.tolist(), tau)
    assert np.allclose(lp, b[:, 0], atol=1e-13)
    assert np.allclose(en, b[:, 1], atol=1e-13)
    assert np.allclose(ls, b[:, 2], atol=1e-13)
    for t in range(T):
        a, e, l = O.token_logprobs_row(H[t], W, y[t], tau)
        assert abs(a - b[t, 0]) < 1e-13 and abs(e - b[t, 1]) < 1e-13 and abs(l - b[t, 2]) < 1e-13


def test_uniform_closed_form():
    V, D, T = 50, 4, 3
    W = rng(2).normal(size=(V, D))
    lp, en, ls = O.token_logprobs(np.zeros((T, D)), W, [0, 7, 49], None, 1.0)
    assert np.allclose(lp, -math.log(V), atol=1e-14)
    assert np.allclose(en, math.log(V), atol=1e-13)
    # all W rows equal -> uniform too
    H = rng(3).normal(size=(T, D))
    lp, en, _ = O.token_logprobs(H, np.tile(W[:1], (V, 1)), [1, 2, 3], None, 0.7)
    assert np.allclose(lp, -math.log(V), atol=1e-13)
    assert np.allclose(en, math.log(V), atol=1e-12)


def test_probabilities_sum_to_one_and_dominant_logit():
    r = rng(4)
    D, V = 5, 33
    h = r.normal(size=(1, D))
    W = r.normal(size=(V, D))
    lp, _, _ = O.token_logprobs(np.repeat(h, V, 0), W, np.arange(V), None, 0.9)
    assert abs(np.exp(lp).sum() - 1.0) < 1e-13
    W2 = np.zeros((V, D))
    W2[5] = 20.0 * h[0] / (h[0] @ h[0])             # one dominant logit: z = [0,..,20,..,0]
    lp, en, _ = O.token_logprobs(h, W2, [5], None, 1.0)
    x = (V - 1) * math.exp(-20.0)
    assert abs(lp[0] + math.log1p(x)) < 1e-15 and 0 < en[0] < 1e-5


def test_library_routines():
    r = rng(5)
    T, D, V = 9, 8, 101
    H, W = r.normal(size=(T, D)), r.normal(size=(V, D))
    y = r.integers(0, V, T)
    tau = 0.7
    lp, en, ls = O.token_logprobs(H, W, y, None, tau)
    z = (H @ W.T) / tau
    ref = scipy.special.log_softmax(z, axis=1)
    assert np.allclose(lp, ref[np.arange(T), y], atol=1e-12)
    assert np.allclose(ls, scipy.special.logsumexp(z, axis=1), atol=1e-12)
    assert np.allclose(en, scipy.stats.entropy(scipy.special.softmax(z, axis=1), axis=1), atol=1e-12)


def test_invariances():
    r = rng(6)
    T, D, V = 7, 6, 41
    H, W = r.normal(size=(T, D)), r.normal(size=(V, D))
    y = r.integers(0, V, T)
    base = O.token_logprobs(H, W, y, None, 1.0)
    # constant added to every logit: extra H column of ones, W column of c
    H1 = np.concatenate([H, np.ones((T, 1))], 1)
    W1 = np.concatenate([W, np.full((V, 1), 3.25)], 1)
    a = O.token_logprobs(H1, W1, y, None, 1.0)
    assert np.allclose(a[0], base[0], atol=1e-12) and np.allclose(a[1], base[1], atol=1e-12)
    assert np.allclose(a[2], base[2] + 3.25, atol=1e-12)
    # (H, tau) == (H/tau, 1)
    b = O.token_logprobs(H, W, y, None, 0.7)
    c = O.token_logprobs(H / 0.7, W, y, None, 1.0)
    for i in range(3):
        assert np.allclose(b[i], c[i], atol=1e-12)
    assert not np.allclose(b[0], base[0], atol=1e-3)
    # vocab permutation with targets remapped
    perm = r.permutation(V)
    inv = np.argsort(perm)
    d = O.token_logprobs(H, W[perm], inv[y], None, 1.0)
    for i in range(3):
        assert np.allclose(d[i], base[i], atol=1e-12)


def test_mask_and_negative_targets_zero_outputs():
    r = rng(7)
    T, D, V = 8, 4, 13
    H, W = r.normal(size=(T, D)), r.normal(size=(V, D))
    y = r.integers(0, V, T)
    y2 = y.copy()
    y2[2] = -100
    m = np.ones(T, np.uint8)
    m[5] = 0
    full = O.token_logprobs(H, W, y, None, 1.0)
    part = O.token_logprobs(H, W, y2, m, 1.0)
    for i in range(3):
        assert part[i][2] == 0.0 and part[i][5] == 0.0
        keep = [0, 1, 3, 4, 6, 7]
        assert np.array_equal(part[i][keep], full[i][keep])


# ------------------------------------------------------------------ steps 4-5: filter, advantages
def test_advantages_golden(golden):
    g = golden("advantages.txt")
    go = [0, 4]
    for key, r in (("1001", [1, 0, 0, 1]), ("1110", [1, 1, 1, 0]), ("2468", [.2, .4, .6, .8])):
        a, _ = O.grpo_advantages(r, go, eps=0.0)
        assert np.allclose(a, g["pop." + key], atol=1e-9)
        if "sample." + key in g:
            a, _ = O.grpo_advantages(r, go, eps=0.0, unbiased_std=True)
            assert np.allclose(a, g["sample." + key], atol=1e-9)
    # closed forms behind the stored decimals
    assert abs(g["sample.1001"][0] - math.sqrt(3) / 2) < 1e-11
    assert abs(g["pop.1110"][3] + math.sqrt(3)) < 1e-11
    assert abs(g["pop.2468"][3] - 3 / math.sqrt(5)) < 1e-9


def test_advantages_properties():
    r = rng(8)
    sizes = [4, 7, 2, 16]
    go = np.concatenate([[0], np.cumsum(sizes)])
    rew = r.random(go[-1])
    eps = 1e-6
    a, keep = O.grpo_advantages(rew, go, eps=eps)
    assert keep.tolist() == [1, 1, 1, 1]
    for g in range(4):
        seg = a[go[g]:go[g + 1]]
        sig = rew[go[g]:go[g + 1]].std()
        assert abs(seg.mean()) < 1e-12
        assert abs(seg.std() - sig / (sig + eps)) < 1e-12          # unit std up to eps/sigma
        au, _ = O.grpo_advantages(rew, go, eps=0.0, unbiased_std=True)
        assert abs(au[go[g]:go[g + 1]].std(ddof=1) - 1.0) < 1e-12
    # n = 2 -> +-1 (population)
    a2 = O.grpo_advantages(rew, go, eps=0.0)[0][go[2]:go[3]]
    assert np.allclose(np.sort(a2), [-1, 1], atol=1e-12)
    # affine invariance r -> a r + b (eps = 0), sign flip for a < 0
    a0, _ = O.grpo_advantages(rew, go, eps=0.0)
    a1, _ = O.grpo_advantages(3.5 * rew - 2.0, go, eps=0.0)
    a3, _ = O.grpo_advantages(-2.0 * rew + 1.0, go, eps=0.0)
    assert np.allclose(a0, a1, atol=1e-11) and np.allclose(a0, -a3, atol=1e-11)


def test_constant_groups_and_filter():
    rew = np.array([1, 1, 1, 1, 0, 1, 0, 0, 0, 0, 0, 0, .5, .5, .5, .25], dtype=np.float32)
    go = [0, 4, 8, 12, 16]
    assert O.group_filter(rew, go).tolist() == [0, 1, 0, 1]
    a, keep = O.grpo_advantages(rew, go, eps=1e-6, drop_constant_groups=False)
    assert keep.tolist() == [1, 1, 1, 1]
    assert np.all(a[0:4] == 0.0) and np.all(a[8:12] == 0.0)        # A = 0 exactly, eps > 0
    a, keep = O.grpo_advantages(rew, go, eps=1e-6, drop_constant_groups=True)
    assert keep.tolist() == [0, 1, 0, 1]
    assert np.all(a[0:4] == 0.0) and abs(a[4:8].mean()) < 1e-12
    with np.errstate(invalid="ignore", divide="ignore"):
        a, _ = O.grpo_advantages(rew, go, eps=0.0)
    assert np.all(np.isnan(a[0:4]))                                 # eps = 0 -> 0/0 (reading 3)


def test_token_to_response():
    cu = [0, 3, 3, 7]
    assert O.token_to_response(cu, 9).tolist() == [0, 0, 0, 2, 2, 2, 2, -1, -1]


# ------------------------------------------------------------------ steps 6-8: loss, g_t
def test_loss_tokens_golden(golden):
    g = golden("loss_tokens.txt")
    for k, (inp, outp) in g.items():
        logp, old, ref, A = inp
        res = O.grpo_loss([logp], [old], [ref], [True], [A], [0, 1], 0.2, 0.2, 0.04)
        assert abs(res["loss"] - outp[0]) < 2e-9, k
        gt = O.grpo_loss_grad_logp([logp], [old], [ref], [True], [A], [0, 1], 0.2, 0.2, 0.04)
        assert abs(gt[0] - outp[1]) < 2e-9, k
    # independent arithmetic for case 1 and case 2 (python floats, formula from the fixture header)
    rho = math.exp(0.1)
    assert abs(-rho + 0.04 * (math.exp(0.1) - 0.1 - 1) - g["case1"][1][0]) < 2e-9
    assert abs(-1.2 + 0.04 * (math.exp(0.1) - 0.1 - 1) - g["case2"][1][0]) < 2e-9
    assert g["case4"][1] == [0.8, 0.0]


def _batch(seed, R=5, ragged=True, old_std=0.3):
    r = rng(seed)
    L = r.integers(1, 9, R) if ragged else np.full(R, 6)
    cu = np.concatenate([[0], np.cumsum(L)])
    T = int(cu[-1])
    logp = -r.random(T) * 3
    old = logp + r.normal(0, old_std, T)
    ref = logp + r.normal(0, 0.1, T)
    adv = r.normal(size=R)
    scored = r.random(T) < 0.75
    return logp, old, ref, scored, adv, cu


def test_loss_identities():
    logp, old, ref, scored, adv, cu = _batch(10)
    resp = O.token_to_response(cu, len(logp))
    A = adv[resp]
    # logp = old and beta = 0  ->  loss = -sum(m A)/sum(m)   (north_star invariant, reading 5)
    res = O.grpo_loss(logp, logp, ref, scored, adv, cu, beta=0.0)
    assert abs(res["loss"] + (A * scored).sum() / scored.sum()) < 1e-14
    assert res["clip_frac"] == 0.0
    # logp = old = ref, beta > 0: same, and KL = 0
    res = O.grpo_loss(logp, logp, logp, scored, adv, cu, beta=0.04)
    assert abs(res["loss"] + (A * scored).sum() / scored.sum()) < 1e-14
    assert res["kl_mean"] == 0.0
    # logp = old != ref: loss = that + beta * kl_mean, k3 >= 0
    res = O.grpo_loss(logp, logp, ref, scored, adv, cu, beta=0.04)
    assert res["kl_mean"] > 0
    assert abs(res["loss"] - (-(A * scored).sum() / scored.sum() + 0.04 * res["kl_mean"])) < 1e-14
    assert abs(res["loss"] - (res["pg_loss"] + 0.04 * res["kl_mean"])) < 1e-15
    assert res["n_scored"] == scored.sum()
    # no clipping when |logp-old| < min(ln 1.2, -ln .8)
    old2 = logp + np.clip(old - logp, -0.18, 0.18)
    assert O.grpo_loss(logp, old2, ref, scored, adv, cu)["clip_frac"] == 0.0
    assert O.grpo_loss(logp, old, ref, scored, adv, cu)["clip_frac"] > 0.0
    # sum m = 0 -> loss 0 (reading 12)
    z = O.grpo_loss(logp, old, ref, np.zeros_like(scored), adv, cu)
    assert z["loss"] == 0.0 and z["n_scored"] == 0.0


def test_clip_fraction_brute_force():
    logp, old, ref, scored, adv, cu = _batch(11)
    resp = O.token_to_response(cu, len(logp))
    n_clip = 0
    for t in range(len(logp)):
        if not scored[t]:
            continue
        rho, A = math.exp(logp[t] - old[t]), adv[resp[t]]
        if (A > 0 and rho > 1.2) or (A < 0 and rho < 0.8):
            n_clip += 1
    res = O.grpo_loss(logp, old, ref, scored, adv, cu)
    assert abs(res["clip_frac"] - n_clip / scored.sum()) < 1e-15


def test_seq_mean_vs_token_mean():
    # equal lengths + full mask: the two aggregations coincide (reading 4)
    logp, old, ref, scored, adv, cu = _batch(12, ragged=False)
    full = np.ones_like(scored)
    a = O.grpo_loss(logp, old, ref, full, adv, cu, agg=O.AGG_TOKEN_MEAN)
    b = O.grpo_loss(logp, old, ref, full, adv, cu, agg=O.AGG_SEQ_MEAN)
    assert abs(a["loss"] - b["loss"]) < 1e-14
    # ragged: brute force seq-mean
    logp, old, ref, scored, adv, cu = _batch(13, ragged=True)
    b = O.grpo_loss(logp, old, ref, scored, adv, cu, agg=O.AGG_SEQ_MEAN)
    per = b["per_token"]
    tot, kept = 0.0, 0
    for r_ in range(len(cu) - 1):
        sl = slice(cu[r_], cu[r_ + 1])
        n = scored[sl].sum()
        if n > 0:
            kept += 1
            tot += per[sl].sum() / n
    assert abs(b["loss"] - tot / kept) < 1e-14


@pytest.mark.parametrize("agg", [O.AGG_TOKEN_MEAN, O.AGG_SEQ_MEAN])
def test_grad_logp_finite_differences(agg):
    logp, old, ref, scored, adv, cu = _batch(14)
    g = O.grpo_loss_grad_logp(logp, old, ref, scored, adv, cu, agg=agg, grad_loss=1.7)
    h = 1e-6
    for t in range(len(logp)):
        e = np.zeros_like(logp)
        e[t] = h
        fp = O.grpo_loss(logp + e, old, ref, scored, adv, cu, agg=agg)["loss"]
        fm = O.grpo_loss(logp - e, old, ref, scored, adv, cu, agg=agg)["loss"]
        assert abs(1.7 * (fp - fm) / (2 * h) - g[t]) < 1e-8
    assert np.all(g[~scored] == 0.0)


# ------------------------------------------------------------------ step 9: dH, dW
def _small_problem(seed=20, tau=0.7):
    r = rng(seed)
    R, D, V = 4, 5, 11
    L = r.integers(2, 6, R)
    cu = np.concatenate([[0], np.cumsum(L)])
    T = int(cu[-1])
    H, W = r.normal(size=(T, D)), r.normal(size=(V, D)) * 0.5
    y = r.integers(0, V, T)
    y[1] = -1
    mask = (r.random(T) < 0.8).astype(np.uint8)
    mask[0] = 1
    lp, _, _ = O.token_logprobs(H, W, np.maximum(y, 0), None, tau)
    old = lp + r.normal(0, 0.3, T)
    ref = lp + r.normal(0, 0.1, T)
    adv = r.normal(size=R)
    return H, W, y, mask, tau, cu, adv, old, ref


@pytest.mark.parametrize("agg", [O.AGG_TOKEN_MEAN, O.AGG_SEQ_MEAN])
def test_backward_finite_differences(agg):
    H, W, y, mask, tau, cu, adv, old, ref = _small_problem()
    out = O.grpo_forward_backward(H, W, y, mask, tau, cu, adv, old, ref, agg=agg)

    def loss(Hx, Wx):
        return O.grpo_forward_backward(Hx, Wx, y, mask, tau, cu, adv, old, ref, agg=agg,
                                       need_grads=False)["loss"]
    h = 1e-5
    r = rng(21)
    for _ in range(4):          # random directions
        dHd, dWd = r.normal(size=H.shape), r.normal(size=W.shape)
        fd = (loss(H + h * dHd, W) - loss(H - h * dHd, W)) / (2 * h)
        assert abs(fd - (out["dH"] * dHd).sum()) < 3e-8 * max(1, abs(fd))
        fd = (loss(H, W + h * dWd) - loss(H, W - h * dWd)) / (2 * h)
        assert abs(fd - (out["dW"] * dWd).sum()) < 3e-8 * max(1, abs(fd))
    for (t, d) in [(0, 0), (2, 3), (H.shape[0] - 1, 4)]:      # single entries
        E = np.zeros_like(H)
        E[t, d] = h
        fd = (loss(H + E, W) - loss(H - E, W)) / (2 * h)
        assert abs(fd - out["dH"][t, d]) < 1e-9
    for (v, d) in [(0, 0), (int(y[0]), 1), (10, 4)]:
        E = np.zeros_like(W)
        E[v, d] = h
        fd = (loss(H, W + E) - loss(H, W - E)) / (2 * h)
        assert abs(fd - out["dW"][v, d]) < 1e-9


def test_backward_identities():
    H, W, y, mask, tau, cu, adv, old, ref = _small_problem(22)
    out = O.grpo_forward_backward(H, W, y, mask, tau, cu, adv, old, ref)
    dH, dW = out["dH"], out["dW"]
    scored = (mask != 0) & (y >= 0)
    assert np.all(dH[~scored] == 0.0)                       # masked rows exactly 0
    assert np.abs(dW.sum(axis=0)).max() < 1e-15 * 50        # every column sum of dW is 0
    assert abs((dH * H).sum() - (dW * W).sum()) < 1e-14     # <dH,H> = <dW,W> (bilinear form)
    for t in np.nonzero(scored)[0]:
        row = O.lm_head_backward_row(H[t], W, y[t], tau, out["g"][t])
        assert np.allclose(row, dH[t], atol=1e-15)


def test_backward_cross_entropy_special_case():
    """logp = old = ref: g_t = -m_t A_t / sum m and the backward is the textbook weighted
    cross-entropy gradient (softmax - onehot) scaled per token."""
    H, W, y, mask, tau, cu, adv, _, _ = _small_problem(23, tau=1.0)
    lp, _, _ = O.token_logprobs(H, W, y, mask, tau)
    out = O.grpo_forward_backward(H, W, y, mask, tau, cu, adv, lp, lp)
    scored = (mask != 0) & (y >= 0)
    A = adv[O.token_to_response(cu, len(y))]
    wgt = np.where(scored, A / scored.sum(), 0.0)           # loss = -sum wgt_t logp_t
    assert np.allclose(out["g"], -wgt, atol=1e-15)
    P = scipy.special.softmax(H @ W.T, axis=1)
    Y = np.zeros_like(P)
    Y[np.arange(len(y)), np.maximum(y, 0)] = 1.0
    dz = wgt[:, None] * (P - Y)                             # d(-sum w logp)/dz
    assert np.allclose(out["dH"], dz @ W, atol=1e-14)
    assert np.allclose(out["dW"], dz.T @ H, atol=1e-14)


def test_backward_wrows_matches_dense_rows_and_finite_differences():
    """lm_head_backward_wrows (step 9 restricted to vocab rows; used by the full-size dW check):
    equal to the dense backward's rows for every row, for target rows and never-target rows, with
    token slices summed; and each entry equal to the central finite difference of the loss."""
    H, W, y, mask, tau, cu, adv, old, ref = _small_problem(24)
    out = O.grpo_forward_backward(H, W, y, mask, tau, cu, adv, old, ref)
    V = W.shape[0]
    scored = (mask != 0) & (y >= 0)
    hit = sorted(set(int(v) for v in y[scored]))
    miss = [v for v in range(V) if v not in hit]
    assert hit and miss
    for ids in (list(range(V)), hit, miss, [miss[0], hit[0], V - 1, 0]):
        rows = O.lm_head_backward_wrows(H, W[ids], ids, y, mask, tau, out["g"], out["lse"])
        assert rows.shape == (len(ids), H.shape[1])
        assert np.allclose(rows, out["dW"][ids], atol=1e-15)
    # a sum over token slices is the same thing (dW is a sum over tokens)
    ids = [hit[0], miss[0]]
    T = len(y)
    acc = np.zeros((2, H.shape[1]))
    for a in range(0, T, 3):
        sl = slice(a, min(T, a + 3))
        acc += O.lm_head_backward_wrows(H[sl], W[ids], ids, y[sl], mask[sl], tau, out["g"][sl],
                                        out["lse"][sl])
    assert np.allclose(acc, out["dW"][ids], atol=1e-15)

    def loss(Wx):
        return O.grpo_forward_backward(H, Wx, y, mask, tau, cu, adv, old, ref,
                                       need_grads=False)["loss"]
    h = 1e-5
    rows = O.lm_head_backward_wrows(H, W[ids], ids, y, mask, tau, out["g"], out["lse"])
    for i, v in enumerate(ids):
        for d in (0, 3):
            E = np.zeros_like(W)
            E[v, d] = h
            fd = (loss(W + E) - loss(W - E)) / (2 * h)
            assert abs(fd - rows[i, d]) < 1e-9
    # a transposed operand, a dropped onehot or a wrong sign would fail the above; a wrong lse
    # must change the result (the function really uses it)
    bad = O.lm_head_backward_wrows(H, W[ids], ids, y, mask, tau, out["g"], out["lse"] + 0.1)
    assert np.abs(bad - rows).max() > 1e-4
