"""Pins of oracle/critic_oracle.py (CPU only): closed forms, brute force, finite differences."""
import numpy as np

from oracle import critic_oracle as CO


def rnd(n, seed):
    return np.random.default_rng(seed).normal(size=n)


def test_gae_hand_worked():
    # one response, 3 tokens, gamma = 0.5, lambda = 0.5, r = (1, 0, 2), v = (0.5, 1, -1)
    # delta_2 = 2 - (-1) = 3;            A_2 = 3
    # delta_1 = 0 + 0.5 (-1) - 1 = -1.5; A_1 = -1.5 + 0.25 * 3 = -0.75
    # delta_0 = 1 + 0.5 (1) - 0.5 = 1;   A_0 = 1 + 0.25 (-0.75) = 0.8125
    adv, ret = CO.gae([1, 0, 2], [0.5, 1, -1], None, [0, 3], 0.5, 0.5)
    assert np.allclose(adv, [0.8125, -0.75, 3.0], atol=1e-15)
    assert np.allclose(ret, [1.3125, 0.25, 2.0], atol=1e-15)


def test_gae_closed_forms():
    r, v = rnd(40, 0), rnd(40, 1)
    cu = [0, 7, 7, 25, 40]                               # incl. an empty response
    # lambda = 1, gamma = 1: A_t = (sum of the rewards from t on) - v_t  (Monte-Carlo return)
    adv, ret = CO.gae(r, v, None, cu, 1.0, 1.0)
    for a, b in zip(cu[:-1], cu[1:]):
        for t in range(a, b):
            assert abs(ret[t] - r[t:b].sum()) < 1e-12 and abs(adv[t] - (r[t:b].sum() - v[t])) < 1e-12
    # lambda = 0: A_t = r_t + gamma v_{t+1} - v_t (one-step TD error)
    adv, _ = CO.gae(r, v, None, cu, 0.9, 0.0)
    for a, b in zip(cu[:-1], cu[1:]):
        for t in range(a, b):
            vn = v[t + 1] if t + 1 < b else 0.0
            assert abs(adv[t] - (r[t] + 0.9 * vn - v[t])) < 1e-12


def test_gae_brute_force_sum_and_mask():
    """A_t = sum_l (gamma lambda)^l delta_{t+l}, over the scored tokens only."""
    r, v = rnd(60, 2), rnd(60, 3)
    mask = (np.random.default_rng(4).random(60) < 0.7).astype(np.uint8)
    mask[:5] = 0                                         # a masked prompt prefix
    cu = [0, 20, 45, 60]
    g, lam = 0.97, 0.9
    adv, ret = CO.gae(r, v, mask, cu, g, lam)
    for a, b in zip(cu[:-1], cu[1:]):
        idx = [t for t in range(a, b) if mask[t]]
        for i, t in enumerate(idx):
            tot = 0.0
            for l, u in enumerate(idx[i:]):
                vn = v[idx[i + l + 1]] if i + l + 1 < len(idx) else 0.0
                tot += (g * lam) ** l * (r[u] + g * vn - v[u])
            assert abs(adv[t] - tot) < 1e-12 and abs(ret[t] - (tot + v[t])) < 1e-12
    assert np.all(adv[mask == 0] == 0) and np.all(ret[mask == 0] == 0)
    # masking is the same as deleting the tokens
    keep = mask != 0
    cu2 = [0] + list(np.cumsum([keep[a:b].sum() for a, b in zip(cu[:-1], cu[1:])]))
    adv2, _ = CO.gae(r[keep], v[keep], None, cu2, g, lam)
    assert np.allclose(adv[keep], adv2, atol=1e-15)


def test_value_loss_hand_and_limits():
    # v = 1.5, v_old = 1, eps = 0.2 -> v_clip = 1.2; ret = 2: l1 = .25, l2 = .64 -> clipped term, 0.32
    # v = 1.1, v_old = 1 -> v_clip = 1.1; ret = 0: l1 = l2 = 1.21 -> unclipped (tie), 0.605
    loss, cf, n = CO.value_loss([1.5, 1.1], [1.0, 1.0], [2.0, 0.0], None, 0.2)
    assert abs(loss - (0.32 + 0.605) / 2) < 1e-15 and cf == 0.5 and n == 2
    g = CO.value_loss_grad([1.5, 1.1], [1.0, 1.0], [2.0, 0.0], None, 0.2)
    assert np.allclose(g, [0.0, 1.1 / 2])               # clipped & outside the range: no gradient
    # clip range so wide that it never binds: plain 0.5 mean squared error
    v, vo, ret = rnd(100, 5), rnd(100, 6), rnd(100, 7)
    m = (np.random.default_rng(8).random(100) < 0.6).astype(np.uint8)
    loss, cf, n = CO.value_loss(v, vo, ret, m, 1e9)
    assert abs(loss - 0.5 * np.mean((v - ret)[m != 0] ** 2)) < 1e-14 and cf == 0.0
    assert np.allclose(CO.value_loss_grad(v, vo, ret, m, 1e9), (v - ret) * m / m.sum())
    assert CO.value_loss(v, vo, ret, np.zeros(100), 0.2) == (0.0, 0.0, 0)


def test_value_loss_gradient_finite_differences():
    v, ret = rnd(50, 9), rnd(50, 10)
    vo = v + 0.3 * rnd(50, 11)
    m = (np.random.default_rng(12).random(50) < 0.8).astype(np.uint8)
    g = CO.value_loss_grad(v, vo, ret, m, 0.2, grad_loss=0.7)
    h = 1e-6
    for t in range(50):
        e = np.zeros(50); e[t] = h
        fd = 0.7 * (CO.value_loss(v + e, vo, ret, m, 0.2)[0] - CO.value_loss(v - e, vo, ret, m, 0.2)[0]) / (2 * h)
        assert abs(fd - g[t]) < 1e-8, t


def test_value_head_and_backward():
    H, w = rnd((30, 16), 13), rnd(16, 14)
    v = CO.value_head(H, w, 0.25)
    assert np.allclose(v, [sum(H[t, d] * w[d] for d in range(16)) + 0.25 for t in range(30)])
    g = rnd(30, 15)
    dH, dw, db = CO.value_head_backward(H, w, g)
    # L = sum_t g_t v_t is linear: its exact derivatives
    assert np.allclose(dH, g[:, None] * w[None, :]) and abs(db - g.sum()) < 1e-13
    assert np.allclose(dw, [sum(g[t] * H[t, d] for t in range(30)) for d in range(16)])
