"""Plain fp64 CPU oracle of the PPO-variant critic path.  TEST
INFRASTRUCTURE: only tests/ may import it; it shares no code with paper_2507_22789_b200.

What the paper says: PAPER.md:96 (sec 2.2) the PPO workflow has a critic that "computes values";
PAPER.md:102-103 stage 3 computes them, stage 4 trains actor and critic.  It gives no formula; the
authority it cites is PPO [18]: generalised advantage estimation and the clipped
value objective.  Readings:

  1 value head        v_t = sum_d H[t,d] w[d] + b
  2 GAE               over the scored tokens of each response, in order (a masked token is not
                      part of the trajectory):  delta_t = r_t + gamma v_next(t) - v_t, with v_next
                      the value at the next scored token of the same response (0 after the last);
                      A_t = delta_t + gamma lambda A_next(t);  return_t = A_t + v_t.
                      adv = returns = 0 at unscored tokens.
  3 value loss        v_clip = clip(v, v_old - eps, v_old + eps);
                      l_t = 0.5 max((v - ret)^2, (v_clip - ret)^2);  loss = sum m l / max(sum m, 1);
                      clip_frac = share of scored tokens where the clipped term is the larger.
  4 d loss / d v_t    = grad_loss m_t / max(sum m,1) * ((v - ret) if (v - ret)^2 >= (v_clip - ret)^2
                      else (v_clip - ret) [v_old - eps < v < v_old + eps])   (ties: unclipped term)
  5 backward          dH[t,:] = g_t w;  dw = sum_t g_t H[t,:];  db = sum_t g_t

Everything is written as the definition: sequential python loops for the recursion (small cases),
numpy for the dot products.  Pins: tests/test_critic_oracle_pins.py.
"""
from __future__ import annotations

import numpy as np


def value_head(H, w, b):
    """Step 1."""
    return np.asarray(H, np.float64) @ np.asarray(w, np.float64) + float(b)


def gae(rewards, values, mask, cu_seqlens, gamma, lam):
    """Step 2: plain reverse loop per response."""
    r = np.asarray(rewards, np.float64)
    v = np.asarray(values, np.float64)
    T = len(r)
    m = np.ones(T, bool) if mask is None else np.asarray(mask) != 0
    adv = np.zeros(T)
    ret = np.zeros(T)
    cu = [int(x) for x in cu_seqlens]
    for s in range(len(cu) - 1):
        a_next, v_next = 0.0, 0.0
        for t in range(cu[s + 1] - 1, cu[s] - 1, -1):
            if not m[t]:
                continue
            delta = r[t] + gamma * v_next - v[t]
            a = delta + gamma * lam * a_next
            adv[t] = a
            ret[t] = a + v[t]
            a_next, v_next = a, v[t]
    return adv, ret


def value_loss(values, old_values, returns, mask, clip_v):
    """Step 3 -> (loss, clip_frac, n_scored)."""
    v = np.asarray(values, np.float64)
    vo = np.asarray(old_values, np.float64)
    ret = np.asarray(returns, np.float64)
    m = np.ones(len(v), bool) if mask is None else np.asarray(mask) != 0
    vc = np.clip(v, vo - clip_v, vo + clip_v)
    l1 = (v - ret) ** 2
    l2 = (vc - ret) ** 2
    n = max(int(m.sum()), 1)
    loss = 0.5 * np.sum(np.maximum(l1, l2)[m]) / n
    clip_frac = float(np.sum((l2 > l1)[m])) / n
    return float(loss), clip_frac, int(m.sum())


def value_loss_grad(values, old_values, returns, mask, clip_v, grad_loss=1.0):
    """Step 4: d loss / d v."""
    v = np.asarray(values, np.float64)
    vo = np.asarray(old_values, np.float64)
    ret = np.asarray(returns, np.float64)
    m = np.ones(len(v), bool) if mask is None else np.asarray(mask) != 0
    vc = np.clip(v, vo - clip_v, vo + clip_v)
    l1 = (v - ret) ** 2
    l2 = (vc - ret) ** 2
    inside = (v > vo - clip_v) & (v < vo + clip_v)
    g = np.where(l1 >= l2, v - ret, (vc - ret) * inside)
    return grad_loss * g * m / max(int(m.sum()), 1)


def value_head_backward(H, w, g):
    """Step 5 -> (dH, dw, db)."""
    H = np.asarray(H, np.float64)
    w = np.asarray(w, np.float64)
    g = np.asarray(g, np.float64)
    return np.outer(g, w), g @ H, float(g.sum())
