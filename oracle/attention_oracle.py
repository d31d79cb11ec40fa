"""Plain fp64 CPU oracle of the distributed attention of G-Core sec 4.5.  TEST INFRASTRUCTURE.

PAPER.md:209 (sec 4.5): "we implemented distributed attention based on CCL all-gather, where we
first all-gather the key (K) and value (V) tensors, and then compute attention output for the
local query (Q) tensor chunk."  PAPER.md:211: "we process only a subset of attention heads at a
time and overlap KV communication with attention computation."  The paper prints no formula and
no mask definition ("more complex attention masks (e.g., Gemma-3)"); the arithmetic is ordinary
scaled-dot-product attention, with the readings of DESIGN.md sec 11 (NEXT-4):

  * the sequence of S tokens is cut into `world` contiguous chunks; rank r holds Q, K, V of its
    chunk; "all-gather" = concatenation of the ranks' K and V in rank order;
  * grouped-query attention: query head h uses key/value head h // (Hq // Hkv);
  * a query at global position q may attend a key at global position k iff
        doc(k) == doc(q)                      (packed documents, cu_seqlens; one document if None)
        and (not causal or k <= q)
        and (window == 0 or q - k < window)   (sliding window, Gemma-3's local layers; with
                                               causal = False the window is two-sided: |q - k| < window)
  * out[q, h, :] = sum_k softmax_k(scale * <Q[q,h,:], K[k,g,:]>) V[k,g,:] over the allowed keys;
    lse[h, q] = log sum_k exp(scale * <.,.>) over the allowed keys (natural log).
    A query with no allowed key cannot occur (k = q is always allowed).

Head-subset chunking and communication overlap change WHEN things are computed, not WHAT: the
oracle is the definition, dense, one head at a time.  It shares no code with the CUDA path.

Pins (tests/test_attention_oracle_pins.py): hand-worked 2-token example; Q = 0 -> mean of the
allowed V rows and lse = log(#allowed); causal first token -> V[0]; window = 1 -> V[q]; key
permutation invariance (bidirectional); documents == attention run per document; GQA == MHA with
repeated K/V heads; scipy.special.softmax / logsumexp as library routines; shards concatenated ==
the unsharded call.
"""
from __future__ import annotations

import numpy as np


def allowed_mask(q_pos, S, cu_seqlens=None, causal=True, window=0):
    """bool [len(q_pos), S]: may the query at global position q_pos[i] attend key k."""
    q_pos = np.asarray(q_pos, dtype=np.int64)
    k_pos = np.arange(S, dtype=np.int64)
    if cu_seqlens is None:
        doc = np.zeros(S, dtype=np.int64)
    else:
        cu = np.asarray(cu_seqlens, dtype=np.int64)
        doc = np.full(S, -1, dtype=np.int64)
        for d in range(len(cu) - 1):
            doc[cu[d]:cu[d + 1]] = d
    ok = doc[q_pos][:, None] == doc[None, :]
    diff = q_pos[:, None] - k_pos[None, :]
    if causal:
        ok &= diff >= 0
        if window > 0:
            ok &= diff < window
    elif window > 0:
        ok &= np.abs(diff) < window
    return ok


def attention(Q, K, V, q_offset=0, cu_seqlens=None, causal=True, window=0, scale=None):
    """Q [Sq, Hq, d] (queries at global positions q_offset .. q_offset+Sq-1), K, V [S, Hkv, d]
    (all keys/values, global order) -> (out [Sq, Hq, d], lse [Hq, Sq]), float64."""
    Q = np.asarray(Q, dtype=np.float64)
    K = np.asarray(K, dtype=np.float64)
    V = np.asarray(V, dtype=np.float64)
    Sq, Hq, d = Q.shape
    S, Hkv, _ = K.shape
    assert Hq % Hkv == 0
    grp = Hq // Hkv
    if scale is None:
        scale = 1.0 / np.sqrt(d)
    ok = allowed_mask(q_offset + np.arange(Sq), S, cu_seqlens, causal, window)
    out = np.zeros((Sq, Hq, d))
    lse = np.zeros((Hq, Sq))
    for h in range(Hq):
        g = h // grp
        s = scale * (Q[:, h, :] @ K[:, g, :].T)                    # [Sq, S]
        s = np.where(ok, s, -np.inf)
        m = s.max(axis=1, keepdims=True)
        e = np.exp(s - m)
        z = e.sum(axis=1, keepdims=True)
        out[:, h, :] = (e / z) @ V[:, g, :]
        lse[h] = (m + np.log(z))[:, 0]
    return out, lse


def attention_allgather(Q_shards, K_shards, V_shards, rank, cu_seqlens=None, causal=True, window=0,
                        scale=None):
    """What rank `rank` computes: its Q chunk against the concatenation of every rank's K, V."""
    K = np.concatenate([np.asarray(k, dtype=np.float64) for k in K_shards], axis=0)
    V = np.concatenate([np.asarray(v, dtype=np.float64) for v in V_shards], axis=0)
    off = int(sum(len(k) for k in K_shards[:rank]))
    return attention(Q_shards[rank], K, V, off, cu_seqlens, causal, window, scale)
