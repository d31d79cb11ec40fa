"""Pins for oracle/attention_oracle.py (NEXT-4) against what the mathematics
fixes: a hand-worked example, closed forms, invariances, library routines.  CPU only."""
import numpy as np
import scipy.special

from oracle import attention_oracle as A


def rng(s=0):
    return np.random.default_rng(s)


def test_hand_worked_two_token_example(golden):
    g = golden("attention_tiny.txt")
    Q = np.array([[[1.0, 0.0]], [[0.0, 1.0]]])
    K = np.array([[[1.0, 0.0]], [[0.0, 2.0]]])
    V = np.array([[[1.0, 2.0]], [[3.0, 4.0]]])
    out, lse = A.attention(Q, K, V, causal=True, scale=1.0)
    assert np.allclose(out[0, 0], g["out0"], atol=1e-14) and np.allclose(out[1, 0], g["out1"], atol=1e-14)
    assert np.allclose(lse[0], g["lse"], atol=1e-14)
    out, lse = A.attention(Q, K, V, causal=False, scale=1.0)
    assert np.allclose(out[0, 0], g["out0_full"], atol=1e-14)
    assert abs(lse[0, 0] - g["lse0_full"][0]) < 1e-14


def brute(Q, K, V, q_off, cu, causal, window, scale):
    """The definition with python loops and math.exp (tiny inputs)."""
    import math
    Sq, Hq, d = Q.shape
    S, Hkv, _ = K.shape
    doc = [0] * S
    if cu is not None:
        for i in range(len(cu) - 1):
            for t in range(cu[i], cu[i + 1]):
                doc[t] = i
    out = np.zeros((Sq, Hq, d))
    lse = np.zeros((Hq, Sq))
    for i in range(Sq):
        q = q_off + i
        for h in range(Hq):
            g = h // (Hq // Hkv)
            ks = [k for k in range(S) if doc[k] == doc[q] and (not causal or k <= q)
                  and (window == 0 or (q - k < window if causal else abs(q - k) < window))]
            sc = [scale * sum(Q[i, h, c] * K[k, g, c] for c in range(d)) for k in ks]
            Z = sum(math.exp(x) for x in sc)
            for k, x in zip(ks, sc):
                out[i, h] += math.exp(x) / Z * V[k, g]
            lse[h, i] = math.log(Z)
    return out, lse


def test_brute_force_small_all_mask_kinds():
    r = rng(1)
    S, Hq, Hkv, d = 13, 4, 2, 3
    Q, K, V = r.normal(size=(S, Hq, d)), r.normal(size=(S, Hkv, d)), r.normal(size=(S, Hkv, d))
    cu = [0, 4, 5, 13]
    for causal in (True, False):
        for window in (0, 1, 3):
            for c in (None, cu):
                o, l = A.attention(Q[3:9], K, V, 3, c, causal, window, 0.7)
                ob, lb = brute(Q[3:9], K, V, 3, c, causal, window, 0.7)
                assert np.allclose(o, ob, atol=1e-13) and np.allclose(l, lb, atol=1e-13)


def test_closed_forms():
    r = rng(2)
    S, H, d = 9, 2, 4
    K, V = r.normal(size=(S, H, d)), r.normal(size=(S, H, d))
    out, lse = A.attention(np.zeros((S, H, d)), K, V, causal=True)
    for q in range(S):                       # Q = 0: uniform over the allowed keys
        assert np.allclose(out[q], V[:q + 1].mean(axis=0), atol=1e-14)
        assert np.allclose(lse[:, q], np.log(q + 1), atol=1e-14)
    Q = r.normal(size=(S, H, d))
    out, _ = A.attention(Q, K, V, causal=True)
    assert np.allclose(out[0], V[0], atol=1e-15)                  # the first token sees itself only
    out, lse = A.attention(Q, K, V, causal=True, window=1)        # window 1: itself only
    assert np.allclose(out, V, atol=1e-15)
    assert np.allclose(lse, np.einsum("shd,shd->hs", Q, K) / np.sqrt(d), atol=1e-14)


def test_library_routines_and_invariances():
    r = rng(3)
    S, H, d = 11, 3, 5
    Q, K, V = r.normal(size=(S, H, d)), r.normal(size=(S, H, d)), r.normal(size=(S, H, d))
    out, lse = A.attention(Q, K, V, causal=False, scale=0.3)
    for h in range(H):
        s = 0.3 * Q[:, h] @ K[:, h].T
        assert np.allclose(out[:, h], scipy.special.softmax(s, axis=1) @ V[:, h], atol=1e-14)
        assert np.allclose(lse[h], scipy.special.logsumexp(s, axis=1), atol=1e-14)
    p = r.permutation(S)                      # bidirectional: key order does not matter
    out2, lse2 = A.attention(Q, K[p], V[p], causal=False, scale=0.3)
    assert np.allclose(out, out2, atol=1e-14) and np.allclose(lse, lse2, atol=1e-14)
    # adding a constant vector to every key shifts every score of a row equally: out unchanged
    out3, _ = A.attention(Q, K + 5.0 * np.ones(d), V, causal=False, scale=0.3)
    assert np.allclose(out, out3, atol=1e-12)
    # GQA == MHA with repeated key/value heads
    Kg, Vg = r.normal(size=(S, 1, d)), r.normal(size=(S, 1, d))
    o1, l1 = A.attention(Q, Kg, Vg, causal=True)
    o2, l2 = A.attention(Q, np.repeat(Kg, H, axis=1), np.repeat(Vg, H, axis=1), causal=True)
    assert np.allclose(o1, o2, atol=1e-15) and np.allclose(l1, l2, atol=1e-15)


def test_documents_equal_separate_calls_and_shards_equal_whole():
    r = rng(4)
    S, Hq, Hkv, d = 20, 4, 2, 4
    Q, K, V = r.normal(size=(S, Hq, d)), r.normal(size=(S, Hkv, d)), r.normal(size=(S, Hkv, d))
    cu = [0, 7, 8, 20]
    out, lse = A.attention(Q, K, V, 0, cu, True, 4)
    for a, b in zip(cu[:-1], cu[1:]):        # packed documents == each document alone
        o, l = A.attention(Q[a:b], K[a:b], V[a:b], 0, None, True, 4)
        assert np.allclose(out[a:b], o, atol=1e-14) and np.allclose(lse[:, a:b], l, atol=1e-14)
    cuts = [0, 6, 11, 20]                    # 3 ranks, unequal chunks: all-gather == unsharded
    Qs = [Q[a:b] for a, b in zip(cuts[:-1], cuts[1:])]
    Ks = [K[a:b] for a, b in zip(cuts[:-1], cuts[1:])]
    Vs = [V[a:b] for a, b in zip(cuts[:-1], cuts[1:])]
    for rank, (a, b) in enumerate(zip(cuts[:-1], cuts[1:])):
        o, l = A.attention_allgather(Qs, Ks, Vs, rank, cu, True, 4)
        assert np.allclose(o, out[a:b], atol=1e-15) and np.allclose(l, lse[:, a:b], atol=1e-15)
