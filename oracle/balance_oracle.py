"""Plain CPU oracle of the step before the scoring path: dynamic-sampling repack + workload
balancing.  TEST INFRASTRUCTURE: only tests/ may import it; it shares
no code with paper_2507_22789_b200.

What the paper says (and all it says):
  PAPER.md:150 (sec 3.2)  dynamic sampling: "filter out prompts with the accuracy equal to 1 and 0"
  PAPER.md:201 (sec 4.4)  "instead of sequence packing, we simply sort data by simulated workload"
  PAPER.md:199            the workload model: attention cost s^2 for a sequence of length s
  PAPER.md:205            "we first bucket data according to the global batch size, then shuffle
                           the buckets to ensure data is randomly distributed"
  PAPER.md:203            "the proportion of wasted compute is less than 10%" (asserted, no formula)
No algorithm box, no tie rule, no RNG: the readings below are DESIGN.md sec 11.

Steps (plain python / numpy, in the paper's order):
  1 kept samples = samples whose group has keep != 0, ascending index
  2 workload w_i = w_lin*L_i + w_quad*L_i^2, arithmetic modulo 2^64 (python ints masked)
  3 stable ascending sort of the kept samples by w  (ties keep ascending index)
  4 consecutive buckets of bucket_size sorted samples; the last bucket may be short
  5 shuffle: buckets reordered by ascending (splitmix64(seed, b) >> 1, b), the counter-based
    generator of Steele, Lea & Flood's SplitMix restated here: z = seed + (b+1)*0x9E3779B97F4A7C15;
    z = (z ^ z>>30)*0xBF58476D1CE4E5B9; z = (z ^ z>>27)*0x94D049BB133111EB; z ^ z>>31 (mod 2^64)
  6 order = buckets concatenated; cu_out = prefix sums of the lengths in that order;
    src_token[cu_out[d] + t] = cu[order[d]] + t

Pins (tests/test_oracle_pins.py): hand-worked example (tests/golden/balance_example.txt); splitmix64
against the published test vector of the generator for seed 0 (first outputs of SplitMix64);
invariants (permutation of the kept set, sorted inside and across unshuffled buckets, multiset of
buckets preserved by the shuffle, token map is a bijection onto the kept tokens); numpy
argsort(kind="stable") as the library routine for step 3.
"""
from __future__ import annotations

import numpy as np

MASK64 = (1 << 64) - 1


def splitmix64(seed: int, b: int) -> int:
    """Step 5's key generator: the SplitMix64 output function applied to seed + (b+1)*gamma."""
    z = (seed + (b + 1) * 0x9E3779B97F4A7C15) & MASK64
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & MASK64
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & MASK64
    return z ^ (z >> 31)


def workload(L: int, w_lin: int, w_quad: int) -> int:
    """Step 2 (s^2 attention term, plus a linear term for everything else)."""
    return (w_lin * L + w_quad * L * L) & MASK64


def balance_plan(cu_seqlens, group_offsets, keep, w_lin, w_quad, bucket_size, seed, shuffle):
    """-> dict(order, n_kept, cu_out, src_token, n_tokens, buckets).  Inputs are 1-D integer
    arrays; group_offsets / keep may be None (every sample kept)."""
    cu = [int(x) for x in cu_seqlens]
    R = len(cu) - 1
    # step 1
    kept = []
    if group_offsets is None:
        kept = list(range(R))
    else:
        go = [int(x) for x in group_offsets]
        for g in range(len(go) - 1):
            if keep is None or int(keep[g]) != 0:
                kept.extend(range(go[g], go[g + 1]))
    # step 2
    w = {i: workload(cu[i + 1] - cu[i], w_lin, w_quad) for i in kept}
    # step 3: python's sort is stable; kept is ascending, so ties keep ascending index
    srt = sorted(kept, key=lambda i: w[i])
    # step 4
    buckets = [srt[a:a + bucket_size] for a in range(0, len(srt), bucket_size)]
    # step 5
    if shuffle:
        keys = [(splitmix64(seed, b) >> 1, b) for b in range(len(buckets))]
        perm = [b for _, b in sorted(keys)]
        buckets = [buckets[b] for b in perm]
    # step 6
    order = [i for bk in buckets for i in bk]
    cu_out = [0]
    src_token = []
    for i in order:
        L = cu[i + 1] - cu[i]
        src_token.extend(range(cu[i], cu[i] + L))
        cu_out.append(cu_out[-1] + L)
    return dict(order=np.array(order, dtype=np.int32), n_kept=len(order),
                cu_out=np.array(cu_out, dtype=np.int32),
                src_token=np.array(src_token, dtype=np.int32), n_tokens=len(src_token),
                buckets=buckets)


def wasted_fraction(lengths, buckets, w_lin, w_quad):
    """PAPER.md:203's quantity under the reading of DESIGN.md sec 11: a bucket is one global batch
    whose samples run in lock-step on data-parallel ranks, so every sample costs the bucket's
    maximum workload; waste = 1 - sum(w) / sum_b (|b| * max_{i in b} w_i)."""
    tot = 0
    padded = 0
    for bk in buckets:
        ws = [w_lin * int(lengths[i]) + w_quad * int(lengths[i]) ** 2 for i in bk]
        tot += sum(ws)
        padded += len(ws) * max(ws)
    return 1.0 - tot / padded if padded else 0.0
