"""Harness-side input synthesis shared by bench.py and the GPU parity tests (so that the tests do not
import the benchmark script): approximate policy log-probs that centre the synthetic old / reference
log-probs, the de-tie of draws that land on a clip bound, and the device-resident batch.  None of it
is the product, none of it is the oracle, and none of it is ever an expected value."""
from __future__ import annotations

import numpy as np
import torch

from paper_2507_22789_b200 import inputs as I


def synth_policy_logp(H, W, y, tau=1.0, chunk=1024):
    """HARNESS-SIDE INPUT SYNTHESIS (not the product, not the oracle): approximate policy
    log-probs by plain torch ops, for batches too large for the oracle.  They only centre the
    synthetic old/ref log-probs ("policy log-probs + N(0, std)", BASELINE.json configs[0]) so that
    the ratio exp(logp - old) is near 1; they are never an expected value.  Lives here, outside the
    package, so that the product holds none of the method's arithmetic twice."""
    T = H.shape[0]
    out = torch.empty(T, dtype=torch.float32, device=H.device)
    Wf = W if H.is_cuda else W.float()
    for a in range(0, T, chunk):
        e = min(T, a + chunk)
        Hc = H[a:e] if H.is_cuda else H[a:e].float()
        z = (Hc @ Wf.T).float() / tau
        lp = z - torch.logsumexp(z, dim=1, keepdim=True)
        out[a:e] = lp.gather(1, y[a:e].clamp(min=0).long().unsqueeze(1)).squeeze(1)
    return out.cpu().numpy().astype(np.float64)


def detie_old(policy_logp, old, clip_lo, clip_hi, margin=1e-4):
    """HARNESS-SIDE INPUT SYNTHESIS: the clip branch is a discontinuous decision on rho =
    exp(logp - old); a synthetic old log-prob that lands within `margin` of a clip bound would let
    fp32-vs-fp64 rounding of logp (~1e-6) flip the branch and change g_t by orders of magnitude
    (reading 19).  Such draws (about 1e-5 of the tokens at std 0.3) are moved 0.01 away
    from the bound, so that both sides take the same branch for every token of a seeded batch."""
    old = np.array(old, dtype=np.float32)
    rho = np.exp(np.asarray(policy_logp, dtype=np.float64) - old.astype(np.float64))
    near = (np.abs(rho - (1.0 + clip_hi)) < margin) | (np.abs(rho - (1.0 - clip_lo)) < margin)
    old[near] -= np.float32(0.01)
    return old


class DeviceBatch:
    def __init__(self, w: I.Workload, seed: int, device, w_seed=None):
        """w_seed: seed of the replicated weight W (multi-GPU: the same on every rank, while the
        tokens follow `seed`)."""
        self.w = w
        lay = I.make_layout(w, seed)
        self.lay = lay
        self.T = lay.T
        self.H, self.W = I.make_hw(lay.T, w.D, w.V, w.dtype, seed, device)
        if w_seed is not None:
            _, self.W = I.make_hw(1, w.D, w.V, w.dtype, w_seed, device)
        self.y = I.sample_targets(self.H, self.W, w.tau, seed)
        self.mask = None if lay.mask.all() else torch.from_numpy(lay.mask).to(device)
        self.n_scored = int(((lay.mask != 0) & (self.y.cpu().numpy() >= 0)).sum())
        self.rewards = torch.from_numpy(I.make_rewards(w, seed)).to(device)
        self.go = torch.from_numpy(lay.group_offsets).to(device)
        self.cu = torch.from_numpy(lay.cu_seqlens).to(device)
        if w.backward:
            pol = synth_policy_logp(self.H, self.W, self.y, w.tau)
            self.old = torch.from_numpy(detie_old(pol, I.perturb_logp(pol, w.old_std, seed + 1),
                                                  w.clip_lo, w.clip_hi)).to(device)
            self.ref = torch.from_numpy(I.perturb_logp(pol, w.ref_std, seed + 2)).to(device)
            self.dH = torch.empty(lay.T, w.D, dtype=self.H.dtype, device=device)
            self.dW = torch.empty(w.V, w.D, dtype=torch.float32, device=device)
