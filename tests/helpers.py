"""Shared test helpers: build a seeded batch for a Workload and run the oracle on it.

Everything the oracle consumes is produced by paper_2507_22789_b200.inputs (seeded recipes) or
by the oracle itself (policy log-probs used to synthesise old/ref); nothing comes from the CUDA
path.
"""
from __future__ import annotations

import numpy as np
import torch

import oracle as O
from paper_2507_22789_b200 import inputs as I
from tests.harness import detie_old


def to_f64(t: torch.Tensor) -> np.ndarray:
    """Exact widening of an fp32/bf16 tensor to float64 on the host."""
    return t.detach().to("cpu", torch.float32).numpy().astype(np.float64)


class Batch:
    pass


def make_batch(w: I.Workload, seed: int = 0, device: str = "cpu", lengths=None, mask=None,
               old_std=None, policy_logp=None) -> Batch:
    """Seeded synthetic micro-batch.  Tensors on `device`; numpy twins on host.

    policy_logp: log-probs used to synthesise old/ref (None -> computed by the ORACLE, which is
    only sensible at sizes the oracle can finish)."""
    b = Batch()
    b.w = w
    lay = I.make_layout(w, seed, lengths)
    if mask is not None:
        lay.mask = np.asarray(mask, dtype=np.uint8)
    b.lay = lay
    b.T, b.R, b.G = lay.T, lay.R, lay.G
    H, W = I.make_hw(b.T, w.D, w.V, w.dtype, seed, device)
    y = I.sample_targets(H, W, w.tau, seed)
    b.H, b.W, b.y = H, W, y
    b.y_np = y.cpu().numpy()
    b.mask_np = lay.mask
    b.all_scored = bool(lay.mask.all())
    b.rewards_np = I.make_rewards(w, seed)
    b.scored_np = (b.mask_np != 0) & (b.y_np >= 0)
    if policy_logp is None:
        policy_logp = O.token_logprobs(to_f64(H), to_f64(W), b.y_np, None, w.tau)[0]
    b.policy_logp = np.asarray(policy_logp, dtype=np.float64)
    b.old_np = detie_old(b.policy_logp,
                         I.perturb_logp(b.policy_logp, w.old_std if old_std is None else old_std, seed + 1),
                         w.clip_lo, w.clip_hi)
    b.ref_np = I.perturb_logp(b.policy_logp, w.ref_std, seed + 2)
    dev = torch.device(device)
    b.mask_t = None if b.all_scored else torch.from_numpy(b.mask_np).to(dev)
    b.old_t = torch.from_numpy(b.old_np).to(dev)
    b.ref_t = torch.from_numpy(b.ref_np).to(dev)
    b.cu_t = torch.from_numpy(lay.cu_seqlens).to(dev)
    b.go_t = torch.from_numpy(lay.group_offsets).to(dev)
    b.rewards_t = torch.from_numpy(b.rewards_np).to(dev)
    return b


def oracle_run(b: Batch, adv_np, agg=O.AGG_TOKEN_MEAN, need_grads=True, grad_loss=1.0):
    w = b.w
    return O.grpo_forward_backward(to_f64(b.H), to_f64(b.W), b.y_np,
                                   None if b.all_scored else b.mask_np, w.tau,
                                   b.lay.cu_seqlens, adv_np, b.old_np, b.ref_np, w.clip_lo,
                                   w.clip_hi, w.beta, agg, grad_loss, need_grads)


def rel_fro(a, b) -> float:
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))


def elem_excess(got, ref, a, b, c=1e-5) -> float:
    """Per-element check beside the Frobenius norm, so that a localised error (one wrong tile of a
    large matrix) cannot hide in the norm: max_ij |got - ref| / (a |ref_ij| + b rms(ref_i,:) +
    c rms(ref)).  a bounds output rounding (relative to the element), b the accumulated rounding of
    the contraction's terms (relative to the row's scale), c is a floor for all-zero rows.  The
    caller asserts the result <= 1."""
    got = np.asarray(got, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    if ref.size == 0:
        return 0.0
    if ref.ndim == 1:
        got, ref = got[None, :], ref[None, :]
    rms_row = np.sqrt((ref ** 2).mean(axis=1, keepdims=True))
    rms_all = float(np.sqrt((ref ** 2).mean()))
    bound = a * np.abs(ref) + b * rms_row + c * rms_all
    bound = np.maximum(bound, 1e-300)
    return float((np.abs(got - ref) / bound).max())


# per-element bars: bf16 path -- dS rounded to bf16 (each term of the
# contraction off by <= 2^-9 relative, random sign: ~1.1e-3 of the row's scale, 6 sigma over
# 1e8 elements ~ 7e-3) and, for dH, the bf16 output rounding (<= 2^-9 |x|)
ELEM_BF16 = dict(a=4e-3, b=1.2e-2)
ELEM_F32 = dict(a=2e-5, b=1e-4)
