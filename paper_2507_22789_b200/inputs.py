"""Seeded synthetic inputs shaped like the RLHF micro-batches of BASELINE.json:configs.

This module is the ONLY code shared by the oracle-side tests and the CUDA path's tests/bench.
It holds none of the method's arithmetic (no softmax, no log-probs, no advantages, no loss): it
draws random tensors, lays out sequences, and samples target ids.  The recipe is DESIGN.md sec 4.

Target sampling needs a draw from Categorical(softmax(z)); it uses a plain ``torch.matmul`` and the
Gumbel-max trick (argmax of z + Gumbel noise -- no normalisation is ever computed) as input
synthesis (``sample_targets``), on whatever device H and W live on.  Policy log-probs needed to
synthesise old/ref log-probs are passed IN by the caller (``perturb_logp``): the tests take them
from the oracle, bench.py from its own harness-side helper.
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace
from typing import Optional

import numpy as np
import torch


@dataclass(frozen=True)
class Workload:
    """One RLHF micro-batch recipe (BASELINE.json:configs[i])."""
    name: str
    D: int
    V: int
    dtype: str                      # "f32" | "bf16"
    groups: int
    group_size: int
    seq_len: int = 0                # fixed tokens per sample (0 -> lognormal lengths)
    prompt_len: int = 0             # leading tokens of each sample with mask 0
    tau: float = 1.0
    rewards: str = "bernoulli"      # "bernoulli" | "uniform" | "bernoulli_nonconst" | "cfg3"
    drop_constant_groups: bool = False
    backward: bool = True
    lognormal: tuple = (6.5, 1.0, 32, 16384)   # mu, sigma, lo, hi (config 3)
    clip_lo: float = 0.2
    clip_hi: float = 0.2
    beta: float = 0.04
    old_std: float = 0.05
    ref_std: float = 0.1


CONFIGS = {
    # configs[0]: tiny fp32 reference
    0: Workload("cfg0_tiny_f32", D=256, V=4096, dtype="f32", groups=4, group_size=4, seq_len=16),
    # configs[1]: 7B-class forward-only scoring
    1: Workload("cfg1_7b_fwd", D=3584, V=152064, dtype="bf16", groups=8, group_size=8,
                seq_len=256, rewards="uniform", backward=False),
    # configs[2]: 8B-class training micro-batch, 75 % response mask
    2: Workload("cfg2_8b_train", D=4096, V=128256, dtype="bf16", groups=4, group_size=8,
                seq_len=1024, prompt_len=256),
    # configs[3]: long-tail dynamic-sampling batch
    3: Workload("cfg3_longtail", D=5120, V=152064, dtype="bf16", groups=16, group_size=16,
                seq_len=0, rewards="cfg3", drop_constant_groups=True),
    # configs[4]: large-vocab stress, tau = 0.7
    4: Workload("cfg4_bigvocab", D=8192, V=256000, dtype="bf16", groups=1, group_size=8,
                seq_len=1024, tau=0.7, rewards="bernoulli_nonconst"),
}


def reduced(w: Workload, **kw) -> Workload:
    """Same recipe with some fields overridden (parity cases at reduced T, odd shapes, ...)."""
    return replace(w, **kw)


def _gen(seed: int, device="cpu") -> torch.Generator:
    g = torch.Generator(device=device)
    g.manual_seed(int(seed))
    return g


def torch_dtype(dtype: str):
    return {"f32": torch.float32, "bf16": torch.bfloat16}[dtype]


# ---------------------------------------------------------------------------------------------
# layout: lengths, cu_seqlens, group_offsets, mask  (integer work, bit-exact by construction)
# ---------------------------------------------------------------------------------------------
def make_lengths(w: Workload, seed: int = 0) -> np.ndarray:
    R = w.groups * w.group_size
    if w.seq_len > 0:
        return np.full(R, w.seq_len, dtype=np.int64)
    mu, sigma, lo, hi = w.lognormal
    rng = np.random.default_rng(seed)
    L = np.rint(rng.lognormal(mu, sigma, R))
    return np.clip(L, lo, hi).astype(np.int64)


@dataclass
class Layout:
    lengths: np.ndarray             # [R]
    cu_seqlens: np.ndarray          # [R+1] int32
    group_offsets: np.ndarray       # [G+1] int32 (in responses)
    mask: np.ndarray                # [T] uint8
    T: int = 0
    R: int = 0
    G: int = 0


def make_layout(w: Workload, seed: int = 0, lengths: Optional[np.ndarray] = None) -> Layout:
    L = make_lengths(w, seed) if lengths is None else np.asarray(lengths, dtype=np.int64)
    R = len(L)
    cu = np.zeros(R + 1, dtype=np.int64)
    cu[1:] = np.cumsum(L)
    T = int(cu[-1])
    assert T < 2 ** 31
    mask = np.ones(T, dtype=np.uint8)
    if w.prompt_len > 0:
        for r in range(R):
            mask[cu[r]:cu[r] + min(w.prompt_len, L[r])] = 0
    G = R // w.group_size
    go = (np.arange(G + 1) * w.group_size).astype(np.int32)
    return Layout(L, cu.astype(np.int32), go, mask, T, R, G)


def make_rewards(w: Workload, seed: int = 0) -> np.ndarray:
    """rewards[R] float32.  Bernoulli(0.5) / U[0,1] / config-3 recipe."""
    rng = np.random.default_rng(seed + 7919)
    G, n = w.groups, w.group_size
    if w.rewards == "uniform":
        return rng.random(G * n).astype(np.float32)
    r = np.zeros((G, n), dtype=np.float32)
    for g in range(G):
        row = (rng.random(n) < 0.5).astype(np.float32)
        if w.rewards in ("bernoulli_nonconst", "cfg3"):
            while np.all(row == row[0]):
                row = (rng.random(n) < 0.5).astype(np.float32)
        if w.rewards == "cfg3" and g % 4 == 3:
            row[:] = float((g // 4) % 2)          # constant groups, alternately all-0 / all-1
        r[g] = row
    return r.reshape(-1)


# ---------------------------------------------------------------------------------------------
# tensors: H, W, targets, perturbed log-probs
# ---------------------------------------------------------------------------------------------
def make_hw(T: int, D: int, V: int, dtype: str, seed: int = 0, device="cpu",
            w_std: float = 0.02):
    """H ~ N(0,1), each row scaled to unit RMS in fp64, THEN rounded to dtype; W ~ N(0, w_std)."""
    g = _gen(seed, device)
    td = torch_dtype(dtype)
    H = torch.empty(T, D, dtype=td, device=device)
    step = max(1, (1 << 24) // max(D, 1))
    for a in range(0, T, step):
        b = min(T, a + step)
        x = torch.randn(b - a, D, generator=g, device=device, dtype=torch.float64)
        x = x / x.pow(2).mean(dim=1, keepdim=True).sqrt()
        H[a:b] = x.to(td)
    W = torch.empty(V, D, dtype=td, device=device)
    for a in range(0, V, step):
        b = min(V, a + step)
        W[a:b] = (torch.randn(b - a, D, generator=g, device=device, dtype=torch.float32)
                  * w_std).to(td)
    return H, W


def sample_targets(H: torch.Tensor, W: torch.Tensor, tau: float = 1.0, seed: int = 0,
                   chunk: int = 1024) -> torch.Tensor:
    """y[t] ~ Categorical(softmax(H[t].W^T / tau)) by Gumbel-max.  Input synthesis only."""
    T = H.shape[0]
    g = _gen(seed + 104729, H.device)
    y = torch.empty(T, dtype=torch.int32, device=H.device)
    Wf = W if W.dtype != torch.bfloat16 or H.is_cuda else W.float()
    for a in range(0, T, chunk):
        b = min(T, a + chunk)
        Hc = H[a:b] if Wf.dtype == H.dtype else H[a:b].float()
        z = (Hc @ Wf.T).float() / tau
        u = torch.rand(z.shape, generator=g, device=H.device, dtype=torch.float32)
        u = u.clamp_(1e-12, 1.0 - 1e-7)
        z = z - torch.log(-torch.log(u))
        y[a:b] = z.argmax(dim=1).to(torch.int32)
    return y


def perturb_logp(policy_logp, std: float, seed: int) -> np.ndarray:
    """old / ref log-probs = policy log-probs + N(0, std), fp32 (configs[0])."""
    rng = np.random.default_rng(seed)
    lp = np.asarray(policy_logp, dtype=np.float64)
    return (lp + rng.normal(0.0, std, lp.shape)).astype(np.float32)


def random_mask(T: int, p_keep: float, seed: int) -> np.ndarray:
    rng = np.random.default_rng(seed + 31)
    return (rng.random(T) < p_keep).astype(np.uint8)


def drop_groups(layout: Layout, keep: np.ndarray, group_size: int):
    """Indices of the responses / tokens that survive the dynamic-sampling filter, plus the
    repacked layout (dropped prompts never reach stage 3/4)."""
    keep = np.asarray(keep).astype(bool)
    resp_keep = np.repeat(keep, group_size)
    resp_idx = np.nonzero(resp_keep)[0]
    cu = layout.cu_seqlens.astype(np.int64)
    tok_idx = np.concatenate([np.arange(cu[r], cu[r + 1]) for r in resp_idx]) \
        if len(resp_idx) else np.zeros(0, dtype=np.int64)
    L = layout.lengths[resp_idx]
    new_cu = np.zeros(len(L) + 1, dtype=np.int64)
    new_cu[1:] = np.cumsum(L)
    G = int(keep.sum())
    new = Layout(L, new_cu.astype(np.int32),
                 (np.arange(G + 1) * group_size).astype(np.int32),
                 layout.mask[tok_idx], int(new_cu[-1]), len(L), G)
    return resp_idx, tok_idx, new
