"""Thin ctypes binding over csrc/libgcore.so (the C ABI of include/gcore.h).

Argument marshalling only: every step of the path runs in the library's CUDA kernels.  PyTorch
provides device memory (tensors, the workspace) and the current stream.  There is no CPU or
eager fallback: a missing library raises ImportError, a non-zero gc_status raises GcoreError.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "csrc", "libgcore.so")

GC_F32, GC_BF16, GC_BF16_SIMT = 0, 1, 2
GC_AGG_TOKEN_MEAN, GC_AGG_SEQ_MEAN = 0, 1
GC_OP_LOGPROBS, GC_OP_LOSS_FWD, GC_OP_LOSS_BWD = 0, 1, 2

EXPORTS = [
    "gc_status_string", "gc_last_cuda_error", "gc_version", "gc_workspace_bytes", "gc_token_logprobs",
    "gc_host_staging_bytes", "gc_logprobs_host_workspace_bytes", "gc_host_band_plan",
    "gc_token_logprobs_host", "gc_grpo_advantages", "gc_grpo_loss_fwd",
    "gc_grpo_loss_bwd", "gc_validate_targets", "gc_compact_rows", "gc_grpo_token_loss",
    "gc_debug_gemm_bf16", "gc_kernel_timing_begin", "gc_kernel_timing_end",
    "gc_balance_workspace_bytes", "gc_balance_plan", "gc_gather_rows", "gc_gather_1d",
    "gc_multi_workspace_bytes", "gc_token_logprobs_multi",
    "gc_grpo_loss_bwd_reduce_scatter",
    "gc_loss_workspace_bytes", "gc_bwd_workspace_bytes",
    "gc_step_host_workspace_bytes", "gc_grpo_step_host",
    "gc_attention_workspace_bytes", "gc_attention_allgather_kv",
    "gc_value_head_fwd", "gc_gae", "gc_critic_workspace_bytes", "gc_value_loss", "gc_value_head_bwd",
    "gc_value_loss_static_scratch",
]


class GcoreError(RuntimeError):
    pass


def _load() -> C.CDLL:
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            f"{LIB_PATH} is missing: build it with `python -m paper_2507_22789_b200.build` "
            "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp, i64, i32, f32, sz = C.c_void_p, C.c_int64, C.c_int32, C.c_float, C.c_size_t
    ci = C.c_int
    lib.gc_status_string.restype = C.c_char_p
    lib.gc_status_string.argtypes = [ci]
    lib.gc_last_cuda_error.restype = C.c_char_p
    lib.gc_last_cuda_error.argtypes = []
    lib.gc_version.restype = ci
    lib.gc_workspace_bytes.restype = sz
    lib.gc_workspace_bytes.argtypes = [ci, i64, i64, i64, ci, i64]
    head = [vp, i64, vp, i64, ci, vp, vp, i64, i64, i64, f32]
    loss = [vp, i32, vp, vp, vp, f32, f32, f32, ci]
    lib.gc_token_logprobs.argtypes = head + [vp, vp, vp, vp, sz, vp]
    lib.gc_host_staging_bytes.restype = sz
    lib.gc_host_staging_bytes.argtypes = [i64, i64, ci]
    lib.gc_logprobs_host_workspace_bytes.restype = sz
    lib.gc_logprobs_host_workspace_bytes.argtypes = [i64, i64, i64, ci]
    lib.gc_host_band_plan.argtypes = [i64, i64, i64, ci, C.POINTER(i64)]
    lib.gc_token_logprobs_host.argtypes = [vp, vp, i64, ci, vp, vp, i64, i64, i64, f32, vp, vp,
                                           vp, sz, vp]
    lib.gc_step_host_workspace_bytes.restype = sz
    lib.gc_step_host_workspace_bytes.argtypes = [i64, i64, i64, ci, i32, i32, ci]
    lib.gc_grpo_step_host.argtypes = [vp, vp, i64, ci, vp, vp, i64, i64, i64, f32, vp, i32, vp, vp, i32,
                                      f32, vp, vp, f32, f32, f32, ci, f32, vp, vp, vp, vp, i64, ci, ci,
                                      vp, sz, vp]
    lib.gc_attention_workspace_bytes.restype = sz
    lib.gc_attention_workspace_bytes.argtypes = [i64, i64, i32]
    lib.gc_attention_allgather_kv.argtypes = [vp, C.POINTER(vp), C.POINTER(vp), C.POINTER(i64), i32, i32,
                                              i32, i32, i32, vp, i32, ci, i32, f32, i32, vp, vp, vp, sz, vp]
    lib.gc_grpo_advantages.argtypes = [vp, vp, i32, f32, ci, ci, vp, vp, vp]
    lib.gc_grpo_loss_fwd.argtypes = head + loss + [vp, vp, vp, vp, vp, sz, vp]
    lib.gc_bwd_workspace_bytes.restype = sz
    lib.gc_bwd_workspace_bytes.argtypes = [i64, i64, i64, ci, i64, ci]
    lib.gc_grpo_loss_bwd.argtypes = head + loss + [vp, vp, f32, vp, i64, vp, i64, ci, ci, i64,
                                                   vp, vp, sz, vp]
    lib.gc_grpo_loss_bwd_reduce_scatter.argtypes = head + loss + [vp, vp, f32, vp, i64, C.POINTER(vp),
                                                                  i32, i64, i64, i64, vp, vp, sz, vp]
    lib.gc_validate_targets.argtypes = [vp, vp, i64, i64, C.POINTER(i64), vp]
    lib.gc_compact_rows.argtypes = [vp, i64, ci, vp, vp, i64, i64, vp, vp, vp, vp, sz, vp]
    lib.gc_grpo_token_loss.argtypes = [vp, vp, vp, vp, vp, i64, vp, i32, vp, f32, f32, f32, ci,
                                       f32, vp, vp, vp, sz, vp]
    lib.gc_loss_workspace_bytes.restype = sz
    lib.gc_loss_workspace_bytes.argtypes = [i64, i32]
    lib.gc_debug_gemm_bf16.argtypes = [vp, i64, ci, vp, i64, ci, vp, i64, i64, i64, i64, ci, ci, ci,
                                       ci, ci, ci, ci, ci, ci, vp]
    u64 = C.c_uint64
    lib.gc_balance_workspace_bytes.restype = sz
    lib.gc_balance_workspace_bytes.argtypes = [i32]
    lib.gc_balance_plan.argtypes = [vp, i32, vp, vp, i32, u64, u64, i32, u64, ci, vp, vp, vp, vp, vp,
                                    vp, sz, vp]
    lib.gc_gather_rows.argtypes = [vp, i64, ci, i64, vp, vp, i64, vp, vp]
    lib.gc_gather_1d.argtypes = [vp, vp, vp, i64, vp, vp]
    lib.gc_multi_workspace_bytes.restype = sz
    lib.gc_multi_workspace_bytes.argtypes = [i64, i64, i64, i32]
    lib.gc_token_logprobs_multi.argtypes = [vp, i64, vp, i64, ci, vp, i32, i64, i64, i64, f32, vp, vp,
                                            vp, vp, sz, vp]
    lib.gc_value_head_fwd.argtypes = [vp, i64, ci, vp, f32, i64, i64, vp, vp]
    lib.gc_gae.argtypes = [vp, vp, vp, vp, i32, i64, f32, f32, vp, vp, vp]
    lib.gc_critic_workspace_bytes.restype = sz
    lib.gc_critic_workspace_bytes.argtypes = [i64, i64]
    lib.gc_value_loss.argtypes = [vp, vp, vp, vp, i64, f32, f32, vp, vp, vp, sz, vp]
    lib.gc_value_head_bwd.argtypes = [vp, i64, ci, vp, vp, i64, i64, vp, i64, vp, vp, vp, sz, vp]
    lib.gc_value_loss_static_scratch.argtypes = [vp, vp, vp, vp, i64, f32, f32, vp, vp, vp]
    lib.gc_kernel_timing_begin.argtypes = []
    lib.gc_kernel_timing_end.argtypes = [C.POINTER(f32), C.POINTER(i32)]
    for name in EXPORTS:
        fn = getattr(lib, name)
        if name not in ("gc_status_string", "gc_last_cuda_error", "gc_workspace_bytes", "gc_host_staging_bytes",
                        "gc_logprobs_host_workspace_bytes",
                        "gc_balance_workspace_bytes", "gc_multi_workspace_bytes",
                        "gc_loss_workspace_bytes", "gc_bwd_workspace_bytes",
                        "gc_step_host_workspace_bytes", "gc_attention_workspace_bytes",
                        "gc_critic_workspace_bytes"):
            fn.restype = ci
    return lib


_lib = _load()


def lib() -> C.CDLL:
    return _lib


def _check(status: int):
    if status != 0:
        msg = _lib.gc_status_string(status).decode()
        if status == 8:
            msg += " (" + _lib.gc_last_cuda_error().decode() + ")"
        raise GcoreError(msg)


def _ptr(t: Optional[torch.Tensor]):
    return None if t is None else C.c_void_p(t.data_ptr())


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def dtype_code(t: torch.Tensor, simt: bool = False) -> int:
    if t.dtype == torch.float32:
        return GC_F32
    if t.dtype == torch.bfloat16:
        return GC_BF16_SIMT if simt else GC_BF16
    raise GcoreError(f"unsupported dtype {t.dtype}")


_ws_cache: dict = {}


def workspace(nbytes: int, device, slot: str = "") -> torch.Tensor:
    """A cached device buffer of at least nbytes (torch caching allocator: 512-byte aligned), one
    per (device, current stream, slot): calls on different streams never share scratch, and a
    buffer that is dropped when a larger one is needed is only ever reused by later work of the
    same stream (the caching allocator's reuse is stream-ordered).  slot "fwd" is the workspace of
    gc_grpo_loss_fwd, kept apart so that the backward can reuse the forward's row selection."""
    key = (str(device), int(torch.cuda.current_stream(device).cuda_stream), slot)
    buf = _ws_cache.get(key)
    if buf is None or buf.numel() < nbytes:
        _ws_cache[key] = buf = torch.empty(max(nbytes, 1 << 20), dtype=torch.uint8, device=device)
    return buf


_fwd_generation: dict = {}


class FwdState:
    """What gc_grpo_loss_fwd leaves for the backward: its workspace (row list, compacted targets and
    H) plus the facts needed to tell whether it still describes the same batch.  The workspace is
    cached per (device, stream), so the NEXT forward on that stream -- another micro-batch --
    overwrites it; a backward handed a state that is no longer the latest one of its slot, or one made
    for other shapes / another mask, silently falls back to recomputing the row selection (the C call
    gets fwd_state = NULL), which is always correct."""

    def __init__(self, ws, key, sig):
        self.ws, self.key, self.sig = ws, key, sig
        self.gen = _fwd_generation[key] = _fwd_generation.get(key, 0) + 1

    def usable_for(self, sig) -> bool:
        return (_fwd_generation.get(self.key) == self.gen and self.sig == sig
                and _ws_cache.get(self.key) is self.ws)


def _state_sig(H, targets, mask, T, D, V, dt):
    return (H.data_ptr(), targets.data_ptr(), None if mask is None else mask.data_ptr(), T, D, V, dt)


def _state_ptr(fwd_state, sig):
    if fwd_state is None:
        return None
    if isinstance(fwd_state, FwdState):
        return _ptr(fwd_state.ws) if fwd_state.usable_for(sig) else None
    return _ptr(fwd_state)          # a raw workspace tensor: the caller vouches for it


def workspace_bytes(op: int, T: int, D: int, V: int, dtype: int, chunk_tokens: int = 0) -> int:
    return int(_lib.gc_workspace_bytes(op, T, D, V, dtype, chunk_tokens))


def _head_args(H, W, targets, mask, tau, simt):
    assert H.dim() == 2 and W.dim() == 2 and H.stride(1) == 1 and W.stride(1) == 1
    T, D = H.shape
    V = W.shape[0]
    assert W.shape[1] == D and H.dtype == W.dtype
    assert targets.dtype == torch.int32 and targets.numel() == T and targets.is_contiguous()
    if mask is not None:
        assert mask.dtype == torch.uint8 and mask.numel() == T and mask.is_contiguous()
    dt = dtype_code(H, simt)
    args = [_ptr(H), H.stride(0) if T > 0 else D, _ptr(W), W.stride(0), dt, _ptr(targets),
            _ptr(mask), T, D, V, float(tau)]
    return args, T, D, V, dt


def gc_token_logprobs(H, W, targets, mask=None, temperature=1.0, *, want_entropy=True,
                      want_lse=True, simt=False):
    """-> (logp, entropy|None, lse|None), float32 [T] on H's device."""
    args, T, D, V, dt = _head_args(H, W, targets, mask, temperature, simt)
    dev = H.device
    logp = torch.empty(T, dtype=torch.float32, device=dev)
    ent = torch.empty(T, dtype=torch.float32, device=dev) if want_entropy else None
    lse = torch.empty(T, dtype=torch.float32, device=dev) if want_lse else None
    nb = workspace_bytes(GC_OP_LOGPROBS, T, D, V, dt)
    ws = workspace(nb, dev)
    _check(_lib.gc_token_logprobs(*args, _ptr(logp), _ptr(ent), _ptr(lse), _ptr(ws), ws.numel(),
                                  _stream()))
    return logp, ent, lse


def gc_token_logprobs_host(H_host, W, targets_host, mask_host=None, temperature=1.0, *,
                           logp_host=None, entropy_host=None, simt=False):
    """Per-step inputs/outputs in (pinned) HOST memory; W on the device.  Enqueues H2D copies,
    the kernels and D2H copies on the current stream; the caller synchronises."""
    T, D = H_host.shape
    V = W.shape[0]
    dt = dtype_code(W, simt)
    assert not H_host.is_cuda and H_host.is_contiguous() and W.is_cuda
    if logp_host is None:
        logp_host = torch.empty(T, dtype=torch.float32).pin_memory()
    nb = int(_lib.gc_logprobs_host_workspace_bytes(T, D, V, dt))
    ws = workspace(nb, W.device)
    _check(_lib.gc_token_logprobs_host(_ptr(H_host), _ptr(W), W.stride(0), dt, _ptr(targets_host),
                                       _ptr(mask_host), T, D, V, float(temperature),
                                       _ptr(logp_host), _ptr(entropy_host), _ptr(ws), ws.numel(),
                                       _stream()))
    return logp_host, entropy_host


def gc_grpo_step_host(H_host, W, targets_host, mask_host, temperature, cu_host, rewards_host,
                      group_offsets_host, old_host, ref_host, dW, *, clip_lo=0.2, clip_hi=0.2,
                      beta=0.04, agg=GC_AGG_TOKEN_MEAN, grad_loss=1.0, adv_eps=1e-6, out5_host=None,
                      logp_host=None, dH_host=None, accumulate_dW=False):
    """One training step of the loss head from (pinned) HOST buffers: -> (out5_host, dH_host);
    dW [V,D] (fp32 or bf16) stays on the device.  Enqueues on the current stream; the caller
    synchronises before reading the host outputs."""
    T, D = H_host.shape
    V = W.shape[0]
    dt = dtype_code(W)
    R, G = cu_host.numel() - 1, group_offsets_host.numel() - 1
    assert not H_host.is_cuda and H_host.is_contiguous() and W.is_cuda and dW.is_cuda
    if out5_host is None:
        out5_host = torch.empty(5, dtype=torch.float32).pin_memory()
    if dH_host is None:
        dH_host = torch.empty(T, D, dtype=H_host.dtype).pin_memory()
    dwt = {torch.float32: GC_F32, torch.bfloat16: GC_BF16}[dW.dtype]
    ws = workspace(int(_lib.gc_step_host_workspace_bytes(T, D, V, dt, R, G, dwt)), W.device, "step")
    _check(_lib.gc_grpo_step_host(
        _ptr(H_host), _ptr(W), W.stride(0), dt, _ptr(targets_host), _ptr(mask_host), T, D, V,
        float(temperature), _ptr(cu_host), R, _ptr(rewards_host), _ptr(group_offsets_host), G,
        float(adv_eps), _ptr(old_host), _ptr(ref_host), float(clip_lo), float(clip_hi), float(beta),
        int(agg), float(grad_loss), _ptr(out5_host), _ptr(logp_host), _ptr(dH_host), _ptr(dW),
        dW.stride(0), dwt, int(accumulate_dW), _ptr(ws), ws.numel(), _stream()))
    return out5_host, dH_host


def gc_grpo_advantages(rewards, group_offsets, eps=1e-6, unbiased_std=False,
                       drop_constant_groups=False):
    """-> (adv float32 [R], keep uint8 [G])."""
    assert rewards.dtype == torch.float32 and group_offsets.dtype == torch.int32
    G = group_offsets.numel() - 1
    adv = torch.empty_like(rewards)
    keep = torch.empty(max(G, 0), dtype=torch.uint8, device=rewards.device)
    _check(_lib.gc_grpo_advantages(_ptr(rewards), _ptr(group_offsets), G, float(eps),
                                   int(unbiased_std), int(drop_constant_groups), _ptr(adv),
                                   _ptr(keep), _stream()))
    return adv, keep


def _loss_args(cu_seqlens, adv, old_logp, ref_logp, clip_lo, clip_hi, beta, agg):
    assert cu_seqlens.dtype == torch.int32 and adv.dtype == torch.float32
    R = cu_seqlens.numel() - 1
    return [_ptr(cu_seqlens), R, _ptr(adv), _ptr(old_logp), _ptr(ref_logp), float(clip_lo),
            float(clip_hi), float(beta), int(agg)]


def gc_grpo_loss_fwd(H, W, targets, mask, temperature, cu_seqlens, adv, old_logp, ref_logp,
                     clip_lo=0.2, clip_hi=0.2, beta=0.04, agg=GC_AGG_TOKEN_MEAN, *, simt=False):
    """-> dict(out5=[loss, pg_loss, kl_mean, clip_frac, n_scored] (device), logp, entropy, lse)."""
    args, T, D, V, dt = _head_args(H, W, targets, mask, temperature, simt)
    dev = H.device
    out5 = torch.empty(5, dtype=torch.float32, device=dev)
    logp = torch.empty(T, dtype=torch.float32, device=dev)
    ent = torch.empty(T, dtype=torch.float32, device=dev)
    lse = torch.empty(T, dtype=torch.float32, device=dev)
    nb = workspace_bytes(GC_OP_LOSS_FWD, T, D, V, dt)
    ws = workspace(nb, dev, "fwd")
    _check(_lib.gc_grpo_loss_fwd(*args, *_loss_args(cu_seqlens, adv, old_logp, ref_logp, clip_lo,
                                                    clip_hi, beta, agg),
                                 _ptr(out5), _ptr(logp), _ptr(ent), _ptr(lse), _ptr(ws),
                                 ws.numel(), _stream()))
    # state: the forward's workspace (row list, compacted H), valid until the next forward on this
    # stream; pass it to gc_grpo_loss_bwd(fwd_state=...) to skip the row selection there
    key = (str(dev), int(torch.cuda.current_stream(dev).cuda_stream), "fwd")
    state = FwdState(ws, key, _state_sig(H, targets, mask, T, D, V, dt))
    return dict(out5=out5, logp=logp, entropy=ent, lse=lse, state=state)


def gc_grpo_loss_bwd(H, W, targets, mask, temperature, cu_seqlens, adv, old_logp, ref_logp,
                     logp, lse, clip_lo=0.2, clip_hi=0.2, beta=0.04, agg=GC_AGG_TOKEN_MEAN,
                     grad_loss=1.0, *, dH=None, dW=None, accumulate_dW=False, chunk_tokens=0,
                     simt=False, dW_dtype=torch.float32, fwd_state=None):
    """-> (dH [T,D] in H's dtype, dW [V,D] float32 or bfloat16).  fwd_state: the "state" entry of
    gc_grpo_loss_fwd's result for the same inputs (optional: reuses its row selection)."""
    args, T, D, V, dt = _head_args(H, W, targets, mask, temperature, simt)
    dev = H.device
    if dH is None:
        dH = torch.empty(T, D, dtype=H.dtype, device=dev)
    if dW is None:
        assert not accumulate_dW
        dW = torch.empty(V, D, dtype=dW_dtype, device=dev)
    dwt = {torch.float32: GC_F32, torch.bfloat16: GC_BF16}[dW.dtype]
    nb = int(_lib.gc_bwd_workspace_bytes(T, D, V, dt, chunk_tokens, dwt))
    ws = workspace(nb, dev)
    _check(_lib.gc_grpo_loss_bwd(*args, *_loss_args(cu_seqlens, adv, old_logp, ref_logp, clip_lo,
                                                    clip_hi, beta, agg),
                                 _ptr(logp), _ptr(lse), float(grad_loss), _ptr(dH),
                                 dH.stride(0) if T > 0 else D, _ptr(dW), dW.stride(0), dwt,
                                 int(accumulate_dW), int(chunk_tokens),
                                 _state_ptr(fwd_state, _state_sig(H, targets, mask, T, D, V, dt)),
                                 _ptr(ws), ws.numel(), _stream()))
    return dH, dW


def gc_grpo_token_loss(logp, old_logp, ref_logp, targets, mask, cu_seqlens, adv, clip_lo=0.2,
                       clip_hi=0.2, beta=0.04, agg=GC_AGG_TOKEN_MEAN, grad_loss=1.0,
                       want_grad=True):
    """The loss kernels alone: -> (out5 device tensor, g [T] or None)."""
    T = logp.numel()
    dev = logp.device
    out5 = torch.empty(5, dtype=torch.float32, device=dev)
    g = torch.empty(T, dtype=torch.float32, device=dev) if want_grad else None
    R = cu_seqlens.numel() - 1
    ws = workspace(int(_lib.gc_loss_workspace_bytes(T, R)), dev)
    _check(_lib.gc_grpo_token_loss(_ptr(logp), _ptr(old_logp), _ptr(ref_logp), _ptr(targets),
                                   _ptr(mask), T, _ptr(cu_seqlens), R, _ptr(adv), float(clip_lo),
                                   float(clip_hi), float(beta), int(agg), float(grad_loss),
                                   _ptr(out5), _ptr(g), _ptr(ws), ws.numel(), _stream()))
    return out5, g


def gc_compact_rows(H, targets, mask, gather=True):
    """-> (rows int32 [T] (first n valid), n_rows int32 [1], Hs [T,D] or None)."""
    T, D = H.shape
    dev = H.device
    rows = torch.empty(max(T, 1), dtype=torch.int32, device=dev)
    n = torch.zeros(1, dtype=torch.int32, device=dev)
    Hs = torch.empty(T, D, dtype=H.dtype, device=dev) if gather else None
    dt = dtype_code(H)
    nb = workspace_bytes(GC_OP_LOGPROBS, T, D, 8, GC_BF16)
    ws = workspace(nb, dev)
    _check(_lib.gc_compact_rows(_ptr(H), H.stride(0) if T > 0 else D, dt, _ptr(targets),
                                _ptr(mask), T, D, _ptr(rows), _ptr(n), _ptr(Hs), _ptr(ws),
                                ws.numel(), _stream()))
    return rows, n, Hs


def gc_validate_targets(targets, mask, V) -> int:
    n = C.c_int64(0)
    _check(_lib.gc_validate_targets(_ptr(targets), _ptr(mask), targets.numel(), int(V),
                                    C.byref(n), _stream()))
    return int(n.value)


def gc_debug_gemm_bf16(A, B, a_mn_major=False, b_mn_major=False, C_out=None, accumulate=False,
                       cta_group=2, dynamic_schedule=True, dual_n=False, cluster4=False,
                       c_major=False, m_band=0, chunk_ntiles=0, n_band=0):
    """C[M,N] f32 = A.B on the tcgen05 tile engine (unit test of the engine, incl. the item
    orders of the path's kernels: c_major/m_band/chunk_ntiles, n_band)."""
    if a_mn_major:
        K, M = A.shape
    else:
        M, K = A.shape
    if b_mn_major:
        Kb, N = B.shape
    else:
        N, Kb = B.shape
    assert K == Kb and A.dtype == torch.bfloat16 and B.dtype == torch.bfloat16
    if C_out is None:
        C_out = torch.zeros(M, N, dtype=torch.float32, device=A.device)
    _check(_lib.gc_debug_gemm_bf16(_ptr(A), A.stride(0), int(a_mn_major), _ptr(B), B.stride(0),
                                   int(b_mn_major), _ptr(C_out), C_out.stride(0), M, N, K,
                                   int(accumulate), int(cta_group), int(dynamic_schedule),
                                   int(dual_n), int(cluster4), int(c_major), int(m_band),
                                   int(chunk_ntiles), int(n_band), _stream()))
    return C_out


KERNEL_KINDS = ("fwd_stats", "recompute_ds", "dh", "dw")


def gc_kernel_timing_begin():
    """Start bracketing every tcgen05 contraction launch with CUDA events on its stream."""
    _check(_lib.gc_kernel_timing_begin())


def gc_kernel_timing_end() -> dict:
    """Waits for the recorded events; -> {kind: (total_ms, launches)} for the four contractions."""
    ms = (C.c_float * len(KERNEL_KINDS))()
    n = (C.c_int32 * len(KERNEL_KINDS))()
    _check(_lib.gc_kernel_timing_end(ms, n))
    return {k: (float(ms[i]), int(n[i])) for i, k in enumerate(KERNEL_KINDS)}


def gc_balance_plan(cu_seqlens, group_offsets=None, keep=None, w_lin=0, w_quad=1, bucket_size=1,
                    seed=0, shuffle=True, n_tokens_max=None):
    """Dynamic-sampling repack + workload balancing plan (device tensors in, device tensors out):
    -> dict(order [R], n_kept [1], cu_out [R+1], src_token [T], n_tokens [1])."""
    assert cu_seqlens.dtype == torch.int32
    dev = cu_seqlens.device
    R = cu_seqlens.numel() - 1
    G = 0 if group_offsets is None else group_offsets.numel() - 1
    T = int(n_tokens_max) if n_tokens_max is not None else int(cu_seqlens[-1].item())
    order = torch.empty(max(R, 1), dtype=torch.int32, device=dev)
    cu_out = torch.empty(R + 1, dtype=torch.int32, device=dev)
    src_token = torch.empty(max(T, 1), dtype=torch.int32, device=dev)
    n_kept = torch.empty(1, dtype=torch.int32, device=dev)
    n_tokens = torch.empty(1, dtype=torch.int32, device=dev)
    ws = workspace(int(_lib.gc_balance_workspace_bytes(R)), dev)
    _check(_lib.gc_balance_plan(_ptr(cu_seqlens), R, _ptr(group_offsets), _ptr(keep), G, int(w_lin),
                                int(w_quad), int(bucket_size), int(seed) & ((1 << 64) - 1),
                                int(bool(shuffle)), _ptr(order), _ptr(n_kept), _ptr(cu_out),
                                _ptr(src_token), _ptr(n_tokens), _ptr(ws), ws.numel(), _stream()))
    return dict(order=order, n_kept=n_kept, cu_out=cu_out, src_token=src_token, n_tokens=n_tokens)


def gc_gather_rows(X, rows, n_rows, y_rows):
    """Y[i] = X[rows[i]] for i < n_rows (device scalar); -> Y [y_rows, D]."""
    assert X.dim() == 2 and X.stride(1) == 1
    Y = torch.empty(y_rows, X.shape[1], dtype=X.dtype, device=X.device)
    _check(_lib.gc_gather_rows(_ptr(X), X.stride(0), dtype_code(X), X.shape[1], _ptr(rows),
                               _ptr(n_rows), y_rows, _ptr(Y), _stream()))
    return Y


def gc_gather_1d(x, rows, n_rows, max_rows):
    """y[i] = x[rows[i]] for i < n_rows; x of a 4-byte dtype."""
    assert x.element_size() == 4 and x.is_contiguous()
    y = torch.zeros(max_rows, dtype=x.dtype, device=x.device)
    _check(_lib.gc_gather_1d(_ptr(x), _ptr(rows), _ptr(n_rows), max_rows, _ptr(y), _stream()))
    return y


def gc_token_logprobs_multi(H, W, targets, temperature=1.0):
    """Verdict-token scoring: targets [T, K] int32 -> (logp [T, K], entropy [T], lse [T])."""
    assert H.dim() == 2 and W.dim() == 2 and targets.dim() == 2 and targets.dtype == torch.int32
    T, D = H.shape
    V, K = W.shape[0], targets.shape[1]
    assert targets.shape[0] == T and targets.is_contiguous()
    dev = H.device
    logp = torch.empty(T, K, dtype=torch.float32, device=dev)
    ent = torch.empty(T, dtype=torch.float32, device=dev)
    lse = torch.empty(T, dtype=torch.float32, device=dev)
    ws = workspace(int(_lib.gc_multi_workspace_bytes(T, D, V, K)), dev)
    _check(_lib.gc_token_logprobs_multi(_ptr(H), H.stride(0) if T > 0 else D, _ptr(W), W.stride(0),
                                        dtype_code(H), _ptr(targets), K, T, D, V, float(temperature),
                                        _ptr(logp), _ptr(ent), _ptr(lse), _ptr(ws), ws.numel(),
                                        _stream()))
    return logp, ent, lse


def gc_value_head_fwd(H, w, bias=0.0):
    """v[t] = H[t,:] . w + bias -> float32 [T]."""
    T, D = H.shape
    assert w.numel() == D and w.dtype == H.dtype and H.stride(1) == 1
    v = torch.empty(T, dtype=torch.float32, device=H.device)
    _check(_lib.gc_value_head_fwd(_ptr(H), H.stride(0) if T > 0 else D, dtype_code(H), _ptr(w),
                                  float(bias), T, D, _ptr(v), _stream()))
    return v


def gc_gae(rewards, values, mask, cu_seqlens, gamma=1.0, lam=0.95):
    """-> (adv [T], returns [T])."""
    T = rewards.numel()
    adv = torch.zeros(T, dtype=torch.float32, device=rewards.device)
    ret = torch.zeros(T, dtype=torch.float32, device=rewards.device)
    _check(_lib.gc_gae(_ptr(rewards), _ptr(values), _ptr(mask), _ptr(cu_seqlens),
                       cu_seqlens.numel() - 1, T, float(gamma), float(lam), _ptr(adv), _ptr(ret),
                       _stream()))
    return adv, ret


def gc_value_loss(values, old_values, returns, mask=None, clip_v=0.2, grad_loss=1.0, want_grad=True):
    """-> (out3 = [loss, clip_frac, n_scored] device tensor, g [T] or None)."""
    T = values.numel()
    dev = values.device
    out3 = torch.empty(3, dtype=torch.float32, device=dev)
    g = torch.empty(T, dtype=torch.float32, device=dev) if want_grad else None
    ws = workspace(int(_lib.gc_critic_workspace_bytes(T, 8)), dev)
    _check(_lib.gc_value_loss(_ptr(values), _ptr(old_values), _ptr(returns), _ptr(mask), T,
                              float(clip_v), float(grad_loss), _ptr(out3), _ptr(g), _ptr(ws),
                              ws.numel(), _stream()))
    return out3, g


GC_VALUE_LOSS_STATIC_MAX_T = 4194304     # include/gcore.h


def gc_value_loss_static_scratch(values, old_values, returns, mask=None, clip_v=0.2, grad_loss=1.0,
                                 *, out3, g=None):
    """gc_value_loss for a caller that cannot allocate device memory (a hook inside someone else's
    training step that owns only its inputs and outputs, a process whose pool already holds all of
    HBM, a loop that must not hit cudaMalloc's device-wide sync): the scratch is a fixed 33 KB array
    inside libgcore.so, so there is no workspace and this wrapper allocates nothing either -- the
    caller passes the outputs: out3 [3] float32 (loss, clip_frac, n_scored) and optionally g [T]
    float32.  T <= GC_VALUE_LOSS_STATIC_MAX_T, else GcoreError.  One array per device, shared by
    all calls: calls that may overlap on the GPU race; keep them on one stream.  The first call on
    a device looks up the array's address: make it with that device current, outside any capture."""
    T = values.numel()
    if T > GC_VALUE_LOSS_STATIC_MAX_T:
        raise GcoreError(f"gc_value_loss_static_scratch: T = {T} exceeds the fixed scratch array's "
                         f"limit GC_VALUE_LOSS_STATIC_MAX_T = {GC_VALUE_LOSS_STATIC_MAX_T}; use "
                         "gc_value_loss (caller workspace) for larger batches")
    assert out3.is_cuda and out3.dtype == torch.float32 and out3.numel() == 3 and out3.is_contiguous()
    assert g is None or (g.is_cuda and g.dtype == torch.float32 and g.numel() == T and g.is_contiguous())
    _check(_lib.gc_value_loss_static_scratch(_ptr(values), _ptr(old_values), _ptr(returns), _ptr(mask),
                                             T, float(clip_v), float(grad_loss), _ptr(out3), _ptr(g),
                                             _stream()))
    return out3, g


def gc_value_head_bwd(H, w, g):
    """-> (dH [T,D] in H's dtype, dw [D] float32, dbias [1] float32)."""
    T, D = H.shape
    dev = H.device
    dH = torch.empty(T, D, dtype=H.dtype, device=dev)
    dw = torch.empty(D, dtype=torch.float32, device=dev)
    db = torch.empty(1, dtype=torch.float32, device=dev)
    ws = workspace(int(_lib.gc_critic_workspace_bytes(T, D)), dev)
    _check(_lib.gc_value_head_bwd(_ptr(H), H.stride(0) if T > 0 else D, dtype_code(H), _ptr(w),
                                  _ptr(g), T, D, _ptr(dH), D, _ptr(dw), _ptr(db), _ptr(ws),
                                  ws.numel(), _stream()))
    return dH, dw, db


def gc_grpo_loss_bwd_reduce_scatter(H, W, targets, mask, temperature, cu_seqlens, adv, old_logp,
                                    ref_logp, logp, lse, shard_ptrs, shard_rows, ld_shard=None,
                                    clip_lo=0.2, clip_hi=0.2, beta=0.04, agg=GC_AGG_TOKEN_MEAN,
                                    grad_loss=1.0, *, dH=None, chunk_tokens=0, fwd_state=None):
    """Backward whose dW tiles are TMA-reduce-added into the owning rank's shard.  shard_ptrs: list of
    `world` device pointers (ints; own tensor.data_ptr() or peer-mapped), shard r = fp32
    [shard_rows, D] holding vocab rows [r*shard_rows, (r+1)*shard_rows).  -> dH."""
    args, T, D, V, dt = _head_args(H, W, targets, mask, temperature, False)
    dev = H.device
    if dH is None:
        dH = torch.empty(T, D, dtype=H.dtype, device=dev)
    world = len(shard_ptrs)
    arr = (C.c_void_p * world)(*[C.c_void_p(int(p)) for p in shard_ptrs])
    nb = workspace_bytes(GC_OP_LOSS_BWD, T, D, V, dt, chunk_tokens)
    ws = workspace(nb, dev)
    _check(_lib.gc_grpo_loss_bwd_reduce_scatter(
        *args, *_loss_args(cu_seqlens, adv, old_logp, ref_logp, clip_lo, clip_hi, beta, agg),
        _ptr(logp), _ptr(lse), float(grad_loss), _ptr(dH), dH.stride(0) if T > 0 else D, arr, world,
        int(shard_rows), int(ld_shard if ld_shard is not None else D), int(chunk_tokens),
        _state_ptr(fwd_state, _state_sig(H, targets, mask, T, D, V, dt)), _ptr(ws), ws.numel(),
        _stream()))
    return dH


def gc_attention_allgather_kv(Q, K_ptrs, V_ptrs, shard_rows, rank, Hkv, cu_seqlens=None, causal=True,
                              window=0, scale=None, heads_per_step=1, want_lse=True):
    """Distributed attention forward (NEXT-4).  Q [S_local, Hq, 128] bf16 on the device; K_ptrs /
    V_ptrs: per rank the device address (int) of its K / V shard [shard_rows[r], Hkv, 128] bf16 --
    own tensors' data_ptr() or peer-mapped memory.  -> (O [S_local, Hq, 128] bf16, lse [Hq, S_local])."""
    S_local, Hq, d = Q.shape
    world = len(shard_rows)
    assert Q.dtype == torch.bfloat16 and Q.is_contiguous() and int(shard_rows[rank]) == S_local
    S = int(sum(shard_rows))
    dev = Q.device
    O = torch.empty_like(Q)
    lse = torch.empty(Hq, S_local, dtype=torch.float32, device=dev) if want_lse else None
    kp = (C.c_void_p * world)(*[C.c_void_p(int(x)) for x in K_ptrs])
    vptr = (C.c_void_p * world)(*[C.c_void_p(int(x)) for x in V_ptrs])
    rows = (C.c_int64 * world)(*[int(x) for x in shard_rows])
    hs = min(int(heads_per_step), Hkv)
    ws = workspace(int(_lib.gc_attention_workspace_bytes(S_local, S, hs)), dev, "attn")
    n_docs = 0 if cu_seqlens is None else cu_seqlens.numel() - 1
    if scale is None:
        scale = 1.0 / (d ** 0.5)
    _check(_lib.gc_attention_allgather_kv(_ptr(Q), kp, vptr, rows, world, int(rank), Hq, int(Hkv), d,
                                          _ptr(cu_seqlens), n_docs, int(bool(causal)), int(window),
                                          float(scale), hs, _ptr(O), _ptr(lse), _ptr(ws), ws.numel(),
                                          _stream()))
    return O, lse
