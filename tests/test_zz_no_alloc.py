"""gc_value_loss_static_scratch: the value loss for callers that cannot allocate device memory.

Who needs it: code that runs inside somebody else's training step and owns nothing but the tensors
it is handed (a hook, a plug-in); a process whose memory pool took all of HBM at start-up, so a
later cudaMalloc fails; a step loop that cannot afford cudaMalloc's device-wide synchronisation.
They cannot give gc_value_loss the workspace it asks for, so this entry point keeps the scratch
(counters + one partial per 1024-token tile) in a fixed 33 KB array inside libgcore.so.

What is checked here: two calls in a row on the same stream -- the second on a different, shorter
batch, so the shared array still holds the first call's counters and partials when it starts --
each against gc_value_loss (caller workspace) on the same inputs, at the tolerances
tests/test_gpu_critic.py uses against the oracle (the two paths run the same kernels, so they are in
fact expected to agree bit for bit, which is asserted for g); and that a batch beyond
GC_VALUE_LOSS_STATIC_MAX_T is refused with a clear error before anything is launched.

This file is named to be collected last: `pytest -x` stops at the first failure, and a failure here
must not hide the parity tests.  It passes alone in a fresh process (the first call then does the
once-per-device address look-up) and after the rest of the suite.
"""
import ctypes

import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    assert torch.cuda.is_available()
    from paper_2507_22789_b200 import binding
    return binding


def _inputs(T, seed):
    r = np.random.default_rng(seed)
    v = r.normal(size=T).astype(np.float32)
    vo = (v + 0.3 * r.normal(size=T)).astype(np.float32)
    ret = r.normal(size=T).astype(np.float32)
    mask = (r.random(T) < 0.7).astype(np.uint8)
    to = lambda a: torch.from_numpy(a).cuda()
    return to(v), to(vo), to(ret), to(mask)


def _agree(B, T, seed, use_mask, clip_v=0.2, grad_loss=0.5):
    v, vo, ret, mask = _inputs(T, seed)
    m = mask if use_mask else None
    ref3, ref_g = B.gc_value_loss(v, vo, ret, m, clip_v, grad_loss)          # caller-workspace path
    out3 = torch.full((3,), float("nan"), dtype=torch.float32, device="cuda")
    g = torch.full((T,), float("nan"), dtype=torch.float32, device="cuda")
    B.gc_value_loss_static_scratch(v, vo, ret, m, clip_v, grad_loss, out3=out3, g=g)
    torch.cuda.synchronize()
    o, e = out3.cpu().numpy().astype(np.float64), ref3.cpu().numpy().astype(np.float64)
    assert abs(o[0] - e[0]) <= 1e-6 + 1e-5 * abs(e[0])                       # loss
    assert abs(o[1] - e[1]) <= 2.0 / max(e[2], 1)                            # clip_frac
    assert o[2] == e[2]                                                      # n_scored (integer)
    gd, ge = g.cpu().numpy(), ref_g.cpu().numpy()
    assert np.abs(gd - ge).max() <= 1e-6 * max(1.0, np.abs(ge).max())
    assert np.array_equal(gd, ge)                                            # same kernels


def test_static_scratch_matches_workspace_path_on_two_calls_in_a_row(B):
    # call 1: 70001 tokens = 69 tiles, masked (the count kernel fills n_scored, blocks take tickets)
    _agree(B, 70001, seed=1, use_mask=True)
    # call 2, straight after, on the same stream: fewer tiles, no mask -- the array still holds
    # call 1's counters, ticket and 69 partials; anything not cleared or rewritten would show here
    _agree(B, 3001, seed=2, use_mask=False)
    # and a masked batch again, larger than both, with a different clip
    _agree(B, 1_000_003, seed=3, use_mask=True, clip_v=0.05, grad_loss=1.0)


def test_static_scratch_rejects_more_tokens_than_the_array_serves(B):
    lim = B.GC_VALUE_LOSS_STATIC_MAX_T
    one = ctypes.c_void_p(256)               # never dereferenced: the size check comes first
    rc = B.lib().gc_value_loss_static_scratch(one, one, one, None, lim + 1, 0.2, 1.0, one, None, None)
    assert rc == 2                           # GC_ERR_SHAPE, reported before any launch
    big = torch.zeros(lim + 1, dtype=torch.float32, device="cuda")
    out3 = torch.zeros(3, dtype=torch.float32, device="cuda")
    with pytest.raises(B.GcoreError, match="GC_VALUE_LOSS_STATIC_MAX_T"):
        B.gc_value_loss_static_scratch(big, big, big, None, out3=out3)
    # exactly at the limit is served
    v = big[:lim]
    B.gc_value_loss_static_scratch(v, v, v, None, out3=out3)
    torch.cuda.synchronize()
    assert out3.cpu().tolist() == [0.0, 0.0, float(lim)]
