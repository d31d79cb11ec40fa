"""Host-only checks of the C-ABI library (no GPU, no compute calls): it builds, loads, and
exports every symbol include/gcore.h declares; host-side argument logic."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2507_22789_b200 import build
    build.build()
    from paper_2507_22789_b200 import binding
    return binding.lib()


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "gcore.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(gc_[a-z0-9_]+)\s*\(", src)))


def test_exports_every_declared_symbol(lib):
    names = declared_symbols()
    assert {"gc_token_logprobs", "gc_grpo_advantages", "gc_grpo_loss_fwd",
            "gc_grpo_loss_bwd"} <= set(names)
    for n in names:
        assert hasattr(lib, n), n
    from paper_2507_22789_b200 import binding
    assert sorted(binding.EXPORTS) == names


def test_status_strings_and_version(lib):
    assert lib.gc_status_string(0) == b"GC_OK"
    for s in range(1, 9):
        assert lib.gc_status_string(s).startswith(b"GC_ERR_")
    assert lib.gc_version() >= 100


def test_workspace_bytes_host_logic(lib):
    from paper_2507_22789_b200 import binding as B
    wb = B.workspace_bytes
    assert wb(B.GC_OP_LOGPROBS, 256, 256, 4096, B.GC_F32) > 0
    # config 1: partial statistics + row list + compacted H copy
    n1 = wb(B.GC_OP_LOGPROBS, 16384, 3584, 152064, B.GC_BF16)
    assert 16384 * 3584 * 2 < n1 < 1 << 30
    # backward adds the bf16 dS chunk buffer: chunk rows * V * 2 bytes
    small = wb(B.GC_OP_LOSS_BWD, 32768, 4096, 128256, B.GC_BF16, 1024)
    big = wb(B.GC_OP_LOSS_BWD, 32768, 4096, 128256, B.GC_BF16, 4096)
    assert big - small == 3072 * 128256 * 2
    auto = wb(B.GC_OP_LOSS_BWD, 32768, 4096, 128256, B.GC_BF16, 0)
    assert auto < 32768 * 128256 * 2            # never the whole [T, V] matrix
    assert wb(99, 1, 8, 8, B.GC_F32) == 0 and wb(B.GC_OP_LOGPROBS, -1, 8, 8, B.GC_F32) == 0
    assert wb(B.GC_OP_LOGPROBS, 1, 8, 8, 7) == 0


def test_host_checkable_errors_before_any_launch(lib):
    """NULL / shape / dtype / argument errors are reported synchronously, without a GPU."""
    from paper_2507_22789_b200 import binding as B
    vp = ctypes.c_void_p
    one = vp(256)
    r = lib.gc_token_logprobs(None, 8, None, 8, B.GC_F32, None, None, 4, 8, 8, 1.0, None, None,
                              None, None, 0, None)
    assert r == 1                                # GC_ERR_NULL
    r = lib.gc_token_logprobs(one, 8, one, 8, 9, one, None, 4, 8, 8, 1.0, one, None, None, None, 0,
                              None)
    assert r == 3                                # GC_ERR_DTYPE
    r = lib.gc_token_logprobs(one, 8, one, 8, B.GC_F32, one, None, 4, 8, 8, 0.0, one, None, None,
                              None, 0, None)
    assert r == 6                                # GC_ERR_ARG (temperature <= 0)
    r = lib.gc_token_logprobs(one, 4, one, 8, B.GC_F32, one, None, 4, 8, 8, 1.0, one, None, None,
                              None, 0, None)
    assert r == 2                                # GC_ERR_SHAPE (ld < D)
    r = lib.gc_token_logprobs(one, 12, one, 12, B.GC_BF16, one, None, 4, 12, 8, 1.0, one, None,
                              None, None, 0, None)
    assert r == 2                                # bf16 needs D % 8 == 0
    r = lib.gc_token_logprobs(vp(260), 16, one, 16, B.GC_BF16, one, None, 4, 16, 8, 1.0, one, None,
                              None, None, 0, None)
    assert r == 4                                # GC_ERR_ALIGN
    assert lib.gc_grpo_advantages(one, one, -1, 1e-6, 0, 0, one, None, None) == 2
    assert lib.gc_grpo_advantages(one, one, 4, -1.0, 0, 0, one, None, None) == 6
    assert lib.gc_grpo_advantages(None, one, 4, 1e-6, 0, 0, one, None, None) == 1
    assert lib.gc_grpo_advantages(None, None, 0, 1e-6, 0, 0, None, None, None) == 0   # empty batch
    assert lib.gc_token_logprobs(None, 8, one, 8, B.GC_F32, None, None, 0, 8, 8, 1.0, None, None,
                                 None, None, 0, None) == 0                             # T = 0


def test_host_entry_workspace_covers_every_band(lib):
    """The *_host entry points score H band by band, one gc_token_logprobs call per band, each with
    its own plan; the plan is not monotonic in the row count, so the carved forward workspace has to
    be the largest query over the bands (it used to be the full-T query: GC_ERR_WORKSPACE at e.g.
    T=6144, D=4096, V=50304).  Host arithmetic only."""
    import itertools
    from paper_2507_22789_b200 import binding as B
    starts = (ctypes.c_int64 * 65)()
    saw_band_above_full = False
    Ts = [1, 300, 513, 5000, 6144, 9000, 16384, 26000, 40000]
    for T, D, V in itertools.product(Ts, (1024, 3584, 4096), (32000, 50304, 152064)):
        n = lib.gc_host_band_plan(T, D, V, B.GC_BF16, starts)
        assert 1 <= n <= 64 and starts[0] == 0 and starts[n] == T
        assert all(starts[b] < starts[b + 1] for b in range(n))
        carved = lib.gc_logprobs_host_workspace_bytes(T, D, V, B.GC_BF16) \
            - lib.gc_host_staging_bytes(T, D, B.GC_BF16)
        full = B.workspace_bytes(B.GC_OP_LOGPROBS, T, D, V, B.GC_BF16)
        assert carved >= full
        for b in range(n):
            need = B.workspace_bytes(B.GC_OP_LOGPROBS, starts[b + 1] - starts[b], D, V, B.GC_BF16)
            assert need <= carved, (T, D, V, b)
            saw_band_above_full |= need > full
        step = lib.gc_step_host_workspace_bytes(T, D, V, B.GC_BF16, 8, 2, B.GC_F32)
        assert step >= carved + lib.gc_bwd_workspace_bytes(T, D, V, B.GC_BF16, 0, B.GC_F32)
    assert saw_band_above_full                  # the sweep does reach the non-monotonic case
    assert lib.gc_host_band_plan(0, 8, 8, B.GC_BF16, starts) == 0
