"""The dW contraction fused with its data-parallel exchange (gc_grpo_loss_bwd_reduce_scatter):
tiles are TMA-reduce-added into the owning rank's shard.  One GPU is all there is here, so:
(a) one process, several shards in its own memory -- the owner mapping, bit-identical to the plain
    backward; (b) two processes on the same GPU, shards opened through CUDA IPC exactly as peers'
    would be -- the cross-process protocol (zero, barrier, add, barrier).  The kernels of the two
    processes never wait on each other; only the hosts meet at barriers."""
import os
import socket

import numpy as np
import pytest
import torch

from paper_2507_22789_b200 import dp, inputs as I
from tests.helpers import make_batch

pytestmark = pytest.mark.gpu


def _fwd_bwd_plain(B, b, chunk=0):
    w = b.w
    adv, _ = B.gc_grpo_advantages(b.rewards_t, b.go_t, 1e-6, False, False)
    f = B.gc_grpo_loss_fwd(b.H, b.W, b.y, b.mask_t, w.tau, b.cu_t, adv, b.old_t, b.ref_t)
    dH, dW = B.gc_grpo_loss_bwd(b.H, b.W, b.y, b.mask_t, w.tau, b.cu_t, adv, b.old_t, b.ref_t,
                                f["logp"], f["lse"], chunk_tokens=chunk)
    return adv, f, dH, dW


@pytest.mark.parametrize("world", [1, 3, 8])
def test_shards_in_one_process_match_plain_backward(world):
    from paper_2507_22789_b200 import binding as B
    w = I.reduced(I.CONFIGS[2], D=256, V=2048 + 8, groups=2, group_size=4, seq_len=96, prompt_len=16)
    b = make_batch(w, seed=3, device="cuda")
    adv, f, dH, dW = _fwd_bwd_plain(B, b, chunk=256)
    sr = dp.shard_rows_for(w.V, world)
    shards = [torch.zeros(sr, w.D, dtype=torch.float32, device="cuda") for _ in range(world)]
    dH2 = B.gc_grpo_loss_bwd_reduce_scatter(b.H, b.W, b.y, b.mask_t, w.tau, b.cu_t, adv, b.old_t,
                                            b.ref_t, f["logp"], f["lse"],
                                            [s.data_ptr() for s in shards], sr, chunk_tokens=256)
    torch.cuda.synchronize()
    got = torch.cat(shards)[:w.V]
    assert torch.equal(dH2, dH)
    assert torch.equal(got, dW)                      # one adder per element: same sums, same order
    assert float(torch.cat(shards)[w.V:].abs().sum()) == 0.0


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _rs_worker(rank, world, port, q):
    import torch.distributed as dist
    from paper_2507_22789_b200 import binding as B
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank),
                      WORLD_SIZE=str(world), LOCAL_RANK="0")
    torch.cuda.set_device(0)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = I.reduced(I.CONFIGS[2], D=256, V=1024 + 72, groups=2, group_size=2, seq_len=70,
                      prompt_len=10)
        # W is replicated (same seed); every rank has its own tokens
        batches = [make_batch(w, seed=10 + r, device="cuda") for r in range(world)]
        for bb in batches[1:]:
            bb.W = batches[0].W
        plain = [_fwd_bwd_plain(B, bb) for bb in batches]          # what each rank would produce
        expect = sum(p[3] for p in plain)
        b = batches[rank]
        adv, f, dH_plain, _ = plain[rank]
        sr = dp.shard_rows_for(w.V, world)
        shard = torch.zeros(sr, w.D, dtype=torch.float32, device="cuda")
        ptrs, keep = dp.exchange_dw_shards(shard)
        torch.cuda.synchronize()
        dist.barrier()                                              # every shard is zero
        dH = B.gc_grpo_loss_bwd_reduce_scatter(b.H, b.W, b.y, b.mask_t, w.tau, b.cu_t, adv, b.old_t,
                                               b.ref_t, f["logp"], f["lse"], ptrs, sr)
        torch.cuda.synchronize()
        dist.barrier()                                              # every rank's adds have landed
        lo, hi = rank * sr, min((rank + 1) * sr, w.V)
        err = (shard[:hi - lo] - expect[lo:hi]).abs().max().item()
        scale = expect.abs().max().item()
        q.put((rank, err, scale, bool(torch.equal(dH, dH_plain)),
               float(shard[hi - lo:].abs().sum())))
        dist.barrier()
        del keep
    finally:
        dist.destroy_process_group()


def test_two_processes_reduce_scatter_through_cuda_ipc():
    import torch.multiprocessing as mp
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_rs_worker, args=(r, world, port, q)) for r in range(world)]
    [p.start() for p in procs]
    res = sorted(q.get(timeout=300) for _ in range(world))
    [p.join(timeout=120) for p in procs]
    assert all(p.exitcode == 0 for p in procs)
    for rank, err, scale, dh_same, pad in res:
        assert err <= 1e-6 * scale, (rank, err, scale)              # fp32 sum of two ranks' tiles
        assert dh_same and pad == 0.0
