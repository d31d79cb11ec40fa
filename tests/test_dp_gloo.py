"""The N > 1 host logic on CPU: 2 ranks over gloo (127.0.0.1)."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2507_22789_b200 import dp, inputs as I


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank),
                      WORLD_SIZE=str(world), LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        assert dp.is_dist() and dp.env_rank_world() == (rank, world, rank)
        w = I.CONFIGS[3]
        mine = dp.shard_groups(w.groups, world, rank)
        lay = I.make_layout(w, 0)
        tok = sum(int(lay.lengths[g * w.group_size:(g + 1) * w.group_size].sum()) for g in mine)
        dp.barrier()
        t_max, tok_sum = dp.reduce_step_stats(10.0 + 5.0 * rank, tok)
        out.put((rank, list(mine), t_max, tok_sum, lay.T))
    finally:
        dist.destroy_process_group()


def test_two_rank_sharding_and_reductions():
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    [p.start() for p in procs]
    res = sorted(q.get(timeout=120) for _ in range(world))
    [p.join(timeout=60) for p in procs]
    assert all(p.exitcode == 0 for p in procs)
    groups = res[0][1] + res[1][1]
    assert groups == list(range(16))                     # whole groups, disjoint, complete
    for _, _, t_max, tok_sum, T in res:
        assert t_max == 15.0                             # max over ranks
        assert tok_sum == T                              # every token counted once


def test_shard_groups_balance():
    for n in (0, 1, 7, 16, 33):
        for world in (1, 2, 3, 8):
            parts = [dp.shard_groups(n, world, r) for r in range(world)]
            flat = [g for p in parts for g in p]
            assert flat == list(range(n))
            sizes = [len(p) for p in parts]
            assert max(sizes) - min(sizes) <= 1
    assert not dp.is_dist() and dp.reduce_step_stats(3.0, 5) == (3.0, 5.0)
