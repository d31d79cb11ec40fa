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


def _train_worker(rank, world, port, out):
    """Each rank runs the ORACLE on its shard (no GPU here); what is under test is the combination
    rule of dp.global_grad_scale + dp.all_reduce_mean against the oracle on the whole batch."""
    import numpy as np
    import oracle as O
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank),
                      WORLD_SIZE=str(world), LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        full = _make_train_case()
        sh = _shard_case(full, dp.shard_groups(full["G"], world, rank))
        n_local = int(sh["scored"].sum())
        gl = dp.global_grad_scale(n_local)
        r = O.grpo_forward_backward(sh["H"], full["W"], sh["y"], sh["mask"], 1.0, sh["cu"], sh["adv"],
                                    sh["old"], sh["ref"], 0.2, 0.2, 0.04, grad_loss=gl)
        dW = torch.from_numpy(r["dW"].copy())
        loss = torch.tensor([r["loss"] * gl], dtype=torch.float64)
        dp.all_reduce_mean(dW, loss)
        out.put((rank, gl, dW.numpy(), float(loss.item()), r["dH"], sh["tok"]))
    finally:
        dist.destroy_process_group()


def _make_train_case():
    import numpy as np
    import oracle as O
    r = np.random.default_rng(0)
    G, gs = 4, 2
    L = np.array([5, 9, 3, 14, 7, 2, 11, 6])             # unequal shards: 31 vs 26 tokens
    cu = np.concatenate([[0], np.cumsum(L)]).astype(np.int32)
    T, D, V = int(cu[-1]), 16, 24
    H = r.normal(size=(T, D)); W = r.normal(size=(V, D)) * 0.3
    y = r.integers(0, V, T).astype(np.int32)
    mask = (r.random(T) < 0.8).astype(np.uint8)
    rewards = r.random(G * gs).astype(np.float32)
    adv, _ = O.grpo_advantages(rewards, np.arange(0, G * gs + 1, gs, dtype=np.int32), 1e-6)
    lp = O.token_logprobs(H, W, y, None, 1.0)[0]
    old = lp + 0.05 * r.normal(size=T); ref = lp + 0.1 * r.normal(size=T)
    return dict(G=G, gs=gs, cu=cu, H=H, W=W, y=y, mask=mask, adv=adv, old=old, ref=ref, T=T)


def _shard_case(c, groups):
    import numpy as np
    resp = [g * c["gs"] + i for g in groups for i in range(c["gs"])]
    tok = np.concatenate([np.arange(c["cu"][i], c["cu"][i + 1]) for i in resp])
    L = [c["cu"][i + 1] - c["cu"][i] for i in resp]
    cu = np.concatenate([[0], np.cumsum(L)]).astype(np.int32)
    scored = (c["mask"][tok] != 0) & (c["y"][tok] >= 0)
    return dict(H=c["H"][tok], y=c["y"][tok], mask=c["mask"][tok], cu=cu, adv=c["adv"][resp],
                old=c["old"][tok], ref=c["ref"][tok], scored=scored, tok=tok)


def test_two_rank_training_exchange_matches_global_objective():
    import numpy as np
    import oracle as O
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_train_worker, args=(r, world, port, q)) for r in range(world)]
    [p.start() for p in procs]
    res = sorted((q.get(timeout=180) for _ in range(world)), key=lambda x: x[0])
    [p.join(timeout=60) for p in procs]
    assert all(p.exitcode == 0 for p in procs)
    c = _make_train_case()
    g = O.grpo_forward_backward(c["H"], c["W"], c["y"], c["mask"], 1.0, c["cu"], c["adv"], c["old"],
                                c["ref"], 0.2, 0.2, 0.04)
    assert abs(sum(x[1] for x in res) - world) < 1e-12     # the scales average to 1
    assert res[0][1] != res[1][1]                          # unequal shards: the scaling matters
    for rank, gl, dW, loss, dH, tok in res:
        assert np.allclose(dW, g["dW"], rtol=1e-12, atol=1e-15)     # both ranks hold the global dW
        assert abs(loss - g["loss"]) < 1e-13
        # dH needs no exchange: it is the gradient of this rank's term of the rank-MEAN, i.e. world x
        # the global gradient, which the trunk's own gradient averaging over ranks divides out
        assert np.allclose(dH / world, g["dH"][tok], rtol=1e-12, atol=1e-15)


def test_dw_shard_rows():
    for V, world in ((128256, 8), (152064, 4), (2056, 3), (31, 2), (256000, 1)):
        sr = dp.shard_rows_for(V, world)
        assert sr % 32 == 0 and sr * world >= V and (sr - 32) * world < V + 32 * world


def test_shard_groups_balance():
    for n in (0, 1, 7, 16, 33):
        for world in (1, 2, 3, 8):
            parts = [dp.shard_groups(n, world, r) for r in range(world)]
            flat = [g for p in parts for g in p]
            assert flat == list(range(n))
            sizes = [len(p) for p in parts]
            assert max(sizes) - min(sizes) <= 1
    assert not dp.is_dist() and dp.reduce_step_stats(3.0, 5) == (3.0, 5.0)


def test_bench_gpus_2_really_starts_two_ranks():
    """`bench.py --gpus 2` outside torchrun re-executes itself under torch.distributed.run with two
    ranks; --dry-run runs the launch path (rendezvous, barriers, max-time / summed-token
    reductions) on CPU over gloo and prints one JSON line from rank 0."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items()
           if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR")}
    env["MASTER_PORT"] = str(_free_port())
    r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--dry-run",
                        "--workload", "cfg2", "--steps", "4"], capture_output=True, text=True,
                       timeout=300, env=env)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1                                  # rank 0 only
    d = json.loads(lines[0])
    assert d["n_gpus"] == 2 and d["ranks_started"] == 2 and d["dry_run"] is True
    assert d["ms_per_step"] == 11.0                         # max over ranks of 10 + rank
    assert d["tokens_all_ranks"] == 2 * 24576               # summed over ranks
    assert abs(d["grad_scale_rank0"] - 1.0) < 1e-12         # equal shards
