"""Multi-process (gloo, world_size 2, CPU) check of the N > 1 path: heads are independent units, so
sharding them across ranks needs no data-path collective. Each rank runs
the recurrence on its head shard; gathering the shards reproduces the unsharded result exactly."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import ttt_inputs as ti
from oracle.ttt_oracle import OracleTTT


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = ti.scaled(ti.CONFIGS["cfg3"], nh=4, tokens_per_frame=40, frames_per_chunk=2, n_frames=4)
    lo, hi = ti.shard_heads(w.nh, world, rank)
    heads = list(range(lo, hi))
    cols = torch.cat([torch.arange(h * w.hd, (h + 1) * w.hd) for h in heads])
    W1, W2, W3 = ti.fast_weights(w)
    ora = OracleTTT(W1[heads], W2[heads], W3[heads], ns_iters=w.ns_iters)
    outs = []
    for (Q, K, V, lr) in ti.TokenStream(w):
        O, _ = ora.chunk_step(Q[:, cols].contiguous(), K[:, cols].contiguous(),
                              V[:, cols].contiguous(), lr[heads].contiguous())
        outs.append(torch.from_numpy(O))
    mine = torch.stack(outs)                                   # [chunks, M, heads*hd]
    gathered = [torch.empty_like(mine) for _ in range(world)]
    dist.all_gather(gathered, mine)                            # test plumbing only, not the data path
    # timing reduction used by bench.py: max over ranks
    t = torch.tensor([float(rank + 1)])
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    if rank == 0:
        np.save(os.path.join(out_dir, "sharded.npy"), torch.cat(gathered, dim=2).numpy())
        np.save(os.path.join(out_dir, "tmax.npy"), t.numpy())
    dist.destroy_process_group()


def test_head_sharding_world_size_2(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    sharded = np.load(tmp_path / "sharded.npy")
    assert float(np.load(tmp_path / "tmax.npy")[0]) == 2.0
    w = ti.scaled(ti.CONFIGS["cfg3"], nh=4, tokens_per_frame=40, frames_per_chunk=2, n_frames=4)
    W1, W2, W3 = ti.fast_weights(w)
    ora = OracleTTT(W1, W2, W3, ns_iters=w.ns_iters)
    full = np.stack([ora.chunk_step(*c)[0] for c in ti.TokenStream(w)])
    np.testing.assert_array_equal(sharded, full)               # heads are bitwise independent
