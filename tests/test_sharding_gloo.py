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


# ------------------------------------------------------------------------------------------------
# Eq. 10, the method's one exchange step: every rank takes the gradient of ITS
# chunk at the shared W, the gradients are summed (all-reduce), every rank commits the same update. The
# library keeps the update split for this (ttt_accumulate / ttt_pending_gradient / ttt_commit); here the
# host-side plumbing is checked on CPU with the oracle standing in for the per-rank gradient kernel.
# ------------------------------------------------------------------------------------------------
def _gcs_worker(rank, world, port, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = ti.scaled(ti.CONFIGS["cfg2"], nh=2, tokens_per_frame=50, frames_per_chunk=1, n_frames=world)
    W1, W2, W3 = ti.fast_weights(w)
    chunks = list(ti.TokenStream(w))
    Q, K, V, lr = chunks[rank]                                 # one chunk per rank
    ora = OracleTTT(W1, W2, W3)
    G = [torch.from_numpy(g) for g in ora.grad(K, V, lr)[:3]]  # = ttt_accumulate + ttt_pending_gradient
    flat = torch.cat([g.reshape(-1) for g in G])
    dist.all_reduce(flat, op=dist.ReduceOp.SUM)                # Eq. 10: g = sum over ranks
    ofs, new = 0, []
    for Wm, g in zip((W1, W2, W3), G):                         # = ttt_commit, identical on every rank
        new.append(Wm.double() - flat[ofs:ofs + g.numel()].reshape(g.shape))
        ofs += g.numel()
    np.save(os.path.join(out_dir, f"w_rank{rank}.npy"), torch.cat([x.reshape(-1) for x in new]).numpy())
    dist.destroy_process_group()


def test_gradient_allreduce_equals_one_update_on_all_chunks(tmp_path):
    world = 2
    mp.spawn(_gcs_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    w = ti.scaled(ti.CONFIGS["cfg2"], nh=2, tokens_per_frame=50, frames_per_chunk=1, n_frames=world)
    W1, W2, W3 = ti.fast_weights(w)
    chunks = list(ti.TokenStream(w))
    ora = OracleTTT(W1, W2, W3)
    K = torch.cat([c[1] for c in chunks]); V = torch.cat([c[2] for c in chunks])
    lr = torch.cat([c[3] for c in chunks], dim=1)
    ora.update(K, V, lr)                                       # one update on the concatenation of all chunks
    expect = np.concatenate([x.reshape(-1) for x in ora.weights()])
    r0, r1 = np.load(tmp_path / "w_rank0.npy"), np.load(tmp_path / "w_rank1.npy")
    np.testing.assert_array_equal(r0, r1)                      # every rank holds the same memory afterwards
    np.testing.assert_allclose(r0, expect, rtol=0, atol=1e-12)
