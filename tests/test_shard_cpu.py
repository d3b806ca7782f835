"""SURVEY 8(e), CPU side: the vocabulary partition and, on a world_size-2 gloo group, the exchange protocol of
paper_2605_09329_b200/sharded.py (all-gather of the per-row tuples in rank order, sum all-reduce of the partial gh,
all-gather of the argmax candidates).  The kernels are not involved: each rank evaluates its vocabulary slice with
the fp64 oracle, so what is checked is that slices + exchange reproduce the unsharded step."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.multiprocessing as mp

from paper_2605_09329_b200 import sharded


def test_shard_range_partitions_the_vocabulary():
    for V, world in ((151936, 8), (151936, 2), (128256, 8), (1024, 3), (128, 1)):
        rs = [sharded.shard_range(V, r, world) for r in range(world)]
        assert rs[0][0] == 0 and rs[-1][1] == V
        for (a0, a1), (b0, b1) in zip(rs[:-1], rs[1:]):
            assert a1 == b0
        sizes = [b - a for a, b in rs]
        assert all(s > 0 and s % 128 == 0 for s in sizes)
        assert max(sizes) - min(sizes) <= 128
    with pytest.raises(ValueError):
        sharded.shard_range(1000, 0, 2)
    with pytest.raises(ValueError):
        sharded.shard_range(256, 0, 3)


def test_single_process_exchange_is_identity():
    x = torch.arange(6.0).reshape(2, 3)
    assert torch.equal(sharded.all_gather_rows(x), x.unsqueeze(0))
    assert torch.equal(sharded.all_reduce_sum_(x.clone()), x)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q, V=1024):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    import torch.distributed as dist
    from oracle import tts_oracle as O
    from paper_2605_09329_b200 import dist_util as D
    from workloads import synth
    D.init("gloo")
    case = synth.make_case(3, V=V, d=64)               # every rank draws the same seeded case
    T = case["T"]
    v0, v1 = sharded.shard_range(V, rank, world)
    t = O.widen(synth.bf16_bits_to_f32(case["teacher"]))
    h = O.widen(synth.bf16_bits_to_f32(case["h"]))
    W = O.widen(synth.bf16_bits_to_f32(case["W"]))
    z_loc = h @ W[v0:v1].T
    # 1. this shard's tuples, 2. gathered in rank order, 3. merged
    st = torch.from_numpy(O.shard_row_stats(t[:, v0:v1], z_loc))
    st_all = sharded.all_gather_rows(st).numpy()
    assert st_all.shape == (world, T, 5)
    np.testing.assert_array_equal(st_all[rank], st.numpy())
    lse_t, lse_z, kl = O.merge_shard_stats(st_all)
    # the shard's rows of the step with the global normalisers, and its part of gh
    om = case["pos_weight"].astype(np.float64)
    z_full = np.zeros((T, V)); z_full[:, v0:v1] = z_loc
    rows = np.arange(v0, v1)
    part = O.distill_step_rows(rows, z_full, lse_t, lse_z, case["teacher"], case["h"], case["W"][v0:v1],
                               case["master"][v0:v1], case["m"][v0:v1], case["v"][v0:v1], om,
                               loss_scale=case["loss_scale"], lr=case["cfg"]["lr"])
    gh = torch.from_numpy(part["dl"] @ W[v0:v1])
    sharded.all_reduce_sum_(gh)
    # mask candidates: (max, lowest global index) of the slice
    am = np.array([v0 + int(np.flatnonzero(t[r, v0:v1] == t[r, v0:v1].max())[0]) for r in range(T)], dtype=np.int32)
    val = torch.from_numpy(t[np.arange(T), am].astype(np.float32))
    val_all = sharded.all_gather_rows(val).numpy()
    idx_all = sharded.all_gather_rows(torch.from_numpy(am)).numpy()
    D.barrier()
    q.put((rank, v0, v1, kl, float(case["loss_scale"] * (om * kl).sum()), gh.numpy(), part["master"], val_all, idx_all))
    dist.destroy_process_group()


@pytest.mark.parametrize("world,V", [(2, 1024), (8, 1152)])
def test_two_rank_exchange_reproduces_the_unsharded_step(world, V):
    """world_size 2, and the node size the driver's scaling run uses (8) with a vocabulary whose 128-row blocks do not
    divide among the ranks (9 blocks over 8 ranks: one shard is twice the others, as 1187 blocks over 8 are uneven)."""
    from oracle import tts_oracle as O
    from workloads import synth
    port = _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, world, port, q, V)) for r in range(world)]
    for p in ps:
        p.start()
    out = sorted((q.get(timeout=180) for _ in range(world)), key=lambda x: x[0])
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert len({o[2] - o[1] for o in out}) == (1 if V % (128 * world) == 0 else 2)      # even / uneven shards
    case = synth.make_case(3, V=V, d=64)
    mask, tau, am = O.accept_mask(case["teacher"], case["draft_tokens"], case["seg_len"])
    ref = O.distill_step(case["teacher"], case["h"], case["W"], case["master"], case["m"], case["v"],
                         case["pos_weight"], mask, seg_len=case["seg_len"], loss_scale=case["loss_scale"],
                         optimizer="adamw", lr=case["cfg"]["lr"])
    master = np.concatenate([o[6] for o in out])
    np.testing.assert_allclose(master, ref["master"], rtol=0, atol=1e-12)
    for rank, v0, v1, kl, loss, gh, _, val_all, idx_all in out:
        np.testing.assert_allclose(kl, ref["kl_rows"], rtol=1e-10)
        assert abs(loss - ref["loss"]) <= 1e-10 * abs(ref["loss"])
        np.testing.assert_allclose(gh, ref["gh"], rtol=0, atol=1e-12 * np.abs(ref["gh"]).max() + 1e-15)
        # lowest global index among the shards' maxima = the unsharded argmax
        assert val_all.shape == idx_all.shape == (world, case["T"])
        top = val_all.max(axis=0)
        best = np.where(val_all == top[None, :], idx_all, np.iinfo(np.int32).max).min(axis=0)
        np.testing.assert_array_equal(best, am)
