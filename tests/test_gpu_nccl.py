"""SURVEY 8(e) on real GPUs: the vocabulary-sharded step over NCCL, one process per GPU, against the UNSHARDED oracle.
Needs at least two CUDA devices (skipped otherwise: this pool leases one GPU per call, so the driver's round-end run
skips it too; on a multi-GPU node `python -m pytest tests/test_gpu_nccl.py -m gpu` runs it).  Every rank draws the same
seeded case, keeps its slice of the vocabulary, runs paper_2605_09329_b200.sharded.VocabShardedStep (tts_shard_* calls
+ the three tiny NCCL collectives) and checks ITS rows of master / m / v / W_out, the global loss and KL rows, the
all-reduced gh and the mask against the oracle's unsharded step at gpu_util.check_step's tolerances."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.multiprocessing as mp

pytestmark = pytest.mark.gpu


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, V, d, n_seq, q):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    sys.path[:0] = [root, os.path.join(root, "tests")]
    import torch.distributed as dist
    from oracle import tts_oracle as O
    from paper_2605_09329_b200 import dist_util as D, sharded, tts
    from workloads import synth
    from gpu_util import _dev, bits, max_abs
    try:
        torch.cuda.set_device(rank)
        dev = torch.device("cuda", rank)
        D.init("nccl", dev)
        case = synth.make_case(3 if n_seq == 1 else 4, V=V, d=d, n_seq=n_seq)
        c, T, C = case["cfg"], case["T"], case["seg_len"]
        v0, v1 = sharded.shard_range(V, rank, world)
        cfg = tts.make_config(v1 - v0, d, T, C, c["param"], c["logits"], c["optimizer"], c["lr"], c["beta1"], c["beta2"],
                              c["eps"], c["weight_decay"])
        with torch.cuda.device(dev):
            sh = sharded.VocabShardedStep(cfg, v0, rank)
            to = lambda a: _dev(a).to(dev)
            teacher = to(np.ascontiguousarray(case["teacher"][:, v0:v1]))
            h, tok, pw = to(case["h"]), to(case["draft_tokens"]), to(case["pos_weight"])
            W_in, master = to(case["W"][v0:v1]), to(case["master"][v0:v1])
            m, v = to(case["m"][v0:v1]), to(case["v"][v0:v1])
            W_out = torch.empty_like(W_in)
            mask = torch.zeros(T, dtype=torch.uint8, device=dev)
            tau = torch.zeros(T // C, dtype=torch.int32, device=dev)
            am = torch.zeros(T, dtype=torch.int32, device=dev)
            loss = torch.zeros(1, device=dev)
            kl = torch.zeros(T, device=dev)
            gh = torch.zeros(T, d, device=dev)
            side = torch.cuda.Stream(device=dev)
            side.wait_stream(torch.cuda.current_stream(dev))
            n = sh.accept_mask(teacher, tok, T, mask, tau, am, side)
            assert n == world
            sh.distill_step(teacher, h, W_in, W_out, master, m, v, pw, mask, T, case["loss_scale"], loss, kl, gh, None,
                            side)
            tts.tts_sync_step(sh.ctx)
            torch.cuda.synchronize(dev)
            # the unsharded oracle
            o_mask, o_tau, o_am = O.accept_mask(case["teacher"], case["draft_tokens"], C)
            o = O.distill_step(case["teacher"], case["h"], case["W"], case["master"], case["m"], case["v"],
                               case["pos_weight"], o_mask, seg_len=C, loss_scale=case["loss_scale"], lr=c["lr"],
                               beta1=c["beta1"], beta2=c["beta2"], eps=c["eps"], weight_decay=c["weight_decay"])
            np.testing.assert_array_equal(mask.cpu().numpy(), o_mask)
            np.testing.assert_array_equal(tau.cpu().numpy(), o_tau)
            np.testing.assert_array_equal(am.cpu().numpy(), o_am)
            assert abs(float(loss.item()) - o["loss"]) <= 1e-3 * abs(o["loss"]) + 1e-6
            assert np.all(np.abs(kl.cpu().numpy() - o["kl_rows"]) <= 1e-3 * np.abs(o["kl_rows"]) + 1e-5)
            assert max_abs(gh.cpu().numpy() - o["gh"]) <= 2e-3 * max_abs(o["gh"])
            for name, g in (("master", master), ("m", m), ("v", v)):
                ref = o[name][v0:v1]
                assert max_abs(g.cpu().numpy().astype(np.float64) - ref) <= 2e-3 * max_abs(o[name]) + 1e-30, name
            np.testing.assert_array_equal(bits(W_out), O.f32_to_bf16_bits(master.cpu().numpy()))
            sh.close()
        D.barrier(dev)
        q.put((rank, "ok"))
    except Exception as e:  # noqa: BLE001
        import traceback
        q.put((rank, "FAILED: %s\n%s" % (e, traceback.format_exc())))
    finally:
        try:
            dist.destroy_process_group()
        except Exception:
            pass


@pytest.mark.skipif(torch.cuda.device_count() < 2, reason="needs two CUDA devices (one process per GPU over NCCL)")
@pytest.mark.parametrize("V,d,n_seq", [(4096 + 128, 1024, 1), (4096 + 384, 256, 32)])
def test_two_gpu_sharded_step_matches_unsharded_oracle(V, d, n_seq):
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, world, port, V, d, n_seq, q)) for r in range(world)]
    for p in ps:
        p.start()
    out = sorted((q.get(timeout=300) for _ in range(world)), key=lambda x: x[0])
    for p in ps:
        p.join(timeout=60)
    for rank, msg in out:
        assert msg == "ok", "rank %d: %s" % (rank, msg)
