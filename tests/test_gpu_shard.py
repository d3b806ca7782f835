"""SURVEY 8(e) on one GPU: the library's shard entry points, driven for G shards ONE AFTER THE OTHER (each shard has
its own ctx over its slice of the vocabulary; the "collectives" are a stack and a sum of the shards' outputs, so no
kernel waits on another rank).  The assembled result must match the fp64 oracle's UNSHARDED step at the tolerances
of gpu_util.check_step; the mask is bit-exact."""
import numpy as np
import pytest
import torch

from oracle import tts_oracle as O
from paper_2605_09329_b200 import sharded, tts
from workloads import synth

from gpu_util import _dev, bits, check_step, run_oracle

pytestmark = pytest.mark.gpu


def _run_sharded(case, G, kernel_path=tts.TTS_PATH_AUTO, align=128, mask_only=False):
    c = case["cfg"]
    T, V, d = case["T"], case["V"], case["d"]
    bf = c["param"] == synth.BF16
    ranges = [sharded.shard_range(V, g, G, align) for g in range(G)]
    teacher = case["teacher"]
    h, tok, pw = _dev(case["h"]), _dev(case["draft_tokens"]), _dev(case["pos_weight"])
    shards = []
    for v0, v1 in ranges:
        cfg = tts.make_config(v1 - v0, d, T, case["seg_len"], c["param"], c["logits"], c["optimizer"], c["lr"],
                              c["beta1"], c["beta2"], c["eps"], c["weight_decay"], tts.TTS_ROWS_ALL, 0, kernel_path)
        sh = dict(ctx=tts.tts_ctx_create(cfg, 0), v0=v0, v1=v1,
                  teacher=_dev(np.ascontiguousarray(teacher[:, v0:v1])), W_in=_dev(case["W"][v0:v1]),
                  master=_dev(case["master"][v0:v1]) if bf else None,
                  m=_dev(case["m"][v0:v1]) if case["m"] is not None else None,
                  v=_dev(case["v"][v0:v1]) if case["v"] is not None else None,
                  stats=torch.zeros(T, 8, device="cuda"), val=torch.zeros(T, device="cuda"),
                  idx=torch.zeros(T, dtype=torch.int32, device="cuda"), loss=torch.zeros(1, device="cuda"),
                  kl=torch.zeros(T, device="cuda"), gh=torch.full((T, d), float("nan"), device="cuda"),
                  gW=torch.full((v1 - v0, d), float("nan"), device="cuda"),
                  mask=torch.zeros(T, dtype=torch.uint8, device="cuda"),
                  tau=torch.zeros(T // case["seg_len"], dtype=torch.int32, device="cuda"),
                  am=torch.zeros(T, dtype=torch.int32, device="cuda"))
        sh["W_out"] = torch.empty_like(sh["W_in"])
        shards.append(sh)
    try:
        # mask: candidates per shard -> stacked -> every shard finalises the same mask
        for sh in shards:
            tts.tts_shard_argmax(sh["ctx"], sh["teacher"], T, sh["v0"], sh["val"], sh["idx"])
        val_all = torch.stack([sh["val"] for sh in shards])
        idx_all = torch.stack([sh["idx"] for sh in shards])
        for sh in shards:
            tts.tts_shard_accept_mask(sh["ctx"], val_all, idx_all, G, tok, T, sh["mask"], sh["tau"], sh["am"])
        if mask_only:
            torch.cuda.synchronize()
            return dict(mask=shards[0]["mask"].cpu().numpy(), tau=shards[0]["tau"].cpu().numpy(),
                        argmax=shards[0]["am"].cpu().numpy(),
                        all_masks=[sh["mask"].cpu().numpy() for sh in shards])
        # step: begin on every shard -> stacked tuples -> finish on every shard -> summed gh
        for sh in shards:
            tts.tts_shard_begin_step(sh["ctx"], sh["teacher"], h, sh["W_in"], T, sh["stats"])
        stats_all = torch.stack([sh["stats"] for sh in shards]).contiguous()
        for sh in shards:
            tts.tts_shard_finish_step(sh["ctx"], stats_all, G, sh["teacher"], h, sh["W_in"], sh["W_out"], sh["master"],
                                      sh["m"], sh["v"], pw, sh["mask"], T, case["loss_scale"], sh["loss"], sh["kl"],
                                      sh["gh"], sh["gW"])
        torch.cuda.synchronize()
        cat = lambda k: np.concatenate([sh[k].cpu().numpy() for sh in shards])
        out = dict(mask=shards[0]["mask"].cpu().numpy(), tau=shards[0]["tau"].cpu().numpy(),
                   argmax=shards[0]["am"].cpu().numpy(), loss=float(shards[0]["loss"].item()),
                   kl_rows=shards[0]["kl"].cpu().numpy(), gh=sum(sh["gh"] for sh in shards).cpu().numpy(), gW=cat("gW"),
                   m=cat("m") if case["m"] is not None else None, v=cat("v") if case["v"] is not None else None,
                   used=[tts.tts_last_step_used_tensor_path(sh["ctx"]) for sh in shards],
                   counts=[tts.tts_get_step_count(sh["ctx"]) for sh in shards])
        if bf:
            out["master"] = cat("master")
            out["W_out"] = np.concatenate([bits(sh["W_out"]) for sh in shards])
        else:
            out["master"] = cat("W_out")
            out["W_out"] = out["master"]
        # every shard reports the same global loss, KL rows and mask
        for sh in shards[1:]:
            assert float(sh["loss"].item()) == out["loss"]
            np.testing.assert_array_equal(sh["kl"].cpu().numpy(), out["kl_rows"])
            np.testing.assert_array_equal(sh["mask"].cpu().numpy(), out["mask"])
            np.testing.assert_array_equal(sh["tau"].cpu().numpy(), out["tau"])
        return out
    finally:
        for sh in shards:
            tts.tts_ctx_destroy(sh["ctx"])


@pytest.mark.parametrize("cfg_id,V,d,n_seq,G", [
    (3, 4096, 1024, 1, 2),        # fused stripe kernel on every shard
    (3, 4096 + 128, 256, 1, 3),   # wide kernel, uneven shards (11 + 11 + 11 blocks of 128 -> 1408 / 1408 / 1408)
    (3, 128 * 7, 256, 1, 3),      # 2 / 2 / 3 blocks
    (4, 2048, 256, 4, 2),         # batched: 64 rows
])
def test_sharded_step_matches_unsharded_oracle(cfg_id, V, d, n_seq, G):
    case = synth.make_case(cfg_id, V=V, d=d, n_seq=n_seq, seg_len=16)
    g = _run_sharded(case, G)
    o = run_oracle(case)
    check_step(g, o, case)
    assert g["used"] == [1] * G and g["counts"] == [1] * G


def test_sharded_step_fp32_sgd_config1():
    case = synth.make_case(1)                      # V = 1024, fp32, SGD: CUDA-core kernels, 4 shards of 256 rows
    g = _run_sharded(case, 4, align=256)
    o = run_oracle(case)
    check_step(g, o, case, fp32=True)
    assert g["used"] == [0] * 4


def test_one_shard_equals_the_plain_step():
    from gpu_util import run_gpu
    case = synth.make_case(3, V=2048, d=1024)
    a = _run_sharded(case, 1)
    b = run_gpu(case)
    # the same kernels on the same data; the only difference is one more fp32 rounding of the eight-number tuple
    assert np.abs(a["master"] - b["master"]).max() <= 0.05 * case["cfg"]["lr"]
    assert np.abs(a["gh"] - b["gh"]).max() <= 1e-5 * np.abs(b["gh"]).max()
    assert a["loss"] == pytest.approx(b["loss"], rel=1e-6)
    np.testing.assert_array_equal(a["mask"], b["mask"])


def test_mask_ties_across_shards_take_the_lowest_global_index():
    V, T, C = 1024, 8, 8
    t = np.full((T, V), -3.0, dtype=np.float32)
    t[0, [700, 100, 900]] = 5.0           # tie between shards 0, 1, 1 (G = 2): 100 wins
    t[1, [600, 513]] = 2.0                # tie inside shard 1
    t[2, :512] = -np.inf; t[2, 800] = 0.0 # shard 0 all -inf
    t[3, :] = -np.inf                     # a row of only -inf resolves to index 0
    tok = np.array([100, 513, 800, 0, 1, 1, 1, 1], dtype=np.int32)
    case = synth.make_case(1)
    case.update(teacher=t, draft_tokens=tok)
    g = _run_sharded(case, 2, align=512, mask_only=True)   # a row of only -inf is outside the step's domain (R23)
    mask, tau, am = O.accept_mask(t, tok, C)
    np.testing.assert_array_equal(g["all_masks"][1], g["all_masks"][0])
    np.testing.assert_array_equal(g["argmax"], am)
    np.testing.assert_array_equal(g["mask"], mask)
    np.testing.assert_array_equal(g["tau"], tau)
    assert am[:4].tolist() == [100, 513, 800, 0]


def test_sharded_step_with_given_logits_and_lambda_term():
    """f1 extras through the shard calls: every shard passes ITS columns of the drafter's logits and of the reference
    logits; the (m_ref, s_ref, b) fields of the exchanged tuples must merge to the whole-row regulariser."""
    case = synth.make_case(3, V=2048, d=256, nonzero_state=True, step=3)
    G, T, V, d = 2, case["T"], case["V"], case["d"]
    rng = np.random.Generator(np.random.PCG64(9))
    W = O.widen(case["W"]); hh = O.widen(case["h"])
    z_given = (hh @ W.T + 0.05 * rng.standard_normal((T, V))).astype(np.float32)
    z_ref = (hh @ W.T + 0.8 * rng.standard_normal((T, V))).astype(np.float32)
    lam = 0.6
    c = case["cfg"]
    mask, _, _ = O.accept_mask(case["teacher"], case["draft_tokens"], case["seg_len"])
    o = O.distill_step(case["teacher"], case["h"], case["W"], case["master"], case["m"], case["v"], case["pos_weight"],
                       mask, seg_len=case["seg_len"], loss_scale=case["loss_scale"], optimizer="adamw", lr=c["lr"],
                       beta1=c["beta1"], beta2=c["beta2"], eps=c["eps"], weight_decay=c["weight_decay"], step=3,
                       draft_logits=z_given, lam=lam, z_ref=z_ref)
    h, pw = _dev(case["h"]), _dev(case["pos_weight"])
    shards = []
    for g in range(G):
        v0, v1 = sharded.shard_range(V, g, G)
        cfg = tts.make_config(v1 - v0, d, T, case["seg_len"], c["param"], c["logits"], c["optimizer"], c["lr"],
                              c["beta1"], c["beta2"], c["eps"], c["weight_decay"])
        ctx = tts.tts_ctx_create(cfg, 0)
        tts.tts_set_step_count(ctx, 2)
        shards.append(dict(ctx=ctx, teacher=_dev(np.ascontiguousarray(case["teacher"][:, v0:v1])),
                           W=_dev(case["W"][v0:v1]), master=_dev(case["master"][v0:v1]), m=_dev(case["m"][v0:v1]),
                           v=_dev(case["v"][v0:v1]), zg=_dev(np.ascontiguousarray(z_given[:, v0:v1])),
                           zr=_dev(np.ascontiguousarray(z_ref[:, v0:v1])), stats=torch.zeros(T, 8, device="cuda"),
                           loss=torch.zeros(1, device="cuda"), kl=torch.zeros(T, device="cuda"),
                           gh=torch.zeros(T, d, device="cuda")))
    try:
        for sh in shards:
            tts.tts_shard_begin_step(sh["ctx"], sh["teacher"], h, sh["W"], T, sh["stats"], draft_logits=sh["zg"],
                                     ref_logits=sh["zr"], lam=lam)
        stats_all = torch.stack([sh["stats"] for sh in shards]).contiguous()
        for sh in shards:
            tts.tts_shard_finish_step(sh["ctx"], stats_all, G, sh["teacher"], h, sh["W"], sh["W"], sh["master"], sh["m"],
                                      sh["v"], pw, None, T, case["loss_scale"], sh["loss"], sh["kl"], sh["gh"], None,
                                      draft_logits=sh["zg"], ref_logits=sh["zr"], lam=lam)
        torch.cuda.synchronize()
        loss = float(shards[0]["loss"].item())
        assert loss == float(shards[1]["loss"].item())
        assert abs(loss - o["loss"]) <= 1e-3 * abs(o["loss"]) + 1e-6
        assert np.all(np.abs(shards[0]["kl"].cpu().numpy() - o["kl_rows"]) <= 1e-3 * np.abs(o["kl_rows"]) + 1e-5)
        cat = lambda k: np.concatenate([sh[k].cpu().numpy() for sh in shards]).astype(np.float64)
        for name, gg, ref in (("master", cat("master"), o["master"]), ("m", cat("m"), o["m"]), ("v", cat("v"), o["v"]),
                              ("gh", sum(sh["gh"] for sh in shards).cpu().numpy().astype(np.float64), o["gh"])):
            assert np.abs(gg - ref).max() <= 2e-3 * np.abs(ref).max(), name
        assert [tts.tts_get_step_count(sh["ctx"]) for sh in shards] == [3, 3]
    finally:
        for sh in shards:
            tts.tts_ctx_destroy(sh["ctx"])
