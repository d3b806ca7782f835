"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (side stream, W_in / W_out
double buffer, no gW dump): the CUDA path against the fp64 oracle on outputs the oracle can compute one by one.

  * mask, tau, teacher argmax     bit-exact over the whole [T, V] input
  * loss, KL_r                    the oracle's full-vocabulary normalisers (row_normalisers, slab by slab)
  * gh [T, d]                     complete (gh_full)
  * master / m / v / W_out        a sample of vocabulary rows (tile edges, the last rows, the canvas tokens and the
                                  teacher's argmax tokens, i.e. the rows with the largest gradients, and random
                                  rows) through distill_step_rows; gW rows from the first-step moment m = (1-b1) g
  * properties over ALL V x d     W_out == rn_bf16(master) bit-exactly, state finite, column sums of m vanish
                                  (sum_v dl[r, v] = 0), v >= 0
Inputs: the seeded device recipe (synth.make_case_device), copied to the host bit for bit.
"""
import numpy as np
import pytest
import torch

from oracle import tts_oracle as O
from paper_2605_09329_b200 import tts
from workloads import synth

from gpu_util import bits, max_abs

pytestmark = pytest.mark.gpu


def _sample_rows(V, rng, tok, am, n_random=192):
    edges = [0, 1, 15, 16, 17, 127, 128, 129, 1023, 1024, V // 2, V - 129, V - 128, V - 17, V - 16, V - 2, V - 1]
    rows = set(int(x) for x in edges if 0 <= x < V)
    rows.update(int(x) for x in tok)
    rows.update(int(x) for x in am)
    rows.update(int(x) for x in rng.integers(0, V, size=n_random))
    return np.array(sorted(rows), dtype=np.int64)


def _run_fullsize(cfg_id, mask_mode_g=tts.TTS_ROWS_ALL, mask_mode_o=O.ROWS_ALL, max_rows=None):
    dev = "cuda:0"
    case = synth.make_case_device(cfg_id, dev)
    c = case["cfg"]
    V, d, T, C = case["V"], case["d"], case["T"], case["seg_len"]
    teacher, h, tok, pw = case["teacher"], case["h"], case["draft_tokens"], case["pos_weight"]
    W_in, master, m, v = case["W"], case["master"], case["m"], case["v"]
    # host copies of the exact bits
    t_bits, h_bits, W_bits = bits(teacher), bits(h), bits(W_in)
    tok_h, pw_h = tok.cpu().numpy(), pw.cpu().numpy()
    o_mask, o_tau, o_am = O.accept_mask(t_bits, tok_h, C)
    rng = np.random.Generator(np.random.PCG64(99 + cfg_id))
    rows = _sample_rows(V, rng, tok_h, o_am)
    rows_t = torch.from_numpy(rows).to(dev)
    master0, m0, v0 = (x[rows_t].cpu().numpy() for x in (master, m, v))

    cfg = tts.make_config(V, d, T, C, tts.TTS_BF16, tts.TTS_BF16, tts.TTS_ADAMW, c["lr"], c["beta1"], c["beta2"],
                          c["eps"], c["weight_decay"], mask_mode_g)
    ctx = tts.tts_ctx_create(cfg, 0)
    try:
        W_out = torch.empty_like(W_in)
        W_before = W_in.clone()
        mask = torch.zeros(T, dtype=torch.uint8, device=dev)
        tau = torch.zeros(T // C, dtype=torch.int32, device=dev)
        am = torch.zeros(T, dtype=torch.int32, device=dev)
        loss = torch.zeros(1, dtype=torch.float32, device=dev)
        kl = torch.zeros(T, dtype=torch.float32, device=dev)
        gh = torch.full((T, d), float("nan"), dtype=torch.float32, device=dev)
        side = torch.cuda.Stream()
        torch.cuda.synchronize()
        tts.tts_accept_mask(ctx, teacher, tok, T, mask, tau, am, side)
        tts.tts_distill_step(ctx, teacher, h, W_in, W_out, master, m, v, pw, mask, T, case["loss_scale"], loss, kl,
                             gh, None, side)
        tts.tts_wait_step(ctx, torch.cuda.current_stream())
        tts.tts_sync_step(ctx)
        torch.cuda.synchronize()
        assert tts.tts_last_step_used_tensor_path(ctx) == 1
    finally:
        tts.tts_ctx_destroy(ctx)

    # ---- a1: bit-exact
    np.testing.assert_array_equal(am.cpu().numpy(), o_am)
    np.testing.assert_array_equal(mask.cpu().numpy(), o_mask)
    np.testing.assert_array_equal(tau.cpu().numpy(), o_tau)
    if case["tau_star"] is not None:
        np.testing.assert_array_equal(o_tau, case["tau_star"])

    # ---- a2-a3: normalisers, KL rows, loss
    z, lse_t, lse_z, o_kl = O.row_normalisers(t_bits, h_bits, W_bits)
    omega = O.row_weights(pw_h, o_mask, mask_mode_o, C)
    o_loss = case["loss_scale"] * float((omega * o_kl).sum())
    g_loss = float(loss.item())
    assert abs(g_loss - o_loss) <= 1e-3 * abs(o_loss) + 1e-6, (g_loss, o_loss)
    assert np.all(np.abs(kl.cpu().numpy() - o_kl) <= 1e-3 * np.abs(o_kl) + 1e-5)

    # ---- a5: gh complete
    o_gh = O.gh_full(z, lse_t, lse_z, t_bits, W_bits, omega, case["loss_scale"])
    g_gh = gh.cpu().numpy().astype(np.float64)
    assert np.all(np.isfinite(g_gh))
    assert max_abs(g_gh - o_gh) <= 2e-3 * max_abs(o_gh), (max_abs(g_gh - o_gh), max_abs(o_gh))

    # ---- a6-a7 on sampled vocabulary rows
    r = O.distill_step_rows(rows, z, lse_t, lse_z, t_bits, h_bits, W_bits[rows], master0, m0, v0, omega,
                            loss_scale=case["loss_scale"], optimizer="adamw", lr=c["lr"], beta1=c["beta1"],
                            beta2=c["beta2"], eps=c["eps"], weight_decay=c["weight_decay"], step=1)
    g_master = master[rows_t].cpu().numpy().astype(np.float64)
    g_m = m[rows_t].cpu().numpy().astype(np.float64)
    g_v = v[rows_t].cpu().numpy().astype(np.float64)
    g_gW = g_m / (1.0 - c["beta1"])                      # first step from m = 0: m = (1 - b1) g
    for name, gg, ref in (("gW", g_gW, r["gW"]), ("master", g_master, r["master"]), ("m", g_m, r["m"]),
                          ("v", g_v, r["v"])):
        assert np.all(np.isfinite(gg)), name
        assert max_abs(gg - ref) <= 2e-3 * max_abs(ref) + 1e-30, (name, max_abs(gg - ref), max_abs(ref))
    # the update itself (R13): on rows with a sizeable gradient the step must agree to 2% of lr
    M_old = master0.astype(np.float64)
    d_ref, d_gpu = r["master"] - M_old, g_master - M_old
    big = np.abs(r["gW"]) >= 1e-2 * max_abs(r["gW"])
    assert big.any()
    ulp = np.spacing(np.abs(master0[big])).astype(np.float64)
    assert np.all(np.abs(d_gpu[big] - d_ref[big]) <= 0.02 * c["lr"] + ulp)
    moved = np.abs(d_ref) > 4 * np.spacing(np.abs(master0)).astype(np.float64)
    badsign = np.sign(d_gpu[moved]) != np.sign(d_ref[moved])
    assert badsign.mean() <= 1e-3, badsign.mean()

    # ---- properties over the whole state
    for x in (master, m, v):
        assert bool(torch.isfinite(x).all())
    assert bool((W_out == master.to(torch.bfloat16)).all())      # rn_bf16 of the GPU's own master, bit for bit
    assert bool((v >= 0).all())
    col = m.sum(dim=0, dtype=torch.float64).abs()
    colabs = m.abs().sum(dim=0, dtype=torch.float64)
    assert float((col / (colabs + 1e-30)).max()) < 1e-3          # sum_v gW[v, j] = 0
    assert bool((W_in == W_before).all())                        # the double buffer's read side is untouched


def test_config3_qwen3_8b_full_size():
    _run_fullsize(3)


def test_config3_full_size_accepted_plus_one():
    _run_fullsize(3, tts.TTS_ROWS_ACCEPTED_PLUS_ONE, O.ROWS_ACCEPTED_PLUS_ONE)


def test_config2_llama31_8b_full_size():
    _run_fullsize(2)


def test_config5_qwen3_32b_head_one_round_full_size():
    _run_fullsize(5)


def test_config4_batched_512_rows_full_size():
    _run_fullsize(4)
