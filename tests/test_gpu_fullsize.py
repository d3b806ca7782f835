"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (side stream, W_in / W_out
double buffer, no gW dump): the CUDA path against the fp64 oracle on outputs the oracle can compute one by one.

  * mask, tau, teacher argmax     bit-exact over the whole [T, V] input
  * loss, KL_r                    the oracle's full-vocabulary normalisers (row_normalisers, slab by slab)
  * gh [T, d]                     complete (gh_full)
  * master / m / v / W_out        EVERY vocabulary row at configs 2, 3 and 5 (slabs of 4096 rows through
                                  distill_step_rows), every fourth slab plus the last one (>= 25% of the rows) at the
                                  512-row config 4; gW rows from the first-step moment m = (1-b1) g.  A sample of rows
                                  (tile edges, the canvas tokens and the teacher's argmax tokens, i.e. the rows with
                                  the largest gradients) fixes the threshold of R13's "sizeable gradient" pin first
  * properties over ALL V x d     W_out == rn_bf16(master) bit-exactly, state finite, column sums of m vanish
                                  (sum_v dl[r, v] = 0), v >= 0
  * config 5, rounds 0, 1, 2      three consecutive rounds of the stream recipe at full size (teacher built on the
                                  device from the CURRENT weights, R16); every round's transition is checked against
                                  the oracle applied to the state the GPU held before that round
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


SLAB = 4096


def _check_rows_in_slabs(slabs, V, z, lse_t, lse_z, t_bits, h_bits, W_bits, pre, post, W_out, omega, c, loss_scale,
                         step, g_thr, gW_from_m):
    """a6 + a7 on whole slabs of vocabulary rows: `pre` / `post` are the device tensors (master, m, v) before and after
    the step.  Accumulates the north_star pins (max abs error over max |ref| for gW, master, m, v) and R13's pins over
    all rows visited; returns the observed figures."""
    lr = c["lr"]

    def one_slab(v0):
        a = dict(err={k: 0.0 for k in ("gW", "master", "m", "v")}, ref={k: 0.0 for k in ("gW", "master", "m", "v")},
                 big_worst=0.0, n_big=0, moved=0, badsign=0, n_w=0, w_gt1=0, rows=0)
        v1 = min(V, v0 + SLAB)
        rows = np.arange(v0, v1)
        p_m, p_a, p_v = (x[v0:v1].cpu().numpy() for x in pre)
        r = O.distill_step_rows(rows, z, lse_t, lse_z, t_bits, h_bits, W_bits[v0:v1], p_m, p_a, p_v, omega,
                                loss_scale=loss_scale, optimizer="adamw", lr=lr, beta1=c["beta1"], beta2=c["beta2"],
                                eps=c["eps"], weight_decay=c["weight_decay"], step=step)
        g_master, g_m, g_v = (x[v0:v1].cpu().numpy().astype(np.float64) for x in post)
        cmp = [("master", g_master, r["master"]), ("m", g_m, r["m"]), ("v", g_v, r["v"])]
        if gW_from_m:                                     # first step from m = 0: m = (1 - b1) g
            cmp.append(("gW", g_m / (1.0 - c["beta1"]), r["gW"]))
        for name, gg, ref in cmp:
            assert np.all(np.isfinite(gg)), (name, v0)
            a["err"][name] = max_abs(gg - ref)
            a["ref"][name] = max_abs(ref)
        M_old = p_m.astype(np.float64)
        d_ref, d_gpu = r["master"] - M_old, g_master - M_old
        big = np.abs(r["gW"]) >= g_thr
        if big.any():
            ulp = np.spacing(np.abs(p_m[big])).astype(np.float64)
            a["big_worst"] = float(np.max(np.abs(d_gpu[big] - d_ref[big]) - ulp)) / lr
            a["n_big"] = int(big.sum())
        moved = np.abs(d_ref) > 4 * np.spacing(np.abs(p_m)).astype(np.float64)
        a["moved"] = int(moved.sum())
        a["badsign"] = int((np.sign(d_gpu[moved]) != np.sign(d_ref[moved])).sum())
        # working copy against the oracle's (R12): <= 1 bf16 ulp + the master difference; > 1 ulp on <= 1e-4 of elements
        wg_bits = bits(W_out[v0:v1])
        wo_bits = O.working_copy_bits(r["master"])
        wg, wo = O.bf16_bits_to_f64(wg_bits), O.bf16_bits_to_f64(wo_bits)
        mag = np.maximum(np.maximum(np.abs(wg), np.abs(wo)), 2.0 ** -126)
        ulp = 2.0 ** (np.floor(np.log2(mag)) - 7)
        assert np.all(np.abs(wg - wo) <= ulp + np.abs(g_master - r["master"])), v0
        a["w_gt1"] = int((np.abs(wg_bits.astype(np.int32) - wo_bits.astype(np.int32)) > 1).sum())
        a["n_w"] = wg_bits.size
        a["rows"] = v1 - v0
        return a

    # the slabs are independent and numpy releases the GIL in its large operations: a few host threads in parallel
    from concurrent.futures import ThreadPoolExecutor
    acc = dict(err={k: 0.0 for k in ("gW", "master", "m", "v")}, ref={k: 0.0 for k in ("gW", "master", "m", "v")},
               big_worst=0.0, n_big=0, moved=0, badsign=0, n_w=0, w_gt1=0, rows=0)
    with ThreadPoolExecutor(max_workers=6) as ex:
        for a in ex.map(one_slab, slabs):
            for k in acc["err"]:
                acc["err"][k] = max(acc["err"][k], a["err"][k])
                acc["ref"][k] = max(acc["ref"][k], a["ref"][k])
            acc["big_worst"] = max(acc["big_worst"], a["big_worst"])
            for k in ("n_big", "moved", "badsign", "n_w", "w_gt1", "rows"):
                acc[k] += a[k]
    for name in acc["err"]:
        if acc["ref"][name] > 0:
            assert acc["err"][name] <= 2e-3 * acc["ref"][name] + 1e-30, (name, acc["err"][name], acc["ref"][name])
    assert acc["n_big"] > 0
    assert acc["big_worst"] <= 0.02, acc["big_worst"]                 # R13: 2% of lr on sizeable gradients
    assert acc["badsign"] <= 1e-3 * max(acc["moved"], 1), (acc["badsign"], acc["moved"])
    assert acc["w_gt1"] <= 1e-4 * acc["n_w"], (acc["w_gt1"], acc["n_w"])
    return acc


def _run_fullsize(cfg_id, mask_mode_g=tts.TTS_ROWS_ALL, mask_mode_o=O.ROWS_ALL, slab_stride=1):
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
    master_pre = master.clone()                    # m = v = 0 before the step: no copies needed

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
        assert tts.tts_last_device_status(ctx) == 0
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

    # ---- a6-a7: the sampled rows (they hold the largest gradients) fix the "sizeable gradient" threshold of R13 ...
    rows_t = torch.from_numpy(rows).to(dev)
    zeros = np.zeros((rows.size, d), dtype=np.float32)
    r = O.distill_step_rows(rows, z, lse_t, lse_z, t_bits, h_bits, W_bits[rows], master_pre[rows_t].cpu().numpy(),
                            zeros, zeros, omega, loss_scale=case["loss_scale"], optimizer="adamw", lr=c["lr"],
                            beta1=c["beta1"], beta2=c["beta2"], eps=c["eps"], weight_decay=c["weight_decay"], step=1)
    g_thr = 1e-2 * max_abs(r["gW"])
    # ... then whole slabs: every row (slab_stride = 1), or every slab_stride-th slab plus the last one
    starts = list(range(0, V, SLAB))
    slabs = [s0 for i, s0 in enumerate(starts) if i % slab_stride == 0 or i == len(starts) - 1]
    zero_dev = torch.zeros_like(master_pre[:1]).expand(V, d)      # m = v = 0 before the step (a view, no memory)
    acc = _check_rows_in_slabs(slabs, V, z, lse_t, lse_z, t_bits, h_bits, W_bits, (master_pre, zero_dev, zero_dev),
                               (master, m, v), W_out, omega, c, case["loss_scale"], 1, g_thr, True)
    assert acc["rows"] >= (V if slab_stride == 1 else V // 4)
    print("config %d: %d of %d rows checked; max err / max|ref| %s; dM(big) worst %.4f lr over %d elements; sign "
          "mismatch %d / %d; W_out > 1 ulp %d / %d" % (
              cfg_id, acc["rows"], V, {k: acc["err"][k] / max(acc["ref"][k], 1e-300) for k in acc["err"]},
              acc["big_worst"], acc["n_big"], acc["badsign"], acc["moved"], acc["w_gt1"], acc["n_w"]))

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
    _run_fullsize(3, tts.TTS_ROWS_ACCEPTED_PLUS_ONE, O.ROWS_ACCEPTED_PLUS_ONE, slab_stride=4)


def test_config2_llama31_8b_full_size():
    _run_fullsize(2)


def test_config4_batched_512_rows_full_size():
    _run_fullsize(4, slab_stride=4)


def test_config5_stream_rounds_0_1_2_full_size():
    """"Oracle parity at full scale on rounds 0, 1, 2".  The stream recipe of bench.py --stream on the
    Qwen3-32B-shaped head (R16): per round h_t ~ N(0,1) and the teacher is built ON THE DEVICE from the CURRENT weights,
    t_t = rn_bf16(h_t W_cur^T + mu_t u + 1.5 eps_t).  Each round's inputs and the state the GPU held before the round
    are copied to the host bit for bit and the oracle's step from THAT state is compared with what the GPU wrote:
    loss, KL rows, mask, gh complete; master / m / v / W_out on every row at round 0 and on every fourth slab at
    rounds 1 and 2 (non-zero moments, Adam counts 2 and 3).  Accumulated drift over many rounds is the scaled-down
    300-round test's job (tests/test_gpu_stream.py)."""
    from paper_2605_09329_b200.scheduler import DraftHeadUpdater
    dev = "cuda:0"
    case = synth.make_case_device(5, dev)
    c = case["cfg"]
    V, d, C = case["V"], case["d"], case["seg_len"]
    T = C
    W0, master, m, v = case["W"], case["master"], case["m"], case["v"]
    pw = case["pos_weight"][:T].contiguous()
    u = torch.from_numpy(synth.stream_direction(V, c["seed"])).to(dev)
    up = DraftHeadUpdater(W0, master, m, v, seg_len=C, T_max=T, stride=1, lr=c["lr"], beta1=c["beta1"],
                          beta2=c["beta2"], eps=c["eps"], weight_decay=c["weight_decay"], want_gh=True)
    try:
        g = torch.Generator(device=dev)
        g.manual_seed(1000003 * (c["seed"] + 1))
        pw_h = pw.cpu().numpy()
        for t in range(3):
            W_cur = up.weights()
            h = torch.empty(T, d, device=dev).normal_(0.0, 1.0, generator=g).to(torch.bfloat16)
            zc = torch.matmul(h, W_cur.T).float()
            tok = torch.argmax(zc, dim=1).to(torch.int32)
            noise = torch.empty(T, V, device=dev).normal_(0.0, 1.0, generator=g)
            teacher = (zc + synth.stream_mu(t, 4000, c.get("mu_max", 3.0)) * u + 1.5 * noise).to(torch.bfloat16)
            del noise, zc
            pre = (master.clone(), m.clone(), v.clone())
            W_bits = bits(W_cur)
            torch.cuda.synchronize()
            assert up.on_round_end(teacher, h, tok, pw, T, 1.0)
            tts.tts_sync_step(up.ctx)
            torch.cuda.synchronize()
            t_bits, h_bits, tok_h = bits(teacher), bits(h), tok.cpu().numpy()
            o_mask, o_tau, _ = O.accept_mask(t_bits, tok_h, C)
            np.testing.assert_array_equal(up.mask.cpu().numpy(), o_mask)
            np.testing.assert_array_equal(up.tau.cpu().numpy(), o_tau)
            z, lse_t, lse_z, o_kl = O.row_normalisers(t_bits, h_bits, W_bits)
            omega = O.row_weights(pw_h, o_mask, O.ROWS_ALL, C)
            o_loss = float((omega * o_kl).sum())
            assert abs(float(up.loss.item()) - o_loss) <= 1e-3 * abs(o_loss) + 1e-6, (t, float(up.loss.item()), o_loss)
            assert np.all(np.abs(up.kl_rows.cpu().numpy() - o_kl) <= 1e-3 * np.abs(o_kl) + 1e-5)
            o_gh = O.gh_full(z, lse_t, lse_z, t_bits, W_bits, omega, 1.0)
            assert max_abs(up.gh.cpu().numpy().astype(np.float64) - o_gh) <= 2e-3 * max_abs(o_gh)
            # threshold of the "sizeable gradient" pin from the canvas-token rows (the largest gradients)
            rows = np.unique(np.concatenate([tok_h.astype(np.int64), np.arange(0, V, 4099)]))
            rows_t = torch.from_numpy(rows).to(dev)
            r = O.distill_step_rows(rows, z, lse_t, lse_z, t_bits, h_bits, W_bits[rows], pre[0][rows_t].cpu().numpy(),
                                    pre[1][rows_t].cpu().numpy(), pre[2][rows_t].cpu().numpy(), omega, loss_scale=1.0,
                                    optimizer="adamw", lr=c["lr"], beta1=c["beta1"], beta2=c["beta2"], eps=c["eps"],
                                    weight_decay=c["weight_decay"], step=t + 1)
            g_thr = 1e-2 * max_abs(r["gW"])
            starts = list(range(0, V, SLAB))
            stride = 1 if t == 0 else 4
            slabs = [s0 for i, s0 in enumerate(starts) if i % stride == 0 or i == len(starts) - 1]
            acc = _check_rows_in_slabs(slabs, V, z, lse_t, lse_z, t_bits, h_bits, W_bits, pre, (master, m, v),
                                       up.weights(), omega, c, 1.0, t + 1, g_thr, t == 0)
            print("config 5 round %d: %d rows; dM(big) worst %.4f lr; sign mismatch %d / %d; W_out > 1 ulp %d / %d" % (
                t, acc["rows"], acc["big_worst"], acc["badsign"], acc["moved"], acc["w_gt1"], acc["n_w"]))
            assert bool((up.weights() == master.to(torch.bfloat16)).all())
            del pre
        assert tts.tts_get_step_count(up.ctx) == 3
    finally:
        up.close()
