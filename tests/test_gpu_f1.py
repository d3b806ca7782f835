"""f1: the step with the drafter's logits taken as given (pass a2 skipped), the
lambda * K~L(q_t || q) term and K > 1 inner steps on one round's signal, against the
oracle on the same seeded inputs.  Tolerances as in gpu_util.check_step (north_star)."""
import numpy as np
import pytest
import torch

from oracle import tts_oracle as O
from paper_2605_09329_b200 import tts
from workloads import synth

from gpu_util import _dev, bits, config_for, max_abs

pytestmark = pytest.mark.gpu


def _setup(case, kernel_path=tts.TTS_PATH_AUTO):
    ctx = tts.tts_ctx_create(config_for(case, kernel_path=kernel_path, max_inner_steps=8), 0)
    bf = case["cfg"]["param"] == synth.BF16
    t = dict(teacher=_dev(case["teacher"]), h=_dev(case["h"]), tok=_dev(case["draft_tokens"]), W_in=_dev(case["W"]),
             master=_dev(case["master"]) if bf else None, m=_dev(case["m"]), v=_dev(case["v"]),
             pw=_dev(case["pos_weight"]))
    t["W_out"] = torch.empty_like(t["W_in"])
    T, d = case["T"], case["d"]
    t["mask"] = torch.zeros(T, dtype=torch.uint8, device="cuda")
    t["tau"] = torch.zeros(T // case["seg_len"], dtype=torch.int32, device="cuda")
    t["kl"] = torch.zeros(T, dtype=torch.float32, device="cuda")
    t["gh"] = torch.full((T, d), float("nan"), dtype=torch.float32, device="cuda")
    return ctx, t


def _oracle_kw(case):
    c = case["cfg"]
    return dict(seg_len=case["seg_len"], loss_scale=case["loss_scale"],
                optimizer="sgd" if c["optimizer"] == synth.SGD else "adamw", lr=c["lr"], beta1=c["beta1"],
                beta2=c["beta2"], eps=c["eps"], weight_decay=c["weight_decay"])


def _check_state(g_master, g_m, g_v, g_gh, o, tol=2e-3):
    for name, gg, ref in (("master", g_master, o["master"]), ("m", g_m, o["m"]), ("v", g_v, o["v"]),
                          ("gh", g_gh, o["gh"])):
        if gg is None or ref is None:
            continue
        gg = gg.cpu().numpy().astype(np.float64)
        assert np.all(np.isfinite(gg)), name
        assert max_abs(gg - ref) <= tol * max_abs(ref) + 1e-30, (name, max_abs(gg - ref), max_abs(ref))


@pytest.mark.parametrize("V,d,path", [(2048 + 128, 1024, tts.TTS_PATH_AUTO), (4096, 256, tts.TTS_PATH_AUTO),
                                      (1000, 72, tts.TTS_PATH_AUTO), (2048, 256, tts.TTS_PATH_SIMT)])
def test_given_draft_logits_skip_pass_a(V, d, path):
    """The caller's z (a perturbed copy of h W^T, so that a silently recomputed z would fail) drives loss, dl, gW,
    gh and the update; the launch count drops by the logits kernel (+ its memset)."""
    case = synth.make_case(3, V=V, d=d)
    rng = np.random.Generator(np.random.PCG64(5))
    W = O.widen(case["W"]); h = O.widen(case["h"])
    z_given = (h @ W.T + 0.05 * rng.standard_normal((case["T"], V))).astype(np.float32)
    mask, tau, _ = O.accept_mask(case["teacher"], case["draft_tokens"], case["seg_len"])
    o = O.distill_step(case["teacher"], case["h"], case["W"], case["master"], case["m"], case["v"], case["pos_weight"],
                       mask, draft_logits=z_given, **_oracle_kw(case))
    ctx, t = _setup(case, path)
    try:
        loss = torch.zeros(1, device="cuda")
        tts.tts_accept_mask(ctx, t["teacher"], t["tok"], case["T"], t["mask"], t["tau"])
        tts.tts_distill_step(ctx, t["teacher"], t["h"], t["W_in"], t["W_out"], t["master"], t["m"].clone(),
                             t["v"].clone(), t["pw"], t["mask"], case["T"], case["loss_scale"], loss, None, t["gh"])
        n_full = tts.tts_last_launch_count(ctx)
        t["master"].copy_(_dev(case["master"]))
        tts.tts_set_step_count(ctx, 0)
        tts.tts_distill_step_ex(ctx, t["teacher"], t["h"], t["W_in"], t["W_out"], t["master"], t["m"], t["v"], t["pw"],
                                t["mask"], case["T"], case["loss_scale"], loss, t["kl"], t["gh"], None,
                                draft_logits=_dev(z_given))
        n_given = tts.tts_last_launch_count(ctx)
        torch.cuda.synchronize()
        # pass a2 is gone; on the tensor path its epilogue carried a3, which now runs as its own sweep
        assert n_given == n_full - 1 if path == tts.TTS_PATH_SIMT else n_given <= n_full
        assert abs(float(loss.item()) - o["loss"]) <= 1e-3 * abs(o["loss"]) + 1e-6
        assert np.all(np.abs(t["kl"].cpu().numpy() - o["kl_rows"]) <= 1e-3 * np.abs(o["kl_rows"]) + 1e-5)
        _check_state(t["master"], t["m"], t["v"], t["gh"], o)
        np.testing.assert_array_equal(bits(t["W_out"]), O.f32_to_bf16_bits(t["master"].cpu().numpy()))
    finally:
        tts.tts_ctx_destroy(ctx)


@pytest.mark.parametrize("V,d,path", [(2048 + 128, 1024, tts.TTS_PATH_AUTO), (4096, 256, tts.TTS_PATH_AUTO),
                                      (2048, 256, tts.TTS_PATH_SIMT)])
def test_lambda_term_with_a_distinct_reference(V, d, path):
    """ref_logits != z: loss gains lam * sum w KL(q_ref || q), dl gains lam (q - q_ref)."""
    case = synth.make_case(3, V=V, d=d, nonzero_state=True, step=4)
    rng = np.random.Generator(np.random.PCG64(6))
    W = O.widen(case["W"]); h = O.widen(case["h"])
    z_ref = (h @ W.T + 0.8 * rng.standard_normal((case["T"], V))).astype(np.float32)
    lam = 0.6
    mask, _, _ = O.accept_mask(case["teacher"], case["draft_tokens"], case["seg_len"])
    o = O.distill_step(case["teacher"], case["h"], case["W"], case["master"], case["m"], case["v"], case["pos_weight"],
                       mask, lam=lam, z_ref=z_ref, step=4, **_oracle_kw(case))
    o0 = O.distill_step(case["teacher"], case["h"], case["W"], case["master"], case["m"], case["v"], case["pos_weight"],
                        mask, step=4, **_oracle_kw(case))
    assert abs(o["loss"] - o0["loss"]) > 0.05 * abs(o0["loss"])      # the term is visible in this case
    ctx, t = _setup(case, path)
    try:
        loss = torch.zeros(1, device="cuda")
        tts.tts_set_step_count(ctx, 3)
        tts.tts_distill_step_ex(ctx, t["teacher"], t["h"], t["W_in"], t["W_out"], t["master"], t["m"], t["v"], t["pw"],
                                None, case["T"], case["loss_scale"], loss, t["kl"], t["gh"], None,
                                ref_logits=_dev(z_ref), lam=lam)
        torch.cuda.synchronize()
        assert abs(float(loss.item()) - o["loss"]) <= 1e-3 * abs(o["loss"]) + 1e-6
        assert np.all(np.abs(t["kl"].cpu().numpy() - o["kl_rows"]) <= 1e-3 * np.abs(o["kl_rows"]) + 1e-5)
        _check_state(t["master"], t["m"], t["v"], t["gh"], o)
    finally:
        tts.tts_ctx_destroy(ctx)


def test_lambda_is_inert_at_one_step():
    """R3: with ref_logits == the step's own z the loss and every gradient are independent of lambda."""
    case = synth.make_case(2, V=2048, d=1024)
    outs = []
    for lam in (0.0, 5.0):
        ctx, t = _setup(case)
        try:
            loss = torch.zeros(1, device="cuda")
            zbuf = torch.empty(16, 2048, device="cuda")
            tts.tts_distill_step_ex(ctx, t["teacher"], t["h"], t["W_in"], t["W_out"], t["master"].clone(),
                                    t["m"].clone(), t["v"].clone(), t["pw"], None, 16, 1.0, loss,
                                    draft_logits_out=zbuf)
            tts.tts_set_step_count(ctx, 0)
            tts.tts_distill_step_ex(ctx, t["teacher"], t["h"], t["W_in"], t["W_out"], t["master"], t["m"], t["v"],
                                    t["pw"], None, 16, 1.0, loss, None, t["gh"], None, draft_logits=zbuf,
                                    ref_logits=zbuf, lam=lam)
            torch.cuda.synchronize()
            outs.append((float(loss.item()), t["m"].cpu().numpy(), t["gh"].cpu().numpy()))
        finally:
            tts.tts_ctx_destroy(ctx)
    assert abs(outs[0][0] - outs[1][0]) <= 1e-6 * abs(outs[0][0])
    assert max_abs(outs[0][1] - outs[1][1]) <= 1e-6 * max_abs(outs[0][1])
    assert max_abs(outs[0][2] - outs[1][2]) <= 1e-5 * max_abs(outs[0][2])


@pytest.mark.parametrize("V,d,K,path", [(2048 + 128, 1024, 3, tts.TTS_PATH_AUTO), (2048, 256, 2, tts.TTS_PATH_AUTO),
                                        (1024, 128, 3, tts.TTS_PATH_SIMT)])
def test_inner_steps_match_oracle(V, d, K, path):
    case = synth.make_case(3, V=V, d=d)
    c = case["cfg"]
    c["lr"] = 1e-3                      # large enough for the K steps to move z visibly
    lam = 0.5
    mask, _, _ = O.accept_mask(case["teacher"], case["draft_tokens"], case["seg_len"])
    o = O.distill_inner_steps(case["teacher"], case["h"], case["W"], case["master"], case["m"], case["v"],
                              case["pos_weight"], mask, K=K, lam=lam, **_oracle_kw(case))
    ctx, t = _setup(case, path)
    try:
        losses = torch.zeros(K, device="cuda")
        tts.tts_accept_mask(ctx, t["teacher"], t["tok"], case["T"], t["mask"], t["tau"])
        tts.tts_distill_inner_steps(ctx, t["teacher"], t["h"], t["W_in"], t["W_out"], t["master"], t["m"], t["v"],
                                    t["pw"], t["mask"], case["T"], case["loss_scale"], K, lam, None, losses, t["kl"],
                                    t["gh"])
        torch.cuda.synchronize()
        assert tts.tts_get_step_count(ctx) == K
        g_losses = losses.cpu().numpy()
        assert np.all(np.abs(g_losses - o["losses"]) <= 1e-3 * np.abs(o["losses"]) + 1e-6), (g_losses, o["losses"])
        assert o["losses"][-1] < o["losses"][0]
        assert np.all(np.abs(t["kl"].cpu().numpy() - o["kl_rows_step1"]) <= 1e-3 * np.abs(o["kl_rows_step1"]) + 1e-5)
        _check_state(t["master"], t["m"], t["v"], t["gh"], o)
        np.testing.assert_array_equal(bits(t["W_out"]), O.f32_to_bf16_bits(t["master"].cpu().numpy()))
        # the accumulated movement agrees (R13: the master tolerance alone would pass a no-op at small lr)
        M0 = case["master"].astype(np.float64)
        d_ref, d_gpu = o["master"] - M0, t["master"].cpu().numpy().astype(np.float64) - M0
        assert np.abs(d_gpu - d_ref).mean() <= 0.02 * np.abs(d_ref).mean()
    finally:
        tts.tts_ctx_destroy(ctx)


def test_extras_argument_checks():
    case = synth.make_case(2, V=2048, d=128)
    ctx, t = _setup(case)
    try:
        loss = torch.zeros(1, device="cuda")
        z = torch.zeros(16, 2048, device="cuda")
        with pytest.raises(tts.TTSError):      # given and out together
            tts.tts_distill_step_ex(ctx, t["teacher"], t["h"], t["W_in"], t["W_out"], t["master"], t["m"], t["v"],
                                    t["pw"], None, 16, 1.0, loss, draft_logits=z, draft_logits_out=z)
        with pytest.raises(tts.TTSError):      # negative lambda
            tts.tts_distill_step_ex(ctx, t["teacher"], t["h"], t["W_in"], t["W_out"], t["master"], t["m"], t["v"],
                                    t["pw"], None, 16, 1.0, loss, ref_logits=z, lam=-1.0)
        with pytest.raises(tts.TTSError):      # K = 0
            tts.tts_distill_inner_steps(ctx, t["teacher"], t["h"], t["W_in"], t["W_out"], t["master"], t["m"], t["v"],
                                        t["pw"], None, 16, 1.0, 0, 0.1, None, loss)
        assert tts.tts_get_step_count(ctx) == 0
    finally:
        tts.tts_ctx_destroy(ctx)
