"""Helpers for the GPU parity tests: run the CUDA path (through the C ABI binding) on a seeded
synthetic case and return numpy arrays; run the fp64 oracle on the same arrays.  Test
infrastructure only."""
from __future__ import annotations

import numpy as np
import torch

from oracle import tts_oracle as O
from paper_2605_09329_b200 import tts
from workloads import synth


def _dev(a, dtype=None):
    """numpy -> cuda tensor; uint16 arrays are bf16 bit patterns."""
    if a is None:
        return None
    if a.dtype == np.uint16:
        return torch.from_numpy(a.view(np.int16).copy()).cuda().view(torch.bfloat16)
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def bits(t: torch.Tensor) -> np.ndarray:
    """bf16 cuda tensor -> uint16 bit patterns."""
    return t.view(torch.int16).cpu().numpy().view(np.uint16)


def config_for(case, *, mask_mode=tts.TTS_ROWS_ALL, kernel_path=tts.TTS_PATH_AUTO, T_max=None, max_ctas=0,
               moment_dtype=tts.TTS_MOMENT_F32, max_inner_steps=0, flags=0):
    c = case["cfg"]
    return tts.make_config(case["V"], case["d"], T_max or case["T"], case["seg_len"], c["param"], c["logits"],
                           c["optimizer"], c["lr"], c["beta1"], c["beta2"], c["eps"], c["weight_decay"], mask_mode,
                           max_ctas, kernel_path, moment_dtype, max_inner_steps, flags)


def run_gpu(case, *, mask_mode=tts.TTS_ROWS_ALL, kernel_path=tts.TTS_PATH_AUTO, want_gW=True, want_gh=True,
            alias_w=False, side_stream=True, max_ctas=0, flags=0, moments="f32", sr_seed=0):
    """One tts_accept_mask + tts_distill_step on cuda:0.  Returns a dict of numpy results."""
    T, V, d = case["T"], case["V"], case["d"]
    bf = case["cfg"]["param"] == synth.BF16
    lowp = moments == "bf16"
    cfg = config_for(case, mask_mode=mask_mode, kernel_path=kernel_path, max_ctas=max_ctas, flags=flags,
                     moment_dtype=tts.TTS_MOMENT_BF16 if lowp else tts.TTS_MOMENT_F32)
    cfg.sr_seed = sr_seed
    ctx = tts.tts_ctx_create(cfg, 0)
    try:
        if case.get("step", 1) > 1:
            tts.tts_set_step_count(ctx, case["step"] - 1)
        teacher, h, tok = _dev(case["teacher"]), _dev(case["h"]), _dev(case["draft_tokens"])
        W_in = _dev(case["W"])
        W_out = W_in if alias_w else torch.empty_like(W_in)
        master = _dev(case["master"]) if bf else None
        if lowp:     # bf16 moment storage: the case's fp32 moments rounded to nearest (uint16 bits -> bf16 tensors)
            m, v = _dev(synth.f32_to_bf16_bits(case["m"])), _dev(synth.f32_to_bf16_bits(case["v"]))
        else:
            m, v = _dev(case["m"]), _dev(case["v"])
        pw = _dev(case["pos_weight"])
        mask = torch.zeros(T, dtype=torch.uint8, device="cuda")
        tau = torch.zeros(T // case["seg_len"], dtype=torch.int32, device="cuda")
        am = torch.zeros(T, dtype=torch.int32, device="cuda")
        loss = torch.zeros(1, dtype=torch.float32, device="cuda")
        kl = torch.zeros(T, dtype=torch.float32, device="cuda")
        gh = torch.full((T, d), float("nan"), dtype=torch.float32, device="cuda") if want_gh else None
        gW = torch.full((V, d), float("nan"), dtype=torch.float32, device="cuda") if want_gW else None
        torch.cuda.synchronize()
        s = torch.cuda.Stream() if side_stream else torch.cuda.current_stream()
        tts.tts_accept_mask(ctx, teacher, tok, T, mask, tau, am, s)
        mask_launches = tts.tts_last_launch_count(ctx)
        tts.tts_distill_step(ctx, teacher, h, W_in, W_out, master, m, v, pw, mask, T, case["loss_scale"], loss, kl,
                             gh, gW, s)
        step_launches = tts.tts_last_launch_count(ctx)
        tts.tts_wait_step(ctx, torch.cuda.current_stream())
        tts.tts_sync_step(ctx)
        torch.cuda.synchronize()
        out = dict(mask=mask.cpu().numpy(), tau=tau.cpu().numpy(), argmax=am.cpu().numpy(),
                   loss=float(loss.item()), kl_rows=kl.cpu().numpy(),
                   gh=gh.cpu().numpy() if want_gh else None, gW=gW.cpu().numpy() if want_gW else None,
                   used_tensor=tts.tts_last_step_used_tensor_path(ctx), step_count=tts.tts_get_step_count(ctx),
                   launches=mask_launches + step_launches, dev_status=tts.tts_last_device_status(ctx))
        if bf:
            out["master"] = master.cpu().numpy()
            out["W_out"] = bits(W_out)
        else:
            out["master"] = W_out.cpu().numpy()
            out["W_out"] = out["master"]
        if lowp:
            out["m_bits"], out["v_bits"] = bits(m), bits(v)
            out["m"], out["v"] = synth.bf16_bits_to_f32(out["m_bits"]), synth.bf16_bits_to_f32(out["v_bits"])
        else:
            out["m"] = m.cpu().numpy() if m is not None else None
            out["v"] = v.cpu().numpy() if v is not None else None
        return out
    finally:
        tts.tts_ctx_destroy(ctx)


def run_oracle(case, *, mask_mode=O.ROWS_ALL, moments="f32", sr_seed=0):
    c = case["cfg"]
    mask, tau, am = O.accept_mask(case["teacher"], case["draft_tokens"], case["seg_len"])
    m_in, v_in = case["m"], case["v"]
    if moments == "bf16":
        m_in, v_in = O.f32_to_bf16_bits(m_in), O.f32_to_bf16_bits(v_in)
    r = O.distill_step(case["teacher"], case["h"], case["W"], case["master"], m_in, v_in,
                       case["pos_weight"], mask, seg_len=case["seg_len"], mask_mode=mask_mode,
                       loss_scale=case["loss_scale"], optimizer="sgd" if c["optimizer"] == synth.SGD else "adamw",
                       lr=c["lr"], beta1=c["beta1"], beta2=c["beta2"], eps=c["eps"], weight_decay=c["weight_decay"],
                       step=case.get("step", 1), moments=moments, sr_seed=sr_seed)
    r.update(mask=mask, tau=tau, argmax=am)
    return r


METRICS = []   # observed error figures of every check_step call; conftest.py writes them to gpurun_out/ at session end


def max_abs(x):
    return float(np.max(np.abs(x))) if x.size else 0.0


def check_step(g, o, case, *, fp32=False):
    """Element-by-element comparison with the tolerances of BASELINE.json north_star (bf16 inputs,
    fp32 accumulation: loss rel <= 1e-3, gW / gh / weights max abs err <= 2e-3 * max|ref|) or, for the
    fp32 configuration, R21 (1e-5).  Mask, tau and argmax are bit-exact."""
    c = case["cfg"]
    obs = dict(V=case["V"], d=case["d"], T=case["T"], step=case.get("step", 1))
    METRICS.append(obs)
    np.testing.assert_array_equal(g["mask"], o["mask"])
    np.testing.assert_array_equal(g["tau"], o["tau"])
    np.testing.assert_array_equal(g["argmax"], o["argmax"])
    rel, aabs, tol = (1e-5, 1e-9, 1e-5) if fp32 else (1e-3, 1e-6, 2e-3)
    obs["loss_rel"] = abs(g["loss"] - o["loss"]) / max(abs(o["loss"]), 1e-30)
    assert abs(g["loss"] - o["loss"]) <= rel * abs(o["loss"]) + aabs, (g["loss"], o["loss"])
    klt = rel * np.abs(o["kl_rows"]) + max(aabs, 1e-6 if not fp32 else 1e-7) * 10
    assert np.all(np.abs(g["kl_rows"] - o["kl_rows"]) <= klt), (g["kl_rows"], o["kl_rows"])
    for name in ("gW", "gh", "master", "m", "v"):
        if g.get(name) is None or o.get(name) is None:
            continue
        ref = o[name]
        err = max_abs(g[name].astype(np.float64) - ref)
        assert np.all(np.isfinite(g[name])), name
        obs[name + "_err_over_max"] = err / max(max_abs(ref), 1e-300)
        assert err <= tol * max_abs(ref) + 1e-30, (name, err, max_abs(ref))
    # the update itself (R13): Delta M on elements with a sizeable gradient, and its sign everywhere
    M_old = O.widen(case["master"]) if case["master"] is not None else O.widen(case["W"])
    d_ref = o["master"] - M_old
    d_gpu = g["master"].astype(np.float64) - M_old
    lr = c["lr"]
    if c["optimizer"] == synth.ADAMW:
        big = np.abs(o["gW"]) >= 1e-2 * max_abs(o["gW"])
        if big.any():
            # fp32 master: one ulp of |M| ~ 0.1 is 7.5e-9, comparable to lr = 1e-5 * 0.02
            ulp = np.spacing(np.abs(M_old[big]).astype(np.float32)).astype(np.float64)
            obs["dM_big_err_over_lr"] = float(np.max(np.abs(d_gpu[big] - d_ref[big]) - ulp)) / lr
            assert np.all(np.abs(d_gpu[big] - d_ref[big]) <= 0.02 * lr + ulp)
        moved = np.abs(d_ref) > 4 * np.spacing(np.abs(M_old).astype(np.float32)).astype(np.float64)
        if moved.any():
            bad = np.sign(d_gpu[moved]) != np.sign(d_ref[moved])
            obs["dM_sign_mismatch_frac"] = float(bad.mean())
            obs["dM_all_err_over_lr"] = float(np.max(np.abs(d_gpu - d_ref))) / lr
            assert bad.mean() <= 1e-3, bad.mean()
    else:
        assert max_abs(d_gpu - d_ref) <= tol * lr * max_abs(o["gW"]) + float(np.spacing(np.float32(max_abs(M_old))))
    if case["master"] is not None:
        # working copy: bit-exactly rn_bf16 of the GPU's own master, and within 1 bf16 ulp of the oracle's (R12)
        np.testing.assert_array_equal(g["W_out"], O.f32_to_bf16_bits(g["master"]))
        # R12: where Adam's step is ill-conditioned (|g| ~ eps: the step is not saturated at +-lr, so a 1e-9 change
        # of g moves M by a sizeable part of lr) and |M| is tiny, a master difference far inside the master
        # tolerance spans several bf16 ulps.  So: value difference <= 1 bf16 ulp + the master difference, and
        # the bit patterns differ by more than 1 ulp on at most 1e-4 of the elements.
        wg, wo = O.bf16_bits_to_f64(g["W_out"]), O.bf16_bits_to_f64(o["W_out"])
        mag = np.maximum(np.maximum(np.abs(wg), np.abs(wo)), 2.0 ** -126)
        ulp = 2.0 ** (np.floor(np.log2(mag)) - 7)
        assert np.all(np.abs(wg - wo) <= ulp + np.abs(g["master"].astype(np.float64) - o["master"]))
        diff = np.abs(g["W_out"].astype(np.int32) - o["W_out"].astype(np.int32))
        obs["W_out_gt1ulp_frac"] = float((diff > 1).mean())
        obs["W_out_ne_frac"] = float((diff > 0).mean())
        assert (diff > 1).mean() <= 1e-4
