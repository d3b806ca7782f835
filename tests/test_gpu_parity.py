"""GPU parity: the CUDA path (through the C ABI) against the fp64 oracle, element by element on the
same seeded inputs.  Sizes are chosen so that the oracle finishes in seconds while the kernels
still see several tiles, several CTAs per role and a ragged tail.  Tolerances: BASELINE.json
north_star for bf16 inputs / fp32 accumulation; R21 for the fp32 configuration; the
mask, tau and argmax are bit-exact."""
import numpy as np
import pytest
import torch

from oracle import tts_oracle as O
from paper_2605_09329_b200 import tts
from workloads import synth

from gpu_util import _dev, check_step, run_gpu, run_oracle

pytestmark = pytest.mark.gpu


def test_library_is_loaded_and_arch_ok():
    assert tts.tts_version() >= 100
    ctx = tts.tts_ctx_create(tts.make_config(1024, 64, 8, 8, tts.TTS_F32, tts.TTS_F32, tts.TTS_SGD, 1e-3), 0)
    assert tts.tts_get_step_count(ctx) == 0
    tts.tts_ctx_destroy(ctx)


# ------------------------------------------------------------------ a1: mask, bit-exact
@pytest.mark.parametrize("dtype", [synth.BF16, synth.F32])
@pytest.mark.parametrize("V,seg_len", [(1024, 8), (151936, 16), (4104, 4), (8, 1)])
def test_accept_mask_planted(dtype, V, seg_len):
    t, tok, expect_tau = synth.planted_mask_cases(V, seg_len, seed=11 + V, dtype=dtype)
    T = t.shape[0]
    o_mask, o_tau, o_am = O.accept_mask(t, tok, seg_len)
    np.testing.assert_array_equal(o_tau, expect_tau)       # the recipe's planted values
    cfg = tts.make_config(V, 64, T, seg_len, tts.TTS_BF16, dtype, tts.TTS_SGD, 1e-3)
    ctx = tts.tts_ctx_create(cfg, 0)
    try:
        mask = torch.zeros(T, dtype=torch.uint8, device="cuda")
        tau = torch.zeros(T // seg_len, dtype=torch.int32, device="cuda")
        am = torch.zeros(T, dtype=torch.int32, device="cuda")
        tts.tts_accept_mask(ctx, _dev(t), _dev(tok), T, mask, tau, am, None)
        torch.cuda.synchronize()
        np.testing.assert_array_equal(am.cpu().numpy(), o_am)
        np.testing.assert_array_equal(mask.cpu().numpy(), o_mask)
        np.testing.assert_array_equal(tau.cpu().numpy(), o_tau)
        # partial T (one segment) and NULL argmax output
        tts.tts_accept_mask(ctx, _dev(t), _dev(tok), seg_len, mask, tau, None, None)
        torch.cuda.synchronize()
        np.testing.assert_array_equal(mask.cpu().numpy()[:seg_len], o_mask[:seg_len])
        assert int(tau[0].item()) == int(o_tau[0])
    finally:
        tts.tts_ctx_destroy(ctx)


# ------------------------------------------------------------------ config 1 exactly (fp32, SGD)
def test_config1_tiny_fp32_sgd():
    case = synth.make_case(1)
    g = run_gpu(case)
    o = run_oracle(case)
    check_step(g, o, case, fp32=True)
    assert g["used_tensor"] == 0 and g["step_count"] == 1


def test_config1_planted_variants_fp32():
    for tau_star in (0, 1, 3, 8):
        case = synth.make_case(1)
        t = case["teacher"]
        synth._plant_prefix(t, case["draft_tokens"], tau_star)
        g = run_gpu(case, mask_mode=tts.TTS_ROWS_ACCEPTED_PLUS_ONE)
        o = run_oracle(case, mask_mode=O.ROWS_ACCEPTED_PLUS_ONE)
        assert int(o["tau"][0]) == tau_star
        check_step(g, o, case, fp32=True)


# ------------------------------------------------------------------ bf16 + master, scaled-down configs 2-4
SMALL = [
    # cfg, V, d, n_seq, seg_len, kwargs
    (2, 4096, 256, 1, 16, {}),                       # several vocab tiles
    (3, 4096 + 128 * 3, 384, 1, 16, {}),             # ragged tile count, d not a power of two
    (3, 2048, 128, 1, 8, {}),                        # T = 8 (EAGLE-3 depth), padded to 16 rows
    (4, 2048, 256, 4, 16, {}),                       # batched: 64 rows, loss_scale 1/32
    (2, 1000, 72, 1, 16, {}),                        # shape outside the tensor-core tiles -> CUDA-core kernels
    (3, 2048 + 16 * 5, 1024, 1, 16, {}),             # V % 128 != 0: CUDA-core kernels at d = 1024
    (3, 2048 + 128 * 3, 1024, 1, 16, {}),            # fused stripe kernel: one 1024-column stripe, 152 bands over 148 CTAs
    (3, 1024 + 128, 2048, 1, 8, {}),                 # fused stripe kernel: two stripes, T = 8 padded to 16 rows
    (4, 2048 + 128, 256, 32, 16, {}),                # 512 rows: CTA-pair logits (17 tiles of 128: the last pair tile is half empty), full-TMEM gh
    (4, 1024, 384, 20, 16, {}),                      # 320 rows: pair pieces of 256 + 64 rows
    (4, 1024, 256, 17, 16, {}),                      # 272 rows: second pair piece of 16 rows (8 per CTA)
    (4, 1024, 128, 3, 16, {}),                       # 48 rows: one fp16 dl plane, K padded to 64
    (4, 1024, 128, 2, 16, {}),                       # 32 rows: hi + lo fp16 planes fill the 64-wide K chunk
    (4, 1024, 128, 12, 16, {}),                      # 192 rows: gh formed inside the wide update kernel, K = 192
    (4, 1024 + 128, 256, 16, 16, {}),                # 256 rows: the most the wide kernel's tensor memory holds next to h^T
]


@pytest.mark.parametrize("cfg_id,V,d,n_seq,seg_len,kw", SMALL)
@pytest.mark.parametrize("path", [tts.TTS_PATH_AUTO, tts.TTS_PATH_SIMT])
def test_bf16_adamw_small(cfg_id, V, d, n_seq, seg_len, kw, path):
    case = synth.make_case(cfg_id, V=V, d=d, n_seq=n_seq, seg_len=seg_len)
    g = run_gpu(case, kernel_path=path)
    o = run_oracle(case)
    check_step(g, o, case)
    if path == tts.TTS_PATH_SIMT:
        assert g["used_tensor"] == 0


@pytest.mark.parametrize("path", [tts.TTS_PATH_AUTO, tts.TTS_PATH_SIMT])
def test_bf16_adamw_nonzero_state_step3(path):
    case = synth.make_case(3, V=4096, d=256, nonzero_state=True, step=3)
    g = run_gpu(case, kernel_path=path)
    o = run_oracle(case)
    check_step(g, o, case)
    assert g["step_count"] == 3


@pytest.mark.parametrize("mode_g,mode_o", [(tts.TTS_ROWS_ACCEPTED, O.ROWS_ACCEPTED),
                                           (tts.TTS_ROWS_ACCEPTED_PLUS_ONE, O.ROWS_ACCEPTED_PLUS_ONE)])
@pytest.mark.parametrize("path", [tts.TTS_PATH_AUTO, tts.TTS_PATH_SIMT])
def test_mask_modes(mode_g, mode_o, path):
    case = synth.make_case(4, V=2048, d=128, n_seq=3, seg_len=16)
    g = run_gpu(case, mask_mode=mode_g, kernel_path=path)
    o = run_oracle(case, mask_mode=mode_o)
    np.testing.assert_array_equal(o["tau"], case["tau_star"])
    check_step(g, o, case)


@pytest.mark.parametrize("path", [tts.TTS_PATH_AUTO, tts.TTS_PATH_SIMT])
def test_bf16_sgd_with_master_and_alias(path):
    case = synth.make_case(2, V=2048, d=256)
    case["cfg"]["optimizer"] = synth.SGD
    case["cfg"]["lr"] = 1e-3
    case["m"] = case["v"] = None
    g = run_gpu(case, kernel_path=path, alias_w=True)
    o = run_oracle(case)
    check_step(g, o, case)


@pytest.mark.parametrize("path", [tts.TTS_PATH_AUTO, tts.TTS_PATH_SIMT])
def test_neg_inf_teacher_entries_and_zero_weight_rows(path):
    case = synth.make_case(3, V=2048, d=128)
    t = synth.bf16_bits_to_f32(case["teacher"])
    t[:, 5::7] = -np.inf                       # masked vocabulary entries: p = 0 (0 log 0 := 0)
    case["teacher"] = synth.f32_to_bf16_bits(t)
    case["pos_weight"][3] = 0.0                # omega_r = 0: the row contributes nothing
    g = run_gpu(case, kernel_path=path)
    o = run_oracle(case)
    check_step(g, o, case)


@pytest.mark.parametrize("d", [256, 1024])
def test_gh_and_gw_outputs_optional(d):
    case = synth.make_case(2, V=2048, d=d)
    g = run_gpu(case, want_gW=False, want_gh=False)
    o = run_oracle(case)
    check_step(g, o, case)


@pytest.mark.parametrize("max_ctas", [1, 3, 7, 64])
def test_fused_kernel_with_capped_grid(max_ctas):
    """max_ctas (the SM budget the main stream keeps) changes how stripes and bands are walked,
    not the result.  3 and 7 are not multiples of the stripe count."""
    case = synth.make_case(3, V=1024 + 128, d=2048, nonzero_state=True, step=2)
    g = run_gpu(case, max_ctas=max_ctas)
    o = run_oracle(case)
    check_step(g, o, case)
    assert g["used_tensor"] == 1


@pytest.mark.parametrize("max_ctas", [1, 3, 8])
def test_several_canvases_with_capped_grid(max_ctas):
    """512 rows under an SM budget: 1 CTA takes the one-CTA-per-tile logits kernel, 3 CTAs one CTA pair (+ an idle
    SM), 8 CTAs four pairs; the wide update's stream-K ranges then span many stripes per CTA."""
    case = synth.make_case(4, V=1024 + 128, d=256, n_seq=32, seg_len=16)
    g = run_gpu(case, max_ctas=max_ctas)
    o = run_oracle(case)
    check_step(g, o, case)
    assert g["used_tensor"] == 1


@pytest.mark.parametrize("V,d,n_seq", [(4096, 512, 4), (4096 + 128, 512, 32), (4096, 1024, 1)])
def test_the_walk_does_not_change_the_update(V, d, n_seq):
    """The several-canvas pass walks fixed stripes on its default grid and windowed stream-K ranges under an SM budget;
    the one-canvas pass one stripe per CTA or two segments.  The order in which (stripe, band) units are visited must
    not touch the arithmetic of any element.  An SM budget also re-partitions a2 / a3 (which CTA folds which tile into
    its running tuple), so the row normalisers may move in their last fp32 bit: the results under budgets of 5 and 37
    CTAs agree with the default grid's 2000 times tighter than with the oracle (gh, an order-dependent fp32 RED sum: 4
    times), and the working copies on all but a handful of elements."""
    case = synth.make_case(4 if n_seq > 1 else 3, V=V, d=d, n_seq=n_seq, nonzero_state="mix", step=4)
    ref = run_gpu(case, want_gW=False)
    check_step(ref, run_oracle(case), case)
    for budget in (5, 37):
        g = run_gpu(case, want_gW=False, max_ctas=budget)
        for k, tol in (("master", 1e-6), ("m", 1e-6), ("v", 1e-6), ("gh", 5e-4)):   # gh: fp32 RED, order-dependent
            err = np.abs(g[k].astype(np.float64) - ref[k].astype(np.float64)).max()
            assert err <= tol * np.abs(ref[k]).max(), "%s differs under max_ctas=%d: %g" % (k, budget, err)
        assert (g["W_out"] != ref["W_out"]).mean() <= 1e-4
        assert abs(g["loss"] - ref["loss"]) <= 1e-6 * abs(ref["loss"])


def test_fused_kernel_sgd_alias_d1024():
    case = synth.make_case(2, V=1024, d=1024)
    case["cfg"]["optimizer"] = synth.SGD
    case["cfg"]["lr"] = 1e-3
    case["m"] = case["v"] = None
    g = run_gpu(case, alias_w=True)
    o = run_oracle(case)
    check_step(g, o, case)


def test_teacher_equals_draft_gives_zero_loss_and_no_move():
    """Closed form: t == z  =>  KL = 0 and zero gradient (to fp32 rounding of z)."""
    case = synth.make_case(2, V=2048, d=128)
    case["cfg"]["sigma"] = ("const", 0.0)
    W = synth.bf16_bits_to_f32(case["W"]).astype(np.float64)
    h = synth.bf16_bits_to_f32(case["h"]).astype(np.float64)
    case["teacher"] = (h @ W.T).astype(np.float32)      # fp32 teacher = exact draft logits (to fp32)
    case["cfg"]["logits"] = synth.F32
    g = run_gpu(case)
    assert abs(g["loss"]) < 1e-5
    assert np.abs(g["gW"]).max() < 1e-6 and np.abs(g["gh"]).max() < 1e-6


def test_invalid_arguments_are_rejected():
    cfg = tts.make_config(2048, 128, 16, 16)
    ctx = tts.tts_ctx_create(cfg, 0)
    try:
        x = torch.zeros(16, device="cuda")
        with pytest.raises(tts.TTSError) as e:
            tts.tts_distill_step(ctx, None, x, x, x, x, x, x, x, None, 16, 1.0, x)
        assert e.value.status == tts.TTS_ERR_INVALID_ARG
        with pytest.raises(tts.TTSError):
            tts.tts_distill_step(ctx, x, x, x, x, x, x, x, x, None, 32, 1.0, x)     # T > T_max
        with pytest.raises(tts.TTSError):
            tts.tts_distill_step(ctx, x, x, x, x, None, x, x, x, None, 16, 1.0, x)  # bf16 needs a master
    finally:
        tts.tts_ctx_destroy(ctx)
    bad = tts.make_config(2048, 128, 16, 16)
    bad.T_max = 15
    with pytest.raises(tts.TTSError):
        tts.tts_ctx_create(bad, 0)


def test_round_host_matches_device_calls():
    case = synth.make_case(3, V=4096, d=256)
    o = run_oracle(case)
    from gpu_util import config_for
    ctx = tts.tts_ctx_create(config_for(case), 0)
    try:
        W_in, master = _dev(case["W"]), _dev(case["master"])
        W_out = torch.empty_like(W_in)
        m, v = _dev(case["m"]), _dev(case["v"])
        gh = torch.zeros(case["T"], case["d"], device="cuda")
        teacher = torch.from_numpy(case["teacher"].view(np.int16)).pin_memory()
        h = torch.from_numpy(case["h"].view(np.int16)).pin_memory()
        tok = torch.from_numpy(case["draft_tokens"]).pin_memory()
        pw = torch.from_numpy(case["pos_weight"]).pin_memory()
        loss = torch.zeros(1).pin_memory()
        tau = torch.zeros(1, dtype=torch.int32).pin_memory()
        mask = torch.zeros(case["T"], dtype=torch.uint8).pin_memory()
        tts.tts_round_host(ctx, teacher, h, tok, pw, case["T"], case["loss_scale"], W_in, W_out, master, m, v, gh,
                           loss, tau, mask, None)
        assert abs(float(loss[0]) - o["loss"]) <= 1e-3 * abs(o["loss"]) + 1e-6
        np.testing.assert_array_equal(tau.numpy(), o["tau"])
        np.testing.assert_array_equal(mask.numpy(), o["mask"])
        err = np.abs(master.cpu().numpy().astype(np.float64) - o["master"]).max()
        assert err <= 2e-3 * np.abs(o["master"]).max()
    finally:
        tts.tts_ctx_destroy(ctx)


def test_round_host_refuses_bad_arguments_before_it_enqueues_anything():
    """A NULL / misaligned parameter tensor or a bad T comes back as TTS_ERR_INVALID_ARG (not as a CUDA error out of
    the tensor-map encoder), with no copy or kernel in flight: the state is untouched, and the very next good round on
    the same slot gives the oracle's step."""
    case = synth.make_case(3, V=4096, d=256)
    o = run_oracle(case)
    from gpu_util import config_for
    ctx = tts.tts_ctx_create(config_for(case), 0)
    try:
        W_in, master = _dev(case["W"]), _dev(case["master"])
        W_out = torch.empty_like(W_in)
        m, v = _dev(case["m"]), _dev(case["v"])
        teacher = torch.from_numpy(case["teacher"].view(np.int16)).pin_memory()
        h = torch.from_numpy(case["h"].view(np.int16)).pin_memory()
        tok = torch.from_numpy(case["draft_tokens"]).pin_memory()
        pw = torch.from_numpy(case["pos_weight"]).pin_memory()
        loss = torch.full((1,), -1.0).pin_memory()
        tau = torch.full((1,), -1, dtype=torch.int32).pin_memory()
        T, ls = case["T"], case["loss_scale"]
        before = master.clone()
        bad = [dict(W_in=None), dict(W_out=W_out.view(torch.int16).view(-1)[1:].data_ptr()), dict(master=None),
               dict(m=None), dict(T=T + 1)]
        for b in bad:
            a = dict(W_in=W_in, W_out=W_out, master=master, m=m, T=T)
            a.update(b)
            with pytest.raises(tts.TTSError) as e:
                tts.tts_round_host_begin(ctx, teacher, h, tok, pw, a["T"], ls, a["W_in"], a["W_out"], a["master"],
                                         a["m"], v, None, loss, tau, None, None)
            assert e.value.status == tts.TTS_ERR_INVALID_ARG, b
        torch.cuda.synchronize()
        assert torch.equal(master, before) and float(loss[0]) == -1.0 and int(tau[0]) == -1
        with pytest.raises(tts.TTSError):
            tts.tts_round_host_end(ctx)                      # nothing was begun
        tts.tts_round_host(ctx, teacher, h, tok, pw, T, ls, W_in, W_out, master, m, v, None, loss, tau, None, None)
        assert abs(float(loss[0]) - o["loss"]) <= 1e-3 * abs(o["loss"]) + 1e-6
        np.testing.assert_array_equal(tau.numpy(), o["tau"])
        assert np.abs(master.cpu().numpy().astype(np.float64) - o["master"]).max() <= 2e-3 * np.abs(o["master"]).max()
    finally:
        tts.tts_ctx_destroy(ctx)


# R12 / VERDICT r1: the non-zero optimiser state spans the whole reachable band |m| / sqrt(v) <= 7.27, including the
# most ordinary state of all (a constant gradient for n steps), through every update kernel: the one-canvas stripe
# kernel (T = 16, d % 1024 == 0), the wide kernel at 16 rows (d = 256), with gh formed in the pass (64 and 256 rows)
# and the 512-row set (one fp16 dl plane, separate gh kernel, CTA-pair logits).
@pytest.mark.parametrize("kind,step", [("mix", 5), ("uniform", 3), ("const2", 3), ("const10", 11), ("const1000", 1001)])
@pytest.mark.parametrize("V,d,n_seq", [(4096, 1024, 1), (4096, 256, 1), (2048 + 128, 256, 4), (2048, 256, 16),
                                       (2048 + 384, 256, 32)])
def test_reachable_adam_states_through_every_update_kernel(kind, step, V, d, n_seq):
    case = synth.make_case(3 if n_seq == 1 else 4, V=V, d=d, n_seq=n_seq, nonzero_state=kind, step=step)
    g, o = run_gpu(case), run_oracle(case)
    assert g["used_tensor"] == 1
    check_step(g, o, case)
