"""tts_accept_mask_static: the accepted-prefix mask for callers that cannot allocate GPU memory.

Why the entry point exists: tts_accept_mask needs a ctx, and tts_ctx_create cudaMallocs the ctx's scratch.  A serving
process whose own pool already owns the whole GPU, code that must not call the CUDA allocator because it synchronises
the device (and with it the decode stream), or an embedder that sends every GPU byte through its own allocator cannot
do that.  The static call keeps its scratch in a fixed array inside the library image (TTS_STATIC_SCRATCH_BYTES per
GPU, T <= TTS_STATIC_T_MAX) and allocates nothing.

What is checked: its outputs are the ctx path's outputs bit for bit (mask, tau, argmax are integer work: the
tolerance of every a1 test is "equal"), on two calls in a row whose shapes differ -- the second call finds the first
call's candidates in the shared array and must not read them.  The file sorts last on purpose: `pytest -x` stops at
the first failure, and a problem here should not hide the parity tests.  It has to pass alone in a fresh process
(where its first call is the first use of the library on the GPU) and after every other test."""
import numpy as np
import pytest
import torch

from paper_2605_09329_b200 import tts
from workloads import synth

from gpu_util import _dev

pytestmark = pytest.mark.gpu


def _ctx_path(t, tok, V, seg_len, dtype):
    """The existing path: a ctx (which allocates) + tts_accept_mask."""
    T = t.shape[0]
    ctx = tts.tts_ctx_create(tts.make_config(V, 64, T, seg_len, tts.TTS_BF16, dtype, tts.TTS_SGD, 1e-3), 0)
    try:
        mask = torch.zeros(T, dtype=torch.uint8, device="cuda")
        tau = torch.zeros(T // seg_len, dtype=torch.int32, device="cuda")
        am = torch.zeros(T, dtype=torch.int32, device="cuda")
        tts.tts_accept_mask(ctx, t, tok, T, mask, tau, am, None)
        torch.cuda.synchronize()
        return mask.cpu().numpy(), tau.cpu().numpy(), am.cpu().numpy()
    finally:
        tts.tts_ctx_destroy(ctx)


def _static_path(t, tok, V, seg_len, dtype, outs, check_no_alloc=False):
    T = t.shape[0]
    mask, tau, am = outs
    mask.fill_(7), tau.fill_(-7), am.fill_(-7)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    tts.tts_accept_mask_static(t, dtype, V, seg_len, tok, T, mask, tau, am, None)
    torch.cuda.synchronize()
    if check_no_alloc:   # not the first call on this device: the amount of free GPU memory does not move
        assert torch.cuda.mem_get_info()[0] == free0
    return mask[:T].cpu().numpy(), tau[:T // seg_len].cpu().numpy(), am[:T].cpu().numpy()


def test_static_mask_equals_ctx_mask_on_two_calls_in_a_row():
    torch.cuda.set_device(0)
    # call 1: the Qwen3 vocabulary in bf16, 16 rows per sequence (many slices per row);
    # call 2: a small fp32 vocabulary with a ragged last slice and more rows (fewer slices per row)
    shapes = [(151936, 16, synth.BF16, 11), (4104, 4, synth.F32, 12)]
    cases = []
    for V, seg_len, dtype, seed in shapes:
        t, tok, _ = synth.planted_mask_cases(V, seg_len, seed=seed, dtype=dtype)
        assert t.shape[0] <= tts.TTS_STATIC_T_MAX
        cases.append((_dev(t), _dev(tok), V, seg_len, dtype))
    # outputs are the caller's: allocated once, before the calls
    outs = (torch.zeros(tts.TTS_STATIC_T_MAX, dtype=torch.uint8, device="cuda"),
            torch.zeros(tts.TTS_STATIC_T_MAX, dtype=torch.int32, device="cuda"),
            torch.zeros(tts.TTS_STATIC_T_MAX, dtype=torch.int32, device="cuda"))
    # the static calls come first (back to back, no ctx exists yet), the ctx path afterwards
    got = [_static_path(*c, outs, check_no_alloc=i > 0) for i, c in enumerate(cases)]
    # and once more in the opposite order: each shape now follows the other one's leftovers
    got_again = [_static_path(*c, outs, check_no_alloc=True) for c in reversed(cases)][::-1]
    for c, g, g2 in zip(cases, got, got_again):
        want = _ctx_path(*c)
        for name, w, a, b in zip(("mask", "tau", "argmax"), want, g, g2):
            np.testing.assert_array_equal(a, w, err_msg=name)
            np.testing.assert_array_equal(b, w, err_msg=name + " (second round)")
        assert want[1].max() > 0 and want[0].min() == 0   # the case has accepted and rejected rows


def test_static_mask_rejects_what_does_not_fit():
    torch.cuda.set_device(0)
    V, seg = 1024, 8
    T = tts.TTS_STATIC_T_MAX + seg
    t = torch.zeros(T, V, dtype=torch.float32, device="cuda")
    tok = torch.zeros(T, dtype=torch.int32, device="cuda")
    mask = torch.full((T,), 7, dtype=torch.uint8, device="cuda")
    tau = torch.zeros(T // seg, dtype=torch.int32, device="cuda")
    with pytest.raises(tts.TTSError) as e:
        tts.tts_accept_mask_static(t, tts.TTS_F32, V, seg, tok, T, mask, tau)
    assert e.value.status == tts.TTS_ERR_INVALID_ARG
    torch.cuda.synchronize()
    assert int(mask.min().item()) == 7        # nothing was enqueued
    with pytest.raises(tts.TTSError) as e:    # rows that do not start 16-byte aligned
        tts.tts_accept_mask_static(t, tts.TTS_F32, 1022, seg, tok, seg, mask, tau)
    assert e.value.status == tts.TTS_ERR_UNSUPPORTED
    # the largest size that fits still works: all-zero logits -> argmax 0 == token 0 everywhere
    tts.tts_accept_mask_static(t, tts.TTS_F32, V, seg, tok, tts.TTS_STATIC_T_MAX, mask, tau)
    torch.cuda.synchronize()
    assert int(mask[:tts.TTS_STATIC_T_MAX].min().item()) == 1 and int(tau[:tts.TTS_STATIC_T_MAX // seg].min().item()) == seg
