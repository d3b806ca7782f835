"""Boundary behaviour of the C-ABI library on the GPU: buffers are written exactly as declared, the
debug-mode precondition checks report into the device status word, the stream-ordered step-count calls, the
no-allocation contract of K > 1 inner steps, and the two flags that change how gh is formed
(TTS_FLAG_SEPARATE_GH: contracted against the W_in buffer; TTS_FLAG_DETERMINISTIC: bit-reproducible)."""
import numpy as np
import pytest
import torch

from oracle import tts_oracle as O
from paper_2605_09329_b200 import tts
from workloads import synth

from gpu_util import _dev, check_step, config_for, max_abs, run_gpu, run_oracle

pytestmark = pytest.mark.gpu


def _buffers(case):
    t = dict(teacher=_dev(case["teacher"]), h=_dev(case["h"]), tok=_dev(case["draft_tokens"]), W_in=_dev(case["W"]),
             master=_dev(case["master"]), m=_dev(case["m"]), v=_dev(case["v"]), pw=_dev(case["pos_weight"]))
    t["W_out"] = torch.empty_like(t["W_in"])
    t["loss"] = torch.zeros(1, device="cuda")
    t["gh"] = torch.zeros(case["T"], case["d"], device="cuda")
    return t


@pytest.mark.parametrize("V,d,T", [(2048 + 128, 1024, 8), (4096, 256, 8), (4096, 256, 24), (1000, 72, 8)])
def test_draft_logits_out_holds_exactly_T_rows(V, d, T):
    """T % 16 != 0 (T = 8 is the EAGLE-3 depth): the tensor-path logits kernels compute ceil16(T) rows
    as MMA padding but must store only T of them into the caller's draft_logits_out [T, V]."""
    case = synth.make_case(3, V=V, d=d, seg_len=8, n_seq=T // 8)
    ctx = tts.tts_ctx_create(config_for(case), 0)
    try:
        t = _buffers(case)
        guard = 4 * V
        buf = torch.full((T * V + guard,), 12345.0, device="cuda")
        z_out = buf[:T * V].view(T, V)
        tts.tts_distill_step_ex(ctx, t["teacher"], t["h"], t["W_in"], t["W_out"], t["master"], t["m"], t["v"], t["pw"],
                                None, T, 1.0, t["loss"], None, t["gh"], None, draft_logits_out=z_out)
        tts.tts_sync_step(ctx)
        assert bool((buf[T * V:] == 12345.0).all()), "rows beyond T were written"
        z_ref = O.widen(case["h"]) @ O.widen(case["W"]).T
        assert max_abs(z_out.cpu().numpy() - z_ref) <= 2e-3 * max_abs(z_ref)
        o = run_oracle(case)
        assert abs(float(t["loss"].item()) - o["loss"]) <= 1e-3 * abs(o["loss"]) + 1e-6
    finally:
        tts.tts_ctx_destroy(ctx)


def test_precondition_checks_report_into_the_status_word():
    case = synth.make_case(3, V=4096, d=1024)
    ctx = tts.tts_ctx_create(config_for(case, flags=tts.TTS_FLAG_CHECK_PRECONDITIONS), 0)
    try:
        T = case["T"]

        def step(t):
            tts.tts_distill_step(ctx, t["teacher"], t["h"], t["W_in"], t["W_out"], t["master"], t["m"], t["v"], t["pw"],
                                 None, T, 1.0, t["loss"], None, t["gh"], None)
            return tts.tts_last_device_status(ctx)

        t = _buffers(case)
        t["teacher"][3, 17] = float("-inf")           # a masked vocabulary entry is legal (R23)
        assert step(t) == 0
        assert tts.tts_last_device_status(ctx) == 0
        t = _buffers(case)
        w = t["W_in"].view(torch.int16)
        w[1234, 77] ^= 1                              # one bf16 ulp off rn_bf16(master)
        assert step(t) == tts.TTS_DEV_W_MISMATCH
        assert tts.tts_last_device_status(ctx) == 0   # read-and-clear
        t = _buffers(case)
        t["teacher"][5, 4000] = float("nan")
        assert step(t) & tts.TTS_DEV_NONFINITE_TEACHER
        t = _buffers(case)
        t["teacher"][0, 0] = float("inf")
        st = step(t)
        assert st & tts.TTS_DEV_NONFINITE_TEACHER and st & tts.TTS_DEV_NONFINITE_LOSS
        t = _buffers(case)
        t["h"][2, 5] = float("inf")
        assert step(t) & tts.TTS_DEV_NONFINITE_H
        # the same checks as one explicit call, no step
        t = _buffers(case)
        t["W_in"].view(torch.int16)[0, 0] ^= 1
        tts.tts_check_preconditions(ctx, t["teacher"], t["h"], t["W_in"], t["master"], T)
        assert tts.tts_last_device_status(ctx) == tts.TTS_DEV_W_MISMATCH
    finally:
        tts.tts_ctx_destroy(ctx)


def test_status_word_sees_work_queued_on_a_non_blocking_stream():
    """A torch.cuda.Stream is cudaStreamNonBlocking: the legacy default stream does not order after it.  The status
    read must still wait for a check (or a stochastic accept) that sits on such a stream behind ~0.1 s of other work,
    through both forms of the call."""
    case = synth.make_case(3, V=4096, d=1024)
    ctx = tts.tts_ctx_create(config_for(case), 0)
    try:
        T, V = case["T"], case["V"]
        t = _buffers(case)
        t["h"][2, 5] = float("inf")
        side = torch.cuda.Stream()
        torch.cuda.synchronize()

        def delayed_check():
            with torch.cuda.stream(side):
                torch.cuda._sleep(200_000_000)    # the check below is still queued when the status is asked for
            tts.tts_check_preconditions(ctx, t["teacher"], t["h"], t["W_in"], t["master"], T, side)

        delayed_check()
        assert tts.tts_last_device_status(ctx) == tts.TTS_DEV_NONFINITE_H
        assert tts.tts_last_device_status(ctx) == 0            # taken: read-and-clear
        delayed_check()
        assert tts.tts_device_status_on(ctx, side) == tts.TTS_DEV_NONFINITE_H
        assert tts.tts_device_status_on(ctx, side) == 0
        # TTS_DEV_BAD_TOKEN from the stochastic accept, same situation
        tok = t["tok"].clone()
        tok[1] = V + 5
        z = torch.randn(T, V, device="cuda")
        u, u2 = torch.rand(T, device="cuda"), torch.rand(T // case["seg_len"], device="cuda")
        mask = torch.zeros(T, dtype=torch.uint8, device="cuda")
        tau = torch.zeros(T // case["seg_len"], dtype=torch.int32, device="cuda")
        nxt = torch.zeros(T // case["seg_len"], dtype=torch.int32, device="cuda")
        torch.cuda.synchronize()
        with torch.cuda.stream(side):
            torch.cuda._sleep(200_000_000)
        tts.tts_accept_stochastic(ctx, t["teacher"], z, tok, u, u2, T, mask, tau, nxt, None, side)
        assert tts.tts_last_device_status(ctx) == tts.TTS_DEV_BAD_TOKEN
        assert tts.tts_last_device_status(ctx) == 0
    finally:
        tts.tts_ctx_destroy(ctx)


def test_host_round_staging_is_allocated_by_the_first_host_round_only():
    """tts_ctx_create no longer reserves the two staging slots of tts_round_host* (2 x T_max x V logits): device-buffer
    steps never pay for them; the first host round allocates them once."""
    case = synth.make_case(4, V=16384, d=256, n_seq=32)
    T, V = case["T"], case["V"]
    slots = 2 * T * V * 2
    ctx = tts.tts_ctx_create(config_for(case), 0)
    try:
        t = _buffers(case)
        mask = torch.zeros(T, dtype=torch.uint8, device="cuda")
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        tts.tts_distill_step(ctx, t["teacher"], t["h"], t["W_in"], t["W_out"], t["master"], t["m"], t["v"], t["pw"],
                             mask, T, 1.0, t["loss"], None, t["gh"], None)
        tts.tts_sync_step(ctx)
        assert torch.cuda.mem_get_info()[0] == free0                     # a step allocates nothing
        host = [torch.from_numpy(case[k].view(np.int16)).pin_memory() for k in ("teacher", "h")]
        tok, pw = torch.from_numpy(case["draft_tokens"]).pin_memory(), torch.from_numpy(case["pos_weight"]).pin_memory()
        loss, tau = torch.zeros(1).pin_memory(), torch.zeros(T // case["seg_len"], dtype=torch.int32).pin_memory()

        def host_round(a, b):
            tts.tts_round_host(ctx, host[0], host[1], tok, pw, T, 1.0, a, b, t["master"], t["m"], t["v"], None, loss,
                               tau, None, None)

        host_round(t["W_out"], t["W_in"])
        free1 = torch.cuda.mem_get_info()[0]
        assert free0 - free1 >= slots                                    # the first host round brought the slots
        host_round(t["W_in"], t["W_out"])
        assert torch.cuda.mem_get_info()[0] == free1                     # and only the first
    finally:
        tts.tts_ctx_destroy(ctx)


def test_checks_are_off_by_default_and_loss_bit_is_always_on():
    case = synth.make_case(3, V=2048, d=256)
    ctx = tts.tts_ctx_create(config_for(case), 0)
    try:
        t = _buffers(case)
        t["W_in"].view(torch.int16)[0, 0] ^= 1
        tts.tts_distill_step(ctx, t["teacher"], t["h"], t["W_in"], t["W_out"], t["master"], t["m"], t["v"], t["pw"],
                             None, case["T"], 1.0, t["loss"], None, t["gh"], None)
        assert tts.tts_last_device_status(ctx) == 0
        t = _buffers(case)
        t["teacher"][0, 0] = float("nan")
        tts.tts_distill_step(ctx, t["teacher"], t["h"], t["W_in"], t["W_out"], t["master"], t["m"], t["v"], t["pw"],
                             None, case["T"], 1.0, t["loss"], None, t["gh"], None)
        assert tts.tts_last_device_status(ctx) == tts.TTS_DEV_NONFINITE_LOSS
    finally:
        tts.tts_ctx_destroy(ctx)


def test_stream_ordered_step_count():
    case = synth.make_case(3, V=2048, d=256)
    ctx = tts.tts_ctx_create(config_for(case), 0)
    try:
        side = torch.cuda.Stream()
        t = _buffers(case)
        assert tts.tts_get_step_count_on(ctx, side) == 0
        tts.tts_set_step_count_async(ctx, 41, side)
        tts.tts_distill_step(ctx, t["teacher"], t["h"], t["W_in"], t["W_out"], t["master"], t["m"], t["v"], t["pw"],
                             None, case["T"], 1.0, t["loss"], None, t["gh"], None, side)
        assert tts.tts_get_step_count_on(ctx, side) == 42
        assert tts.tts_get_step_count(ctx) == 42
        # the step really ran with n = 42: compare m against the oracle at that count (m does not depend on n, the
        # master does)
        case2 = dict(case, step=42)
        o = run_oracle(case2)
        err = max_abs(t["master"].cpu().numpy().astype(np.float64) - o["master"])
        assert err <= 2e-3 * max_abs(o["master"])
        d_ref = o["master"] - O.widen(case["master"])
        d_gpu = t["master"].cpu().numpy().astype(np.float64) - O.widen(case["master"])
        big = np.abs(o["gW"]) >= 1e-2 * max_abs(o["gW"])
        assert np.all(np.abs(d_gpu[big] - d_ref[big]) <= 0.02 * case["cfg"]["lr"] + 1e-8)
    finally:
        tts.tts_ctx_destroy(ctx)


def test_inner_steps_never_allocate():
    case = synth.make_case(3, V=2048, d=256)
    t = _buffers(case)
    losses = torch.zeros(3, device="cuda")
    ctx = tts.tts_ctx_create(config_for(case), 0)             # max_inner_steps = 0: no z_ref scratch
    try:
        with pytest.raises(tts.TTSError) as e:
            tts.tts_distill_inner_steps(ctx, t["teacher"], t["h"], t["W_in"], t["W_out"], t["master"], t["m"], t["v"],
                                        t["pw"], None, case["T"], 1.0, 3, 0.5, None, losses)
        assert e.value.status == tts.TTS_ERR_INVALID_ARG
        # with the drafter's own logits as z_ref no scratch is needed
        z = torch.from_numpy((O.widen(case["h"]) @ O.widen(case["W"]).T).astype(np.float32)).cuda()
        tts.tts_distill_inner_steps(ctx, t["teacher"], t["h"], t["W_in"], t["W_out"], t["master"], t["m"], t["v"],
                                    t["pw"], None, case["T"], 1.0, 3, 0.5, z, losses)
        tts.tts_sync_step(ctx)
        assert bool(torch.isfinite(losses).all()) and float(losses[0]) > 0
    finally:
        tts.tts_ctx_destroy(ctx)
    ctx = tts.tts_ctx_create(config_for(case, max_inner_steps=3), 0)
    try:
        t = _buffers(case)
        free0, _ = torch.cuda.mem_get_info()
        tts.tts_distill_inner_steps(ctx, t["teacher"], t["h"], t["W_in"], t["W_out"], t["master"], t["m"], t["v"],
                                    t["pw"], None, case["T"], 1.0, 3, 0.5, None, losses)
        tts.tts_sync_step(ctx)
        free1, _ = torch.cuda.mem_get_info()
        assert free1 == free0, "a step call allocated device memory"
    finally:
        tts.tts_ctx_destroy(ctx)


@pytest.mark.parametrize("V,d,n_seq", [(4096, 1024, 1), (4096 + 128, 256, 4), (2048, 512, 24)])
@pytest.mark.parametrize("flag", [tts.TTS_FLAG_SEPARATE_GH, tts.TTS_FLAG_DETERMINISTIC])
def test_gh_from_its_own_kernel_matches_oracle(V, d, n_seq, flag):
    case = synth.make_case(4 if n_seq > 1 else 3, V=V, d=d, n_seq=n_seq)
    g, o = run_gpu(case, flags=flag), run_oracle(case)
    check_step(g, o, case)


def test_separate_gh_reads_the_W_in_buffer():
    """With TTS_FLAG_SEPARATE_GH a W_in that is NOT rn_bf16(master) still gives gh = dl . W_in (the default path would
    contract against rn_bf16(master) instead: precondition 1)."""
    case = synth.make_case(3, V=4096, d=1024)
    rng = np.random.Generator(np.random.PCG64(3))
    case["master"] = (case["master"] * (1.0 + 0.05 * rng.standard_normal(case["master"].shape))).astype(np.float32)
    o = run_oracle(case)                       # the oracle's z and gh use W_in; its update starts from the master
    g = run_gpu(case, flags=tts.TTS_FLAG_SEPARATE_GH)
    assert max_abs(g["gh"] - o["gh"]) <= 2e-3 * max_abs(o["gh"])
    assert abs(g["loss"] - o["loss"]) <= 1e-3 * abs(o["loss"]) + 1e-6
    g0 = run_gpu(case)                         # default: gh from rn_bf16(master), visibly different here
    assert max_abs(g0["gh"] - o["gh"]) > 2e-3 * max_abs(o["gh"])


@pytest.mark.parametrize("V,d,n_seq", [(19072, 256, 32), (4096 + 384, 512, 32), (4096, 1024, 1), (8192, 256, 8)])
def test_deterministic_mode_is_bit_reproducible(V, d, n_seq):
    """Two runs of the same step give bit-identical loss, gh, master, m, v and W_out, including at 512 rows with a
    vocabulary whose pair-tile count does not divide the number of CTA pairs (leftover tiles cut along K), which is
    where the draft logits used to collect ~37 unordered fp32 addends per entry."""
    case = synth.make_case(4 if n_seq > 1 else 3, V=V, d=d, n_seq=n_seq)
    a = run_gpu(case, flags=tts.TTS_FLAG_DETERMINISTIC, want_gW=False)
    for _ in range(2):
        b = run_gpu(case, flags=tts.TTS_FLAG_DETERMINISTIC, want_gW=False)
        assert a["loss"] == b["loss"]
        for k in ("gh", "master", "m", "v", "W_out", "kl_rows"):
            np.testing.assert_array_equal(a[k], b[k], err_msg=k)


@pytest.mark.parametrize("V,d,n_seq", [(19072, 256, 32), (4096 + 384, 512, 32)])
def test_default_mode_weights_are_bit_reproducible(V, d, n_seq):
    """Without the flag only gh (fp32 RED from many CTAs) may differ between runs; z, the loss and every weight-state
    tensor are order-free."""
    case = synth.make_case(4, V=V, d=d, n_seq=n_seq)
    a = run_gpu(case, want_gW=False)
    b = run_gpu(case, want_gW=False)
    assert a["loss"] == b["loss"]
    for k in ("master", "m", "v", "W_out", "kl_rows"):
        np.testing.assert_array_equal(a[k], b[k], err_msg=k)


def test_a_stalled_pipeline_traps_instead_of_hanging():
    """A protocol slip inside a tensor-path kernel (a wait nobody satisfies) ends in TTS_ERR_CUDA after the watchdog's
    limit, not in a hung GPU.  The trap kills the CUDA context, so the probe runs in a process of its own, with the
    limit lowered through TTS_WATCHDOG_CYCLES to 2^31 cycles (~1.1 s) so that the GPU is held only that long; a value
    that is not a cycle count is refused by tts_ctx_create."""
    import os
    import subprocess
    import sys
    import time
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    code = ("import sys; sys.path.insert(0, %r)\n"
            "import torch\n"
            "from paper_2605_09329_b200 import tts\n"
            "ctx = tts.tts_ctx_create(tts.make_config(2048, 128, 16, 16), 0)\n"
            "torch.cuda.synchronize(); import time; t0 = time.time()\n"
            "st = tts.tts_debug_trip_watchdog(ctx, torch.cuda.Stream())\n"
            "print('STATUS', st, tts.tts_last_cuda_error(ctx), time.time() - t0)\n" % root)
    env = dict(os.environ, TTS_WATCHDOG_CYCLES=str(1 << 31))
    r = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True, timeout=120, env=env)
    line = [l for l in r.stdout.splitlines() if l.startswith("STATUS")]
    assert line, (r.stdout, r.stderr[-500:])
    _, st, cuda_err, dt = line[0].split()
    assert int(st) == tts.TTS_ERR_CUDA and int(cuda_err) != 0
    assert 0.5 < float(dt) < 5.0, dt          # 2^31 cycles at 1.0 - 2.0 GHz
    os.environ["TTS_WATCHDOG_CYCLES"] = "soon"
    try:
        with pytest.raises(tts.TTSError) as e:
            tts.tts_ctx_create(tts.make_config(2048, 128, 16, 16), 0)
        assert e.value.status == tts.TTS_ERR_INVALID_ARG
    finally:
        del os.environ["TTS_WATCHDOG_CYCLES"]
    # this process's context is untouched: a step still runs
    case = synth.make_case(3, V=2048, d=256)
    g, o = run_gpu(case), run_oracle(case)
    check_step(g, o, case)


@pytest.mark.parametrize("V,d,n_seq", [(4096, 1024, 1), (2048 + 128, 256, 32)])
def test_pipelined_host_rounds_equal_serial_host_rounds(V, d, n_seq):
    """tts_round_host_begin / _end with two rounds in flight (the next round's teacher logits travel under this round's
    step) give the rounds of tts_round_host bit for bit: per-round loss, tau and mask, and the final
    master / m / v / working copy.  Also: a third pending round and a plain tts_round_host next to pending rounds are
    refused."""
    n_rounds = 5
    cases = [synth.make_case(4 if n_seq > 1 else 3, V=V, d=d, n_seq=n_seq, seed=900 + r) for r in range(n_rounds)]
    c0 = cases[0]
    T, C = c0["T"], c0["seg_len"]
    host = []
    for c in cases:
        host.append(dict(teacher=torch.from_numpy(c["teacher"].view(np.int16)).pin_memory(),
                         h=torch.from_numpy(c["h"].view(np.int16)).pin_memory(),
                         tok=torch.from_numpy(c["draft_tokens"]).pin_memory(),
                         pw=torch.from_numpy(c["pos_weight"]).pin_memory()))

    def run(pipelined):
        ctx = tts.tts_ctx_create(config_for(c0), 0)
        try:
            W = [_dev(c0["W"]), torch.empty_like(_dev(c0["W"]))]
            master, m, v = _dev(c0["master"]), _dev(c0["m"]), _dev(c0["v"])
            out = [dict(loss=torch.zeros(1).pin_memory(), tau=torch.zeros(T // C, dtype=torch.int32).pin_memory(),
                        mask=torch.zeros(T, dtype=torch.uint8).pin_memory()) for _ in range(n_rounds)]
            side = torch.cuda.Stream()

            def args(r):
                hb, ob = host[r], out[r]
                return (ctx, hb["teacher"], hb["h"], hb["tok"], hb["pw"], T, c0["loss_scale"], W[r & 1], W[1 - (r & 1)],
                        master, m, v, None, ob["loss"], ob["tau"], ob["mask"], side)

            if not pipelined:
                for r in range(n_rounds):
                    tts.tts_round_host(*args(r))
            else:
                tts.tts_round_host_begin(*args(0))
                for r in range(1, n_rounds):
                    tts.tts_round_host_begin(*args(r))
                    if r == 1:
                        with pytest.raises(tts.TTSError):          # both slots are in flight
                            tts.tts_round_host_begin(*args(2))
                        with pytest.raises(tts.TTSError):          # the synchronous form next to pending rounds
                            tts.tts_round_host(*args(2))
                    tts.tts_round_host_end(ctx)
                tts.tts_round_host_end(ctx)
                with pytest.raises(tts.TTSError):                  # nothing pending
                    tts.tts_round_host_end(ctx)
            torch.cuda.synchronize()
            res = dict(loss=[float(o["loss"][0]) for o in out], tau=[o["tau"].numpy().copy() for o in out],
                       mask=[o["mask"].numpy().copy() for o in out], master=master.cpu().numpy(),
                       m=m.cpu().numpy(), v=v.cpu().numpy(), W=W[n_rounds & 1].cpu().view(torch.int16).numpy())
            return res
        finally:
            tts.tts_ctx_destroy(ctx)

    a, b = run(False), run(True)
    assert a["loss"] == b["loss"] and all(np.isfinite(a["loss"])) and len(set(a["loss"])) == n_rounds
    for r in range(n_rounds):
        np.testing.assert_array_equal(a["tau"][r], b["tau"][r])
        np.testing.assert_array_equal(a["mask"][r], b["mask"][r])
    for k in ("master", "m", "v", "W"):
        np.testing.assert_array_equal(a[k], b[k])
    # and the first round is the oracle's
    o = run_oracle(cases[0])
    assert abs(a["loss"][0] - o["loss"]) <= 1e-3 * abs(o["loss"]) + 1e-6
    np.testing.assert_array_equal(a["tau"][0], o["tau"])
