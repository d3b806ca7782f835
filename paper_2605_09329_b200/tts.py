"""Thin ctypes binding over libtts_b200.so (include/tts.h).  Argument marshalling only: every
function has the name and argument order of its C counterpart, tensors are passed as their
device (or, where the header says "host", host) pointers, and every step of the path runs in
the library's CUDA kernels.  There is no fallback: if the library is missing or cannot be
loaded, ``lib()`` raises.
"""
from __future__ import annotations

import ctypes as C
import os

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libtts_b200.so")

# enums of include/tts.h
TTS_OK, TTS_ERR_INVALID_ARG, TTS_ERR_UNSUPPORTED, TTS_ERR_CUDA, TTS_ERR_ARCH = 0, 1, 2, 3, 4
TTS_F32, TTS_BF16 = 0, 1
TTS_SGD, TTS_ADAMW = 0, 1
TTS_ROWS_ALL, TTS_ROWS_ACCEPTED, TTS_ROWS_ACCEPTED_PLUS_ONE = 0, 1, 2
TTS_PATH_AUTO, TTS_PATH_SIMT = 0, 1
TTS_MOMENT_F32, TTS_MOMENT_BF16 = 0, 1
TTS_FLAG_CHECK_PRECONDITIONS, TTS_FLAG_DETERMINISTIC, TTS_FLAG_SEPARATE_GH = 1, 2, 4
TTS_DEV_W_MISMATCH, TTS_DEV_NONFINITE_TEACHER, TTS_DEV_NONFINITE_H, TTS_DEV_BAD_TOKEN, TTS_DEV_NONFINITE_LOSS = 1, 2, 4, 8, 16
TTS_NUM_PHASES = 5
TTS_SHARD_STAT_FIELDS = 8
TTS_STATIC_T_MAX, TTS_STATIC_SCRATCH_BYTES = 512, 264192
PHASE_NAMES = ("a2_logits", "a3_row_stats", "a4_dlogits", "a5_gh", "a6a7_gW_update")


class tts_step_extras(C.Structure):
    _fields_ = [("draft_logits", C.c_void_p), ("draft_logits_out", C.c_void_p), ("ref_logits", C.c_void_p),
                ("lambda_", C.c_float)]


class tts_config(C.Structure):
    _fields_ = [("V", C.c_int32), ("d", C.c_int32), ("T_max", C.c_int32), ("seg_len", C.c_int32),
                ("param_dtype", C.c_int32), ("logits_dtype", C.c_int32), ("optimizer", C.c_int32),
                ("lr", C.c_float), ("beta1", C.c_float), ("beta2", C.c_float), ("eps", C.c_float),
                ("weight_decay", C.c_float), ("mask_mode", C.c_int32), ("max_ctas", C.c_int32),
                ("kernel_path", C.c_int32), ("moment_dtype", C.c_int32), ("max_inner_steps", C.c_int32),
                ("flags", C.c_int32), ("sr_seed", C.c_int32)]


EXPORTS = {
    # name: (restype, argtypes)
    "tts_status_string": (C.c_char_p, [C.c_int32]),
    "tts_version": (C.c_int32, []),
    "tts_ctx_create": (C.c_int32, [C.POINTER(tts_config), C.c_int32, C.POINTER(C.c_void_p)]),
    "tts_ctx_destroy": (C.c_int32, [C.c_void_p]),
    "tts_set_lr": (C.c_int32, [C.c_void_p, C.c_float]),
    "tts_set_step_count": (C.c_int32, [C.c_void_p, C.c_int64]),
    "tts_get_step_count": (C.c_int64, [C.c_void_p]),
    "tts_set_step_count_async": (C.c_int32, [C.c_void_p, C.c_int64, C.c_void_p]),
    "tts_get_step_count_on": (C.c_int64, [C.c_void_p, C.c_void_p]),
    "tts_last_device_status": (C.c_int32, [C.c_void_p]),
    "tts_device_status_on": (C.c_int32, [C.c_void_p, C.c_void_p]),
    "tts_check_preconditions": (C.c_int32, [C.c_void_p] * 5 + [C.c_int32, C.c_void_p]),
    "tts_debug_trip_watchdog": (C.c_int32, [C.c_void_p, C.c_void_p]),
    "tts_last_cuda_error": (C.c_int32, [C.c_void_p]),
    "tts_last_step_used_tensor_path": (C.c_int32, [C.c_void_p]),
    "tts_last_launch_count": (C.c_int32, [C.c_void_p]),
    "tts_accept_mask": (C.c_int32, [C.c_void_p] * 3 + [C.c_int32] + [C.c_void_p] * 4),
    "tts_accept_mask_static": (C.c_int32, [C.c_void_p] + [C.c_int32] * 3 + [C.c_void_p, C.c_int32] + [C.c_void_p] * 4),
    "tts_static_last_cuda_error": (C.c_int32, []),
    "tts_accept_stochastic": (C.c_int32, [C.c_void_p] * 6 + [C.c_int32] + [C.c_void_p] * 5),
    "tts_distill_step": (C.c_int32, [C.c_void_p] * 10 + [C.c_int32, C.c_float] + [C.c_void_p] * 5),
    "tts_distill_step_ex": (C.c_int32, [C.c_void_p] * 10 + [C.c_int32, C.c_float] + [C.c_void_p] * 6),
    "tts_distill_inner_steps": (C.c_int32, [C.c_void_p] * 10 + [C.c_int32, C.c_float, C.c_int32, C.c_float] +
                                [C.c_void_p] * 5),
    "tts_profile_enable": (C.c_int32, [C.c_void_p, C.c_int32]),
    "tts_profile_read": (C.c_int32, [C.c_void_p, C.POINTER(C.c_float), C.POINTER(C.c_int32)]),
    "tts_wait_step": (C.c_int32, [C.c_void_p, C.c_void_p]),
    "tts_sync_step": (C.c_int32, [C.c_void_p]),
    "tts_record_done": (C.c_int32, [C.c_void_p, C.c_void_p]),
    "tts_round_host": (C.c_int32, [C.c_void_p] * 5 + [C.c_int32, C.c_float] + [C.c_void_p] * 10),
    "tts_round_host_begin": (C.c_int32, [C.c_void_p] * 5 + [C.c_int32, C.c_float] + [C.c_void_p] * 10),
    "tts_round_host_end": (C.c_int32, [C.c_void_p]),
    "tts_shard_begin_step": (C.c_int32, [C.c_void_p] * 4 + [C.c_int32] + [C.c_void_p] * 3),
    "tts_shard_finish_step": (C.c_int32, [C.c_void_p] * 2 + [C.c_int32] + [C.c_void_p] * 9 + [C.c_int32, C.c_float] +
                              [C.c_void_p] * 6),
    "tts_shard_argmax": (C.c_int32, [C.c_void_p] * 2 + [C.c_int32, C.c_int32] + [C.c_void_p] * 3),
    "tts_shard_accept_mask": (C.c_int32, [C.c_void_p] * 3 + [C.c_int32, C.c_void_p, C.c_int32] + [C.c_void_p] * 4),
}

_lib = None


def lib() -> C.CDLL:
    """Loads the CUDA library; raises (never falls back) when it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError("%s not found: build it with `python -m paper_2605_09329_b200.build` "
                               "(there is no CPU fallback)" % LIB_PATH)
        l = C.CDLL(LIB_PATH)
        for name, (res, args) in EXPORTS.items():
            f = getattr(l, name)
            f.restype, f.argtypes = res, args
        _lib = l
    return _lib


class TTSError(RuntimeError):
    def __init__(self, status, where, cuda_error=0):
        self.status, self.cuda_error = status, cuda_error
        name = lib().tts_status_string(status).decode()
        super().__init__("%s failed: %s%s" % (where, name, " (cudaError %d)" % cuda_error if cuda_error else ""))


def _ptr(x):
    """torch tensor / numpy array / int / None -> address."""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    if hasattr(x, "data_ptr"):
        return x.data_ptr()
    if hasattr(x, "ctypes"):
        return x.ctypes.data
    raise TypeError("cannot take the address of %r" % type(x))


_ctx_device = {}   # ctx address -> CUDA ordinal (a process may hold ctxs on several GPUs)


def _stream(s, ctx=None):
    """None -> the current stream OF THE CTX'S DEVICE (not of whatever device is current)."""
    if s is None:
        import torch
        dev = _ctx_device.get(getattr(ctx, "value", None))
        return torch.cuda.current_stream(dev).cuda_stream
    if isinstance(s, int):
        return s
    return s.cuda_stream


def _check(ctx, st, where):
    if st != TTS_OK:
        raise TTSError(st, where, lib().tts_last_cuda_error(ctx) if ctx else 0)


def tts_status_string(status: int) -> str:
    return lib().tts_status_string(status).decode()


def tts_version() -> int:
    return lib().tts_version()


def tts_ctx_create(cfg: tts_config, device: int = 0):
    out = C.c_void_p()
    st = lib().tts_ctx_create(C.byref(cfg), device, C.byref(out))
    _check(None, st, "tts_ctx_create")
    _ctx_device[out.value] = device
    return out


def tts_ctx_destroy(ctx):
    _ctx_device.pop(getattr(ctx, "value", None), None)
    _check(None, lib().tts_ctx_destroy(ctx), "tts_ctx_destroy")


def tts_set_lr(ctx, lr: float):
    _check(ctx, lib().tts_set_lr(ctx, lr), "tts_set_lr")


def tts_set_step_count(ctx, n: int):
    _check(ctx, lib().tts_set_step_count(ctx, n), "tts_set_step_count")


def tts_get_step_count(ctx) -> int:
    return lib().tts_get_step_count(ctx)


def tts_set_step_count_async(ctx, n: int, stream=None):
    _check(ctx, lib().tts_set_step_count_async(ctx, n, _stream(stream, ctx)), "tts_set_step_count_async")


def tts_get_step_count_on(ctx, stream=None) -> int:
    return lib().tts_get_step_count_on(ctx, _stream(stream, ctx))


def tts_last_device_status(ctx) -> int:
    return lib().tts_last_device_status(ctx)


def tts_device_status_on(ctx, stream=None) -> int:
    return lib().tts_device_status_on(ctx, _stream(stream, ctx))


def tts_check_preconditions(ctx, teacher_logits, h, W_in, W_master, T, stream=None):
    st = lib().tts_check_preconditions(ctx, _ptr(teacher_logits), _ptr(h), _ptr(W_in), _ptr(W_master), T,
                                       _stream(stream, ctx))
    _check(ctx, st, "tts_check_preconditions")


def tts_debug_trip_watchdog(ctx, stream=None) -> int:
    """Returns the status (TTS_ERR_CUDA expected); the CUDA context is dead afterwards."""
    return lib().tts_debug_trip_watchdog(ctx, _stream(stream, ctx))


def tts_last_cuda_error(ctx) -> int:
    return lib().tts_last_cuda_error(ctx)


def tts_last_step_used_tensor_path(ctx) -> int:
    return lib().tts_last_step_used_tensor_path(ctx)


def tts_last_launch_count(ctx) -> int:
    return lib().tts_last_launch_count(ctx)


def tts_accept_mask(ctx, teacher_logits, draft_tokens, T, mask_out, tau_out, teacher_argmax_out=None, stream=None):
    st = lib().tts_accept_mask(ctx, _ptr(teacher_logits), _ptr(draft_tokens), T, _ptr(mask_out), _ptr(tau_out),
                               _ptr(teacher_argmax_out), _stream(stream, ctx))
    _check(ctx, st, "tts_accept_mask")


def tts_accept_mask_static(teacher_logits, logits_dtype, V, seg_len, draft_tokens, T, mask_out, tau_out,
                           teacher_argmax_out=None, stream=None):
    """tts_accept_mask for callers that may not allocate on the GPU (no ctx: tts_ctx_create calls cudaMalloc, which a
    process whose pool owns the whole GPU, or code that must not synchronise the device, cannot afford).  Runs on the
    CURRENT device with the library's built-in scratch; T <= TTS_STATIC_T_MAX.  Calls on one device share that
    scratch, so keep them ordered (one stream)."""
    st = lib().tts_accept_mask_static(_ptr(teacher_logits), logits_dtype, V, seg_len, _ptr(draft_tokens), T,
                                      _ptr(mask_out), _ptr(tau_out), _ptr(teacher_argmax_out), _stream(stream))
    if st != TTS_OK:
        raise TTSError(st, "tts_accept_mask_static", lib().tts_static_last_cuda_error())


def tts_static_last_cuda_error() -> int:
    return lib().tts_static_last_cuda_error()


def tts_accept_stochastic(ctx, teacher_logits, draft_logits, draft_tokens, uniforms, uniforms_resample, T, mask_out,
                          tau_out, next_token_out, diag_out=None, stream=None):
    st = lib().tts_accept_stochastic(ctx, _ptr(teacher_logits), _ptr(draft_logits), _ptr(draft_tokens), _ptr(uniforms),
                                     _ptr(uniforms_resample), T, _ptr(mask_out), _ptr(tau_out), _ptr(next_token_out),
                                     _ptr(diag_out), _stream(stream, ctx))
    _check(ctx, st, "tts_accept_stochastic")


def tts_distill_step(ctx, teacher_logits, h, W_in, W_out, W_master, adam_m, adam_v, pos_weight, mask, T, loss_scale,
                     loss_out, kl_rows_out=None, gh_out=None, gW_debug_out=None, side_stream=None):
    st = lib().tts_distill_step(ctx, _ptr(teacher_logits), _ptr(h), _ptr(W_in), _ptr(W_out), _ptr(W_master),
                                _ptr(adam_m), _ptr(adam_v), _ptr(pos_weight), _ptr(mask), T, loss_scale,
                                _ptr(loss_out), _ptr(kl_rows_out), _ptr(gh_out), _ptr(gW_debug_out),
                                _stream(side_stream, ctx))
    _check(ctx, st, "tts_distill_step")


def tts_distill_step_ex(ctx, teacher_logits, h, W_in, W_out, W_master, adam_m, adam_v, pos_weight, mask, T, loss_scale,
                        loss_out, kl_rows_out=None, gh_out=None, gW_debug_out=None, *, draft_logits=None,
                        draft_logits_out=None, ref_logits=None, lam=0.0, side_stream=None):
    ex = tts_step_extras(_ptr(draft_logits), _ptr(draft_logits_out), _ptr(ref_logits), lam)
    st = lib().tts_distill_step_ex(ctx, _ptr(teacher_logits), _ptr(h), _ptr(W_in), _ptr(W_out), _ptr(W_master),
                                   _ptr(adam_m), _ptr(adam_v), _ptr(pos_weight), _ptr(mask), T, loss_scale,
                                   _ptr(loss_out), _ptr(kl_rows_out), _ptr(gh_out), _ptr(gW_debug_out),
                                   C.addressof(ex), _stream(side_stream, ctx))
    _check(ctx, st, "tts_distill_step_ex")


def tts_distill_inner_steps(ctx, teacher_logits, h, W_in, W_out, W_master, adam_m, adam_v, pos_weight, mask, T,
                            loss_scale, K, lam, draft_logits, loss_out, kl_rows_out=None, gh_out=None,
                            side_stream=None):
    st = lib().tts_distill_inner_steps(ctx, _ptr(teacher_logits), _ptr(h), _ptr(W_in), _ptr(W_out), _ptr(W_master),
                                       _ptr(adam_m), _ptr(adam_v), _ptr(pos_weight), _ptr(mask), T, loss_scale, K,
                                       lam, _ptr(draft_logits), _ptr(loss_out), _ptr(kl_rows_out), _ptr(gh_out),
                                       _stream(side_stream, ctx))
    _check(ctx, st, "tts_distill_inner_steps")


def tts_profile_enable(ctx, enable: int):
    _check(ctx, lib().tts_profile_enable(ctx, int(enable)), "tts_profile_enable")


def tts_profile_read(ctx):
    """-> (list of mean ms per phase, number of steps averaged)"""
    ms = (C.c_float * TTS_NUM_PHASES)()
    n = C.c_int32()
    _check(ctx, lib().tts_profile_read(ctx, ms, C.byref(n)), "tts_profile_read")
    return list(ms), n.value


def tts_wait_step(ctx, main_stream=None):
    _check(ctx, lib().tts_wait_step(ctx, _stream(main_stream, ctx)), "tts_wait_step")


def tts_record_done(ctx, stream=None):
    _check(ctx, lib().tts_record_done(ctx, _stream(stream, ctx)), "tts_record_done")


def tts_sync_step(ctx):
    _check(ctx, lib().tts_sync_step(ctx), "tts_sync_step")


def tts_round_host(ctx, teacher_logits_host, h_host, draft_tokens_host, pos_weight_host, T, loss_scale, W_in, W_out,
                   W_master, adam_m, adam_v, gh_dev, loss_host, tau_host, mask_host=None, stream=None):
    st = lib().tts_round_host(ctx, _ptr(teacher_logits_host), _ptr(h_host), _ptr(draft_tokens_host),
                              _ptr(pos_weight_host), T, loss_scale, _ptr(W_in), _ptr(W_out), _ptr(W_master),
                              _ptr(adam_m), _ptr(adam_v), _ptr(gh_dev), _ptr(loss_host), _ptr(tau_host),
                              _ptr(mask_host), _stream(stream, ctx))
    _check(ctx, st, "tts_round_host")


def tts_round_host_begin(ctx, teacher_logits_host, h_host, draft_tokens_host, pos_weight_host, T, loss_scale, W_in,
                         W_out, W_master, adam_m, adam_v, gh_dev, loss_host, tau_host, mask_host=None, stream=None):
    st = lib().tts_round_host_begin(ctx, _ptr(teacher_logits_host), _ptr(h_host), _ptr(draft_tokens_host),
                                    _ptr(pos_weight_host), T, loss_scale, _ptr(W_in), _ptr(W_out), _ptr(W_master),
                                    _ptr(adam_m), _ptr(adam_v), _ptr(gh_dev), _ptr(loss_host), _ptr(tau_host),
                                    _ptr(mask_host), _stream(stream, ctx))
    _check(ctx, st, "tts_round_host_begin")


def tts_round_host_end(ctx):
    _check(ctx, lib().tts_round_host_end(ctx), "tts_round_host_end")


def _extras(draft_logits, draft_logits_out, ref_logits, lam):
    return tts_step_extras(_ptr(draft_logits), _ptr(draft_logits_out), _ptr(ref_logits), lam)


def tts_shard_begin_step(ctx, teacher_logits_local, h, W_in_local, T, stats_out, *, draft_logits=None,
                         draft_logits_out=None, ref_logits=None, lam=0.0, side_stream=None):
    ex = _extras(draft_logits, draft_logits_out, ref_logits, lam)
    st = lib().tts_shard_begin_step(ctx, _ptr(teacher_logits_local), _ptr(h), _ptr(W_in_local), T, C.addressof(ex),
                                    _ptr(stats_out), _stream(side_stream, ctx))
    _check(ctx, st, "tts_shard_begin_step")


def tts_shard_finish_step(ctx, stats_all, n_shards, teacher_logits_local, h, W_in_local, W_out_local, W_master_local,
                          adam_m_local, adam_v_local, pos_weight, mask, T, loss_scale, loss_out, kl_rows_out=None,
                          gh_partial_out=None, gW_debug_out=None, *, draft_logits=None, draft_logits_out=None,
                          ref_logits=None, lam=0.0, side_stream=None):
    ex = _extras(draft_logits, draft_logits_out, ref_logits, lam)
    st = lib().tts_shard_finish_step(ctx, _ptr(stats_all), n_shards, _ptr(teacher_logits_local), _ptr(h),
                                     _ptr(W_in_local), _ptr(W_out_local), _ptr(W_master_local), _ptr(adam_m_local),
                                     _ptr(adam_v_local), _ptr(pos_weight), _ptr(mask), T, loss_scale, _ptr(loss_out),
                                     _ptr(kl_rows_out), _ptr(gh_partial_out), _ptr(gW_debug_out), C.addressof(ex),
                                     _stream(side_stream, ctx))
    _check(ctx, st, "tts_shard_finish_step")


def tts_shard_argmax(ctx, teacher_logits_local, T, v_offset, val_out, idx_out, stream=None):
    st = lib().tts_shard_argmax(ctx, _ptr(teacher_logits_local), T, v_offset, _ptr(val_out), _ptr(idx_out),
                                _stream(stream, ctx))
    _check(ctx, st, "tts_shard_argmax")


def tts_shard_accept_mask(ctx, val_all, idx_all, n_shards, draft_tokens, T, mask_out, tau_out, teacher_argmax_out=None,
                          stream=None):
    st = lib().tts_shard_accept_mask(ctx, _ptr(val_all), _ptr(idx_all), n_shards, _ptr(draft_tokens), T, _ptr(mask_out),
                                     _ptr(tau_out), _ptr(teacher_argmax_out), _stream(stream, ctx))
    _check(ctx, st, "tts_shard_accept_mask")


def make_config(V, d, T_max, seg_len, param_dtype=TTS_BF16, logits_dtype=TTS_BF16, optimizer=TTS_ADAMW, lr=1e-5,
                beta1=0.9, beta2=0.999, eps=1e-8, weight_decay=0.0, mask_mode=TTS_ROWS_ALL, max_ctas=0,
                kernel_path=TTS_PATH_AUTO, moment_dtype=TTS_MOMENT_F32, max_inner_steps=0, flags=0,
                sr_seed=0) -> tts_config:
    return tts_config(V, d, T_max, seg_len, param_dtype, logits_dtype, optimizer, lr, beta1, beta2, eps,
                      weight_decay, mask_mode, max_ctas, kernel_path, moment_dtype, max_inner_steps, flags, sr_seed)
