// C-ABI entry points of libtts_b200.so (include/tts.h): context, validation, dispatch.
// All arithmetic lives in the kernels (tts_mask.cu, tts_stats.cu, tts_simt.cu, tts_tc.cu).
#include <math.h>
#include <new>
#include <stdlib.h>
#include <string.h>

#include "tts_internal.h"

namespace {

inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

inline int32_t cuda_fail(tts_ctx* c, cudaError_t e) {
  if (c) c->last_cuda_error = static_cast<int>(e);
  return TTS_ERR_CUDA;
}

size_t elem_size(int dtype) { return dtype == TTS_BF16 ? 2 : 4; }

template <typename T>
cudaError_t dmalloc(T** p, size_t n) {
  *p = nullptr;
  if (n == 0) return cudaSuccess;
  return cudaMalloc(reinterpret_cast<void**>(p), n * sizeof(T));
}

void free_all(tts_ctx* c) {
  if (!c) return;
  tts::tc_destroy(c);
  cudaFree(c->step_count_dev); cudaFree(c->step_scalars); cudaFree(c->dev_status);
  if (c->host_slot) cudaFreeHost(c->host_slot);
  cudaFree(c->z); cudaFree(c->z_ref_buf); cudaFree(c->dl32); cudaFree(c->stat_part); cudaFree(c->row_stats);
  cudaFree(c->row_loss); cudaFree(c->merge_ticket);
  cudaFree(c->arg_val); cudaFree(c->arg_idx); cudaFree(c->argmax_tmp);
  cudaFree(c->acc_rows); cudaFree(c->acc_rej); cudaFree(c->acc_rpart);
  for (int k = 0; k < 2; ++k) {
    tts_ctx::RoundSlot& r = c->rs[k];
    cudaFree(r.teacher); cudaFree(r.h); cudaFree(r.tok); cudaFree(r.pw); cudaFree(r.mask); cudaFree(r.tau); cudaFree(r.loss);
    if (r.copy_done) cudaEventDestroy(r.copy_done);
    if (r.round_done) cudaEventDestroy(r.round_done);
  }
  if (c->done_event) cudaEventDestroy(c->done_event);
  if (c->status_event) cudaEventDestroy(c->status_event);
  if (c->status_stream) cudaStreamDestroy(c->status_stream);
  if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
  if (c->prof_events) {
    for (int i = 0; i < tts::kProfSlots * (TTS_NUM_PHASES + 1); ++i) cudaEventDestroy(c->prof_events[i]);
    free(c->prof_events);
  }
}

// Staging of the host-buffer rounds, allocated on first use (the one place outside tts_ctx_create that allocates;
// include/tts.h says so at tts_round_host).
cudaError_t ensure_round_slots(tts_ctx* c) {
  if (c->rs_ready) return cudaSuccess;
  const tts_config& cfg = c->cfg;
  const size_t V = cfg.V, Tm = cfg.T_max;
  cudaError_t e = cudaSuccess;
  for (int k = 0; k < 2 && e == cudaSuccess; ++k) {
    tts_ctx::RoundSlot& r = c->rs[k];
    if (e == cudaSuccess) e = cudaMalloc(&r.teacher, Tm * V * elem_size(cfg.logits_dtype));
    if (e == cudaSuccess) e = cudaMalloc(&r.h, Tm * cfg.d * elem_size(cfg.param_dtype));
    if (e == cudaSuccess) e = dmalloc(&r.tok, Tm);
    if (e == cudaSuccess) e = dmalloc(&r.pw, Tm);
    if (e == cudaSuccess) e = dmalloc(&r.mask, Tm);
    if (e == cudaSuccess) e = dmalloc(&r.tau, Tm / cfg.seg_len);
    if (e == cudaSuccess) e = dmalloc(&r.loss, 1);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&r.copy_done, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&r.round_done, cudaEventDisableTiming);
  }
  if (e != cudaSuccess) {   // all or nothing: a later call may try again
    for (int k = 0; k < 2; ++k) {
      tts_ctx::RoundSlot& r = c->rs[k];
      cudaFree(r.teacher); cudaFree(r.h); cudaFree(r.tok); cudaFree(r.pw); cudaFree(r.mask); cudaFree(r.tau); cudaFree(r.loss);
      if (r.copy_done) cudaEventDestroy(r.copy_done);
      if (r.round_done) cudaEventDestroy(r.round_done);
      memset(&r, 0, sizeof(r));
    }
    return e;
  }
  c->rs_ready = true;
  return cudaSuccess;
}

}  // namespace

extern "C" {

const char* tts_status_string(int32_t s) {
  switch (s) {
    case TTS_OK: return "TTS_OK";
    case TTS_ERR_INVALID_ARG: return "TTS_ERR_INVALID_ARG";
    case TTS_ERR_UNSUPPORTED: return "TTS_ERR_UNSUPPORTED";
    case TTS_ERR_CUDA: return "TTS_ERR_CUDA";
    case TTS_ERR_ARCH: return "TTS_ERR_ARCH";
    default: return "TTS_ERR_UNKNOWN";
  }
}

int32_t tts_version(void) { return 300; /* 0.3.0 */ }

int32_t tts_ctx_create(const tts_config* cfg, int32_t device, tts_ctx** out) {
  if (!cfg || !out) return TTS_ERR_INVALID_ARG;
  *out = nullptr;
  if (cfg->V <= 0 || cfg->d <= 0 || cfg->T_max <= 0 || cfg->seg_len <= 0) return TTS_ERR_INVALID_ARG;
  if (cfg->T_max > 4096 || cfg->T_max % cfg->seg_len != 0) return TTS_ERR_INVALID_ARG;
  if (cfg->param_dtype != TTS_F32 && cfg->param_dtype != TTS_BF16) return TTS_ERR_UNSUPPORTED;
  if (cfg->logits_dtype != TTS_F32 && cfg->logits_dtype != TTS_BF16) return TTS_ERR_UNSUPPORTED;
  if (cfg->optimizer != TTS_SGD && cfg->optimizer != TTS_ADAMW) return TTS_ERR_UNSUPPORTED;
  if (cfg->mask_mode < TTS_ROWS_ALL || cfg->mask_mode > TTS_ROWS_ACCEPTED_PLUS_ONE) return TTS_ERR_UNSUPPORTED;
  if (cfg->kernel_path != TTS_PATH_AUTO && cfg->kernel_path != TTS_PATH_SIMT) return TTS_ERR_UNSUPPORTED;
  if (cfg->max_ctas < 0 || cfg->max_inner_steps < 0) return TTS_ERR_INVALID_ARG;
  if (cfg->flags & ~(TTS_FLAG_CHECK_PRECONDITIONS | TTS_FLAG_DETERMINISTIC | TTS_FLAG_SEPARATE_GH)) return TTS_ERR_INVALID_ARG;
  if (cfg->moment_dtype != TTS_MOMENT_F32 && cfg->moment_dtype != TTS_MOMENT_BF16) return TTS_ERR_UNSUPPORTED;
  if (cfg->moment_dtype != TTS_MOMENT_F32 && cfg->optimizer != TTS_ADAMW) return TTS_ERR_UNSUPPORTED;
  // rows of every [*, V] / [*, d] tensor must start 16-byte aligned
  if ((static_cast<size_t>(cfg->V) * elem_size(cfg->logits_dtype)) % 16 != 0) return TTS_ERR_UNSUPPORTED;
  if ((static_cast<size_t>(cfg->d) * elem_size(cfg->param_dtype)) % 16 != 0) return TTS_ERR_UNSUPPORTED;

  int ndev = 0;
  cudaError_t e = cudaGetDeviceCount(&ndev);
  if (e != cudaSuccess) return TTS_ERR_CUDA;   // no driver / no device: there is no CPU fallback
  if (device < 0 || device >= ndev) return TTS_ERR_INVALID_ARG;
  cudaDeviceProp prop;
  if ((e = cudaGetDeviceProperties(&prop, device)) != cudaSuccess) return TTS_ERR_CUDA;
  if (prop.major != 10) return TTS_ERR_ARCH;
  if ((e = cudaSetDevice(device)) != cudaSuccess) return TTS_ERR_CUDA;

  tts_ctx* c = new (std::nothrow) tts_ctx();
  if (!c) return TTS_ERR_INVALID_ARG;
  memset(c, 0, sizeof(*c));
  c->cfg = *cfg;
  c->device = device;
  c->sm_count = prop.multiProcessorCount;
  c->T_pad_max = (cfg->T_max + 15) / 16 * 16;
  c->tensor_ok = cfg->kernel_path == TTS_PATH_AUTO && tts::tc_supported(*cfg);
  c->watchdog_cycles = 1ll << 34;
  if (const char* w = getenv("TTS_WATCHDOG_CYCLES")) {   // include/tts.h, tts_debug_trip_watchdog
    char* end = nullptr;
    const long long v = strtoll(w, &end, 10);
    if (end == w || *end != '\0' || v < 0) { delete c; return TTS_ERR_INVALID_ARG; }
    c->watchdog_cycles = v;
  }

  const size_t V = cfg->V, Tm = cfg->T_max, Tp = c->T_pad_max;
  bool ok = true;
  ok = ok && cudaEventCreateWithFlags(&c->done_event, cudaEventDisableTiming) == cudaSuccess;
  ok = ok && cudaEventCreateWithFlags(&c->status_event, cudaEventDisableTiming) == cudaSuccess;
  ok = ok && cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking) == cudaSuccess;
  ok = ok && cudaStreamCreateWithFlags(&c->status_stream, cudaStreamNonBlocking) == cudaSuccess;
  ok = ok && dmalloc(&c->step_count_dev, 1) == cudaSuccess;
  ok = ok && dmalloc(&c->step_scalars, 2) == cudaSuccess;
  ok = ok && cudaMemset(c->step_count_dev, 0, sizeof(unsigned long long)) == cudaSuccess;
  ok = ok && dmalloc(&c->dev_status, 2) == cudaSuccess;
  ok = ok && cudaMemset(c->dev_status, 0, 2 * sizeof(int)) == cudaSuccess;
  ok = ok && cudaHostAlloc(reinterpret_cast<void**>(&c->host_slot), 16, cudaHostAllocDefault) == cudaSuccess;
  ok = ok && dmalloc(&c->z, Tp * V) == cudaSuccess;
  // K > 1 inner steps keep step 1's logits as z_ref: reserved here so that no step call allocates
  if (cfg->max_inner_steps > 1) ok = ok && dmalloc(&c->z_ref_buf, Tp * V) == cudaSuccess;
  if (!c->tensor_ok) ok = ok && dmalloc(&c->dl32, Tm * V) == cudaSuccess;   // fp32 dlogits: CUDA-core kernels only
  ok = ok && dmalloc(&c->stat_part, Tm * tts::kStatTuplesMax * tts::kStatFields) == cudaSuccess;
  ok = ok && dmalloc(&c->row_stats, tts::kRowStatFields * Tm) == cudaSuccess;
  ok = ok && dmalloc(&c->row_loss, Tm) == cudaSuccess;
  ok = ok && dmalloc(&c->merge_ticket, 1) == cudaSuccess;
  ok = ok && cudaMemset(c->merge_ticket, 0, sizeof(unsigned int)) == cudaSuccess;
  ok = ok && dmalloc(&c->arg_val, Tm * tts::kArgSplitsMax) == cudaSuccess;
  ok = ok && dmalloc(&c->arg_idx, Tm * tts::kArgSplitsMax) == cudaSuccess;
  ok = ok && dmalloc(&c->argmax_tmp, Tm) == cudaSuccess;
  ok = ok && dmalloc(&c->acc_rows, 2 * Tm) == cudaSuccess;
  ok = ok && dmalloc(&c->acc_rej, Tm / cfg->seg_len) == cudaSuccess;
  ok = ok && dmalloc(&c->acc_rpart, (Tm / cfg->seg_len) * tts::kStatSplitsMax) == cudaSuccess;
  // the staging slots of tts_round_host* (2 x T_max x V logits: 311 MB at T_max = 512) are allocated by the first
  // such call (ensure_round_slots): callers that keep their data on the device never pay for them
  // the low-precision moment formats live in the tcgen05 update kernels only
  if (ok && !c->tensor_ok && cfg->moment_dtype != TTS_MOMENT_F32) {
    free_all(c);
    delete c;
    return TTS_ERR_UNSUPPORTED;
  }
  if (ok) ok = tts::check_init(c) == cudaSuccess;
  if (ok && c->tensor_ok) ok = tts::tc_init(c) == cudaSuccess;
  if (!ok) {
    cudaGetLastError();
    free_all(c);
    delete c;
    return TTS_ERR_CUDA;
  }
  *out = c;
  return TTS_OK;
}

int32_t tts_ctx_destroy(tts_ctx* c) {
  if (!c) return TTS_ERR_INVALID_ARG;
  cudaSetDevice(c->device);
  cudaDeviceSynchronize();
  free_all(c);
  delete c;
  return TTS_OK;
}

int32_t tts_set_lr(tts_ctx* c, float lr) {
  if (!c || !(lr >= 0.f)) return TTS_ERR_INVALID_ARG;
  c->cfg.lr = lr;
  return TTS_OK;
}

int32_t tts_set_step_count(tts_ctx* c, int64_t n) {
  if (!c || n < 0) return TTS_ERR_INVALID_ARG;
  const unsigned long long v = static_cast<unsigned long long>(n);
  cudaError_t e = cudaSetDevice(c->device);
  if (e == cudaSuccess) e = cudaDeviceSynchronize();
  if (e == cudaSuccess) e = cudaMemcpy(c->step_count_dev, &v, sizeof(v), cudaMemcpyHostToDevice);
  return e == cudaSuccess ? TTS_OK : cuda_fail(c, e);
}

int64_t tts_get_step_count(const tts_ctx* c) {
  if (!c) return -1;
  unsigned long long v = 0;
  if (cudaSetDevice(c->device) != cudaSuccess || cudaDeviceSynchronize() != cudaSuccess ||
      cudaMemcpy(&v, c->step_count_dev, sizeof(v), cudaMemcpyDeviceToHost) != cudaSuccess)
    return -1;
  return static_cast<int64_t>(v);
}
int32_t tts_set_step_count_async(tts_ctx* c, int64_t n, void* stream) {
  if (!c || n < 0) return TTS_ERR_INVALID_ARG;
  tts_device_guard g(c->device);
  cudaError_t e = tts::launch_set_count(c, static_cast<unsigned long long>(n), static_cast<cudaStream_t>(stream));
  return e == cudaSuccess ? TTS_OK : cuda_fail(c, e);
}

int64_t tts_get_step_count_on(tts_ctx* c, void* stream) {
  if (!c) return -1;
  tts_device_guard g(c->device);
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  unsigned long long* slot = reinterpret_cast<unsigned long long*>(c->host_slot);
  cudaError_t e = cudaMemcpyAsync(slot, c->step_count_dev, sizeof(*slot), cudaMemcpyDeviceToHost, s);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  if (e != cudaSuccess) { cuda_fail(c, e); return -1; }
  return static_cast<int64_t>(*slot);
}

// The word is exchanged with 0 by a one-thread kernel on `s` and copied into the pinned slot behind it; the host then
// waits for `s` alone.
static int32_t take_status(tts_ctx* c, cudaStream_t s) {
  int* slot = c->host_slot + 2;   // the step-count read uses the first 8 bytes of the 16-byte slot
  cudaError_t e = tts::launch_take_status(c, s);
  if (e == cudaSuccess) e = cudaMemcpyAsync(slot, c->dev_status + 1, sizeof(int), cudaMemcpyDeviceToHost, s);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  if (e != cudaSuccess) { cuda_fail(c, e); return -1; }
  return *slot;
}

int32_t tts_last_device_status(tts_ctx* c) {
  if (!c) return -1;
  tts_device_guard g(c->device);
  // Host-side waits on the two events that stand behind every kernel able to set a bit: the last step's done-event and
  // the event of the last tts_check_preconditions / tts_accept_stochastic.  (The legacy default stream would NOT order
  // this read after work on cudaStreamNonBlocking streams, which is what every torch.cuda.Stream is.)
  cudaError_t e = cudaSuccess;
  if (c->done_recorded) e = cudaEventSynchronize(c->done_event);
  if (e == cudaSuccess && c->status_recorded) e = cudaEventSynchronize(c->status_event);
  if (e != cudaSuccess) { cuda_fail(c, e); return -1; }
  return take_status(c, c->status_stream);
}

int32_t tts_device_status_on(tts_ctx* c, void* stream) {
  if (!c) return -1;
  tts_device_guard g(c->device);
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
  if (cudaStreamIsCapturing(s, &cap) != cudaSuccess || cap != cudaStreamCaptureStatusNone) return -1;
  return take_status(c, s);
}

// status bits can also come from calls that are not steps: an event behind them for tts_last_device_status
static cudaError_t mark_status_source(tts_ctx* c, cudaStream_t s) {
  cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
  cudaError_t e = cudaStreamIsCapturing(s, &cap);
  if (e != cudaSuccess || cap != cudaStreamCaptureStatusNone) return e;   // inside a capture: see tts_record_done
  if ((e = cudaEventRecord(c->status_event, s)) == cudaSuccess) c->status_recorded = true;
  return e;
}

int32_t tts_check_preconditions(tts_ctx* c, const void* teacher, const void* h, const void* W_in, const float* W_master,
                                int32_t T, void* stream) {
  if (!c) return TTS_ERR_INVALID_ARG;
  if (T <= 0 || T > c->cfg.T_max) return TTS_ERR_INVALID_ARG;
  if (!aligned16(teacher) || !aligned16(h) || !aligned16(W_in) || !aligned16(W_master)) return TTS_ERR_INVALID_ARG;
  tts_device_guard g(c->device);
  int launches = 0;
  cudaError_t e = tts::launch_check_preconditions(c, teacher, h, W_in, W_master, T, static_cast<cudaStream_t>(stream),
                                                  &launches);
  c->last_launches = launches;
  if (e == cudaSuccess) e = mark_status_source(c, static_cast<cudaStream_t>(stream));
  return e == cudaSuccess ? TTS_OK : cuda_fail(c, e);
}

int32_t tts_debug_trip_watchdog(tts_ctx* c, void* stream) {
  if (!c) return TTS_ERR_INVALID_ARG;
  tts_device_guard g(c->device);
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  cudaError_t e = tts::launch_stalled_pipeline(s);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  return e == cudaSuccess ? TTS_OK : cuda_fail(c, e);
}

int32_t tts_last_cuda_error(const tts_ctx* c) { return c ? c->last_cuda_error : 0; }
int32_t tts_last_step_used_tensor_path(const tts_ctx* c) { return c ? c->last_used_tensor : 0; }
int32_t tts_last_launch_count(const tts_ctx* c) { return c ? c->last_launches : 0; }

int32_t tts_accept_mask(tts_ctx* c, const void* teacher, const int32_t* tok, int32_t T, uint8_t* mask_out,
                        int32_t* tau_out, int32_t* am_out, void* stream) {
  if (!c || !teacher || !tok || !mask_out || !tau_out) return TTS_ERR_INVALID_ARG;
  if (T <= 0 || T > c->cfg.T_max || T % c->cfg.seg_len != 0) return TTS_ERR_INVALID_ARG;
  if (!aligned16(teacher)) return TTS_ERR_INVALID_ARG;
  tts_device_guard g(c->device);
  int launches = 0;
  cudaError_t e = tts::launch_accept_mask(c, teacher, tok, T, mask_out, tau_out, am_out,
                                          static_cast<cudaStream_t>(stream), &launches);
  c->last_launches = launches;
  if (e != cudaSuccess) return cuda_fail(c, e);
  return TTS_OK;
}

int32_t tts_accept_stochastic(tts_ctx* c, const void* teacher, const float* draft_logits, const int32_t* tok,
                              const float* uniforms, const float* uniforms_resample, int32_t T, uint8_t* mask_out,
                              int32_t* tau_out, int32_t* next_token_out, float* diag_out, void* stream) {
  if (!c || !teacher || !draft_logits || !tok || !uniforms || !uniforms_resample || !mask_out || !tau_out ||
      !next_token_out)
    return TTS_ERR_INVALID_ARG;
  if (T <= 0 || T > c->cfg.T_max || T % c->cfg.seg_len != 0) return TTS_ERR_INVALID_ARG;
  if (!aligned16(teacher) || !aligned16(draft_logits)) return TTS_ERR_INVALID_ARG;
  if ((static_cast<size_t>(c->cfg.V) * sizeof(float)) % 16 != 0) return TTS_ERR_UNSUPPORTED;
  tts_device_guard g(c->device);
  int launches = 0;
  cudaError_t e = tts::launch_accept_stochastic(c, teacher, draft_logits, tok, uniforms, uniforms_resample, T,
                                                mask_out, tau_out, next_token_out, diag_out,
                                                static_cast<cudaStream_t>(stream), &launches);
  c->last_launches = launches;
  if (e == cudaSuccess) e = mark_status_source(c, static_cast<cudaStream_t>(stream));
  if (e != cudaSuccess) return cuda_fail(c, e);
  return TTS_OK;
}

int32_t tts_distill_step(tts_ctx* c, const void* teacher, const void* h, const void* W_in, void* W_out,
                         float* W_master, void* adam_m, void* adam_v, const float* pos_weight,
                         const uint8_t* mask, int32_t T, float loss_scale, float* loss_out, float* kl_rows_out,
                         float* gh_out, float* gW_debug_out, void* side_stream) {
  return tts_distill_step_ex(c, teacher, h, W_in, W_out, W_master, adam_m, adam_v, pos_weight, mask, T, loss_scale,
                             loss_out, kl_rows_out, gh_out, gW_debug_out, nullptr, side_stream);
}

// Everything a step call can reject without touching the GPU (so that callers which enqueue other work first, like
// tts_round_host, can ask BEFORE their first enqueue).
static int32_t check_step_args(const tts_ctx* c, const void* teacher, const void* h, const void* W_in, const void* W_out,
                               const float* W_master, const void* adam_m, const void* adam_v, const float* pos_weight,
                               const uint8_t* mask, int32_t T, const float* loss_out, const float* gh_out,
                               const float* gW_debug_out, const tts_step_extras* ex, int phase, const float* stats_out,
                               const float* stats_all, int32_t n_shards) {
  if (!c || !teacher || !h || !W_in) return TTS_ERR_INVALID_ARG;
  if (phase != tts::kPhaseBegin && (!W_out || !pos_weight || !loss_out)) return TTS_ERR_INVALID_ARG;
  if (phase == tts::kPhaseBegin && !stats_out) return TTS_ERR_INVALID_ARG;
  if (phase == tts::kPhaseFinish && (!stats_all || n_shards < 1 || n_shards > 1024)) return TTS_ERR_INVALID_ARG;
  if (ex) {
    if (!(ex->lambda >= 0.f)) return TTS_ERR_INVALID_ARG;
    if (ex->draft_logits && ex->draft_logits_out) return TTS_ERR_INVALID_ARG;   // nothing is computed to write out
    if (!aligned16(ex->draft_logits) || !aligned16(ex->draft_logits_out) || !aligned16(ex->ref_logits))
      return TTS_ERR_INVALID_ARG;
  }
  const tts_config& cfg = c->cfg;
  if (T <= 0 || T > cfg.T_max || T % cfg.seg_len != 0) return TTS_ERR_INVALID_ARG;
  if (phase != tts::kPhaseBegin) {
    if ((cfg.param_dtype == TTS_BF16) != (W_master != nullptr)) return TTS_ERR_INVALID_ARG;
    if ((cfg.optimizer == TTS_ADAMW) != (adam_m != nullptr && adam_v != nullptr)) return TTS_ERR_INVALID_ARG;
    if (cfg.optimizer == TTS_SGD && (adam_m || adam_v)) return TTS_ERR_INVALID_ARG;
    if (cfg.mask_mode != TTS_ROWS_ALL && !mask) return TTS_ERR_INVALID_ARG;
  }
  if (!aligned16(teacher) || !aligned16(h) || !aligned16(W_in) || !aligned16(W_out) || !aligned16(W_master) ||
      !aligned16(adam_m) || !aligned16(adam_v) || !aligned16(gh_out) || !aligned16(gW_debug_out))
    return TTS_ERR_INVALID_ARG;
  return TTS_OK;
}

// The step of include/tts.h in one piece (phase 0) or as the two halves of the vocabulary-sharded step.
static int32_t run_step(tts_ctx* c, const void* teacher, const void* h, const void* W_in, void* W_out,
                        float* W_master, void* adam_m, void* adam_v, const float* pos_weight,
                        const uint8_t* mask, int32_t T, float loss_scale, float* loss_out, float* kl_rows_out,
                        float* gh_out, float* gW_debug_out, const tts_step_extras* ex, void* side_stream, int phase,
                        float* stats_out, const float* stats_all, int32_t n_shards) {
  const int32_t ok = check_step_args(c, teacher, h, W_in, W_out, W_master, adam_m, adam_v, pos_weight, mask, T, loss_out,
                                     gh_out, gW_debug_out, ex, phase, stats_out, stats_all, n_shards);
  if (ok != TTS_OK) return ok;
  const tts_config& cfg = c->cfg;

  tts_device_guard guard(c->device);
  cudaStream_t s = static_cast<cudaStream_t>(side_stream);
  cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
  cudaError_t e = cudaStreamIsCapturing(s, &cap);
  if (e != cudaSuccess) return cuda_fail(c, e);
  const bool capturing = cap != cudaStreamCaptureStatusNone;
  tts::StepArgs a;
  a.step_scalars = c->step_scalars;
  a.phase = phase; a.shard_stats_out = stats_out; a.shard_stats_all = stats_all; a.n_shards = n_shards;
  a.teacher = teacher; a.h = h; a.W_in = W_in; a.W_out = W_out;
  a.master = W_master; a.adam_m = adam_m; a.adam_v = adam_v;
  a.pos_weight = pos_weight; a.mask = mask; a.T = T; a.loss_scale = loss_scale;
  a.loss_out = loss_out; a.kl_rows_out = kl_rows_out; a.gh_out = gh_out; a.gW_debug = gW_debug_out;
  a.z_given = ex ? ex->draft_logits : nullptr;
  a.z_keep = ex ? ex->draft_logits_out : nullptr;
  a.z_ref = (ex && ex->lambda > 0.f) ? ex->ref_logits : nullptr;   // lambda = 0: the term vanishes, skip its sweep
  a.lambda = a.z_ref ? ex->lambda : 0.f;
  a.lr = cfg.lr; a.beta1 = cfg.beta1; a.beta2 = cfg.beta2; a.eps = cfg.eps; a.wd = cfg.weight_decay;

  int launches = 0;
  const bool prof_saved = c->prof_on;
  if (phase != tts::kPhaseAll || capturing) c->prof_on = false;   // the phase events describe whole, eager steps only
  // Adam's count advances once per step, ON THE DEVICE: in the merge kernel of a3 (second half of a sharded step)
  tts::prof_mark(c, -1, s);
  if ((cfg.flags & TTS_FLAG_CHECK_PRECONDITIONS) && phase != tts::kPhaseFinish) {   // debug mode: SURVEY 8(b) 1 and 5
    if ((e = tts::launch_check_preconditions(c, teacher, h, W_in, phase == tts::kPhaseAll ? W_master : nullptr, T, s,
                                             &launches)) != cudaSuccess) {
      c->prof_on = prof_saved;
      return cuda_fail(c, e);
    }
  }
  if (c->tensor_ok) {
    c->last_used_tensor = 1;
    e = tts::tc_step(c, a, s, &launches);
  } else {
    c->last_used_tensor = 0;
    e = tts::simt_step(c, a, s, &launches);
  }
  c->last_launches = launches;
  if (e != cudaSuccess) { c->prof_on = prof_saved; return cuda_fail(c, e); }
  if (c->prof_on) c->prof_count += 1;
  c->prof_on = prof_saved;
  if (capturing) return TTS_OK;   // an event recorded inside a capture cannot be waited on outside: tts_record_done
  if ((e = cudaEventRecord(c->done_event, s)) != cudaSuccess) return cuda_fail(c, e);
  c->done_recorded = true;
  return TTS_OK;
}

int32_t tts_record_done(tts_ctx* c, void* stream) {
  if (!c) return TTS_ERR_INVALID_ARG;
  tts_device_guard g(c->device);
  cudaError_t e = cudaEventRecord(c->done_event, static_cast<cudaStream_t>(stream));
  if (e != cudaSuccess) return cuda_fail(c, e);
  c->done_recorded = true;
  return TTS_OK;
}

int32_t tts_distill_step_ex(tts_ctx* c, const void* teacher, const void* h, const void* W_in, void* W_out,
                            float* W_master, void* adam_m, void* adam_v, const float* pos_weight,
                            const uint8_t* mask, int32_t T, float loss_scale, float* loss_out, float* kl_rows_out,
                            float* gh_out, float* gW_debug_out, const tts_step_extras* ex, void* side_stream) {
  return run_step(c, teacher, h, W_in, W_out, W_master, adam_m, adam_v, pos_weight, mask, T, loss_scale, loss_out,
                  kl_rows_out, gh_out, gW_debug_out, ex, side_stream, tts::kPhaseAll, nullptr, nullptr, 0);
}

int32_t tts_shard_begin_step(tts_ctx* c, const void* teacher_local, const void* h, const void* W_in_local, int32_t T,
                             const tts_step_extras* ex, float* stats_out, void* side_stream) {
  if (stats_out && !aligned16(stats_out)) return TTS_ERR_INVALID_ARG;
  return run_step(c, teacher_local, h, W_in_local, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, T, 1.f, nullptr,
                  nullptr, nullptr, nullptr, ex, side_stream, tts::kPhaseBegin, stats_out, nullptr, 0);
}

int32_t tts_shard_finish_step(tts_ctx* c, const float* stats_all, int32_t n_shards, const void* teacher_local,
                              const void* h, const void* W_in_local, void* W_out_local, float* W_master_local,
                              void* adam_m_local, void* adam_v_local, const float* pos_weight, const uint8_t* mask,
                              int32_t T, float loss_scale, float* loss_out, float* kl_rows_out, float* gh_partial_out,
                              float* gW_debug_out, const tts_step_extras* ex, void* side_stream) {
  return run_step(c, teacher_local, h, W_in_local, W_out_local, W_master_local, adam_m_local, adam_v_local, pos_weight,
                  mask, T, loss_scale, loss_out, kl_rows_out, gh_partial_out, gW_debug_out, ex, side_stream,
                  tts::kPhaseFinish, nullptr, stats_all, n_shards);
}

int32_t tts_shard_argmax(tts_ctx* c, const void* teacher_local, int32_t T, int32_t v_offset, float* val_out,
                         int32_t* idx_out, void* stream) {
  if (!c || !teacher_local || !val_out || !idx_out || v_offset < 0) return TTS_ERR_INVALID_ARG;
  if (T <= 0 || T > c->cfg.T_max || T % c->cfg.seg_len != 0 || !aligned16(teacher_local)) return TTS_ERR_INVALID_ARG;
  tts_device_guard g(c->device);
  int launches = 0;
  cudaError_t e = tts::launch_shard_argmax(c, teacher_local, T, v_offset, val_out, idx_out,
                                           static_cast<cudaStream_t>(stream), &launches);
  c->last_launches = launches;
  return e == cudaSuccess ? TTS_OK : cuda_fail(c, e);
}

int32_t tts_shard_accept_mask(tts_ctx* c, const float* val_all, const int32_t* idx_all, int32_t n_shards,
                              const int32_t* tok, int32_t T, uint8_t* mask_out, int32_t* tau_out, int32_t* am_out,
                              void* stream) {
  if (!c || !val_all || !idx_all || !tok || !mask_out || !tau_out || n_shards < 1) return TTS_ERR_INVALID_ARG;
  if (T <= 0 || T > c->cfg.T_max || T % c->cfg.seg_len != 0) return TTS_ERR_INVALID_ARG;
  tts_device_guard g(c->device);
  int launches = 0;
  cudaError_t e = tts::launch_shard_mask(c, val_all, idx_all, n_shards, tok, T, mask_out, tau_out, am_out,
                                         static_cast<cudaStream_t>(stream), &launches);
  c->last_launches = launches;
  return e == cudaSuccess ? TTS_OK : cuda_fail(c, e);
}

int32_t tts_distill_inner_steps(tts_ctx* c, const void* teacher, const void* h, const void* W_in, void* W_out,
                                float* W_master, void* adam_m, void* adam_v, const float* pos_weight,
                                const uint8_t* mask, int32_t T, float loss_scale, int32_t K, float lambda,
                                const float* draft_logits, float* loss_out, float* kl_rows_out, float* gh_out,
                                void* side_stream) {
  if (!c || K < 1 || !(lambda >= 0.f) || !loss_out) return TTS_ERR_INVALID_ARG;
  // K > 1 keeps step 1's logits as z_ref: the caller's own draft_logits, or the scratch reserved by
  // tts_config.max_inner_steps (no step call allocates)
  if (K > 1 && !draft_logits && !c->z_ref_buf) return TTS_ERR_INVALID_ARG;
  int launches = 0;
  for (int k = 0; k < K; ++k) {
    tts_step_extras ex;
    ex.draft_logits = nullptr; ex.draft_logits_out = nullptr; ex.ref_logits = nullptr; ex.lambda = 0.f;
    if (k == 0) {
      // step 1 at q = q_t: the lambda term and its gradient vanish (R3).  Its logits become z_ref.
      if (draft_logits) ex.draft_logits = draft_logits;
      else if (K > 1) ex.draft_logits_out = c->z_ref_buf;
    } else {
      ex.ref_logits = draft_logits ? draft_logits : c->z_ref_buf;
      ex.lambda = lambda;
    }
    // step 1 reads W_in and writes W_out; later steps update W_out in place (W_out may alias W_in, include/tts.h)
    const int32_t st = tts_distill_step_ex(c, teacher, h, k == 0 ? W_in : W_out, W_out, W_master, adam_m, adam_v,
                                           pos_weight, mask, T, loss_scale, loss_out + k,
                                           k == 0 ? kl_rows_out : nullptr, k == K - 1 ? gh_out : nullptr, nullptr,
                                           &ex, side_stream);
    if (st != TTS_OK) return st;
    launches += c->last_launches;
  }
  c->last_launches = launches;
  return TTS_OK;
}

int32_t tts_profile_enable(tts_ctx* c, int32_t enable) {
  if (!c) return TTS_ERR_INVALID_ARG;
  if (enable && !c->prof_events) {
    const int n = tts::kProfSlots * (TTS_NUM_PHASES + 1);
    c->prof_events = static_cast<cudaEvent_t*>(calloc(n, sizeof(cudaEvent_t)));
    if (!c->prof_events) return TTS_ERR_INVALID_ARG;
    for (int i = 0; i < n; ++i) {
      cudaError_t e = cudaEventCreate(&c->prof_events[i]);
      if (e != cudaSuccess) return cuda_fail(c, e);
    }
  }
  c->prof_on = enable != 0;
  c->prof_count = 0;
  return TTS_OK;
}

int32_t tts_profile_read(tts_ctx* c, float* ms_out, int32_t* n_steps_out) {
  if (!c || !ms_out) return TTS_ERR_INVALID_ARG;
  for (int p = 0; p < TTS_NUM_PHASES; ++p) ms_out[p] = 0.f;
  const int n = c->prof_count < tts::kProfSlots ? c->prof_count : tts::kProfSlots;
  if (n_steps_out) *n_steps_out = n;
  if (n == 0 || !c->prof_events) return TTS_OK;
  if (c->done_recorded) {
    cudaError_t e = cudaEventSynchronize(c->done_event);
    if (e != cudaSuccess) return cuda_fail(c, e);
  }
  for (int i = 0; i < n; ++i) {
    const cudaEvent_t* ev = c->prof_events + i * (TTS_NUM_PHASES + 1);
    for (int p = 0; p < TTS_NUM_PHASES; ++p) {
      float ms = 0.f;
      cudaError_t e = cudaEventElapsedTime(&ms, ev[p], ev[p + 1]);
      if (e != cudaSuccess) return cuda_fail(c, e);
      ms_out[p] += ms / n;
    }
  }
  c->prof_count = 0;
  return TTS_OK;
}

int32_t tts_wait_step(tts_ctx* c, void* main_stream) {
  if (!c) return TTS_ERR_INVALID_ARG;
  if (!c->done_recorded) return TTS_OK;
  tts_device_guard g(c->device);
  cudaError_t e = cudaStreamWaitEvent(static_cast<cudaStream_t>(main_stream), c->done_event, 0);
  return e == cudaSuccess ? TTS_OK : cuda_fail(c, e);
}

int32_t tts_sync_step(tts_ctx* c) {
  if (!c) return TTS_ERR_INVALID_ARG;
  if (!c->done_recorded) return TTS_OK;
  cudaError_t e = cudaEventSynchronize(c->done_event);
  return e == cudaSuccess ? TTS_OK : cuda_fail(c, e);
}

// One round through host buffers, enqueued only: inputs into staging slot (rounds begun & 1), a1 + the step on `stream`,
// results back into the caller's host buffers, the slot's round_done event behind them.
static int32_t round_host_body(tts_ctx* c, tts_ctx::RoundSlot& r, bool reused, const void* teacher_host,
                               const void* h_host, const int32_t* tok_host, const float* pw_host, int32_t T,
                               float loss_scale, const void* W_in, void* W_out, float* W_master, void* adam_m,
                               void* adam_v, float* gh_dev, float* loss_host, int32_t* tau_host, uint8_t* mask_host,
                               void* stream) {
  const tts_config& cfg = c->cfg;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  const size_t V = cfg.V, d = cfg.d;
  cudaError_t e;
  // The teacher logits (the bulk: 160 MB at 512 rows, ~3 ms of PCIe) travel on the ctx's copy stream.  That copy waits
  // only for the round that used this slot two rounds ago, NOT for the caller's stream: it runs under the previous
  // round's step and under this round's pass a2, which needs only h and W_in (tensor path).  That is why the host
  // buffers must be complete ON THE HOST when this is called (include/tts.h).  The small inputs go on the caller's
  // stream (their slot's last readers are earlier kernels of that stream).
  if (reused && (e = cudaStreamWaitEvent(c->copy_stream, r.round_done, 0)) != cudaSuccess) return cuda_fail(c, e);
  if ((e = cudaMemcpyAsync(r.teacher, teacher_host, (size_t)T * V * elem_size(cfg.logits_dtype),
                           cudaMemcpyHostToDevice, c->copy_stream)) != cudaSuccess) return cuda_fail(c, e);
  if ((e = cudaEventRecord(r.copy_done, c->copy_stream)) != cudaSuccess) return cuda_fail(c, e);
  if ((e = cudaMemcpyAsync(r.h, h_host, (size_t)T * d * elem_size(cfg.param_dtype), cudaMemcpyHostToDevice, s)) !=
      cudaSuccess)
    return cuda_fail(c, e);
  if ((e = cudaMemcpyAsync(r.tok, tok_host, (size_t)T * 4, cudaMemcpyHostToDevice, s)) != cudaSuccess)
    return cuda_fail(c, e);
  if ((e = cudaMemcpyAsync(r.pw, pw_host, (size_t)T * 4, cudaMemcpyHostToDevice, s)) != cudaSuccess)
    return cuda_fail(c, e);
  int early_launches = 0;
  tts_step_extras ex;
  ex.draft_logits = nullptr; ex.draft_logits_out = nullptr; ex.ref_logits = nullptr; ex.lambda = 0.f;
  if (c->tensor_ok) {
    tts::StepArgs a0;
    memset(&a0, 0, sizeof(a0));
    a0.h = r.h; a0.W_in = W_in; a0.T = T;
    if ((e = tts::tc_logits_only(c, a0, s, &early_launches)) != cudaSuccess) return cuda_fail(c, e);
    ex.draft_logits = c->z;                          // the step below takes z as given: a2 is done
  }
  if ((e = cudaStreamWaitEvent(s, r.copy_done, 0)) != cudaSuccess) return cuda_fail(c, e);
  int32_t st = tts_accept_mask(c, r.teacher, r.tok, T, r.mask, r.tau, nullptr, stream);
  if (st != TTS_OK) return st;
  const int mask_launches = c->last_launches;
  st = tts_distill_step_ex(c, r.teacher, r.h, W_in, W_out, W_master, adam_m, adam_v, r.pw, r.mask, T, loss_scale, r.loss,
                           nullptr, gh_dev, nullptr, &ex, stream);
  if (st != TTS_OK) return st;
  c->last_launches += mask_launches + early_launches;
  if ((e = cudaMemcpyAsync(loss_host, r.loss, 4, cudaMemcpyDeviceToHost, s)) != cudaSuccess) return cuda_fail(c, e);
  if ((e = cudaMemcpyAsync(tau_host, r.tau, (size_t)(T / cfg.seg_len) * 4, cudaMemcpyDeviceToHost, s)) != cudaSuccess)
    return cuda_fail(c, e);
  if (mask_host && (e = cudaMemcpyAsync(mask_host, r.mask, (size_t)T, cudaMemcpyDeviceToHost, s)) != cudaSuccess)
    return cuda_fail(c, e);
  if ((e = cudaEventRecord(r.round_done, s)) != cudaSuccess) return cuda_fail(c, e);
  return TTS_OK;
}

static int32_t round_host_enqueue(tts_ctx* c, const void* teacher_host, const void* h_host, const int32_t* tok_host,
                                  const float* pw_host, int32_t T, float loss_scale, const void* W_in, void* W_out,
                                  float* W_master, void* adam_m, void* adam_v, float* gh_dev, float* loss_host,
                                  int32_t* tau_host, uint8_t* mask_host, void* stream) {
  if (!c || !teacher_host || !h_host || !tok_host || !pw_host || !loss_host || !tau_host) return TTS_ERR_INVALID_ARG;
  if (c->rh_begun - c->rh_ended >= 2) return TTS_ERR_INVALID_ARG;   // both slots are in flight: end a round first
  // Everything the step could refuse is refused here, BEFORE anything is allocated or enqueued.  The step's device
  // inputs will be a slot's staging buffers (never NULL, cudaMalloc-aligned: `staged` stands in for them, it is only
  // compared, never dereferenced) and the caller's parameter tensors.
  alignas(16) static const unsigned char staged[16] = {0};
  const float* sf = reinterpret_cast<const float*>(staged);
  const int32_t ok = check_step_args(c, staged, staged, W_in, W_out, W_master, adam_m, adam_v, sf, staged, T, sf, gh_dev,
                                     nullptr, nullptr, tts::kPhaseAll, nullptr, nullptr, 0);
  if (ok != TTS_OK) return ok;
  tts_device_guard guard(c->device);
  if (!c->rs_ready) {   // first host-buffer round on this ctx: allocate the two staging slots (nothing is in flight yet)
    const cudaError_t ea = ensure_round_slots(c);
    if (ea != cudaSuccess) return cuda_fail(c, ea);
  }
  tts_ctx::RoundSlot& r = c->rs[c->rh_begun & 1];
  const int32_t st = round_host_body(c, r, c->rh_begun >= 2, teacher_host, h_host, tok_host, pw_host, T, loss_scale,
                                     W_in, W_out, W_master, adam_m, adam_v, gh_dev, loss_host, tau_host, mask_host,
                                     stream);
  if (st != TTS_OK) {
    // A CUDA call failed after copies / kernels of this round were enqueued.  The round does not count (rh_begun stays),
    // so nothing would ever wait for them: drain both streams here, while the caller's host buffers and this slot are
    // still what the in-flight work expects, and leave the slot's events in a state the next begin can wait on.
    cudaStreamSynchronize(c->copy_stream);
    cudaStreamSynchronize(static_cast<cudaStream_t>(stream));
    cudaEventRecord(r.round_done, static_cast<cudaStream_t>(stream));
    return st;
  }
  ++c->rh_begun;
  return TTS_OK;
}

int32_t tts_round_host_begin(tts_ctx* c, const void* teacher_host, const void* h_host, const int32_t* tok_host,
                             const float* pw_host, int32_t T, float loss_scale, const void* W_in, void* W_out,
                             float* W_master, void* adam_m, void* adam_v, float* gh_dev, float* loss_host,
                             int32_t* tau_host, uint8_t* mask_host, void* stream) {
  return round_host_enqueue(c, teacher_host, h_host, tok_host, pw_host, T, loss_scale, W_in, W_out, W_master, adam_m,
                            adam_v, gh_dev, loss_host, tau_host, mask_host, stream);
}

int32_t tts_round_host_end(tts_ctx* c) {
  if (!c || c->rh_begun == c->rh_ended) return TTS_ERR_INVALID_ARG;
  tts_device_guard guard(c->device);
  const cudaError_t e = cudaEventSynchronize(c->rs[c->rh_ended & 1].round_done);
  ++c->rh_ended;
  return e == cudaSuccess ? TTS_OK : cuda_fail(c, e);
}

int32_t tts_round_host(tts_ctx* c, const void* teacher_host, const void* h_host, const int32_t* tok_host,
                       const float* pw_host, int32_t T, float loss_scale, const void* W_in, void* W_out,
                       float* W_master, void* adam_m, void* adam_v, float* gh_dev, float* loss_host,
                       int32_t* tau_host, uint8_t* mask_host, void* stream) {
  if (c && c->rh_begun != c->rh_ended) return TTS_ERR_INVALID_ARG;   // rounds begun with tts_round_host_begin are pending
  const int32_t st = round_host_enqueue(c, teacher_host, h_host, tok_host, pw_host, T, loss_scale, W_in, W_out,
                                        W_master, adam_m, adam_v, gh_dev, loss_host, tau_host, mask_host, stream);
  return st != TTS_OK ? st : tts_round_host_end(c);
}

}  // extern "C"
