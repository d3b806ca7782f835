// Internal declarations shared by the translation units of libtts_b200.so.
// Not part of the ABI (include/tts.h is).
#pragma once

#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <stdint.h>

#include "../../include/tts.h"

namespace tts {

constexpr int kStatSplitsMax = 64;   // V-splits per row in the row-statistics sweep
constexpr int kStatFixMax = 160;     // tiles whose statistics come from the fix-up sweep (cut by a stream-K walk)
constexpr int kStatTuplesMax = 320;  // tuples per canvas row in stat_part: one per CTA of a logits kernel + the fix-ups
constexpr int kArgSplitsMax = 64;    // V-splits per row in the argmax sweep
constexpr int kStatFields = 8;       // (m_t, s_t, a, m_z, s_z) of SURVEY §8(a) a3 + (m_ref, s_ref, b) of the lambda term
constexpr int kRowStatFields = 5;    // row_stats planes: lse_t, lse_z, kl, coef, lse_ref
constexpr int kProfSlots = 256;      // profiled steps kept between two tts_profile_read calls
constexpr int kKPad = 64;            // K extent (bf16 elements) of one 128-byte swizzle atom

struct StepArgs {
  const void* teacher;
  const void* h;
  const void* W_in;
  void* W_out;
  float* master;
  void* adam_m;   // [V,d] cfg.moment_dtype (fp32, or bf16 bits with TTS_MOMENT_BF16)
  void* adam_v;
  const float* pos_weight;
  const uint8_t* mask;
  int T;
  float loss_scale;
  float* loss_out;
  float* kl_rows_out;
  float* gh_out;
  float* gW_debug;
  // f1: optional extras of tts_distill_step_ex
  const float* z_given;   // [T,V] fp32 draft logits supplied by the caller (a2 is skipped) or NULL
  float* z_keep;          // [T,V] fp32: a2 writes z here instead of the ctx scratch (it becomes z_ref of later inner steps) or NULL
  const float* z_ref;     // [T,V] fp32 logits of q_t for the lambda term or NULL
  float lambda;           // weight of K~L(q_t || q)
  // SURVEY 8(e), the step sharded over the vocabulary: phase 1 = a2 + this shard's a3 sweep -> shard_stats_out;
  // phase 2 = merge of all shards' tuples -> a4 .. a7 on this shard; 0 = the whole step on one GPU
  int phase;
  float* shard_stats_out;        // [T, kStatFields]            (phase 1)
  const float* shard_stats_all;  // [n_shards, T, kStatFields]  (phase 2)
  int n_shards;
  // optimiser scalars for this step (bias corrections precomputed on the host in fp64)
  float lr, beta1, beta2, eps, wd;
  const float* step_scalars;   // device: {1 / (1 - beta1^n), 1 / sqrt(1 - beta2^n)} of THIS step, written by the
                               // row-statistics merge kernel earlier in the same stream (so a captured CUDA graph of the step
                               // advances Adam's count on every replay)
};

// where a2 writes the draft logits, and where a3 / a4 read them
inline float* z_dst(const StepArgs& a, float* scratch) { return a.z_keep ? a.z_keep : scratch; }
inline const float* z_src(const StepArgs& a, float* scratch) { return a.z_given ? a.z_given : z_dst(a, scratch); }

}  // namespace tts

// Makes the ctx's device current for the lifetime of the object (a process may hold ctxs on several GPUs).
struct tts_device_guard {
  int prev;
  bool switched;
  explicit tts_device_guard(int device) : prev(-1), switched(false) {
    if (cudaGetDevice(&prev) == cudaSuccess && prev != device) switched = cudaSetDevice(device) == cudaSuccess;
  }
  ~tts_device_guard() { if (switched) cudaSetDevice(prev); }
};

struct tts_ctx {
  tts_config cfg;
  int device;
  int sm_count;
  unsigned long long* step_count_dev;   // Adam's step count n lives on the device (see step_scalars)
  float* step_scalars;                  // [2]
  int last_cuda_error;
  int last_used_tensor;
  int last_launches;
  int T_pad_max;          // T_max rounded up to 16
  long long watchdog_cycles;   // limit of the kernels' watchdog (TTS_WATCHDOG_CYCLES at create; 0 = off)
  bool tensor_ok;         // shape/dtype qualifies for the tcgen05 kernels
  cudaEvent_t done_event;
  bool done_recorded;
  cudaEvent_t status_event;   // behind the last tts_check_preconditions / tts_accept_stochastic (they set status bits too)
  bool status_recorded;
  cudaStream_t status_stream; // non-blocking: the read-and-clear of the status word runs here, never on the legacy stream
  // ---- scratch (device) ----
  float* z;               // [T_pad_max, V] draft logits (fp32)
  float* dl32;            // [T_max, V] fp32 dlogits                (CUDA-core path)
  float* stat_part;       // [T_max, kStatTuplesMax, kStatFields]
  float* row_stats;       // [kRowStatFields, T_max]: lse_t, lse_z, kl, coef (= loss_scale * omega), lse_ref
  double* row_loss;       // [T_max] omega_r (KL_r + lambda KL_ref,r): summed in a fixed order by the merge kernel's last CTA
  unsigned int* merge_ticket;
  float* z_ref_buf;       // [T_pad_max, V] fp32, reserved by tts_ctx_create when cfg.max_inner_steps > 1, else NULL
  float* arg_val;         // [T_max, kArgSplitsMax]
  int32_t* arg_idx;       // [T_max, kArgSplitsMax]
  int32_t* argmax_tmp;    // [T_max]
  int* dev_status;        // [2]: device status word (bits TTS_DEV_*) + the slot its read-and-clear exchanges it into
  int* host_slot;         // pinned host scratch (16 bytes) for the stream-ordered status / step-count reads
  float* gh_part;         // TTS_FLAG_DETERMINISTIC: [units][T16][128] per-unit parts of gh (tts_tc_gemm.cu)
  float* acc_rows;        // [T_max, 2] lse_t, lse_z of tts_accept_stochastic
  int32_t* acc_rej;       // [T_max / seg_len] first rejected row per sequence
  double* acc_rpart;      // [T_max / seg_len, kStatSplitsMax] residual mass per slice
  // ---- staging for tts_round_host / tts_round_host_begin: two slots, so that the next round's inputs can travel while
  // this round's step runs ----
  struct RoundSlot {
    void* teacher;
    void* h;
    int32_t* tok;
    float* pw;
    uint8_t* mask;
    int32_t* tau;
    float* loss;
    cudaEvent_t copy_done;    // the teacher's H2D copy into this slot has landed
    cudaEvent_t round_done;   // the round that used this slot has finished (results copied back): the slot is free
  } rs[2];
  bool rs_ready;                // the slots exist (allocated by the first tts_round_host* call, not by tts_ctx_create)
  unsigned rh_begun, rh_ended;  // rounds begun / ended through the host API (slot = count & 1; at most 2 outstanding)
  cudaStream_t copy_stream;   // the teacher's H2D copy runs here, next to a2 (and the previous round) on the caller's stream
  // ---- per-phase profiling (tts_profile_*) ----
  bool prof_on;
  int prof_count;                                   // steps recorded since the last read
  cudaEvent_t* prof_events;                         // [kProfSlots][TTS_NUM_PHASES + 1], created lazily
  // ---- tensor-path state (opaque, owned by tts_tc.cu) ----
  void* tc_state;
};

namespace tts {

// Phase boundary: records the profiling event that ENDS phase `phase` (phase = -1: step start).
inline void prof_mark(tts_ctx* c, int phase, cudaStream_t s) {
  if (!c->prof_on || !c->prof_events) return;
  const int slot = c->prof_count % kProfSlots;
  cudaEventRecord(c->prof_events[slot * (TTS_NUM_PHASES + 1) + phase + 1], s);
}

// tts_check.cu: precondition checks (debug mode)
cudaError_t launch_check_preconditions(tts_ctx* c, const void* teacher, const void* h, const void* W_in,
                                       const float* master, int T, cudaStream_t s, int* launches);
cudaError_t launch_set_count(tts_ctx* c, unsigned long long n, cudaStream_t s);
cudaError_t launch_take_status(tts_ctx* c, cudaStream_t s);   // dev_status[1] = atomicExch(&dev_status[0], 0)
cudaError_t launch_stalled_pipeline(cudaStream_t s);
cudaError_t check_init(tts_ctx* c);   // this unit's copy of the watchdog limit (tts_tc_ptx.cuh)
// tts_mask.cu
cudaError_t launch_accept_mask(tts_ctx* c, const void* teacher, const int32_t* tok, int T, uint8_t* mask,
                               int32_t* tau, int32_t* am_out, cudaStream_t s, int* launches);
cudaError_t launch_shard_argmax(tts_ctx* c, const void* teacher, int T, int v_offset, float* val, int32_t* idx,
                                cudaStream_t s, int* launches);
cudaError_t launch_shard_mask(tts_ctx* c, const float* val_all, const int32_t* idx_all, int n_shards,
                              const int32_t* tok, int T, uint8_t* mask, int32_t* tau, int32_t* am_out, cudaStream_t s,
                              int* launches);
// tts_accept.cu (f2)
cudaError_t launch_accept_stochastic(tts_ctx* c, const void* teacher, const float* z, const int32_t* tok,
                                     const float* u, const float* u2, int T, uint8_t* mask, int32_t* tau,
                                     int32_t* next_tok, float* diag, cudaStream_t s, int* launches);
// tts_stats.cu: row statistics + merge + loss (CUDA-core sweeps shared by both paths).
// z_ld = leading dimension (row stride in floats) of the z scratch.
cudaError_t launch_row_stats(tts_ctx* c, const StepArgs& a, const float* z, int z_ld, cudaStream_t s, int* launches);
cudaError_t launch_row_stats_shard(tts_ctx* c, const StepArgs& a, const float* z, int z_ld, float* stats_out,
                                   cudaStream_t s, int* launches);
cudaError_t launch_row_stats_merge_shards(tts_ctx* c, const StepArgs& a, const float* stats_all, int n_shards,
                                          cudaStream_t s, int* launches);
// a3 fused into a2 (tts_tc_epi.cuh): the logits kernel left `splits` tuples per row in c->stat_part.
//   tiles:  the fix-up sweep over n 128-column tiles whose z was completed by fp32 RED (tuples slot0 .. slot0 + n - 1)
//   finish: merge -> normalisers, KL, omega, loss (whole step) or -> one tuple per row in stats_out (shard, phase 1)
cudaError_t launch_row_stats_tiles(tts_ctx* c, const StepArgs& a, const float* z, int z_ld, const int* col0, int n,
                                   int slot0, int splits, cudaStream_t s, int* launches);
cudaError_t launch_row_stats_finish(tts_ctx* c, const StepArgs& a, int splits, float* shard_stats_out, cudaStream_t s,
                                    int* launches);
// a2 + a3 of either path for the phase of `a`: returns after phase 1, or leaves the row normalisers in c->row_stats
enum { kPhaseAll = 0, kPhaseBegin = 1, kPhaseFinish = 2 };
// tts_simt.cu
cudaError_t simt_step(tts_ctx* c, const StepArgs& a, cudaStream_t s, int* launches);
// tts_tc.cu
bool tc_supported(const tts_config& cfg);
cudaError_t tc_init(tts_ctx* c);
void tc_destroy(tts_ctx* c);
cudaError_t tc_step(tts_ctx* c, const StepArgs& a, cudaStream_t s, int* launches);
// a2 alone into the ctx's z scratch (no statistics): what tts_round_host runs while the round's teacher logits are
// still on their way from the host
cudaError_t tc_logits_only(tts_ctx* c, const StepArgs& a, cudaStream_t s, int* launches);

}  // namespace tts
