// Tensor path of the distillation step (sm_100a): context state and dispatch.  The kernels live in
//   tts_tc_gemm.cu   a2 draft logits and a5 gh as W-streaming tcgen05 GEMMs
//   tts_tc_fused.cu  one canvas (T <= 16, d % 1024 == 0): a5 + a6 + a7 in one pass over the optimiser state
//   tts_tc_wide.cu   several canvases (T <= 512) and the remaining one-canvas shapes: a6 + a7 with the stripe's h^T
//                    resident in tensor memory and one fp16 dl plane
#include <new>
#include <string.h>

#include "tts_common.cuh"
#include "tts_tc_state.h"

namespace tts {

bool tc_supported(const tts_config& cfg) {
  return cfg.param_dtype == TTS_BF16 && cfg.V % kTileMN == 0 && cfg.d % kTileMN == 0 && cfg.T_max <= 512;
}

cudaError_t tc_init(tts_ctx* c) {
  TcState* st = new (std::nothrow) TcState();
  if (!st) return cudaErrorMemoryAllocation;
  memset(st, 0, sizeof(*st));
  c->tc_state = st;
  const int T16 = c->T_pad_max;
  st->Kp = (T16 + kKC - 1) / kKC * kKC;
  st->P = T16 > 32 ? (T16 > 64 ? T16 : 64) : 2 * T16;   // >= planes(t) * t for every step size t <= T16
  cudaError_t e;
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  if ((e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres)) != cudaSuccess) return e;
  if (!fn || qres != cudaDriverEntryPointSuccess) return cudaErrorNotSupported;
  st->encode = reinterpret_cast<PFN_cuTensorMapEncodeTiled_v12000>(fn);
  const size_t V = c->cfg.V, d = c->cfg.d;
  if ((e = cudaMalloc(&st->dlT, V * st->Kp * 2)) != cudaSuccess) return e;
  if ((e = cudaMalloc(&st->hTT, d * st->Kp * 2)) != cudaSuccess) return e;
  if ((e = cudaMalloc(&st->dlR, (size_t)st->P * V * 2)) != cudaSuccess) return e;
  if ((e = cudaMalloc(&st->dl_scale, 8 * sizeof(float))) != cudaSuccess) return e;
  if ((e = cudaMemset(st->dlR, 0, (size_t)st->P * V * 2)) != cudaSuccess) return e;
  if ((e = cudaMemset(st->dlT, 0, V * st->Kp * 2)) != cudaSuccess) return e;
  if ((e = cudaMemset(st->hTT, 0, d * st->Kp * 2)) != cudaSuccess) return e;
  if (c->cfg.flags & TTS_FLAG_DETERMINISTIC) {
    if ((e = cudaMalloc(&c->gh_part, tc_gh_part_floats(c, T16) * sizeof(float))) != cudaSuccess) return e;
  }
  if ((e = tc_gemm_init(c)) != cudaSuccess) return e;
  if ((e = tc_wide_init(c)) != cudaSuccess) return e;
  if ((e = tc_pair_init(c)) != cudaSuccess) return e;
  return tc_fused_init(c);
}

void tc_destroy(tts_ctx* c) {
  TcState* st = static_cast<TcState*>(c->tc_state);
  if (!st) return;
  cudaFree(st->dlT);
  cudaFree(st->hTT);
  cudaFree(st->dlR);
  cudaFree(st->dl_scale);
  cudaFree(st->hTc);
  cudaFree(st->dlC);
  cudaFree(c->gh_part);
  c->gh_part = nullptr;
  delete st;
  c->tc_state = nullptr;
}

cudaError_t tc_logits_only(tts_ctx* c, const StepArgs& a, cudaStream_t s, int* launches) {
  const int T16 = (a.T + 15) / 16 * 16;
  int n_tuples = 0;
  return tc_pair_eligible(c, T16) ? tc_launch_logits_pair(c, a, c->z, false, s, launches, &n_tuples)
                                  : tc_launch_logits(c, a, c->z, false, s, launches, &n_tuples);
}

cudaError_t tc_step(tts_ctx* c, const StepArgs& a, cudaStream_t s, int* launches) {
  const int V = c->cfg.V, T = a.T;
  const int T16 = (T + 15) / 16 * 16;
  cudaError_t e;

  // a2: draft logits on tcgen05 (skipped when the caller supplies them), a3: row statistics + loss
  const float* z = z_src(a, c->z);
  if (a.phase != kPhaseFinish) {
    // a3 rides in a2's epilogue (north_star (1): one TMA-staged sweep, no second pass over [T, V]) unless the lambda
    // term needs the reference distribution's statistics too (K > 1 inner steps) or the caller supplies z
    int n_tuples = 0;
    if (!a.z_given) {
      const bool fuse = a.z_ref == nullptr;
      e = tc_pair_eligible(c, T16) ? tc_launch_logits_pair(c, a, z_dst(a, c->z), fuse, s, launches, &n_tuples)
                                   : tc_launch_logits(c, a, z_dst(a, c->z), fuse, s, launches, &n_tuples);
      if (e != cudaSuccess) return e;
    }
    prof_mark(c, 0, s);
    if (n_tuples > 0) {
      if (a.phase == kPhaseBegin) return launch_row_stats_finish(c, a, n_tuples, a.shard_stats_out, s, launches);
      if ((e = launch_row_stats_finish(c, a, n_tuples, nullptr, s, launches)) != cudaSuccess) return e;
    } else {
      if (a.phase == kPhaseBegin) return launch_row_stats_shard(c, a, z, V, a.shard_stats_out, s, launches);
      if ((e = launch_row_stats(c, a, z, V, s, launches)) != cudaSuccess) return e;
    }
  } else {
    prof_mark(c, 0, s);
    if ((e = launch_row_stats_merge_shards(c, a, a.shard_stats_all, a.n_shards, s, launches)) != cudaSuccess) return e;
  }
  prof_mark(c, 1, s);

  // a4: operands of the gradient contractions
  // one canvas (T <= 16): one fused pass over the optimiser state (tts_tc_fused.cu) with its own pre-tiled operands
  // TTS_FLAG_SEPARATE_GH / TTS_FLAG_DETERMINISTIC: gh comes from its own kernel (reads the W_in buffer; per-unit parts
  // reduced in a fixed order), which consumes the wide path's dl planes
  const bool own_gh_kernel = a.gh_out && (c->cfg.flags & (TTS_FLAG_SEPARATE_GH | TTS_FLAG_DETERMINISTIC)) != 0;
  const int fused_grid = own_gh_kernel ? 0 : tc_fused_grid(c, T16);
  if (fused_grid > 0) {
    if ((e = tc_launch_prep_fused(c, a, z, s, launches)) != cudaSuccess) return e;
    prof_mark(c, 2, s);
    prof_mark(c, 3, s);
    if ((e = tc_launch_update_fused(c, a, fused_grid, s, launches)) != cudaSuccess) return e;
    prof_mark(c, 4, s);
    return cudaGetLastError();
  }
  // several canvases, or a one-canvas shape outside the fused kernel's stripes
  if ((e = tc_launch_prep_wide(c, a, z, s, launches)) != cudaSuccess) return e;
  prof_mark(c, 2, s);
  // a5: gh on tcgen05 (reads W_in before the update may overwrite an aliased W_out)
  if (a.gh_out && !tc_wide_fuses_gh(c, T16)) {
    if ((e = tc_launch_gh(c, a, s, launches)) != cudaSuccess) return e;
  }
  prof_mark(c, 3, s);
  // a6 + a7
  if ((e = tc_launch_update_wide(c, a, s, launches)) != cudaSuccess) return e;
  prof_mark(c, 4, s);
  return cudaGetLastError();
}

}  // namespace tts
