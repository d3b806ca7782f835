// Host-side state of the tensor-path kernels (tts_tc.cu, tts_tc_gemm.cu): the operand scratch the
// gradient contractions read, the tensor maps over it and the driver entry point that encodes
// tensor maps.  Internal to the library.
#pragma once

#include <cuda.h>
#include <cudaTypedefs.h>

#include "tts_internal.h"

namespace tts {

constexpr int kKC = 64;          // bf16 elements per K chunk = one 128-byte swizzle row
constexpr int kTileMN = 128;     // MMA M of every tensor-path kernel (vocabulary rows or hidden columns per tile)

struct TcState {
  void* dlT;            // [V, Kp] fp16   B operand of gW (wide path): row v = S dl[0..Kp, v], this step's Kp as row pitch
  void* hTT;            // [d, Kp] fp16   A operand of gW (wide path): row j = S_h h[0..Kp, j]
  __nv_bfloat16* hTc;   // [d][16]        h^T rows, the A operand of gW (tts_tc_fused.cu, T <= 16; copied into tensor memory)
  __nv_bfloat16* dlC;   // [V / 16][2][2][2][8][8]        dl hi / lo planes, pre-tiled in core-matrix order (tts_tc_fused.cu)
  void* dlR;            // [P, V] fp16    B operand of gh: S dl[r, v] (rows T16 .. 2 T16: the lo plane when there are two)
  float* dl_scale;      // {S, 1 / S, S_h, 1 / S_h, bits of max|h|}: power-of-two scales of the fp16 dl and h^T planes (a4 kernels)
  int Kp;               // largest K extent of dlT / hTT (T_pad_max rounded up to kKC)
  int P;                // rows of dlR (T_pad_max, twice that up to 32 rows)
  PFN_cuTensorMapEncodeTiled_v12000 encode;
};

// 2-D row-major tensor map: inner extent `inner` (contiguous), `outer` rows, box [box_inner x box_outer].
inline CUresult make_map_2d(const TcState* st, CUtensorMap* m, CUtensorMapDataType dt, int esize, const void* base,
                            uint64_t inner, uint64_t outer, uint32_t box_inner, uint32_t box_outer,
                            CUtensorMapSwizzle sw) {
  const cuuint64_t dims[2] = {inner, outer};
  const cuuint64_t strides[1] = {inner * esize};
  const cuuint32_t box[2] = {box_inner, box_outer};
  const cuuint32_t estr[2] = {1, 1};
  return st->encode(m, dt, 2, const_cast<void*>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, sw,
                    CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
}

// CTAs of an update pass (tc_update_gh_kernel, tc_update_wide_kernel) when the caller sets no SM budget.
// With fp32 moments the pass is HBM-bound and the memory system, not the SM count, sets its speed: measured on B200
// (Qwen3-8B head, profiles/r2_README.md) the one-canvas pass runs 2.46 ms on 132 CTAs whatever the ring depth (5-7
// stages) and 2.51 / 2.68 / 2.74 ms on 148 CTAs with 5 / 6 / 7 stages; every grid of 136 CTAs and more shows that
// cliff, every grid from 124 to 132 does not; the several-canvas pass behaves the same way (2.69 against 2.73-2.91 ms
// at 64 rows).  So those passes leave a tenth of the SMs idle ON THAT PART: the figure is one measurement of the
// 148-SM B200 (and the driver's box of round 2 ran 2.66 ms at the same 132 CTAs), not a rule, so any other
// SM count gets one CTA per SM and a caller's max_ctas always wins.  With bf16 moments the pass is bound by its
// epilogue warps (18 bytes per parameter in this pass, 20 per step with a2's read of W_in) and wants every SM.
constexpr int kB200Sms = 148, kB200UpdateCtas = 132;
inline int tc_update_ctas(const tts_ctx* c, bool lowp_moments) {
  if (c->cfg.max_ctas > 0) return c->cfg.max_ctas < c->sm_count ? c->cfg.max_ctas : c->sm_count;
  if (lowp_moments || c->sm_count != kB200Sms) return c->sm_count;
  return kB200UpdateCtas;
}

// CTAs of a logits kernel (tc_logits_kernel, tc_logits_pair_kernel): the caller's SM budget, never more than the SMs
// there are, and never more than the per-row statistics scratch can describe.  A stream-K walk over `grid` ranges cuts
// at most grid - 1 tiles (the pair kernel's K-split tail: at most grid / 2), each cut tile adds one fix-up tuple, so
// grid <= kStatFixMax keeps the fix-up list within kStatFixMax entries and grid + cuts within kStatTuplesMax tuples
// on any part (B200: 148 + 147 = 295).
static_assert(2 * kStatFixMax <= kStatTuplesMax, "stat_part holds one tuple per CTA plus one per cut tile");
inline int tc_logits_ctas(const tts_ctx* c) {
  const int g = (c->cfg.max_ctas > 0 && c->cfg.max_ctas < c->sm_count) ? c->cfg.max_ctas : c->sm_count;
  return g < kStatFixMax ? g : kStatFixMax;
}

// tts_tc_gemm.cu
cudaError_t tc_gemm_init(tts_ctx* c);
// a2: z[r, v] = sum_j h[r, j] W_in[v, j] on tcgen05 (fp32 accumulation), z scratch [T16, V]
// fuse_stats: the a3 online statistics are taken in the kernel's epilogue (tts_tc_epi.cuh) and *n_split_out tuples per
// canvas row are left in c->stat_part for launch_row_stats_finish; otherwise *n_split_out = 0
cudaError_t tc_launch_logits(tts_ctx* c, const StepArgs& a, float* z_out, bool fuse_stats, cudaStream_t s, int* launches,
                             int* n_split_out);
// a5: gh[r, j] = sum_v dl[r, v] W_in[v, j] on tcgen05, split over the vocabulary, fp32 atomics into gh
cudaError_t tc_launch_gh(tts_ctx* c, const StepArgs& a, cudaStream_t s, int* launches);
// floats of the deterministic-mode scratch (per-unit parts of gh) for steps of up to T16 rows
size_t tc_gh_part_floats(const tts_ctx* c, int T16);

// tts_tc_fused.cu: a5 + a6 + a7 in one pass over the optimiser state (T <= 16, d % 1024 == 0, V % 16 == 0)
cudaError_t tc_fused_init(tts_ctx* c);
int tc_fused_grid(const tts_ctx* c, int T16);
cudaError_t tc_launch_prep_fused(tts_ctx* c, const StepArgs& a, const float* z, cudaStream_t s, int* launches);   // a4: operands
cudaError_t tc_launch_update_fused(tts_ctx* c, const StepArgs& a, int grid, cudaStream_t s, int* launches);

// tts_tc_wide.cu: a4 operands (h^T rows, fp16 dl planes) and a6 + a7 for T <= 512
cudaError_t tc_wide_init(tts_ctx* c);
int tc_wide_planes(int T16);   // 2: dl S = hi + lo (T16 <= 32), 1: one fp16 plane
int tc_wide_fuses_gh(const tts_ctx* c, int T16); // 1: the wide update kernel forms gh itself (planes * T16 <= 256, and
                                                 // neither TTS_FLAG_SEPARATE_GH nor TTS_FLAG_DETERMINISTIC): no gh kernel
cudaError_t tc_launch_prep_wide(tts_ctx* c, const StepArgs& a, const float* z, cudaStream_t s, int* launches);
cudaError_t tc_launch_update_wide(tts_ctx* c, const StepArgs& a, cudaStream_t s, int* launches);

// tts_tc_pair.cu: CTA-pair (cta_group::2) a2 for 256 < T16 <= 512
cudaError_t tc_pair_init(tts_ctx* c);
int tc_pair_eligible(const tts_ctx* c, int T16);
cudaError_t tc_launch_logits_pair(tts_ctx* c, const StepArgs& a, float* z_out, bool fuse_stats, cudaStream_t s,
                                  int* launches, int* n_split_out);

}  // namespace tts
