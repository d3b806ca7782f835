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
constexpr int kGhNB = 128;       // canvas rows (MMA N) per accumulator block of the gh contraction

struct TcState {
  __nv_bfloat16* dlT;   // [V, Kp]        B operand of gW: row v = (dl_hi[0..T16), dl_lo[0..T16)) of vocabulary row v
  __nv_bfloat16* hTT;   // [d, Kp]        A operand of gW: row j = (h[0..T16, j], h[0..T16, j])
  __nv_bfloat16* hTc;   // [d / 128][2][16][8][8]        A tiles of gW in core-matrix order (tts_tc_fused.cu, T <= 16)
  __nv_bfloat16* dlC;   // [V / 16][2][2][2][8][8]        dl hi / lo planes, pre-tiled in core-matrix order (tts_tc_fused.cu)
  __nv_bfloat16* dlR;   // [2, P, V]      B operand of gh: plane 0 = dl_hi[r, v], plane 1 = dl_lo[r, v]
  int Kp;               // K extent of dlT / hTT (multiple of kKC)
  int P;                // rows per dlR plane (T_pad_max, rounded up to kGhNB when larger)
  CUtensorMap tm_dlT, tm_hTT;
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

// tts_tc_gemm.cu
cudaError_t tc_gemm_init(tts_ctx* c);
// a2: z[r, v] = sum_j h[r, j] W_in[v, j] on tcgen05 (fp32 accumulation), z scratch [T16, V]
cudaError_t tc_launch_logits(tts_ctx* c, const StepArgs& a, float* z_out, cudaStream_t s, int* launches);
// a5: gh[r, j] = sum_v (dl_hi + dl_lo)[r, v] W_in[v, j] on tcgen05, split over the vocabulary, fp32 atomics into gh
cudaError_t tc_launch_gh(tts_ctx* c, const StepArgs& a, cudaStream_t s, int* launches);

// tts_tc_fused.cu: a5 + a6 + a7 in one pass over the optimiser state (T <= 16, d % 1024 == 0, V % 16 == 0)
cudaError_t tc_fused_init(tts_ctx* c);
int tc_fused_grid(const tts_ctx* c, int T16);
cudaError_t tc_launch_prep_fused(tts_ctx* c, const StepArgs& a, const float* z, cudaStream_t s, int* launches);   // a4: operands
cudaError_t tc_launch_update_fused(tts_ctx* c, const StepArgs& a, int grid, cudaStream_t s, int* launches);

}  // namespace tts
