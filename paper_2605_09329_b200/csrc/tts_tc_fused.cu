// Pass B of the distillation step for small canvases (T16 <= 32): ONE persistent kernel per step that streams the
// optimiser state exactly once and does, per [128 vocabulary rows x 128 hidden columns] tile,
//
//   a6  gW^T tile = h^T . dl            tcgen05, accumulator in TMEM (never in HBM)
//   a7  SGD / AdamW on the fp32 master  epilogue straight out of TMEM, state tiles staged by TMA,
//       + bf16 working-copy write-back  results leave by coalesced 128-byte stores
//   a5  gh^T[j, r] += W_in[v, j] dl[r, v]   tcgen05 as well: the bf16 tile of W_in is RE-DERIVED from the
//                                       fp32 master tile the epilogue already holds in registers
//                                       (precondition W_in == rn_bf16(W_master), include/tts.h), written to
//                                       shared memory as the A operand, so bf16 W is not read from HBM again.
//
// gh accumulators persist in TMEM across a CTA's tiles: CTA b visits tiles t = b, b + grid, ..., whose hidden
// tile index t mod n_jt takes only n_jt / gcd(grid, n_jt) distinct values (8 for grid 148, d = 4096), each
// owning T16 TMEM columns next to the two gW accumulators; they are reduced into gh with fp32 atomics once,
// at the end of the kernel.
//
// Operands: hTT [d, Kp] (K-major A of gW) and the dl planes dlR [2, P, V] (hi / lo bf16 split of dl).  One
// shared-memory copy of the dlR tile serves both contractions: as the MN-major B of gW (N = vocabulary,
// K = canvas row) and as the K-major B of gh (N = canvas row, K = vocabulary).
#include <string.h>

#include "tts_common.cuh"
#include "tts_tc_ptx.cuh"
#include "tts_tc_state.h"

namespace tts {
namespace {

constexpr int kMJ = 128;         // hidden columns per tile  = MMA M = TMEM lanes
constexpr int kNV = 128;         // vocabulary rows per tile = MMA N of gW
constexpr int kSV = 16;          // vocabulary rows per optimiser-state sub-tile (one pipeline stage)
constexpr int kSubs = kNV / kSV;
constexpr int kStages = 6;       // state ring depth
constexpr int kOpStages = 2;     // operand ring depth
constexpr int kWt = 4;           // ring of re-derived bf16 W sub-tiles (A operand of gh)
constexpr int kHBytes = kMJ * kKC * 2;               // 16 KB hTT tile
constexpr int kStateTileBytes = kSV * kMJ * 4;       // 8 KB per tensor per stage
constexpr int kWtBytes = kMJ * kSV * 2;              // 4 KB
constexpr int kThreads = 384;    // warp 0 state TMA, 1 MMA, 2 TMEM alloc, 3 operand TMA, 4-11 epilogue
constexpr int kGhCol0 = 2 * kNV; // first TMEM column of the gh accumulators
constexpr int kTmemCols = 512;

struct FusedParams {
  float* master;
  float* am;
  float* av;
  __nv_bfloat16* W_out;
  float* gW_debug;
  float* gh;
  int V, d, T, T16, P;
  int n_jt;     // d / 128
  int jt_gcd;   // gcd(grid, n_jt): the hidden tiles a CTA visits are congruent mod jt_gcd
  float lr, b1, b2, eps, decay, c1, inv_sqrt_bc2;   // decay = 1 - lr wd, c1 = lr / (1 - b1^n)
};

__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
  const __nv_bfloat162 p = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<const uint32_t*>(&p);
}

template <bool ADAM>
__global__ void __launch_bounds__(kThreads, 1)
tc_update_gh_kernel(const __grid_constant__ CUtensorMap tm_hTT, const __grid_constant__ CUtensorMap tm_dl,
                    const __grid_constant__ CUtensorMap tm_master, const __grid_constant__ CUtensorMap tm_m,
                    const __grid_constant__ CUtensorMap tm_v, const FusedParams p) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  const int box_bytes = p.T16 * kKC * 2;     // one dlR box: [T16 rows x 64 v]
  const int dl_bytes = 4 * box_bytes;        // (hi, lo) x (v 0..63, v 64..127)
  uint8_t* opA = smem;                                  // [kOpStages][16 KB]   hTT tiles (SW128, K-major)
  uint8_t* opB = opA + kOpStages * kHBytes;             // [kOpStages][dl_bytes] dlR tiles (SW128)
  uint8_t* st = opB + kOpStages * dl_bytes;             // [kStages][3][kSV][128] fp32
  uint8_t* wt = st + kStages * 3 * kStateTileBytes;     // [kWt][2 k-groups][16 j-groups][8 x 16 B]
  uint64_t* bars = reinterpret_cast<uint64_t*>(wt + kWt * kWtBytes);
  uint64_t* op_full = bars;                  // [kOpStages]
  uint64_t* op_empty = op_full + kOpStages;  // [kOpStages]
  uint64_t* acc_full = op_empty + kOpStages; // [2]
  uint64_t* acc_empty = acc_full + 2;        // [2]
  uint64_t* st_full = acc_empty + 2;         // [kStages]
  uint64_t* st_empty = st_full + kStages;    // [kStages]
  uint64_t* wt_full = st_empty + kStages;    // [kWt]
  uint64_t* wt_empty = wt_full + kWt;        // [kWt]
  uint64_t* gh_full = wt_empty + kWt;        // [1]
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(gh_full + 1);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int n_jt = p.n_jt;
  const int n_tiles = (p.V / kNV) * n_jt;
  const int n_my = (n_tiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;

  if (warp == 0 && lane == 0) {
    ptx::prefetch_tensormap(&tm_master);
    if (ADAM) { ptx::prefetch_tensormap(&tm_m); ptx::prefetch_tensormap(&tm_v); }
  }
  if (warp == 3 && lane == 0) {
    ptx::prefetch_tensormap(&tm_hTT);
    ptx::prefetch_tensormap(&tm_dl);
  }
  if (warp == 1 && lane == 0) {
    for (int i = 0; i < kOpStages; ++i) { ptx::mbar_init(&op_full[i], 1); ptx::mbar_init(&op_empty[i], 1); }
    for (int i = 0; i < 2; ++i) { ptx::mbar_init(&acc_full[i], 1); ptx::mbar_init(&acc_empty[i], 8); }
    for (int i = 0; i < kStages; ++i) { ptx::mbar_init(&st_full[i], 1); ptx::mbar_init(&st_empty[i], 4); }
    for (int i = 0; i < kWt; ++i) { ptx::mbar_init(&wt_full[i], 4); ptx::mbar_init(&wt_empty[i], 1); }
    ptx::mbar_init(gh_full, 1);
    ptx::fence_barrier_init();
  }
  if (warp == 2) {
    ptx::tmem_alloc(tmem_slot, kTmemCols);
    ptx::tmem_relinquish();
  }
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;

  if (warp == 0) {
    // ===== optimiser-state producer: master / m / v sub-tiles [kSV rows x 128 floats] by TMA =====
    if (lane == 0) {
      uint32_t n = 0;
      for (int t = blockIdx.x; t < n_tiles; t += gridDim.x) {
        const int v0 = (t / n_jt) * kNV, j0 = (t % n_jt) * kMJ;
        for (int sub = 0; sub < kSubs; ++sub, ++n) {
          const int s = n % kStages;
          ptx::mbar_wait(&st_empty[s], ((n / kStages) & 1) ^ 1);
          uint8_t* dst = st + s * 3 * kStateTileBytes;
          ptx::mbar_expect_tx(&st_full[s], (ADAM ? 3 : 1) * kStateTileBytes);
          ptx::tma_load_2d(dst, &tm_master, &st_full[s], j0, v0 + sub * kSV);
          if (ADAM) {
            ptx::tma_load_2d(dst + kStateTileBytes, &tm_m, &st_full[s], j0, v0 + sub * kSV);
            ptx::tma_load_2d(dst + 2 * kStateTileBytes, &tm_v, &st_full[s], j0, v0 + sub * kSV);
          }
        }
      }
    }
  } else if (warp == 3) {
    // ===== operand producer: hTT tile [128 j x 64 k] and the dlR tile (4 boxes [T16 r x 64 v]) =====
    if (lane == 0) {
      uint32_t it = 0;
      for (int t = blockIdx.x; t < n_tiles; t += gridDim.x, ++it) {
        const int v0 = (t / n_jt) * kNV, j0 = (t % n_jt) * kMJ;
        const int s = it % kOpStages;
        ptx::mbar_wait(&op_empty[s], ((it / kOpStages) & 1) ^ 1);
        ptx::mbar_expect_tx(&op_full[s], kHBytes + dl_bytes);
        ptx::tma_load_2d(opA + s * kHBytes, &tm_hTT, &op_full[s], 0, j0);
        uint8_t* b = opB + s * dl_bytes;
        for (int pl = 0; pl < 2; ++pl)
          for (int kh = 0; kh < 2; ++kh)
            ptx::tma_load_2d(b + (pl * 2 + kh) * box_bytes, &tm_dl, &op_full[s], v0 + kh * kKC, pl * p.P);
      }
    }
  } else if (warp == 1) {
    // ===== MMA issuer =====
    if (lane == 0 && n_my > 0) {
      const uint32_t idesc_gw = ptx::make_idesc_bf16(kMJ, kNV, 0, 1);      // A = hTT K-major, B = dl MN-major
      const uint32_t idesc_gh = ptx::make_idesc_bf16(kMJ, p.T16, 0, 0);    // A = W (re-derived) K-major, B = dl K-major
      const int k_steps = p.T16 / 16;
      // acc[j, v] = sum_r hTT[j, r] (dl_hi + dl_lo)[r, v]
      auto issue_gw = [&](uint32_t it) {
        const int ab = it & 1;
        ptx::mbar_wait(&acc_empty[ab], ((it >> 1) & 1) ^ 1);
        const int s = it % kOpStages;
        ptx::mbar_wait(&op_full[s], (it / kOpStages) & 1);
        ptx::tc_fence_after();
        const uint32_t a0 = ptx::smem_u32(opA + s * kHBytes), b0 = ptx::smem_u32(opB + s * dl_bytes);
        uint32_t acc = 0;
        for (int pl = 0; pl < 2; ++pl)
          for (int kk = 0; kk < k_steps; ++kk) {
            const uint64_t ad = ptx::make_smem_desc(a0 + kk * 32, 16, 1024, ptx::kSwizzle128B);
            // MN-major: 64 v per 128-byte row, one row per canvas row; the second 64 v are one box further (LBO)
            const uint64_t bd =
                ptx::make_smem_desc(b0 + pl * 2 * box_bytes + kk * 2048, box_bytes, 1024, ptx::kSwizzle128B);
            ptx::mma_f16_ss(tmem_base + ab * kNV, ad, bd, idesc_gw, acc);
            acc = 1;
          }
        ptx::mma_commit(&acc_full[ab]);
      };
      uint32_t slot_mask = 0;
      issue_gw(0);
      for (uint32_t it = 0; it < (uint32_t)n_my; ++it) {
        const int t = blockIdx.x + it * gridDim.x;
        const int slot = (t % n_jt) / p.jt_gcd;
        const int s = it % kOpStages;
        const uint32_t b0 = ptx::smem_u32(opB + s * dl_bytes);
        for (int sub = 0; sub < kSubs; ++sub) {
          if (sub == 3 && it + 1 < (uint32_t)n_my) issue_gw(it + 1);
          const uint32_t n = it * kSubs + sub;
          const int buf = n % kWt;
          ptx::mbar_wait(&wt_full[buf], (n / kWt) & 1);
          ptx::tc_fence_after();
          // A: K-major, no swizzle: core matrices [8 j x 8 v] of 128 B; j-groups 128 B apart (SBO), the two
          // v-groups 2 KB apart (LBO)
          const uint64_t ad = ptx::make_smem_desc(ptx::smem_u32(wt + buf * kWtBytes), 2048, 128, 0);
          for (int pl = 0; pl < 2; ++pl) {
            const uint64_t bd = ptx::make_smem_desc(b0 + (pl * 2 + (sub >> 2)) * box_bytes + (sub & 3) * 32, 16, 1024,
                                                    ptx::kSwizzle128B);
            ptx::mma_f16_ss(tmem_base + kGhCol0 + slot * p.T16, ad, bd, idesc_gh, ((slot_mask >> slot) & 1) | pl);
          }
          slot_mask |= 1u << slot;
          ptx::mma_commit(&wt_empty[buf]);
        }
        ptx::mma_commit(&op_empty[s]);
      }
      ptx::mma_commit(gh_full);
    }
  } else if (warp >= 4) {
    // ===== epilogue: 2 groups x 4 warps; group g takes sub-tiles sub % 2 == g; warp quarter q owns lanes 32q.. =====
    const int q = warp & 3, g = (warp - 4) >> 2;
    const int col = q * 32 + lane;
    uint8_t* wt_thr = wt + (col >> 3) * 128 + (col & 7) * 16;
    uint32_t slot_mask = 0;
    uint32_t it = 0;
    for (int t = blockIdx.x; t < n_tiles; t += gridDim.x, ++it) {
      const int v0 = (t / n_jt) * kNV, j0 = (t % n_jt) * kMJ;
      slot_mask |= 1u << ((t % n_jt) / p.jt_gcd);
      const int ab = it & 1;
      ptx::mbar_wait(&acc_full[ab], (it >> 1) & 1);
      ptx::tc_fence_after();
      for (int sub = g; sub < kSubs; sub += 2) {
        const uint32_t n = it * kSubs + sub;
        const int s = n % kStages;
        uint32_t gr[kSV];
        ptx::tmem_ld_32x32b_x16(tmem_base + ab * kNV + sub * kSV + (static_cast<uint32_t>(q * 32) << 16), gr);
        ptx::mbar_wait(&st_full[s], (n / kStages) & 1);
        const float* sM = reinterpret_cast<const float*>(st + s * 3 * kStateTileBytes) + col;
        float M[kSV], mm[kSV], vv[kSV];
#pragma unroll
        for (int r = 0; r < kSV; ++r) {
          M[r] = sM[r * kMJ];
          if (ADAM) { mm[r] = sM[kSV * kMJ + r * kMJ]; vv[r] = sM[2 * kSV * kMJ + r * kMJ]; }
        }
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(&st_empty[s]);   // the stage's smem is in registers now
        // a5 operand: W_in[v, j] = rn_bf16(master[v, j]) for this thread's column j, 16 consecutive v
        const int buf = n % kWt;
        ptx::mbar_wait(&wt_empty[buf], ((n / kWt) & 1) ^ 1);
        {
          uint4 w0, w1;
          w0.x = pack_bf16(M[0], M[1]);   w0.y = pack_bf16(M[2], M[3]);
          w0.z = pack_bf16(M[4], M[5]);   w0.w = pack_bf16(M[6], M[7]);
          w1.x = pack_bf16(M[8], M[9]);   w1.y = pack_bf16(M[10], M[11]);
          w1.z = pack_bf16(M[12], M[13]); w1.w = pack_bf16(M[14], M[15]);
          uint8_t* dst = wt_thr + buf * kWtBytes;
          *reinterpret_cast<uint4*>(dst) = w0;
          *reinterpret_cast<uint4*>(dst + 2048) = w1;
        }
        ptx::fence_proxy_async_smem();
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(&wt_full[buf]);
        ptx::tmem_ld_wait();
        size_t idx = (size_t)(v0 + sub * kSV) * p.d + j0 + col;
#pragma unroll
        for (int r = 0; r < kSV; ++r, idx += p.d) {
          const float gg = __uint_as_float(gr[r]);
          float Mn;
          if (ADAM) {
            const float m1 = p.b1 * mm[r] + (1.f - p.b1) * gg;
            const float v1 = p.b2 * vv[r] + (1.f - p.b2) * gg * gg;
            const float den = __fsqrt_rn(v1) * p.inv_sqrt_bc2 + p.eps;
            Mn = M[r] * p.decay - __fdividef(p.c1 * m1, den);
            p.am[idx] = m1;
            p.av[idx] = v1;
          } else {
            Mn = M[r] - p.lr * gg;
          }
          p.master[idx] = Mn;
          p.W_out[idx] = __float2bfloat16_rn(Mn);
          if (p.gW_debug) p.gW_debug[idx] = gg;
        }
      }
      ptx::tc_fence_before();
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive(&acc_empty[ab]);
    }
    // ===== gh flush: the CTA's persistent accumulators -> fp32 atomics (group 0: one warp per lane quarter) =====
    if (g == 0 && it > 0) {
      ptx::mbar_wait(gh_full, 0);
      ptx::tc_fence_after();
      const int n_slots = n_jt / p.jt_gcd;
      for (int slot = 0; slot < n_slots; ++slot) {
        if (!((slot_mask >> slot) & 1)) continue;
        const int jt = (blockIdx.x % p.jt_gcd) + p.jt_gcd * slot;
        float* gc = p.gh + jt * kMJ + col;
        for (int c0 = 0; c0 < p.T16; c0 += 16) {
          uint32_t r[16];
          ptx::tmem_ld_32x32b_x16(tmem_base + kGhCol0 + slot * p.T16 + c0 + (static_cast<uint32_t>(q * 32) << 16), r);
          ptx::tmem_ld_wait();
#pragma unroll
          for (int i = 0; i < 16; ++i)
            if (c0 + i < p.T) atomicAdd(gc + (size_t)(c0 + i) * p.d, __uint_as_float(r[i]));
        }
      }
    }
  }
  ptx::tc_fence_before();
  __syncthreads();
  if (warp == 2) {
    ptx::tc_fence_after();
    ptx::tmem_dealloc(tmem_base, kTmemCols);
  }
}

int gcd_int(int a, int b) {
  while (b) { const int t = a % b; a = b; b = t; }
  return a;
}

size_t fused_smem(int T16) {
  return 1024 + (size_t)kOpStages * (kHBytes + 4 * T16 * kKC * 2) + (size_t)kStages * 3 * kStateTileBytes +
         (size_t)kWt * kWtBytes + 512;
}

}  // namespace

cudaError_t tc_fused_init(tts_ctx*) {
  cudaError_t e;
  const int smem = (int)fused_smem(32);
  if ((e = cudaFuncSetAttribute(tc_update_gh_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem)) !=
      cudaSuccess)
    return e;
  return cudaFuncSetAttribute(tc_update_gh_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
}

// Largest grid <= the wanted one whose CTAs each visit few enough distinct hidden tiles for their gh
// accumulators to fit the TMEM columns left beside the gW accumulators.  0: no such grid.
int tc_fused_grid(const tts_ctx* c, int T16) {
  if (T16 > 32) return 0;
  const int n_jt = c->cfg.d / kMJ;
  const long n_tiles = (long)(c->cfg.V / kNV) * n_jt;
  int grid = c->cfg.max_ctas > 0 ? c->cfg.max_ctas : c->sm_count;
  if (grid > n_tiles) grid = (int)n_tiles;
  for (; grid >= 1; --grid)
    if ((n_jt / gcd_int(grid, n_jt)) * T16 <= kTmemCols - kGhCol0) return grid;
  return 0;
}

cudaError_t tc_launch_update_fused(tts_ctx* c, const StepArgs& a, int grid, cudaStream_t s, int* launches) {
  TcState* st = static_cast<TcState*>(c->tc_state);
  const int V = c->cfg.V, d = c->cfg.d, T = a.T;
  const int T16 = (T + 15) / 16 * 16;
  const bool adam = c->cfg.optimizer == TTS_ADAMW;
  cudaError_t e;
  if ((e = cudaMemsetAsync(a.gh_out, 0, (size_t)T * d * sizeof(float), s)) != cudaSuccess) return e;
  CUtensorMap tm_master, tm_m, tm_v, tm_dl;
  if (make_map_2d(st, &tm_master, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, a.master, d, V, kMJ, kSV,
                  CU_TENSOR_MAP_SWIZZLE_NONE) != CUDA_SUCCESS)
    return cudaErrorInvalidValue;
  tm_m = tm_master;
  tm_v = tm_master;
  if (adam) {
    if (make_map_2d(st, &tm_m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, a.adam_m, d, V, kMJ, kSV,
                    CU_TENSOR_MAP_SWIZZLE_NONE) != CUDA_SUCCESS)
      return cudaErrorInvalidValue;
    if (make_map_2d(st, &tm_v, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, a.adam_v, d, V, kMJ, kSV,
                    CU_TENSOR_MAP_SWIZZLE_NONE) != CUDA_SUCCESS)
      return cudaErrorInvalidValue;
  }
  if (make_map_2d(st, &tm_dl, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, st->dlR, V, (uint64_t)2 * st->P, kKC, T16,
                  CU_TENSOR_MAP_SWIZZLE_128B) != CUDA_SUCCESS)
    return cudaErrorInvalidValue;
  FusedParams p;
  p.master = a.master; p.am = a.adam_m; p.av = a.adam_v;
  p.W_out = static_cast<__nv_bfloat16*>(a.W_out);
  p.gW_debug = a.gW_debug; p.gh = a.gh_out;
  p.V = V; p.d = d; p.T = T; p.T16 = T16; p.P = st->P;
  p.n_jt = d / kMJ;
  p.jt_gcd = gcd_int(grid, p.n_jt);
  p.lr = a.lr; p.b1 = a.beta1; p.b2 = a.beta2; p.eps = a.eps;
  p.decay = 1.f - a.lr * a.wd;
  p.c1 = a.lr * a.inv_bc1;
  p.inv_sqrt_bc2 = a.inv_sqrt_bc2;
  const size_t smem = fused_smem(T16);
  if (adam)
    tc_update_gh_kernel<true><<<grid, kThreads, smem, s>>>(st->tm_hTT, tm_dl, tm_master, tm_m, tm_v, p);
  else
    tc_update_gh_kernel<false><<<grid, kThreads, smem, s>>>(st->tm_hTT, tm_dl, tm_master, tm_m, tm_v, p);
  *launches += 1;
  return cudaGetLastError();
}

}  // namespace tts
