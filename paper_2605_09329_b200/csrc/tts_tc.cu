// Tensor-path kernels of the distillation step (sm_100a): tcgen05.mma with TMEM accumulators, operands
// and optimiser state staged by TMA, mbarrier pipelines, warp-specialised persistent CTAs.
//
//   prep      (a4)     dl = coef_r (q - p) from z, teacher and the row normalisers; written as the bf16
//                      operands of the two gradient contractions (hi/lo split: dl = hi + lo to 2^-16):
//                      dlT [V, Kp] (vocabulary-major, for gW) and dlR [2, P, V] (row-major planes, for gh)
//   update    (a6+a7)  gW^T tile = h^T . dl   on the tensor cores (accumulator in TMEM, never in HBM),
//                      epilogue = SGD / AdamW on the fp32 master + bf16 working-copy write-back; the
//                      master / m / v tiles arrive by TMA, results leave by coalesced 128-byte stores
//
// Tile orientation of the update: TMEM lane = hidden column j, TMEM column = vocabulary row v, so that a
// warp's 32 lanes touch 32 consecutive floats of one parameter row: every global access is a full line.
#include <new>
#include <string.h>

#include "tts_common.cuh"
#include "tts_tc_ptx.cuh"
#include "tts_tc_state.h"

namespace tts {
namespace {

constexpr int kMJ = 128;         // hidden columns per tile  = MMA M = TMEM lanes
constexpr int kNV = 128;         // vocabulary rows per tile = MMA N = TMEM columns per accumulator
constexpr int kSV = 16;          // vocabulary rows per optimiser-state sub-tile (one pipeline stage)
constexpr int kStages = 6;       // state ring depth
constexpr int kOpStages = 2;     // operand ring depth
constexpr int kOpBytes = kMJ * kKC * 2;              // 16 KB per operand tile (A and B alike: kMJ == kNV)
constexpr int kStateTileBytes = kSV * kMJ * 4;       // 8 KB per tensor per stage
constexpr int kUpdThreads = 384; // warp 0 state TMA, 1 MMA, 2 TMEM alloc, 3 operand TMA, 4-11 epilogue
constexpr int kTmemCols = 2 * kNV;
constexpr int kUpdSmem = 1024 + 2 * kOpStages * kOpBytes + kStages * 3 * kStateTileBytes + 256;

// ------------------------------------------------------------------ a4: operand preparation
// One thread per vocabulary row v (coalesced over v for every canvas row r).
template <bool BF16>
__global__ void __launch_bounds__(256) tc_prep_dl_kernel(const void* __restrict__ teacher, const float* __restrict__ z,
                                                         const float* __restrict__ z_ref, float lam,
                                                         int V, int z_ld, int T, int T16, int Kp, int T_max,
                                                         const float* __restrict__ row_stats,
                                                         __nv_bfloat16* __restrict__ dlT,
                                                         __nv_bfloat16* __restrict__ dlR, int P) {
  extern __shared__ float sh[];   // lse_t[T16], lse_z[T16], coef[T16], lse_ref[T16]
  for (int r = threadIdx.x; r < T16; r += blockDim.x) {
    sh[r] = r < T ? row_stats[0 * T_max + r] : 0.f;
    sh[T16 + r] = r < T ? row_stats[1 * T_max + r] : 0.f;
    sh[2 * T16 + r] = r < T ? row_stats[3 * T_max + r] : 0.f;
    sh[3 * T16 + r] = r < T ? row_stats[4 * T_max + r] : 0.f;
  }
  __syncthreads();
  const int v = blockIdx.x * blockDim.x + threadIdx.x;
  if (v >= V) return;
  uint4* out = dlT ? reinterpret_cast<uint4*>(dlT + (size_t)v * Kp) : nullptr;
  for (int r0 = 0; r0 < T16; r0 += 8) {
    uint32_t hi[4], lo[4];
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      const int r = r0 + u;
      float dl = 0.f;
      if (r < T) {
        const float t = BF16 ? __bfloat162float(static_cast<const __nv_bfloat16*>(teacher)[(size_t)r * V + v])
                             : static_cast<const float*>(teacher)[(size_t)r * V + v];
        const float q = expf(z[(size_t)r * z_ld + v] - sh[T16 + r]);
        const float p = expf(t - sh[r]);   // t = -inf -> 0
        float g = q - p;
        if (z_ref) g += lam * (q - expf(z_ref[(size_t)r * z_ld + v] - sh[3 * T16 + r]));
        dl = sh[2 * T16 + r] * g;
      }
      const __nv_bfloat16 h = __float2bfloat16_rn(dl);
      const __nv_bfloat16 l = __float2bfloat16_rn(dl - __bfloat162float(h));
      if (dlR) {   // row-major planes for the gh contraction (coalesced over v)
        dlR[(size_t)r * V + v] = h;
        dlR[(size_t)(P + r) * V + v] = l;
      }
      const uint32_t hb = __bfloat16_as_ushort(h), lb = __bfloat16_as_ushort(l);
      if (u & 1) { hi[u >> 1] |= hb << 16; lo[u >> 1] |= lb << 16; }
      else       { hi[u >> 1] = hb;        lo[u >> 1] = lb; }
    }
    if (out) {
      out[r0 / 8] = make_uint4(hi[0], hi[1], hi[2], hi[3]);
      out[(T16 + r0) / 8] = make_uint4(lo[0], lo[1], lo[2], lo[3]);
    }
  }
}

// hTT[j, k] = h[k mod T16, j] for k < 2 T16 (rows >= T are zero).  One thread per hidden column j.
__global__ void __launch_bounds__(256) tc_prep_h_kernel(const __nv_bfloat16* __restrict__ h, int d, int T, int T16,
                                                        int Kp, __nv_bfloat16* __restrict__ hTT) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= d) return;
  __nv_bfloat16* row = hTT + (size_t)j * Kp;
  for (int r = 0; r < T16; ++r) {
    const __nv_bfloat16 x = r < T ? h[(size_t)r * d + j] : __float2bfloat16_rn(0.f);
    row[r] = x;
    row[T16 + r] = x;
  }
}

// ------------------------------------------------------------------ a6 + a7: gW on tcgen05 fused with the update
struct UpdParams {
  float* master;
  float* am;
  float* av;
  __nv_bfloat16* W_out;
  float* gW_debug;
  int V, d;
  int k_chunks;       // K chunks of 64 per tile
  int k_steps_last;   // MMA K-steps (of 16) in the last chunk
  float lr, b1, b2, eps, decay, c1, inv_sqrt_bc2;   // decay = 1 - lr wd, c1 = lr / (1 - b1^n)
};

template <bool ADAM>
__global__ void __launch_bounds__(kUpdThreads, 1)
tc_update_kernel(const __grid_constant__ CUtensorMap tm_hTT, const __grid_constant__ CUtensorMap tm_dlT,
                 const __grid_constant__ CUtensorMap tm_master, const __grid_constant__ CUtensorMap tm_m,
                 const __grid_constant__ CUtensorMap tm_v, const UpdParams p) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t* opA = smem;                                  // [kOpStages][16 KB]  hTT tiles (SW128, K-major)
  uint8_t* opB = opA + kOpStages * kOpBytes;            // [kOpStages][16 KB]  dlT tiles
  uint8_t* st = opB + kOpStages * kOpBytes;             // [kStages][3][kSV][128] fp32
  uint64_t* bars = reinterpret_cast<uint64_t*>(st + kStages * 3 * kStateTileBytes);
  uint64_t* op_full = bars;                  // [kOpStages]
  uint64_t* op_empty = op_full + kOpStages;  // [kOpStages]
  uint64_t* acc_full = op_empty + kOpStages; // [2]
  uint64_t* acc_empty = acc_full + 2;        // [2]
  uint64_t* st_full = acc_empty + 2;         // [kStages]
  uint64_t* st_empty = st_full + kStages;    // [kStages]
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(st_empty + kStages);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int n_jt = p.d / kMJ;
  const int n_tiles = (p.V / kNV) * n_jt;
  constexpr int kSubs = kNV / kSV;

  if (warp == 0 && lane == 0) {
    ptx::prefetch_tensormap(&tm_master);
    if (ADAM) { ptx::prefetch_tensormap(&tm_m); ptx::prefetch_tensormap(&tm_v); }
  }
  if (warp == 3 && lane == 0) {
    ptx::prefetch_tensormap(&tm_hTT);
    ptx::prefetch_tensormap(&tm_dlT);
  }
  if (warp == 1 && lane == 0) {
    for (int i = 0; i < kOpStages; ++i) { ptx::mbar_init(&op_full[i], 1); ptx::mbar_init(&op_empty[i], 1); }
    for (int i = 0; i < 2; ++i) { ptx::mbar_init(&acc_full[i], 1); ptx::mbar_init(&acc_empty[i], 8); }
    for (int i = 0; i < kStages; ++i) { ptx::mbar_init(&st_full[i], 1); ptx::mbar_init(&st_empty[i], 4); }
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
    // ===== operand producer: hTT [128 j x 64 k] and dlT [128 v x 64 k] tiles (L2-resident scratch) =====
    if (lane == 0) {
      uint32_t n = 0;
      for (int t = blockIdx.x; t < n_tiles; t += gridDim.x) {
        const int v0 = (t / n_jt) * kNV, j0 = (t % n_jt) * kMJ;
        for (int kc = 0; kc < p.k_chunks; ++kc, ++n) {
          const int s = n % kOpStages;
          ptx::mbar_wait(&op_empty[s], ((n / kOpStages) & 1) ^ 1);
          ptx::mbar_expect_tx(&op_full[s], 2 * kOpBytes);
          ptx::tma_load_2d(opA + s * kOpBytes, &tm_hTT, &op_full[s], kc * kKC, j0);
          ptx::tma_load_2d(opB + s * kOpBytes, &tm_dlT, &op_full[s], kc * kKC, v0);
        }
      }
    }
  } else if (warp == 1) {
    // ===== MMA issuer: acc[j, v] = sum_k hTT[j, k] dlT[v, k]  (M = 128, N = 128, K = 16 per instruction) =====
    if (lane == 0) {
      constexpr uint32_t idesc = ptx::make_idesc_bf16(kMJ, kNV, 0, 0);
      uint32_t n = 0, it = 0;
      for (int t = blockIdx.x; t < n_tiles; t += gridDim.x, ++it) {
        const int ab = it & 1;
        ptx::mbar_wait(&acc_empty[ab], ((it >> 1) & 1) ^ 1);
        ptx::tc_fence_after();
        const uint32_t d_tmem = tmem_base + ab * kNV;
        for (int kc = 0; kc < p.k_chunks; ++kc, ++n) {
          const int s = n % kOpStages;
          ptx::mbar_wait(&op_full[s], (n / kOpStages) & 1);
          ptx::tc_fence_after();
          const int steps = (kc == p.k_chunks - 1) ? p.k_steps_last : kKC / 16;
          const uint32_t a0 = ptx::smem_u32(opA + s * kOpBytes), b0 = ptx::smem_u32(opB + s * kOpBytes);
          for (int ks = 0; ks < steps; ++ks) {
            const uint64_t ad = ptx::make_smem_desc(a0 + ks * 32, 16, 1024, ptx::kSwizzle128B);
            const uint64_t bd = ptx::make_smem_desc(b0 + ks * 32, 16, 1024, ptx::kSwizzle128B);
            ptx::mma_f16_ss(d_tmem, ad, bd, idesc, (kc | ks) != 0);
          }
          ptx::mma_commit(&op_empty[s]);
        }
        ptx::mma_commit(&acc_full[ab]);
      }
    }
  } else if (warp >= 4) {
    // ===== epilogue: 2 groups x 4 warps; group g takes sub-tiles sub % 2 == g; warp quarter q owns lanes 32q.. =====
    const int q = warp & 3, g = (warp - 4) >> 2;
    const int col = q * 32 + lane;
    uint32_t it = 0;
    for (int t = blockIdx.x; t < n_tiles; t += gridDim.x, ++it) {
      const int v0 = (t / n_jt) * kNV, j0 = (t % n_jt) * kMJ;
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
  }
  ptx::tc_fence_before();
  __syncthreads();
  if (warp == 2) {
    ptx::tc_fence_after();
    ptx::tmem_dealloc(tmem_base, kTmemCols);
  }
}

}  // namespace

bool tc_supported(const tts_config& cfg) {
  return cfg.param_dtype == TTS_BF16 && cfg.V % kNV == 0 && cfg.d % kMJ == 0 && cfg.T_max <= 512;
}

cudaError_t tc_init(tts_ctx* c) {
  TcState* st = new (std::nothrow) TcState();
  if (!st) return cudaErrorMemoryAllocation;
  memset(st, 0, sizeof(*st));
  c->tc_state = st;
  const int T16 = c->T_pad_max;
  st->Kp = (2 * T16 + kKC - 1) / kKC * kKC;
  cudaError_t e;
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  if ((e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres)) != cudaSuccess) return e;
  if (!fn || qres != cudaDriverEntryPointSuccess) return cudaErrorNotSupported;
  st->encode = reinterpret_cast<PFN_cuTensorMapEncodeTiled_v12000>(fn);
  const size_t V = c->cfg.V, d = c->cfg.d;
  if ((e = cudaMalloc(&st->dlT, V * st->Kp * 2)) != cudaSuccess) return e;
  if ((e = cudaMalloc(&st->hTT, d * st->Kp * 2)) != cudaSuccess) return e;
  st->P = T16 <= kGhNB ? T16 : (T16 + kGhNB - 1) / kGhNB * kGhNB;
  if ((e = cudaMalloc(&st->dlR, (size_t)2 * st->P * V * 2)) != cudaSuccess) return e;
  if ((e = cudaMemset(st->dlR, 0, (size_t)2 * st->P * V * 2)) != cudaSuccess) return e;
  if ((e = cudaMemset(st->dlT, 0, V * st->Kp * 2)) != cudaSuccess) return e;
  if ((e = cudaMemset(st->hTT, 0, d * st->Kp * 2)) != cudaSuccess) return e;
  if (make_map_2d(st, &st->tm_dlT, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, st->dlT, st->Kp, V, kKC, kNV,
                  CU_TENSOR_MAP_SWIZZLE_128B) != CUDA_SUCCESS)
    return cudaErrorInvalidValue;
  if (make_map_2d(st, &st->tm_hTT, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, st->hTT, st->Kp, d, kKC, kMJ,
                  CU_TENSOR_MAP_SWIZZLE_128B) != CUDA_SUCCESS)
    return cudaErrorInvalidValue;
  if ((e = cudaFuncSetAttribute(tc_update_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kUpdSmem)) !=
      cudaSuccess)
    return e;
  if ((e = cudaFuncSetAttribute(tc_update_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, kUpdSmem)) !=
      cudaSuccess)
    return e;
  if ((e = tc_gemm_init(c)) != cudaSuccess) return e;
  return tc_fused_init(c);
}

void tc_destroy(tts_ctx* c) {
  TcState* st = static_cast<TcState*>(c->tc_state);
  if (!st) return;
  cudaFree(st->dlT);
  cudaFree(st->hTT);
  cudaFree(st->dlR);
  cudaFree(st->hTc);
  cudaFree(st->dlC);
  delete st;
  c->tc_state = nullptr;
}

cudaError_t tc_step(tts_ctx* c, const StepArgs& a, cudaStream_t s, int* launches) {
  TcState* st = static_cast<TcState*>(c->tc_state);
  const int V = c->cfg.V, d = c->cfg.d, T = a.T;
  const int T16 = (T + 15) / 16 * 16;
  const bool adam = c->cfg.optimizer == TTS_ADAMW;
  cudaError_t e;

  // a2: draft logits on tcgen05 (skipped when the caller supplies them), a3: row statistics + loss
  const float* z = z_src(a, c->z);
  if (!a.z_given && (e = tc_launch_logits(c, a, z_dst(a, c->z), s, launches)) != cudaSuccess) return e;
  prof_mark(c, 0, s);
  if ((e = launch_row_stats(c, a, z, V, s, launches)) != cudaSuccess) return e;
  prof_mark(c, 1, s);

  // a4: operands of the gradient contractions
  // one canvas (T <= 16): one fused pass over the optimiser state (tts_tc_fused.cu) with its own pre-tiled operands
  const int fused_grid = tc_fused_grid(c, T16);
  if (fused_grid > 0) {
    if ((e = tc_launch_prep_fused(c, a, z, s, launches)) != cudaSuccess) return e;
    prof_mark(c, 2, s);
    prof_mark(c, 3, s);
    if ((e = tc_launch_update_fused(c, a, fused_grid, s, launches)) != cudaSuccess) return e;
    prof_mark(c, 4, s);
    return cudaGetLastError();
  }
  const size_t sh = 4 * T16 * sizeof(float);
  __nv_bfloat16* dlR = a.gh_out ? st->dlR : nullptr;
  if (c->cfg.logits_dtype == TTS_BF16)
    tc_prep_dl_kernel<true><<<(V + 255) / 256, 256, sh, s>>>(a.teacher, z, a.z_ref, a.lambda, V, V, T, T16, st->Kp, c->cfg.T_max,
                                                               c->row_stats, st->dlT, dlR, st->P);
  else
    tc_prep_dl_kernel<false><<<(V + 255) / 256, 256, sh, s>>>(a.teacher, z, a.z_ref, a.lambda, V, V, T, T16, st->Kp, c->cfg.T_max,
                                                                c->row_stats, st->dlT, dlR, st->P);
  *launches += 1;
  tc_prep_h_kernel<<<(d + 255) / 256, 256, 0, s>>>(static_cast<const __nv_bfloat16*>(a.h), d, T, T16, st->Kp,
                                                   st->hTT);
  *launches += 1;
  prof_mark(c, 2, s);
  // a5: gh on tcgen05 (reads W_in before the update may overwrite an aliased W_out)
  if (a.gh_out) {
    if ((e = tc_launch_gh(c, a, s, launches)) != cudaSuccess) return e;
  }
  prof_mark(c, 3, s);

  // a6 + a7
  CUtensorMap tm_master, tm_m, tm_v;
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
  UpdParams p;
  p.master = a.master; p.am = a.adam_m; p.av = a.adam_v;
  p.W_out = static_cast<__nv_bfloat16*>(a.W_out);
  p.gW_debug = a.gW_debug;
  p.V = V; p.d = d;
  const int K = 2 * T16;
  p.k_chunks = (K + kKC - 1) / kKC;
  p.k_steps_last = (K - (p.k_chunks - 1) * kKC) / 16;
  p.lr = a.lr; p.b1 = a.beta1; p.b2 = a.beta2; p.eps = a.eps;
  p.decay = 1.f - a.lr * a.wd;
  p.c1 = a.lr * a.inv_bc1;
  p.inv_sqrt_bc2 = a.inv_sqrt_bc2;
  const int n_tiles = (V / kNV) * (d / kMJ);
  int grid = c->cfg.max_ctas > 0 ? c->cfg.max_ctas : c->sm_count;
  if (grid > n_tiles) grid = n_tiles;
  if (adam)
    tc_update_kernel<true><<<grid, kUpdThreads, kUpdSmem, s>>>(st->tm_hTT, st->tm_dlT, tm_master, tm_m, tm_v, p);
  else
    tc_update_kernel<false><<<grid, kUpdThreads, kUpdSmem, s>>>(st->tm_hTT, st->tm_dlT, tm_master, tm_m, tm_v, p);
  *launches += 1;
  prof_mark(c, 4, s);
  return cudaGetLastError();
}

}  // namespace tts
