// CUDA-core (fp32 FMA) kernel set of the distillation step: the dtype variant for fp32 parameters
// (BASELINE config 1, "fp32 throughout" has no tcgen05 equivalent) and for shapes outside the
// tensor-core kernels' tile constraints.  Same mathematics as tts_tc.cu (include/tts.h):
//   z = h W^T (a2) -> row statistics (a3, tts_stats.cu) -> dl (a4) -> gh = dl W (a5)
//   -> gW = dl^T h fused with the SGD / AdamW update and the working-copy write-back (a6, a7).
#include "tts_common.cuh"
#include "tts_internal.h"

namespace tts {

// ---------------------------------------------------------------- a2: z[r,v] = sum_j h[r,j] W[v,j]
// CTA: 64 vocab rows x 16 canvas rows, 256 threads; K marched in slabs of 32 through shared memory.
// thread (tv = tid & 63, tr = tid >> 6) accumulates rows 4*tr .. 4*tr+3 of vocab row tv.
template <typename PT>
__global__ void __launch_bounds__(256) simt_logits_kernel(const PT* __restrict__ h, const PT* __restrict__ W, int T,
                                                          int V, int d, float* __restrict__ z, int z_ld) {
  constexpr int KS = 32;
  __shared__ float Ws[64][KS + 1];
  __shared__ float Hs[16][KS];
  const int v0 = blockIdx.x * 64, r0 = blockIdx.y * 16;
  const int tv = threadIdx.x & 63, tr = threadIdx.x >> 6;
  float acc[4] = {0.f, 0.f, 0.f, 0.f};
  for (int k0 = 0; k0 < d; k0 += KS) {
    for (int i = threadIdx.x; i < 64 * KS; i += 256) {
      const int vv = i / KS, kk = i % KS;
      const int v = v0 + vv, k = k0 + kk;
      Ws[vv][kk] = (v < V && k < d) ? ldf(W, (size_t)v * d + k) : 0.f;
    }
    for (int i = threadIdx.x; i < 16 * KS; i += 256) {
      const int rr = i / KS, kk = i % KS;
      const int r = r0 + rr, k = k0 + kk;
      Hs[rr][kk] = (r < T && k < d) ? ldf(h, (size_t)r * d + k) : 0.f;
    }
    __syncthreads();
#pragma unroll
    for (int kk = 0; kk < KS; ++kk) {
      const float w = Ws[tv][kk];
#pragma unroll
      for (int q = 0; q < 4; ++q) acc[q] = fmaf(Hs[4 * tr + q][kk], w, acc[q]);
    }
    __syncthreads();
  }
  const int v = v0 + tv;
  if (v < V) {
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      const int r = r0 + 4 * tr + q;
      if (r < T) z[(size_t)r * z_ld + v] = acc[q];
    }
  }
}

// ---------------------------------------------------------------- a4: dl = coef_r (q - p)
template <bool BF16>
__global__ void __launch_bounds__(256) simt_dl_kernel(const void* __restrict__ teacher, const float* __restrict__ z,
                                                      const float* __restrict__ z_ref, float lam, int V, int z_ld,
                                                      int T_max, const float* __restrict__ row_stats,
                                                      float* __restrict__ dl) {
  const int r = blockIdx.y;
  const float lse_t = row_stats[0 * T_max + r], lse_z = row_stats[1 * T_max + r], coef = row_stats[3 * T_max + r];
  const float lse_ref = row_stats[4 * T_max + r];
  for (int v = blockIdx.x * blockDim.x + threadIdx.x; v < V; v += gridDim.x * blockDim.x) {
    const float t = BF16 ? __bfloat162float(static_cast<const __nv_bfloat16*>(teacher)[(size_t)r * V + v])
                         : static_cast<const float*>(teacher)[(size_t)r * V + v];
    const float q = expf(z[(size_t)r * z_ld + v] - lse_z);
    const float p = expf(t - lse_t);   // t = -inf -> 0
    float g = q - p;
    if (z_ref) g += lam * (q - expf(z_ref[(size_t)r * z_ld + v] - lse_ref));   // + lambda (q - q_ref)
    dl[(size_t)r * V + v] = coef * g;
  }
}

// ---------------------------------------------------------------- a5: gh[r,j] = sum_v dl[r,v] W_in[v,j]
// grid (ceil(d/128), v-splits, ceil(T/16)); thread = one hidden column j, 16 row accumulators.
template <typename PT>
__global__ void __launch_bounds__(128) simt_gh_kernel(const float* __restrict__ dl, const PT* __restrict__ W, int T,
                                                      int V, int d, int vchunk, float* __restrict__ gh) {
  constexpr int VT = 64;
  __shared__ float dls[16][VT];
  const int j = blockIdx.x * 128 + threadIdx.x;
  const int r0 = blockIdx.z * 16;
  const int vbeg = blockIdx.y * vchunk, vend = min(V, vbeg + vchunk);
  float acc[16];
#pragma unroll
  for (int q = 0; q < 16; ++q) acc[q] = 0.f;
  for (int v0 = vbeg; v0 < vend; v0 += VT) {
    for (int i = threadIdx.x; i < 16 * VT; i += 128) {
      const int rr = i / VT, vv = i % VT;
      dls[rr][vv] = (r0 + rr < T && v0 + vv < vend) ? dl[(size_t)(r0 + rr) * V + v0 + vv] : 0.f;
    }
    __syncthreads();
    if (j < d) {
      const int n = min(VT, vend - v0);
      for (int vv = 0; vv < n; ++vv) {
        const float w = ldf(W, (size_t)(v0 + vv) * d + j);
#pragma unroll
        for (int q = 0; q < 16; ++q) acc[q] = fmaf(dls[q][vv], w, acc[q]);
      }
    }
    __syncthreads();
  }
  if (j < d) {
#pragma unroll
    for (int q = 0; q < 16; ++q)
      if (r0 + q < T) atomicAdd(&gh[(size_t)(r0 + q) * d + j], acc[q]);
  }
}

// ---------------------------------------------------------------- a6 + a7: gW = dl^T h fused with the update
// CTA: 8 vocab rows x 128 hidden columns; thread = one column j; canvas rows marched in slabs of 16.
//   SGD   : M <- M - lr g
//   AdamW : M <- M (1 - lr wd); m <- b1 m + (1-b1) g; v <- b2 v + (1-b2) g^2;
//           M <- M - lr (m / bc1) / (sqrt(v / bc2) + eps)                         (R5)
//   W_out = rn_bf16(M) when a master exists, else W_out = M.
template <typename PT, bool ADAM>
__global__ void __launch_bounds__(128) simt_update_kernel(const float* __restrict__ dl, const PT* __restrict__ h,
                                                          int T, int V, int d, const PT* __restrict__ W_in,
                                                          PT* __restrict__ W_out, float* __restrict__ master,
                                                          float* __restrict__ am, float* __restrict__ av,
                                                          float* __restrict__ gW_debug, float lr, float b1, float b2,
                                                          float eps, float wd, const float* __restrict__ step_scalars) {
  const float inv_bc1 = ADAM ? step_scalars[0] : 1.f, inv_sqrt_bc2 = ADAM ? step_scalars[1] : 1.f;
  constexpr int VT = 8;
  __shared__ float dls[16][VT];
  const int j = blockIdx.x * 128 + threadIdx.x;
  const int v0 = blockIdx.y * VT;
  float g[VT];
#pragma unroll
  for (int q = 0; q < VT; ++q) g[q] = 0.f;
  for (int r0 = 0; r0 < T; r0 += 16) {
    __syncthreads();
    if (threadIdx.x < 16 * VT) {
      const int rr = threadIdx.x / VT, vv = threadIdx.x % VT;
      dls[rr][vv] = (r0 + rr < T && v0 + vv < V) ? dl[(size_t)(r0 + rr) * V + v0 + vv] : 0.f;
    }
    __syncthreads();
    if (j < d) {
#pragma unroll
      for (int rr = 0; rr < 16; ++rr) {
        const float hv = (r0 + rr < T) ? ldf(h, (size_t)(r0 + rr) * d + j) : 0.f;
#pragma unroll
        for (int q = 0; q < VT; ++q) g[q] = fmaf(dls[rr][q], hv, g[q]);
      }
    }
  }
  if (j >= d) return;
#pragma unroll
  for (int q = 0; q < VT; ++q) {
    const int v = v0 + q;
    if (v >= V) break;
    const size_t idx = (size_t)v * d + j;
    const float gg = g[q];
    if (gW_debug) gW_debug[idx] = gg;
    float M = master ? master[idx] : ldf(W_in, idx);
    if (ADAM) {
      M *= (1.f - lr * wd);
      const float m = b1 * am[idx] + (1.f - b1) * gg;
      const float vv = b2 * av[idx] + (1.f - b2) * gg * gg;
      am[idx] = m;
      av[idx] = vv;
      M -= lr * (m * inv_bc1) / (sqrtf(vv) * inv_sqrt_bc2 + eps);
    } else {
      M -= lr * gg;
    }
    if (master) master[idx] = M;
    W_out[idx] = from_float<PT>(M);   // float -> bf16 conversion is round-to-nearest-even
  }
}

template <typename PT>
static cudaError_t simt_step_t(tts_ctx* c, const StepArgs& a, cudaStream_t s, int* launches) {
  const int V = c->cfg.V, d = c->cfg.d, T = a.T;
  const PT* h = static_cast<const PT*>(a.h);
  const PT* W_in = static_cast<const PT*>(a.W_in);
  PT* W_out = static_cast<PT*>(a.W_out);
  const bool bf_logits = c->cfg.logits_dtype == TTS_BF16;

  const float* z = z_src(a, c->z);
  cudaError_t e;
  if (a.phase != kPhaseFinish) {
    if (!a.z_given) {
      simt_logits_kernel<PT><<<dim3((V + 63) / 64, (T + 15) / 16), 256, 0, s>>>(h, W_in, T, V, d, z_dst(a, c->z), V);
      *launches += 1;
    }
    prof_mark(c, 0, s);
    if (a.phase == kPhaseBegin) return launch_row_stats_shard(c, a, z, V, a.shard_stats_out, s, launches);
    e = launch_row_stats(c, a, z, V, s, launches);
  } else {
    prof_mark(c, 0, s);
    e = launch_row_stats_merge_shards(c, a, a.shard_stats_all, a.n_shards, s, launches);
  }
  if (e != cudaSuccess) return e;
  prof_mark(c, 1, s);
  {
    const int gx = max(1, min((V + 255) / 256, (4 * c->sm_count + T - 1) / T));
    if (bf_logits)
      simt_dl_kernel<true><<<dim3(gx, T), 256, 0, s>>>(a.teacher, z, a.z_ref, a.lambda, V, V, c->cfg.T_max,
                                                       c->row_stats, c->dl32);
    else
      simt_dl_kernel<false><<<dim3(gx, T), 256, 0, s>>>(a.teacher, z, a.z_ref, a.lambda, V, V, c->cfg.T_max,
                                                        c->row_stats, c->dl32);
    *launches += 1;
  }
  prof_mark(c, 2, s);
  if (a.gh_out) {
    if ((e = cudaMemsetAsync(a.gh_out, 0, (size_t)T * d * sizeof(float), s)) != cudaSuccess) return e;
    const int jb = (d + 127) / 128, rb = (T + 15) / 16;
    int vs = max(1, (4 * c->sm_count) / (jb * rb));
    int vchunk = ((V + vs - 1) / vs + 63) / 64 * 64;
    vs = (V + vchunk - 1) / vchunk;
    simt_gh_kernel<PT><<<dim3(jb, vs, rb), 128, 0, s>>>(c->dl32, W_in, T, V, d, vchunk, a.gh_out);
    *launches += 1;
  }
  prof_mark(c, 3, s);
  dim3 grid((d + 127) / 128, (V + 7) / 8);
  if (c->cfg.optimizer == TTS_ADAMW)
    simt_update_kernel<PT, true><<<grid, 128, 0, s>>>(c->dl32, h, T, V, d, W_in, W_out, a.master, static_cast<float*>(a.adam_m), static_cast<float*>(a.adam_v),
                                                      a.gW_debug, a.lr, a.beta1, a.beta2, a.eps, a.wd,
                                                      a.step_scalars);
  else
    simt_update_kernel<PT, false><<<grid, 128, 0, s>>>(c->dl32, h, T, V, d, W_in, W_out, a.master, nullptr, nullptr,
                                                       a.gW_debug, a.lr, a.beta1, a.beta2, a.eps, a.wd,
                                                       a.step_scalars);
  *launches += 1;
  prof_mark(c, 4, s);
  return cudaGetLastError();
}

cudaError_t simt_step(tts_ctx* c, const StepArgs& a, cudaStream_t s, int* launches) {
  if (c->cfg.param_dtype == TTS_BF16) return simt_step_t<__nv_bfloat16>(c, a, s, launches);
  return simt_step_t<float>(c, a, s, launches);
}

}  // namespace tts
