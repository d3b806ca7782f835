// a1: greedy accepted-prefix mask (include/tts.h tts_accept_mask; Alg. 1 "Accept"
// PAPER.md:152, greedy rule per north_star (4)).  Integer / compare only: bit-exact.
//
// Kernel 1 (argmax_partial): grid (splits, T).  Each CTA sweeps a contiguous slice of one teacher row
//   with 128-bit loads and keeps (max value, lowest index) per thread, then reduces with warp
//   shuffles.  Kernel 2 (mask_finalize): one CTA merges the splits per row, compares with the draft
//   tokens and runs the per-segment prefix-AND.
#include "tts_common.cuh"
#include "tts_internal.h"

namespace tts {

struct ArgPair {
  float v;
  int i;
};

// larger value wins; equal values: lower index wins (R11).  (-inf, INT_MAX) is the identity.
__device__ __forceinline__ ArgPair arg_better(ArgPair a, ArgPair b) {
  return (b.v > a.v || (b.v == a.v && b.i < a.i)) ? b : a;
}

__device__ __forceinline__ ArgPair warp_argmax(ArgPair p) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    ArgPair q;
    q.v = __shfl_xor_sync(0xffffffffu, p.v, o);
    q.i = __shfl_xor_sync(0xffffffffu, p.i, o);
    p = arg_better(p, q);
  }
  return p;
}

template <bool BF16>
__global__ void __launch_bounds__(256) argmax_partial_kernel(const void* __restrict__ teacher, int V, int chunk,
                                                             float* __restrict__ out_val, int* __restrict__ out_idx) {
  const int r = blockIdx.y, sp = blockIdx.x;
  const int v0 = sp * chunk;
  const int v1 = min(V, v0 + chunk);
  ArgPair best{-CUDART_INF_F, 0x7fffffff};
  if (BF16) {
    const __nv_bfloat16* row = static_cast<const __nv_bfloat16*>(teacher) + (size_t)r * V;
    // chunk is a multiple of 8 and rows start 16-byte aligned (V * 2 % 16 == 0)
    const int nvec = (v1 - v0) / 8;
    const uint4* p = reinterpret_cast<const uint4*>(row + v0);
    for (int i = threadIdx.x; i < nvec; i += blockDim.x) {
      const uint4 q = __ldg(p + i);
      float f[8];
      unpack_bf16x8(q, f);
      const int base = v0 + i * 8;
#pragma unroll
      for (int k = 0; k < 8; ++k)
        if (f[k] > best.v || (f[k] == best.v && base + k < best.i)) { best.v = f[k]; best.i = base + k; }
    }
    for (int v = v0 + nvec * 8 + threadIdx.x; v < v1; v += blockDim.x) {
      const float f = __bfloat162float(row[v]);
      if (f > best.v || (f == best.v && v < best.i)) { best.v = f; best.i = v; }
    }
  } else {
    const float* row = static_cast<const float*>(teacher) + (size_t)r * V;
    const int nvec = (v1 - v0) / 4;
    const float4* p = reinterpret_cast<const float4*>(row + v0);
    for (int i = threadIdx.x; i < nvec; i += blockDim.x) {
      const float4 q = __ldg(p + i);
      const float f[4] = {q.x, q.y, q.z, q.w};
      const int base = v0 + i * 4;
#pragma unroll
      for (int k = 0; k < 4; ++k)
        if (f[k] > best.v || (f[k] == best.v && base + k < best.i)) { best.v = f[k]; best.i = base + k; }
    }
    for (int v = v0 + nvec * 4 + threadIdx.x; v < v1; v += blockDim.x) {
      const float f = row[v];
      if (f > best.v || (f == best.v && v < best.i)) { best.v = f; best.i = v; }
    }
  }
  __shared__ float sv[8];
  __shared__ int si[8];
  best = warp_argmax(best);
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  if (lane == 0) { sv[w] = best.v; si[w] = best.i; }
  __syncthreads();
  if (w == 0) {
    ArgPair p{-CUDART_INF_F, 0x7fffffff};
    if (lane < (blockDim.x >> 5)) { p.v = sv[lane]; p.i = si[lane]; }
    p = warp_argmax(p);
    if (lane == 0) {
      out_val[(size_t)r * gridDim.x + sp] = p.v;
      out_idx[(size_t)r * gridDim.x + sp] = p.i;
    }
  }
}

// the splits of one row merged into this shard's (max value, GLOBAL index = local index + v_offset)
__global__ void __launch_bounds__(256) argmax_reduce_kernel(const float* __restrict__ pv, const int* __restrict__ pi,
                                                            int splits, int T, int v_offset, float* __restrict__ val,
                                                            int32_t* __restrict__ idx) {
  for (int r = blockIdx.x * blockDim.x + threadIdx.x; r < T; r += gridDim.x * blockDim.x) {
    ArgPair best{-CUDART_INF_F, 0x7fffffff};
    for (int s = 0; s < splits; ++s) best = arg_better(best, ArgPair{pv[(size_t)r * splits + s], pi[(size_t)r * splits + s]});
    val[r] = best.v;
    idx[r] = best.i == 0x7fffffff ? 0x7fffffff : best.i + v_offset;
  }
}

// pv / pi hold `splits` candidates per row: element (r, s) at r * row_stride + s * split_stride
__global__ void __launch_bounds__(256) mask_finalize_kernel(const float* __restrict__ pv, const int* __restrict__ pi,
                                                            int splits, long row_stride, long split_stride,
                                                            const int32_t* __restrict__ tok, int T,
                                                            int seg_len, uint8_t* __restrict__ mask,
                                                            int32_t* __restrict__ tau, int32_t* __restrict__ am_out,
                                                            int32_t* __restrict__ am_tmp) {
  for (int r = threadIdx.x; r < T; r += blockDim.x) {
    ArgPair best{-CUDART_INF_F, 0x7fffffff};
    for (int s = 0; s < splits; ++s)
      best = arg_better(best, ArgPair{pv[r * row_stride + s * split_stride], pi[r * row_stride + s * split_stride]});
    // a row of only -inf (or an empty slice everywhere) resolves to index 0, like the lowest-index rule
    const int am = best.i == 0x7fffffff ? 0 : best.i;
    am_tmp[r] = am;
    if (am_out) am_out[r] = am;
  }
  __syncthreads();
  const int S = T / seg_len;
  for (int s = threadIdx.x; s < S; s += blockDim.x) {
    bool alive = true;   // "if x_{t+k} rejected then break"
    int n = 0;
    for (int k = 0; k < seg_len; ++k) {
      const int r = s * seg_len + k;
      alive = alive && (am_tmp[r] == tok[r]);
      mask[r] = alive ? 1 : 0;
      n += alive ? 1 : 0;
    }
    tau[s] = n;
  }
}

static int launch_argmax_partial(tts_ctx* c, const void* teacher, int T, cudaStream_t s) {
  const int V = c->cfg.V;
  const bool bf = c->cfg.logits_dtype == TTS_BF16;
  // enough CTAs to fill the machine at small T, at most kArgSplitsMax per row, slices a multiple of 8
  int splits = (2 * c->sm_count + T - 1) / T;
  splits = max(1, min(splits, kArgSplitsMax));
  int chunk = (V + splits - 1) / splits;
  chunk = (chunk + 7) / 8 * 8;
  splits = (V + chunk - 1) / chunk;
  dim3 grid(splits, T);
  if (bf)
    argmax_partial_kernel<true><<<grid, 256, 0, s>>>(teacher, V, chunk, c->arg_val, c->arg_idx);
  else
    argmax_partial_kernel<false><<<grid, 256, 0, s>>>(teacher, V, chunk, c->arg_val, c->arg_idx);
  return splits;
}

cudaError_t launch_accept_mask(tts_ctx* c, const void* teacher, const int32_t* tok, int T, uint8_t* mask,
                               int32_t* tau, int32_t* am_out, cudaStream_t s, int* launches) {
  const int splits = launch_argmax_partial(c, teacher, T, s);
  mask_finalize_kernel<<<1, 256, 0, s>>>(c->arg_val, c->arg_idx, splits, splits, 1, tok, T, c->cfg.seg_len, mask, tau,
                                         am_out, c->argmax_tmp);
  *launches += 2;
  return cudaGetLastError();
}

// shard: (max, global index) of this shard's columns per row
cudaError_t launch_shard_argmax(tts_ctx* c, const void* teacher, int T, int v_offset, float* val, int32_t* idx,
                                cudaStream_t s, int* launches) {
  const int splits = launch_argmax_partial(c, teacher, T, s);
  argmax_reduce_kernel<<<(T + 255) / 256, 256, 0, s>>>(c->arg_val, c->arg_idx, splits, T, v_offset, val, idx);
  *launches += 2;
  return cudaGetLastError();
}

// shard: candidates of all shards [n_shards, T] -> mask, tau (lowest global index wins ties, as on one GPU)
cudaError_t launch_shard_mask(tts_ctx* c, const float* val_all, const int32_t* idx_all, int n_shards,
                              const int32_t* tok, int T, uint8_t* mask, int32_t* tau, int32_t* am_out, cudaStream_t s,
                              int* launches) {
  mask_finalize_kernel<<<1, 256, 0, s>>>(val_all, idx_all, n_shards, 1, T, tok, T, c->cfg.seg_len, mask, tau, am_out,
                                         c->argmax_tmp);
  *launches += 1;
  return cudaGetLastError();
}

}  // namespace tts
