// a3: the vocab-wide sweep.  One pass over a teacher row t and the draft-logit row z keeps the
// online statistics (m_t, s_t, a, m_z, s_z):
//     m_t = max t,  s_t = sum e^{t-m_t},  a = sum e^{t-m_t} (t - z),  m_z = max z,  s_z = sum e^{z-m_z}
// so that  lse_t = m_t + log s_t,  lse_z = m_z + log s_z,
//          KL_r  = sum_v p (log p - log q) = a / s_t - lse_t + lse_z
// without ever storing a [T,V] probability tensor.  Partial tuples from different CTAs merge
// associatively (rescale to the larger maximum).  The merge kernel also forms the row weights
// omega_r (mask_mode per DESIGN.md R2), coef_r = loss_scale * omega_r and
// loss = loss_scale * sum_r omega_r KL_r  (a sum), and advances Adam's step count.
#include "tts_common.cuh"
#include "tts_internal.h"

namespace tts {

struct RowStat {
  float mt, st, a, mz, sz;
  float mr, sr, b;   // reference distribution q_ref = softmax(z_ref): max, sum e^{zr-mr}, sum e^{zr-mr} (zr - z)
};

__device__ __forceinline__ void stat_init(RowStat& s) {
  s.mt = -CUDART_INF_F; s.st = 0.f; s.a = 0.f; s.mz = -CUDART_INF_F; s.sz = 0.f;
  s.mr = -CUDART_INF_F; s.sr = 0.f; s.b = 0.f;
}

// one element; teacher entries equal to -inf have p = 0 and are dropped (0 log 0 := 0)
__device__ __forceinline__ void stat_push(RowStat& s, float t, float z) {
  if (t != -CUDART_INF_F) {
    const float e = expf(-fabsf(t - s.mt));   // s.mt = -inf  ->  e = 0
    if (t > s.mt) { s.st = s.st * e + 1.f; s.a = s.a * e + (t - z); s.mt = t; }
    else          { s.st += e;             s.a += e * (t - z); }
  }
  const float e = expf(-fabsf(z - s.mz));
  if (z > s.mz) { s.sz = s.sz * e + 1.f; s.mz = z; }
  else          { s.sz += e; }
}
// the lambda term's statistics: K~L(q_ref || q)_r = b / s_ref - lse_ref + lse_z
__device__ __forceinline__ void stat_push_ref(RowStat& s, float zr, float z) {
  const float e = expf(-fabsf(zr - s.mr));
  if (zr > s.mr) { s.sr = s.sr * e + 1.f; s.b = s.b * e + (zr - z); s.mr = zr; }
  else           { s.sr += e;             s.b += e * (zr - z); }
}

// N elements at once: one rescale of the running sums to the new maxima, then one exp per element (the per-element
// form above costs a compare / select chain and an exp of the correction per element).  Same quantities.
template <int N>
__device__ __forceinline__ void stat_push_vec(RowStat& s, const float (&t)[N], const float (&z)[N]) {
  float mt = s.mt, mz = s.mz;
#pragma unroll
  for (int k = 0; k < N; ++k) { mt = fmaxf(mt, t[k]); mz = fmaxf(mz, z[k]); }
  if (mt != -CUDART_INF_F) {          // all teacher entries so far -inf: nothing to add (p = 0)
    const float c = s.mt == -CUDART_INF_F ? 0.f : expf(s.mt - mt);
    float st = s.st * c, a = s.a * c;
#pragma unroll
    for (int k = 0; k < N; ++k) {
      const float e = expf(t[k] - mt);   // t = -inf -> 0
      st += e;
      a += t[k] == -CUDART_INF_F ? 0.f : e * (t[k] - z[k]);
    }
    s.st = st; s.a = a; s.mt = mt;
  }
  const float cz = s.mz == -CUDART_INF_F ? 0.f : expf(s.mz - mz);
  float sz = s.sz * cz;
#pragma unroll
  for (int k = 0; k < N; ++k) sz += expf(z[k] - mz);
  s.sz = sz; s.mz = mz;
}

__device__ __forceinline__ RowStat stat_merge(const RowStat& x, const RowStat& y) {
  RowStat o;
  o.mt = fmaxf(x.mt, y.mt);
  const float ex = (x.mt == -CUDART_INF_F) ? 0.f : expf(x.mt - o.mt);
  const float ey = (y.mt == -CUDART_INF_F) ? 0.f : expf(y.mt - o.mt);
  o.st = x.st * ex + y.st * ey;
  o.a = x.a * ex + y.a * ey;
  o.mz = fmaxf(x.mz, y.mz);
  const float fx = (x.mz == -CUDART_INF_F) ? 0.f : expf(x.mz - o.mz);
  const float fy = (y.mz == -CUDART_INF_F) ? 0.f : expf(y.mz - o.mz);
  o.sz = x.sz * fx + y.sz * fy;
  o.mr = fmaxf(x.mr, y.mr);
  const float gx = (x.mr == -CUDART_INF_F) ? 0.f : expf(x.mr - o.mr);
  const float gy = (y.mr == -CUDART_INF_F) ? 0.f : expf(y.mr - o.mr);
  o.sr = x.sr * gx + y.sr * gy;
  o.b = x.b * gx + y.b * gy;
  return o;
}

__device__ __forceinline__ RowStat warp_stat(RowStat s) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    RowStat q;
    q.mt = __shfl_xor_sync(0xffffffffu, s.mt, o);
    q.st = __shfl_xor_sync(0xffffffffu, s.st, o);
    q.a = __shfl_xor_sync(0xffffffffu, s.a, o);
    q.mz = __shfl_xor_sync(0xffffffffu, s.mz, o);
    q.sz = __shfl_xor_sync(0xffffffffu, s.sz, o);
    q.mr = __shfl_xor_sync(0xffffffffu, s.mr, o);
    q.sr = __shfl_xor_sync(0xffffffffu, s.sr, o);
    q.b = __shfl_xor_sync(0xffffffffu, s.b, o);
    s = stat_merge(s, q);
  }
  return s;
}

// grid (splits, T), 256 threads.  128-bit loads of the teacher (8 bf16 / 4 fp32) and of z (2 x / 1 x float4).
template <bool BF16>
__global__ void __launch_bounds__(256) row_stats_partial_kernel(const void* __restrict__ teacher,
                                                                const float* __restrict__ z,
                                                                const float* __restrict__ z_ref, int V, int z_ld,
                                                                int chunk, float* __restrict__ part) {
  const int r = blockIdx.y, sp = blockIdx.x;
  const int v0 = sp * chunk, v1 = min(V, v0 + chunk);
  const float* zr = z + (size_t)r * z_ld;
  const float* zf = z_ref ? z_ref + (size_t)r * z_ld : nullptr;
  RowStat s;
  stat_init(s);
  if (BF16) {
    const __nv_bfloat16* row = static_cast<const __nv_bfloat16*>(teacher) + (size_t)r * V;
    const int nvec = (v1 - v0) / 8;
    const uint4* pt = reinterpret_cast<const uint4*>(row + v0);
    const float4* pz = reinterpret_cast<const float4*>(zr + v0);
    for (int i = threadIdx.x; i < nvec; i += blockDim.x) {
      const uint4 q = __ldg(pt + i);
      const float4 z0 = __ldg(pz + 2 * i), z1 = __ldg(pz + 2 * i + 1);
      float f[8];
      unpack_bf16x8(q, f);
      const float zz[8] = {z0.x, z0.y, z0.z, z0.w, z1.x, z1.y, z1.z, z1.w};
      stat_push_vec<8>(s, f, zz);
      if (zf) {
        const float4 r0 = __ldg(reinterpret_cast<const float4*>(zf + v0) + 2 * i);
        const float4 r1 = __ldg(reinterpret_cast<const float4*>(zf + v0) + 2 * i + 1);
        const float rr[8] = {r0.x, r0.y, r0.z, r0.w, r1.x, r1.y, r1.z, r1.w};
#pragma unroll
        for (int k = 0; k < 8; ++k) stat_push_ref(s, rr[k], zz[k]);
      }
    }
    for (int v = v0 + nvec * 8 + threadIdx.x; v < v1; v += blockDim.x) {
      stat_push(s, __bfloat162float(row[v]), zr[v]);
      if (zf) stat_push_ref(s, zf[v], zr[v]);
    }
  } else {
    const float* row = static_cast<const float*>(teacher) + (size_t)r * V;
    const int nvec = (v1 - v0) / 4;
    const float4* pt = reinterpret_cast<const float4*>(row + v0);
    const float4* pz = reinterpret_cast<const float4*>(zr + v0);
    for (int i = threadIdx.x; i < nvec; i += blockDim.x) {
      const float4 q = __ldg(pt + i);
      const float4 z0 = __ldg(pz + i);
      {
        const float tq[4] = {q.x, q.y, q.z, q.w}, zq[4] = {z0.x, z0.y, z0.z, z0.w};
        stat_push_vec<4>(s, tq, zq);
      }
      if (zf) {
        const float4 r0 = __ldg(reinterpret_cast<const float4*>(zf + v0) + i);
        stat_push_ref(s, r0.x, z0.x); stat_push_ref(s, r0.y, z0.y); stat_push_ref(s, r0.z, z0.z);
        stat_push_ref(s, r0.w, z0.w);
      }
    }
    for (int v = v0 + nvec * 4 + threadIdx.x; v < v1; v += blockDim.x) {
      stat_push(s, row[v], zr[v]);
      if (zf) stat_push_ref(s, zf[v], zr[v]);
    }
  }
  __shared__ RowStat sh[8];
  s = warp_stat(s);
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  if (lane == 0) sh[w] = s;
  __syncthreads();
  if (w == 0) {
    RowStat q;
    stat_init(q);
    if (lane < (blockDim.x >> 5)) q = sh[lane];
    q = warp_stat(q);
    if (lane == 0) {
      float* o = part + ((size_t)r * gridDim.x + sp) * kStatFields;
      o[0] = q.mt; o[1] = q.st; o[2] = q.a; o[3] = q.mz; o[4] = q.sz; o[5] = q.mr; o[6] = q.sr; o[7] = q.b;
    }
  }
}

// A warp merges one row with its lanes spread over the row's tuples (8 rows per CTA); with few tuples and many rows
// (several canvases from the unfused sweep; vocabulary shards) a THREAD merges one row (256 rows per CTA).
// row_stats planes ([kRowStatFields][T_max]): 0 = lse_t, 1 = lse_z, 2 = kl, 3 = coef (= loss_scale * omega), 4 = lse_ref.
// The maxima are exact in fp32; the rescaled sums and the final a / s_t - lse_t + lse_z (a difference of numbers
// ~10 for a result that can be ~0.01) are formed in double.  With z_ref (has_ref) the loss gains
// lambda * sum_r omega_r K~L(q_ref || q)_r.
// The loss is a sum over rows in a FIXED order: every CTA leaves omega_r (KL_r + lambda KL_ref,r) per row, and the CTA
// that finishes last (a ticket) adds them up, advances Adam's count and resets the ticket for the next launch.
constexpr int kMergeThreads = 256;
__global__ void __launch_bounds__(kMergeThreads) row_stats_merge_kernel(
    const float* __restrict__ part, int splits, long row_stride, long split_stride, int T, int T_max, int seg_len,
    int mask_mode, const float* __restrict__ pos_weight, const uint8_t* __restrict__ mask, float loss_scale, int has_ref,
    float lambda, float* __restrict__ row_stats, float* __restrict__ kl_rows_out, float* __restrict__ loss_out,
    unsigned long long* __restrict__ step_count, float* __restrict__ step_scalars, float b1, float b2,
    int* __restrict__ dev_status, double* __restrict__ row_loss, unsigned int* __restrict__ ticket, int thread_rows) {
  __shared__ double red[kMergeThreads / 32];
  __shared__ int is_last;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, n_warps = kMergeThreads >> 5;
  const int r = thread_rows ? blockIdx.x * kMergeThreads + (int)threadIdx.x : blockIdx.x * n_warps + warp;
  const int l_first = thread_rows ? 0 : lane, l_step = thread_rows ? 1 : 32;
  if (r < T) {
    const float* pr = part + (size_t)r * row_stride;
    float mt = -CUDART_INF_F, mz = -CUDART_INF_F, mr = -CUDART_INF_F;
    for (int s = l_first; s < splits; s += l_step) {
      const float* p = pr + s * split_stride;
      mt = fmaxf(mt, p[0]); mz = fmaxf(mz, p[3]); mr = fmaxf(mr, p[5]);
    }
    if (!thread_rows) { mt = warp_max(mt); mz = warp_max(mz); mr = warp_max(mr); }
    double st = 0.0, a = 0.0, sz = 0.0, sr = 0.0, b = 0.0;
    for (int s = l_first; s < splits; s += l_step) {
      const float* p = pr + s * split_stride;
      // rescale factors in fp32 (expf, ~1 ulp: 6e-8 relative per term, against a loss tolerance of 1e-3), sums in double
      if (p[0] != -CUDART_INF_F) {
        const double e = (double)expf(p[0] - mt);
        st += (double)p[1] * e; a += (double)p[2] * e;
      }
      if (p[3] != -CUDART_INF_F) sz += (double)p[4] * (double)expf(p[3] - mz);
      if (has_ref && p[5] != -CUDART_INF_F) {
        const double e = (double)expf(p[5] - mr);
        sr += (double)p[6] * e; b += (double)p[7] * e;
      }
    }
    if (!thread_rows) {
      st = warp_sum(st); a = warp_sum(a); sz = warp_sum(sz);
      if (has_ref) { sr = warp_sum(sr); b = warp_sum(b); }
    }
    if (thread_rows || lane == 0) {
      const double lse_t = (double)mt + log(st), lse_z = (double)mz + log(sz);
      const double kl = a / st - lse_t + lse_z;
      double lse_ref = 0.0, kl_ref = 0.0;
      if (has_ref) {
        lse_ref = (double)mr + log(sr);
        kl_ref = b / sr - lse_ref + lse_z;
      }
      // omega_r = w_k * mask factor (R2)
      double f = 1.0;
      if (mask_mode != TTS_ROWS_ALL) {
        f = mask[r] ? 1.0 : 0.0;
        if (mask_mode == TTS_ROWS_ACCEPTED_PLUS_ONE && !mask[r]) {
          const int k = r % seg_len;
          if (k == 0 || mask[r - 1]) f = 1.0;   // the first rejected row of the segment
        }
      }
      const double omega = (double)pos_weight[r] * f;
      row_stats[0 * T_max + r] = (float)lse_t;
      row_stats[1 * T_max + r] = (float)lse_z;
      row_stats[2 * T_max + r] = (float)kl;
      row_stats[3 * T_max + r] = (float)((double)loss_scale * omega);
      row_stats[4 * T_max + r] = (float)lse_ref;
      if (kl_rows_out) kl_rows_out[r] = (float)kl;
      row_loss[r] = omega * (kl + (double)lambda * kl_ref);
    }
  }
  __threadfence();
  __syncthreads();
  if (threadIdx.x == 0) is_last = atomicAdd(ticket, 1u) == gridDim.x - 1;
  __syncthreads();
  if (!is_last) return;
  __threadfence();
  double local = 0.0;
  for (int q = threadIdx.x; q < T; q += kMergeThreads) local += __ldcg(row_loss + q);   // fixed order per thread
  local = warp_sum(local);                                                              // fixed shuffle tree
  if (lane == 0) red[warp] = local;
  __syncthreads();
  if (threadIdx.x == 0) {
    double sum = 0.0;
    for (int w = 0; w < n_warps; ++w) sum += red[w];   // fixed order
    const float loss = (float)((double)loss_scale * sum);
    loss_out[0] = loss;
    if (!isfinite(loss)) atomicOr(dev_status, TTS_DEV_NONFINITE_LOSS);
    // Adam's count and bias corrections live on the device (a replayed CUDA graph of the step keeps counting):
    // n <- n + 1, {1 / (1 - b1^n), 1 / sqrt(1 - b2^n)} in double, read by the update kernel later in the stream
    const unsigned long long n = *step_count + 1ull;
    *step_count = n;
    step_scalars[0] = (float)(1.0 / (1.0 - pow((double)b1, (double)n)));
    step_scalars[1] = (float)(1.0 / sqrt(1.0 - pow((double)b2, (double)n)));
    *ticket = 0u;
  }
}

// the splits of one row merged into ONE tuple (m_t, s_t, a, m_z, s_z, m_ref, s_ref, b) instead of the
// normalisers: what a vocabulary shard hands to the other shards.  Same arithmetic as the merge kernel (maxima exact,
// rescaled sums in double), so merging the shards' tuples equals merging all their splits up to fp32 rounding of
// the eight numbers.  One warp per row.
__global__ void __launch_bounds__(1024) row_stats_reduce_kernel(const float* __restrict__ part, int splits, int T,
                                                                float* __restrict__ out) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, n_warps = blockDim.x >> 5;
  for (int r = warp; r < T; r += n_warps) {
    const float* pr = part + (size_t)r * splits * kStatFields;
    float mt = -CUDART_INF_F, mz = -CUDART_INF_F, mr = -CUDART_INF_F;
    for (int s = lane; s < splits; s += 32) {
      const float* p = pr + s * kStatFields;
      mt = fmaxf(mt, p[0]); mz = fmaxf(mz, p[3]); mr = fmaxf(mr, p[5]);
    }
    mt = warp_max(mt); mz = warp_max(mz); mr = warp_max(mr);
    double st = 0.0, a = 0.0, sz = 0.0, sr = 0.0, b = 0.0;
    for (int s = lane; s < splits; s += 32) {
      const float* p = pr + s * kStatFields;
      if (p[0] != -CUDART_INF_F) {
        const double e = exp((double)p[0] - (double)mt);
        st += (double)p[1] * e; a += (double)p[2] * e;
      }
      if (p[3] != -CUDART_INF_F) sz += (double)p[4] * exp((double)p[3] - (double)mz);
      if (p[5] != -CUDART_INF_F) {
        const double e = exp((double)p[5] - (double)mr);
        sr += (double)p[6] * e; b += (double)p[7] * e;
      }
    }
    st = warp_sum(st); a = warp_sum(a); sz = warp_sum(sz); sr = warp_sum(sr); b = warp_sum(b);
    if (lane == 0) {
      float* o = out + (size_t)r * kStatFields;
      o[0] = mt; o[1] = (float)st; o[2] = (float)a; o[3] = mz; o[4] = (float)sz; o[5] = mr; o[6] = (float)sr; o[7] = (float)b;
    }
  }
}

// Fix-up sweep of the fused a2 + a3 path: block (k, r) takes the 128 columns [col0[k], col0[k] + 128) of canvas row r
// (tiles whose z was completed by fp32 RED from two CTAs, so that neither epilogue saw whole logits) and writes the
// row's tuple slot0 + k.  One element per thread, shuffle merge.
struct FixTiles { int col0[kStatFixMax]; };
template <bool BF16>
__global__ void __launch_bounds__(128) row_stats_tiles_kernel(const void* __restrict__ teacher,
                                                              const float* __restrict__ z, int V, int z_ld,
                                                              const FixTiles tiles, int slot0, int splits,
                                                              float* __restrict__ part) {
  const int r = blockIdx.y, v = tiles.col0[blockIdx.x] + threadIdx.x;
  RowStat s;
  stat_init(s);
  const float t = BF16 ? __bfloat162float(static_cast<const __nv_bfloat16*>(teacher)[(size_t)r * V + v])
                       : static_cast<const float*>(teacher)[(size_t)r * V + v];
  stat_push(s, t, z[(size_t)r * z_ld + v]);
  __shared__ RowStat sh[4];
  s = warp_stat(s);
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = s;
  __syncthreads();
  if (threadIdx.x == 0) {
    RowStat q = stat_merge(stat_merge(sh[0], sh[1]), stat_merge(sh[2], sh[3]));
    float* o = part + ((size_t)r * splits + slot0 + blockIdx.x) * kStatFields;
    o[0] = q.mt; o[1] = q.st; o[2] = q.a; o[3] = q.mz; o[4] = q.sz; o[5] = -CUDART_INF_F; o[6] = 0.f; o[7] = 0.f;
  }
}

static int launch_partial(tts_ctx* c, const StepArgs& a, const float* z, int z_ld, cudaStream_t s) {
  const int V = c->cfg.V, T = a.T;
  int splits = (2 * c->sm_count + T - 1) / T;
  splits = max(1, min(splits, kStatSplitsMax));
  int chunk = (V + splits - 1) / splits;
  chunk = (chunk + 7) / 8 * 8;
  splits = (V + chunk - 1) / chunk;
  dim3 grid(splits, T);
  if (c->cfg.logits_dtype == TTS_BF16)
    row_stats_partial_kernel<true><<<grid, 256, 0, s>>>(a.teacher, z, a.z_ref, V, z_ld, chunk, c->stat_part);
  else
    row_stats_partial_kernel<false><<<grid, 256, 0, s>>>(a.teacher, z, a.z_ref, V, z_ld, chunk, c->stat_part);
  return splits;
}

static void launch_merge(tts_ctx* c, const StepArgs& a, const float* part, int splits, long row_stride,
                         long split_stride, cudaStream_t s) {
  const int T = a.T;
  const int thread_rows = splits <= 8 && T > kMergeThreads / 32;
  const int rows_per_cta = thread_rows ? kMergeThreads : kMergeThreads / 32;
  row_stats_merge_kernel<<<(T + rows_per_cta - 1) / rows_per_cta, kMergeThreads, 0, s>>>(
      part, splits, row_stride, split_stride, T, c->cfg.T_max, c->cfg.seg_len, c->cfg.mask_mode, a.pos_weight, a.mask,
      a.loss_scale, a.z_ref != nullptr, a.lambda, c->row_stats, a.kl_rows_out, a.loss_out, c->step_count_dev,
      c->step_scalars, c->cfg.beta1, c->cfg.beta2, c->dev_status, c->row_loss, c->merge_ticket, thread_rows);
}

cudaError_t launch_row_stats(tts_ctx* c, const StepArgs& a, const float* z, int z_ld, cudaStream_t s, int* launches) {
  const int splits = launch_partial(c, a, z, z_ld, s);
  launch_merge(c, a, c->stat_part, splits, (long)splits * kStatFields, kStatFields, s);
  *launches += 2;
  return cudaGetLastError();
}

// shard: this shard's sweep, one tuple per row into stats_out [T, kStatFields]
cudaError_t launch_row_stats_shard(tts_ctx* c, const StepArgs& a, const float* z, int z_ld, float* stats_out,
                                   cudaStream_t s, int* launches) {
  const int splits = launch_partial(c, a, z, z_ld, s);
  row_stats_reduce_kernel<<<1, a.T >= 32 ? 1024 : 32 * a.T, 0, s>>>(c->stat_part, splits, a.T, stats_out);
  *launches += 2;
  return cudaGetLastError();
}

cudaError_t launch_row_stats_tiles(tts_ctx* c, const StepArgs& a, const float* z, int z_ld, const int* col0, int n,
                                   int slot0, int splits, cudaStream_t s, int* launches) {
  FixTiles ft;
  for (int i = 0; i < n; ++i) ft.col0[i] = col0[i];
  const dim3 grid(n, a.T);
  if (c->cfg.logits_dtype == TTS_BF16)
    row_stats_tiles_kernel<true><<<grid, 128, 0, s>>>(a.teacher, z, c->cfg.V, z_ld, ft, slot0, splits, c->stat_part);
  else
    row_stats_tiles_kernel<false><<<grid, 128, 0, s>>>(a.teacher, z, c->cfg.V, z_ld, ft, slot0, splits, c->stat_part);
  *launches += 1;
  return cudaGetLastError();
}

cudaError_t launch_row_stats_finish(tts_ctx* c, const StepArgs& a, int splits, float* shard_stats_out, cudaStream_t s,
                                    int* launches) {
  if (shard_stats_out)
    row_stats_reduce_kernel<<<1, a.T >= 32 ? 1024 : 32 * a.T, 0, s>>>(c->stat_part, splits, a.T, shard_stats_out);
  else
    launch_merge(c, a, c->stat_part, splits, (long)splits * kStatFields, kStatFields, s);
  *launches += 1;
  return cudaGetLastError();
}

// shard: the tuples of all shards, stats_all [n_shards, T, kStatFields] -> normalisers, KL, omega, loss
cudaError_t launch_row_stats_merge_shards(tts_ctx* c, const StepArgs& a, const float* stats_all, int n_shards,
                                          cudaStream_t s, int* launches) {
  launch_merge(c, a, stats_all, n_shards, kStatFields, (long)a.T * kStatFields, s);
  *launches += 1;
  return cudaGetLastError();
}

}  // namespace tts
