// a3: the vocab-wide sweep.  One pass over a teacher row t and the draft-logit row z keeps the
// online statistics (m_t, s_t, a, m_z, s_z):
//     m_t = max t,  s_t = sum e^{t-m_t},  a = sum e^{t-m_t} (t - z),  m_z = max z,  s_z = sum e^{z-m_z}
// so that  lse_t = m_t + log s_t,  lse_z = m_z + log s_z,
//          KL_r  = sum_v p (log p - log q) = a / s_t - lse_t + lse_z
// without ever storing a [T,V] probability tensor.  Partial tuples from different CTAs merge
// associatively (rescale to the larger maximum).  The merge kernel also forms the row weights
// omega_r (mask_mode per DESIGN.md R2), coef_r = loss_scale * omega_r and
// loss = loss_scale * sum_r omega_r KL_r  (a sum).
#include "tts_common.cuh"
#include "tts_internal.h"

namespace tts {

struct RowStat {
  float mt, st, a, mz, sz;
};

__device__ __forceinline__ void stat_init(RowStat& s) {
  s.mt = -CUDART_INF_F; s.st = 0.f; s.a = 0.f; s.mz = -CUDART_INF_F; s.sz = 0.f;
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
    s = stat_merge(s, q);
  }
  return s;
}

// grid (splits, T), 256 threads.  128-bit loads of the teacher (8 bf16 / 4 fp32) and of z (2 x / 1 x float4).
template <bool BF16>
__global__ void __launch_bounds__(256) row_stats_partial_kernel(const void* __restrict__ teacher,
                                                                const float* __restrict__ z, int V, int z_ld,
                                                                int chunk, float* __restrict__ part) {
  const int r = blockIdx.y, sp = blockIdx.x;
  const int v0 = sp * chunk, v1 = min(V, v0 + chunk);
  const float* zr = z + (size_t)r * z_ld;
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
#pragma unroll
      for (int k = 0; k < 8; ++k) stat_push(s, f[k], zz[k]);
    }
    for (int v = v0 + nvec * 8 + threadIdx.x; v < v1; v += blockDim.x) stat_push(s, __bfloat162float(row[v]), zr[v]);
  } else {
    const float* row = static_cast<const float*>(teacher) + (size_t)r * V;
    const int nvec = (v1 - v0) / 4;
    const float4* pt = reinterpret_cast<const float4*>(row + v0);
    const float4* pz = reinterpret_cast<const float4*>(zr + v0);
    for (int i = threadIdx.x; i < nvec; i += blockDim.x) {
      const float4 q = __ldg(pt + i);
      const float4 z0 = __ldg(pz + i);
      stat_push(s, q.x, z0.x); stat_push(s, q.y, z0.y); stat_push(s, q.z, z0.z); stat_push(s, q.w, z0.w);
    }
    for (int v = v0 + nvec * 4 + threadIdx.x; v < v1; v += blockDim.x) stat_push(s, row[v], zr[v]);
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
      o[0] = q.mt; o[1] = q.st; o[2] = q.a; o[3] = q.mz; o[4] = q.sz;
    }
  }
}

// One CTA.  row_stats layout: [0]=lse_t, [1]=lse_z, [2]=kl, [3]=coef, each [T_max].
__global__ void __launch_bounds__(256) row_stats_merge_kernel(const float* __restrict__ part, int splits, int T,
                                                              int T_max, int seg_len, int mask_mode,
                                                              const float* __restrict__ pos_weight,
                                                              const uint8_t* __restrict__ mask, float loss_scale,
                                                              float* __restrict__ row_stats,
                                                              float* __restrict__ kl_rows_out,
                                                              float* __restrict__ loss_out) {
  __shared__ double red[256];
  double local = 0.0;
  for (int r = threadIdx.x; r < T; r += blockDim.x) {
    // merge in double: the partials are few and this fixes the cancellation in a/s_t - lse_t + lse_z
    double mt = -CUDART_INF, st = 0.0, a = 0.0, mz = -CUDART_INF, sz = 0.0;
    for (int s = 0; s < splits; ++s) {
      const float* p = part + ((size_t)r * splits + s) * kStatFields;
      const double pmt = p[0], pst = p[1], pa = p[2], pmz = p[3], psz = p[4];
      if (pmt != -CUDART_INF) {
        const double nm = fmax(mt, pmt);
        const double e0 = (mt == -CUDART_INF) ? 0.0 : exp(mt - nm), e1 = exp(pmt - nm);
        st = st * e0 + pst * e1; a = a * e0 + pa * e1; mt = nm;
      }
      if (pmz != -CUDART_INF) {
        const double nm = fmax(mz, pmz);
        const double e0 = (mz == -CUDART_INF) ? 0.0 : exp(mz - nm), e1 = exp(pmz - nm);
        sz = sz * e0 + psz * e1; mz = nm;
      }
    }
    const double lse_t = mt + log(st), lse_z = mz + log(sz);
    const double kl = a / st - lse_t + lse_z;
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
    if (kl_rows_out) kl_rows_out[r] = (float)kl;
    local += omega * kl;
  }
  red[threadIdx.x] = local;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if (threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
    __syncthreads();
  }
  if (threadIdx.x == 0) loss_out[0] = (float)((double)loss_scale * red[0]);
}

cudaError_t launch_row_stats(tts_ctx* c, const StepArgs& a, int z_ld, cudaStream_t s, int* launches) {
  const int V = c->cfg.V, T = a.T;
  int splits = (2 * c->sm_count + T - 1) / T;
  splits = max(1, min(splits, kStatSplitsMax));
  int chunk = (V + splits - 1) / splits;
  chunk = (chunk + 7) / 8 * 8;
  splits = (V + chunk - 1) / chunk;
  dim3 grid(splits, T);
  if (c->cfg.logits_dtype == TTS_BF16)
    row_stats_partial_kernel<true><<<grid, 256, 0, s>>>(a.teacher, c->z, V, z_ld, chunk, c->stat_part);
  else
    row_stats_partial_kernel<false><<<grid, 256, 0, s>>>(a.teacher, c->z, V, z_ld, chunk, c->stat_part);
  row_stats_merge_kernel<<<1, 256, 0, s>>>(c->stat_part, splits, T, c->cfg.T_max, c->cfg.seg_len, c->cfg.mask_mode,
                                           a.pos_weight, a.mask, a.loss_scale, c->row_stats, a.kl_rows_out,
                                           a.loss_out);
  *launches += 2;
  return cudaGetLastError();
}

}  // namespace tts
