// f2: the paper's own accept rule and its section-3 diagnostics (include/tts.h tts_accept_stochastic).
//
//   accept x_{t+k} with probability min{1, p(x_{t+k}) / q(x_{t+k})}, left to right, break at the first rejection
//   (Alg. 1 "standard speculative rejection sampling"); at the first rejected
//   position the replacement token is drawn from the residual norm(max(0, p - q)).  The uniforms are the caller's.
//
//   diagnostics per row (Fig. 4): H(p_r), -log q_r(argmax p_r), p_r(tok_r), q_r(tok_r).
//
// Kernels
//   accept_stats_partial   grid (splits, T): one 128-bit-vectorised sweep of a teacher row t and the draft-logit row z:
//                          online (m_t, s_t, w_t = sum e^{t-m_t} t), teacher argmax (lowest index on ties), (m_z, s_z)
//   accept_finalize        one CTA: a warp merges a row's splits (sums in double), forms lse_t, lse_z and the four
//                          diagnostics; then one thread per sequence runs the accept loop and notes the rejected row
//   residual_partial       grid (splits, S): sum_v max(0, p - q) over a slice of each sequence's rejected row (double)
//   residual_pick          grid S: inverse CDF, the smallest v with cumsum_{v' <= v} max(0, p - q) >= u2 * total
#include "tts_common.cuh"
#include "tts_internal.h"

namespace tts {
namespace {

constexpr int kAccFields = 7;   // m_t, s_t, w_t, argmax value, argmax index (int bits), m_z, s_z

struct AccStat {
  float mt, st, wt, av;
  int ai;
  float mz, sz;
};

__device__ __forceinline__ void acc_init(AccStat& s) {
  s.mt = -CUDART_INF_F; s.st = 0.f; s.wt = 0.f; s.av = -CUDART_INF_F; s.ai = 0x7fffffff;
  s.mz = -CUDART_INF_F; s.sz = 0.f;
}

__device__ __forceinline__ void acc_push(AccStat& s, float t, float z, int v) {
  if (t != -CUDART_INF_F) {   // p = 0: contributes nothing to lse_t or to sum p t (0 * -inf := 0)
    const float e = expf(-fabsf(t - s.mt));
    if (t > s.mt) { s.st = s.st * e + 1.f; s.wt = s.wt * e + t; s.mt = t; }
    else          { s.st += e;             s.wt += e * t; }
  }
  if (t > s.av || (t == s.av && v < s.ai)) { s.av = t; s.ai = v; }
  const float e = expf(-fabsf(z - s.mz));
  if (z > s.mz) { s.sz = s.sz * e + 1.f; s.mz = z; }
  else          { s.sz += e; }
}

__device__ __forceinline__ AccStat acc_merge(const AccStat& x, const AccStat& y) {
  AccStat o;
  o.mt = fmaxf(x.mt, y.mt);
  const float ex = (x.mt == -CUDART_INF_F) ? 0.f : expf(x.mt - o.mt);
  const float ey = (y.mt == -CUDART_INF_F) ? 0.f : expf(y.mt - o.mt);
  o.st = x.st * ex + y.st * ey;
  o.wt = x.wt * ex + y.wt * ey;
  const bool yb = y.av > x.av || (y.av == x.av && y.ai < x.ai);
  o.av = yb ? y.av : x.av;
  o.ai = yb ? y.ai : x.ai;
  o.mz = fmaxf(x.mz, y.mz);
  const float fx = (x.mz == -CUDART_INF_F) ? 0.f : expf(x.mz - o.mz);
  const float fy = (y.mz == -CUDART_INF_F) ? 0.f : expf(y.mz - o.mz);
  o.sz = x.sz * fx + y.sz * fy;
  return o;
}

__device__ __forceinline__ AccStat warp_acc(AccStat s) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    AccStat q;
    q.mt = __shfl_xor_sync(0xffffffffu, s.mt, o);
    q.st = __shfl_xor_sync(0xffffffffu, s.st, o);
    q.wt = __shfl_xor_sync(0xffffffffu, s.wt, o);
    q.av = __shfl_xor_sync(0xffffffffu, s.av, o);
    q.ai = __shfl_xor_sync(0xffffffffu, s.ai, o);
    q.mz = __shfl_xor_sync(0xffffffffu, s.mz, o);
    q.sz = __shfl_xor_sync(0xffffffffu, s.sz, o);
    s = acc_merge(s, q);
  }
  return s;
}

template <bool BF16>
__device__ __forceinline__ float load_t(const void* teacher, size_t i) {
  return BF16 ? __bfloat162float(static_cast<const __nv_bfloat16*>(teacher)[i]) : static_cast<const float*>(teacher)[i];
}

template <bool BF16>
__global__ void __launch_bounds__(256) accept_stats_partial_kernel(const void* __restrict__ teacher,
                                                                   const float* __restrict__ z, int V, int chunk,
                                                                   float* __restrict__ part) {
  const int r = blockIdx.y, sp = blockIdx.x;
  const int v0 = sp * chunk, v1 = min(V, v0 + chunk);
  const float* zr = z + (size_t)r * V;
  AccStat s;
  acc_init(s);
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
      for (int k = 0; k < 8; ++k) acc_push(s, f[k], zz[k], v0 + i * 8 + k);
    }
    for (int v = v0 + nvec * 8 + threadIdx.x; v < v1; v += blockDim.x) acc_push(s, __bfloat162float(row[v]), zr[v], v);
  } else {
    const float* row = static_cast<const float*>(teacher) + (size_t)r * V;
    const int nvec = (v1 - v0) / 4;
    const float4* pt = reinterpret_cast<const float4*>(row + v0);
    const float4* pz = reinterpret_cast<const float4*>(zr + v0);
    for (int i = threadIdx.x; i < nvec; i += blockDim.x) {
      const float4 q = __ldg(pt + i), z0 = __ldg(pz + i);
      const int b = v0 + i * 4;
      acc_push(s, q.x, z0.x, b); acc_push(s, q.y, z0.y, b + 1); acc_push(s, q.z, z0.z, b + 2);
      acc_push(s, q.w, z0.w, b + 3);
    }
    for (int v = v0 + nvec * 4 + threadIdx.x; v < v1; v += blockDim.x) acc_push(s, row[v], zr[v], v);
  }
  __shared__ AccStat sh[8];
  s = warp_acc(s);
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  if (lane == 0) sh[w] = s;
  __syncthreads();
  if (w == 0) {
    AccStat q;
    acc_init(q);
    if (lane < (blockDim.x >> 5)) q = sh[lane];
    q = warp_acc(q);
    if (lane == 0) {
      float* o = part + ((size_t)r * gridDim.x + sp) * kAccFields;
      o[0] = q.mt; o[1] = q.st; o[2] = q.wt; o[3] = q.av; o[4] = __int_as_float(q.ai); o[5] = q.mz; o[6] = q.sz;
    }
  }
}

// rows[r] = (lse_t, lse_z) kept for the residual kernels; rej_row[s] = the first rejected row of sequence s or -1.
template <bool BF16>
__global__ void __launch_bounds__(1024) accept_finalize_kernel(const float* __restrict__ part, int splits,
                                                               const void* __restrict__ teacher,
                                                               const float* __restrict__ z, int V,
                                                               const int32_t* __restrict__ tok,
                                                               const float* __restrict__ u, int T, int seg_len,
                                                               uint8_t* __restrict__ mask, int32_t* __restrict__ tau,
                                                               int32_t* __restrict__ next_tok, float* __restrict__ diag,
                                                               float* __restrict__ rows, int32_t* __restrict__ rej_row,
                                                               int* __restrict__ dev_status) {
  extern __shared__ float pq[];   // [T][2]: p_r(tok), q_r(tok)
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, n_warps = blockDim.x >> 5;
  for (int r = warp; r < T; r += n_warps) {
    const float* pr = part + (size_t)r * splits * kAccFields;
    float mt = -CUDART_INF_F, mz = -CUDART_INF_F, av = -CUDART_INF_F;
    int ai = 0x7fffffff;
    for (int s = lane; s < splits; s += 32) {
      const float* p = pr + s * kAccFields;
      mt = fmaxf(mt, p[0]); mz = fmaxf(mz, p[5]);
      const int pi = __float_as_int(p[4]);
      if (p[3] > av || (p[3] == av && pi < ai)) { av = p[3]; ai = pi; }
    }
    mt = warp_max(mt); mz = warp_max(mz);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      const float ov = __shfl_xor_sync(0xffffffffu, av, o);
      const int oi = __shfl_xor_sync(0xffffffffu, ai, o);
      if (ov > av || (ov == av && oi < ai)) { av = ov; ai = oi; }
    }
    double st = 0.0, wt = 0.0, sz = 0.0;
    for (int s = lane; s < splits; s += 32) {
      const float* p = pr + s * kAccFields;
      if (p[0] != -CUDART_INF_F) {
        const double e = exp((double)p[0] - (double)mt);
        st += (double)p[1] * e; wt += (double)p[2] * e;
      }
      if (p[5] != -CUDART_INF_F) sz += (double)p[6] * exp((double)p[5] - (double)mz);
    }
    st = warp_sum(st); wt = warp_sum(wt); sz = warp_sum(sz);
    if (lane == 0) {
      const double lse_t = (double)mt + log(st), lse_z = (double)mz + log(sz);
      const int am = ai == 0x7fffffff ? 0 : ai;
      const size_t row = (size_t)r * V;
      // a draft token outside [0, V) (e.g. a GLOBAL id handed to a vocabulary shard: this call is not shard-aware)
      // is never dereferenced: p(tok) = 0, q(tok) = +inf, so the row is rejected for every u, and the status word says so
      const int tk = tok[r];
      const bool tok_ok = tk >= 0 && tk < V;
      if (!tok_ok) atomicOr(dev_status, TTS_DEV_BAD_TOKEN);
      const float tt = tok_ok ? load_t<BF16>(teacher, row + tk) : -CUDART_INF_F;
      const float p_tok = tt == -CUDART_INF_F ? 0.f : (float)exp((double)tt - lse_t);
      const float q_tok = tok_ok ? (float)exp((double)z[row + tk] - lse_z) : CUDART_INF_F;
      pq[2 * r] = p_tok;
      pq[2 * r + 1] = q_tok;
      rows[2 * r] = (float)lse_t;
      rows[2 * r + 1] = (float)lse_z;
      if (diag) {
        diag[4 * r + 0] = (float)(lse_t - wt / st);                    // H(p_r) = lse_t - sum_v p t
        diag[4 * r + 1] = (float)(lse_z - (double)z[row + am]);        // -log q_r(argmax_v p_r)
        diag[4 * r + 2] = p_tok;
        diag[4 * r + 3] = q_tok;
      }
    }
  }
  __syncthreads();
  const int S = T / seg_len;
  for (int s = threadIdx.x; s < S; s += blockDim.x) {
    int n = 0, rej = -1;
    for (int k = 0; k < seg_len; ++k) {
      const int r = s * seg_len + k;
      // accept with probability min{1, p/q}: u <= p / q, written without the division (q = 0 accepts)
      const bool ok = rej < 0 && u[r] * pq[2 * r + 1] <= pq[2 * r];
      if (rej < 0 && !ok) rej = r;   // "if x_{t+k} rejected then break"
      mask[r] = ok ? 1 : 0;
      n += ok ? 1 : 0;
    }
    tau[s] = n;
    rej_row[s] = rej;
    if (rej < 0) next_tok[s] = -1;   // the whole canvas was accepted: the bonus token needs p at position C + 1
  }
}

template <bool BF16>
__device__ __forceinline__ float residual_at(const void* teacher, const float* z, size_t i, float lse_t, float lse_z) {
  const float t = load_t<BF16>(teacher, i);
  const float p = t == -CUDART_INF_F ? 0.f : expf(t - lse_t);
  return fmaxf(0.f, p - expf(z[i] - lse_z));
}

template <bool BF16>
__global__ void __launch_bounds__(256) residual_partial_kernel(const void* __restrict__ teacher,
                                                               const float* __restrict__ z, int V, int chunk,
                                                               const float* __restrict__ rows,
                                                               const int32_t* __restrict__ rej_row,
                                                               double* __restrict__ rpart) {
  const int s = blockIdx.y, sp = blockIdx.x;
  const int r = rej_row[s];
  if (r < 0) return;
  const float lse_t = rows[2 * r], lse_z = rows[2 * r + 1];
  const int v0 = sp * chunk, v1 = min(V, v0 + chunk);
  double acc = 0.0;
  for (int v = v0 + threadIdx.x; v < v1; v += blockDim.x)
    acc += (double)residual_at<BF16>(teacher, z, (size_t)r * V + v, lse_t, lse_z);
  __shared__ double sh[8];
  acc = warp_sum(acc);
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = acc;
  __syncthreads();
  if (threadIdx.x == 0) {
    double t = 0.0;
    for (int w = 0; w < (blockDim.x >> 5); ++w) t += sh[w];
    rpart[(size_t)s * gridDim.x + sp] = t;
  }
}

// One CTA per sequence.  Thread i owns a contiguous run of its slice; an exclusive scan of the run sums locates the
// run that contains the target mass, and that thread walks its run.
template <bool BF16>
__global__ void __launch_bounds__(256) residual_pick_kernel(const void* __restrict__ teacher,
                                                            const float* __restrict__ z, int V, int chunk, int splits,
                                                            const float* __restrict__ rows,
                                                            const int32_t* __restrict__ rej_row,
                                                            const double* __restrict__ rpart,
                                                            const float* __restrict__ u2,
                                                            int32_t* __restrict__ next_tok) {
  const int s = blockIdx.x;
  const int r = rej_row[s];
  if (r < 0) return;
  const float lse_t = rows[2 * r], lse_z = rows[2 * r + 1];
  __shared__ double sh_run[256];
  __shared__ double sh_base;
  __shared__ int sh_split, sh_pick;
  if (threadIdx.x == 0) {
    double total = 0.0;
    for (int i = 0; i < splits; ++i) total += rpart[(size_t)s * splits + i];
    const double target = (double)u2[s] * total;
    double cum = 0.0;
    int pick = -1;
    for (int i = 0; i < splits; ++i) {
      const double c = rpart[(size_t)s * splits + i];
      if (c > 0.0 && cum + c >= target) { pick = i; break; }
      cum += c;
    }
    bool take_last = false;
    if (pick < 0) {   // rounding pushed the target past the end: the last slice with any mass, its last element
      for (int i = 0; i < splits; ++i)
        if (rpart[(size_t)s * splits + i] > 0.0) pick = i;
      if (pick < 0) pick = 0;   // no residual mass at all (p <= q everywhere): unreachable in exact arithmetic
      take_last = true;
    }
    sh_split = pick;
    sh_base = take_last ? -1.0 : target - cum;     // mass to cover inside the slice (< 0: take the last element)
    sh_pick = -1;
  }
  __syncthreads();
  const int v0 = sh_split * chunk, v1 = min(V, v0 + chunk);
  const int per = (v1 - v0 + blockDim.x - 1) / blockDim.x;
  const int a = min(v1, v0 + (int)threadIdx.x * per), b = min(v1, a + per);
  double run = 0.0;
  for (int v = a; v < b; ++v) run += (double)residual_at<BF16>(teacher, z, (size_t)r * V + v, lse_t, lse_z);
  sh_run[threadIdx.x] = run;
  __syncthreads();
  if (threadIdx.x == 0) {
    // serial scan over 256 run sums: find the first run whose inclusive sum reaches the target
    double cum = 0.0;
    int owner = -1, last_pos = -1;
    for (int i = 0; i < (int)blockDim.x; ++i) {
      if (sh_run[i] > 0.0) last_pos = i;
      if (sh_base >= 0.0 && sh_run[i] > 0.0 && cum + sh_run[i] >= sh_base) { owner = i; break; }
      cum += sh_run[i];
    }
    if (owner < 0) {            // target beyond the slice's mass by rounding: the last run with mass, its last element
      owner = last_pos;
      sh_base = -1.0;
    } else {
      sh_base -= cum;
    }
    sh_pick = owner;
    if (owner < 0) next_tok[s] = -1;   // no residual mass (see above)
  }
  __syncthreads();
  if ((int)threadIdx.x == sh_pick) {
    const double need = sh_base;
    double cum = 0.0;
    int pick = -1, last_pos = -1;
    for (int v = a; v < b; ++v) {
      const double x = (double)residual_at<BF16>(teacher, z, (size_t)r * V + v, lse_t, lse_z);
      if (x > 0.0) {
        last_pos = v;
        cum += x;
        if (need >= 0.0 && cum >= need) { pick = v; break; }
      }
    }
    next_tok[s] = pick >= 0 ? pick : last_pos;
  }
}

}  // namespace

cudaError_t launch_accept_stochastic(tts_ctx* c, const void* teacher, const float* z, const int32_t* tok,
                                     const float* u, const float* u2, int T, uint8_t* mask, int32_t* tau,
                                     int32_t* next_tok, float* diag, cudaStream_t s, int* launches) {
  const int V = c->cfg.V, S = T / c->cfg.seg_len;
  const bool bf = c->cfg.logits_dtype == TTS_BF16;
  int splits = (2 * c->sm_count + T - 1) / T;
  splits = max(1, min(splits, kStatSplitsMax));
  int chunk = (V + splits - 1) / splits;
  chunk = (chunk + 7) / 8 * 8;
  splits = (V + chunk - 1) / chunk;
  // scratch: stat_part holds [T][splits][kAccFields <= kStatFields]; acc_rows [T][2]; acc_rej [S]; acc_rpart [S][64]
  dim3 g1(splits, T);
  const int nt = T >= 32 ? 1024 : 32 * T;
  const size_t sh = (size_t)2 * T * sizeof(float);
  // residual slices: kStatSplitsMax per sequence, multiples of 8
  int rsplits = kStatSplitsMax;
  int rchunk = ((V + rsplits - 1) / rsplits + 7) / 8 * 8;
  rsplits = (V + rchunk - 1) / rchunk;
  dim3 g3(rsplits, S);
  if (bf) {
    accept_stats_partial_kernel<true><<<g1, 256, 0, s>>>(teacher, z, V, chunk, c->stat_part);
    accept_finalize_kernel<true><<<1, nt, sh, s>>>(c->stat_part, splits, teacher, z, V, tok, u, T, c->cfg.seg_len, mask,
                                                   tau, next_tok, diag, c->acc_rows, c->acc_rej, c->dev_status);
    residual_partial_kernel<true><<<g3, 256, 0, s>>>(teacher, z, V, rchunk, c->acc_rows, c->acc_rej, c->acc_rpart);
    residual_pick_kernel<true><<<S, 256, 0, s>>>(teacher, z, V, rchunk, rsplits, c->acc_rows, c->acc_rej, c->acc_rpart,
                                                 u2, next_tok);
  } else {
    accept_stats_partial_kernel<false><<<g1, 256, 0, s>>>(teacher, z, V, chunk, c->stat_part);
    accept_finalize_kernel<false><<<1, nt, sh, s>>>(c->stat_part, splits, teacher, z, V, tok, u, T, c->cfg.seg_len,
                                                    mask, tau, next_tok, diag, c->acc_rows, c->acc_rej, c->dev_status);
    residual_partial_kernel<false><<<g3, 256, 0, s>>>(teacher, z, V, rchunk, c->acc_rows, c->acc_rej, c->acc_rpart);
    residual_pick_kernel<false><<<S, 256, 0, s>>>(teacher, z, V, rchunk, rsplits, c->acc_rows, c->acc_rej,
                                                  c->acc_rpart, u2, next_tok);
  }
  *launches += 4;
  return cudaGetLastError();
}

}  // namespace tts
