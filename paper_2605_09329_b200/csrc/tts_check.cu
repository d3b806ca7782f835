// Boundary hardening (SURVEY 8(b) preconditions 1 and 5): debug-mode checks of what tts_distill_step assumes, the
// device status word they report into.
//   precondition 1   W_in == rn_bf16(W_master) element-wise: the update pass re-derives the bf16 tile the gh
//                    contraction needs from the master it already holds (the gradient is "evaluated at
//                    q = q_t", the W_in that produced z), so a caller whose two copies disagree gets a gh that does not
//                    belong to its logits.  Complete compare, one pass over both tensors.
//   precondition 5   teacher logits finite or -inf (R23), hidden states finite.
#include "tts_common.cuh"
#include "tts_internal.h"
#include "tts_tc_ptx.cuh"

namespace tts {
namespace {

__global__ void __launch_bounds__(256) check_w_kernel(const uint4* __restrict__ W, const float4* __restrict__ M,
                                                      size_t nvec, int* __restrict__ status) {
  bool bad = false;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += (size_t)gridDim.x * blockDim.x) {
    const uint4 w = __ldg(W + i);
    const float4 a = __ldg(M + 2 * i), b = __ldg(M + 2 * i + 1);
    const __nv_bfloat162 p0 = __floats2bfloat162_rn(a.x, a.y), p1 = __floats2bfloat162_rn(a.z, a.w);
    const __nv_bfloat162 p2 = __floats2bfloat162_rn(b.x, b.y), p3 = __floats2bfloat162_rn(b.z, b.w);
    bad |= w.x != *reinterpret_cast<const uint32_t*>(&p0) || w.y != *reinterpret_cast<const uint32_t*>(&p1) ||
           w.z != *reinterpret_cast<const uint32_t*>(&p2) || w.w != *reinterpret_cast<const uint32_t*>(&p3);
  }
  if (__any_sync(0xffffffffu, bad) && (threadIdx.x & 31) == 0) atomicOr(status, TTS_DEV_W_MISMATCH);
}

// NaN / +inf (and, unless allowed, -inf) anywhere in x[0..n)
template <typename T>
__global__ void __launch_bounds__(256) check_finite_kernel(const T* __restrict__ x, size_t n, int allow_neg_inf, int bit,
                                                           int* __restrict__ status) {
  bool bad = false;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const float f = ldf(x, i);
    bad |= !(isfinite(f) || (allow_neg_inf && f == -CUDART_INF_F));
  }
  if (__any_sync(0xffffffffu, bad) && (threadIdx.x & 31) == 0) atomicOr(status, bit);
}

// A pipeline that never completes: warp 1 waits on an mbarrier nobody arrives at (the shape of a protocol slip in the
// tensor-path kernels), so the "epilogue" never reports and the watchdog warp must trap.
__global__ void __launch_bounds__(96) stalled_pipeline_kernel() {
  __shared__ uint64_t bar;
  __shared__ uint64_t done;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x == 0) { ptx::mbar_init(&bar, 1); ptx::mbar_init(&done, 1); ptx::fence_barrier_init(); }
  __syncthreads();
  if (warp == 1) {
    ptx::mbar_wait(&bar, 0);
    if (lane == 0) ptx::watchdog_arrive(&done);
  } else if (warp == 2) {
    ptx::watchdog_wait(&done);
  }
  __syncthreads();
}

__global__ void set_count_kernel(unsigned long long* p, unsigned long long n) { *p = n; }

// read-and-clear in one atomic: a bit that a still-running kernel sets around it lands either in this read or in the next
__global__ void take_status_kernel(int* status) { status[1] = atomicExch(status, 0); }

}  // namespace

cudaError_t launch_check_preconditions(tts_ctx* c, const void* teacher, const void* h, const void* W_in,
                                       const float* master, int T, cudaStream_t s, int* launches) {
  const size_t V = c->cfg.V, d = c->cfg.d;
  const int grid = 8 * c->sm_count;
  if (c->cfg.param_dtype == TTS_BF16 && master && W_in) {   // rows are 16-byte aligned: d * 2 % 16 == 0
    check_w_kernel<<<grid, 256, 0, s>>>(static_cast<const uint4*>(W_in), reinterpret_cast<const float4*>(master),
                                        V * d / 8, c->dev_status);
    *launches += 1;
  }
  if (teacher) {
    if (c->cfg.logits_dtype == TTS_BF16)
      check_finite_kernel<<<grid, 256, 0, s>>>(static_cast<const __nv_bfloat16*>(teacher), (size_t)T * V, 1,
                                               TTS_DEV_NONFINITE_TEACHER, c->dev_status);
    else
      check_finite_kernel<<<grid, 256, 0, s>>>(static_cast<const float*>(teacher), (size_t)T * V, 1,
                                               TTS_DEV_NONFINITE_TEACHER, c->dev_status);
    *launches += 1;
  }
  if (h) {
    if (c->cfg.param_dtype == TTS_BF16)
      check_finite_kernel<<<64, 256, 0, s>>>(static_cast<const __nv_bfloat16*>(h), (size_t)T * d, 0,
                                             TTS_DEV_NONFINITE_H, c->dev_status);
    else
      check_finite_kernel<<<64, 256, 0, s>>>(static_cast<const float*>(h), (size_t)T * d, 0, TTS_DEV_NONFINITE_H,
                                             c->dev_status);
    *launches += 1;
  }
  return cudaGetLastError();
}

cudaError_t check_init(tts_ctx* c) { return ptx::set_watchdog_cycles(c->watchdog_cycles); }

cudaError_t launch_stalled_pipeline(cudaStream_t s) {
  stalled_pipeline_kernel<<<1, 96, 0, s>>>();
  return cudaGetLastError();
}

cudaError_t launch_take_status(tts_ctx* c, cudaStream_t s) {
  take_status_kernel<<<1, 1, 0, s>>>(c->dev_status);
  return cudaGetLastError();
}

cudaError_t launch_set_count(tts_ctx* c, unsigned long long n, cudaStream_t s) {
  set_count_kernel<<<1, 1, 0, s>>>(c->step_count_dev, n);
  return cudaGetLastError();
}

}  // namespace tts
