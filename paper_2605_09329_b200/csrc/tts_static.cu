// tts_accept_mask_static (include/tts.h): the greedy accepted-prefix mask of a1 (Alg. 1 "Accept"
// PAPER.md:152; readings R8, R9, R11) for callers that must not allocate device memory.
//
// Who that is.  tts_accept_mask needs a tts_ctx, and tts_ctx_create cudaMallocs the ctx's scratch.  Some hosts of
// this library cannot do that at the point where they need the mask: a serving process whose memory pool has
// already claimed the whole GPU (a cudaMalloc there fails, or succeeds only by stealing from the KV cache), code
// that runs inside a region where the CUDA allocator is off limits (it synchronises the device, which stalls the
// decode stream the mask sits on), and embedders whose policy is that every byte on the GPU goes through their own
// allocator.  For them this file carries the split-argmax partials in a file-scope __device__ array that is part of
// the library image: the driver places it when the module is loaded on a GPU, and it stays there until the process
// exits.  The call itself takes no ctx, and issues no cudaMalloc / cudaFree / allocating library routine.
//
// The two kernels below are variants of argmax_partial_kernel / mask_finalize_kernel (tts_mask.cu) that take their
// scratch as one struct; the ctx-based path is untouched and the tests compare the two.
#include <mutex>

#include "tts_common.cuh"
#include "tts_internal.h"

namespace {

constexpr int kSplitsMax = 64;   // vocabulary slices per row (as tts::kArgSplitsMax)

// One (value, index) candidate per (row, slice), then the merged argmax per row.  Every slot the second kernel
// reads is written by the first kernel of the SAME call, so nothing here has to start at zero and the previous
// call's contents are never observed.
struct MaskScratch {
  float val[TTS_STATIC_T_MAX * kSplitsMax];
  int32_t idx[TTS_STATIC_T_MAX * kSplitsMax];
  int32_t am[TTS_STATIC_T_MAX];
};
static_assert(sizeof(MaskScratch) == TTS_STATIC_SCRATCH_BYTES, "include/tts.h states the size of the static scratch");

// In host code this name is only a handle for cudaGetSymbolAddress; it is NOT a device address and must never be
// passed to a kernel.  Device code may name it directly, but the kernels below take the address as an argument so
// that what they use is exactly what the host resolved for the current device.
static __device__ __align__(256) unsigned char g_mask_scratch[sizeof(MaskScratch)];

struct Cand {
  float v;
  int i;
};

// larger value wins, equal values: lower index wins (R11); (-inf, INT_MAX) is the identity
__device__ __forceinline__ Cand better(Cand a, Cand b) { return (b.v > a.v || (b.v == a.v && b.i < a.i)) ? b : a; }

__device__ __forceinline__ Cand warp_best(Cand p) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    Cand q;
    q.v = __shfl_xor_sync(0xffffffffu, p.v, o);
    q.i = __shfl_xor_sync(0xffffffffu, p.i, o);
    p = better(p, q);
  }
  return p;
}

// grid (splits, T): CTA (sp, r) sweeps columns [sp * chunk, min(V, (sp + 1) * chunk)) of teacher row r
template <bool BF16>
__global__ void __launch_bounds__(256) static_argmax_partial_kernel(const void* __restrict__ teacher, int V, int chunk,
                                                                    MaskScratch* __restrict__ sc) {
  const int r = blockIdx.y, sp = blockIdx.x;
  const int v0 = sp * chunk, v1 = min(V, v0 + chunk);
  Cand best{-CUDART_INF_F, 0x7fffffff};
  constexpr int kVec = BF16 ? 8 : 4;   // elements per 16-byte load; chunk % 8 == 0 and rows start 16-byte aligned
  const int nvec = (v1 - v0) / kVec;
  if (BF16) {
    const __nv_bfloat16* row = static_cast<const __nv_bfloat16*>(teacher) + (size_t)r * V;
    const uint4* p = reinterpret_cast<const uint4*>(row + v0);
    for (int i = threadIdx.x; i < nvec; i += blockDim.x) {
      float f[8];
      tts::unpack_bf16x8(__ldg(p + i), f);
#pragma unroll
      for (int k = 0; k < 8; ++k) best = better(best, Cand{f[k], v0 + i * 8 + k});
    }
    for (int v = v0 + nvec * 8 + threadIdx.x; v < v1; v += blockDim.x) best = better(best, Cand{__bfloat162float(row[v]), v});
  } else {
    const float* row = static_cast<const float*>(teacher) + (size_t)r * V;
    const float4* p = reinterpret_cast<const float4*>(row + v0);
    for (int i = threadIdx.x; i < nvec; i += blockDim.x) {
      const float4 q = __ldg(p + i);
      const float f[4] = {q.x, q.y, q.z, q.w};
#pragma unroll
      for (int k = 0; k < 4; ++k) best = better(best, Cand{f[k], v0 + i * 4 + k});
    }
    for (int v = v0 + nvec * 4 + threadIdx.x; v < v1; v += blockDim.x) best = better(best, Cand{row[v], v});
  }
  __shared__ float sv[8];
  __shared__ int si[8];
  best = warp_best(best);
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  if (lane == 0) { sv[w] = best.v; si[w] = best.i; }
  __syncthreads();
  if (w == 0) {
    Cand p{-CUDART_INF_F, 0x7fffffff};
    if (lane < (blockDim.x >> 5)) { p.v = sv[lane]; p.i = si[lane]; }
    p = warp_best(p);
    if (lane == 0) {
      sc->val[r * kSplitsMax + sp] = p.v;
      sc->idx[r * kSplitsMax + sp] = p.i;
    }
  }
}

// one CTA: merge the slices of every row, compare with the draft tokens, prefix-AND per sequence
__global__ void __launch_bounds__(256) static_mask_finalize_kernel(MaskScratch* __restrict__ sc, int splits,
                                                                   const int32_t* __restrict__ tok, int T, int seg_len,
                                                                   uint8_t* __restrict__ mask, int32_t* __restrict__ tau,
                                                                   int32_t* __restrict__ am_out) {
  for (int r = threadIdx.x; r < T; r += blockDim.x) {
    Cand best{-CUDART_INF_F, 0x7fffffff};
    for (int s = 0; s < splits; ++s) best = better(best, Cand{sc->val[r * kSplitsMax + s], sc->idx[r * kSplitsMax + s]});
    const int am = best.i == 0x7fffffff ? 0 : best.i;   // a row of only -inf resolves to index 0 (lowest-index rule)
    sc->am[r] = am;
    if (am_out) am_out[r] = am;
  }
  __syncthreads();
  for (int s = threadIdx.x; s < T / seg_len; s += blockDim.x) {
    bool alive = true;   // "if x_{t+k} rejected then break"
    int n = 0;
    for (int k = 0; k < seg_len; ++k) {
      const int r = s * seg_len + k;
      alive = alive && (sc->am[r] == tok[r]);
      mask[r] = alive ? 1 : 0;
      n += alive ? 1 : 0;
    }
    tau[s] = n;
  }
}

// ---- per-device set-up: resolved once per GPU, under a lock, with that GPU current ----
constexpr int kMaxDevices = 64;
struct DeviceSetup {
  bool ready;
  MaskScratch* scratch;   // device address of g_mask_scratch ON THIS GPU (every GPU holds its own copy)
  int sm_count;
};
DeviceSetup g_setup[kMaxDevices];
std::mutex g_setup_lock;
thread_local int t_last_cuda_error = 0;

int32_t fail(cudaError_t e) {
  t_last_cuda_error = static_cast<int>(e);
  cudaGetLastError();   // a failed launch / query leaves a sticky-looking "last error": clear the non-sticky ones
  return TTS_ERR_CUDA;
}

// Looks up (first call on this device: resolves) the scratch address and the SM count of the CURRENT device.
int32_t setup_for_current_device(DeviceSetup* out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail(e);
  if (dev < 0 || dev >= kMaxDevices) return TTS_ERR_UNSUPPORTED;
  std::lock_guard<std::mutex> hold(g_setup_lock);
  DeviceSetup& d = g_setup[dev];
  if (!d.ready) {
    int major = 0, sms = 0;
    if ((e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev)) != cudaSuccess) return fail(e);
    if (major != 10) return TTS_ERR_ARCH;   // the image holds sm_100a code only; there is no fallback
    if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return fail(e);
    void* p = nullptr;
    // The symbol is a host-side stand-in; this call (which also makes the driver load the module on this GPU if it
    // has not yet) returns where the array lives in THIS device's memory.
    if ((e = cudaGetSymbolAddress(&p, g_mask_scratch)) != cudaSuccess) return fail(e);
    if (!p) return fail(cudaErrorInvalidSymbol);
    d.scratch = static_cast<MaskScratch*>(p);
    d.sm_count = sms;
    d.ready = true;
  }
  *out = d;
  return TTS_OK;
}

}  // namespace

extern "C" {

int32_t tts_static_last_cuda_error(void) { return t_last_cuda_error; }

int32_t tts_accept_mask_static(const void* teacher, int32_t logits_dtype, int32_t V, int32_t seg_len,
                               const int32_t* tok, int32_t T, uint8_t* mask_out, int32_t* tau_out, int32_t* am_out,
                               void* stream) {
  if (!teacher || !tok || !mask_out || !tau_out) return TTS_ERR_INVALID_ARG;
  if (V <= 0 || seg_len <= 0 || T <= 0 || T % seg_len != 0) return TTS_ERR_INVALID_ARG;
  if (T > TTS_STATIC_T_MAX) return TTS_ERR_INVALID_ARG;   // the fixed scratch holds TTS_STATIC_T_MAX rows, no more
  if (logits_dtype != TTS_F32 && logits_dtype != TTS_BF16) return TTS_ERR_UNSUPPORTED;
  const bool bf = logits_dtype == TTS_BF16;
  if ((static_cast<size_t>(V) * (bf ? 2 : 4)) % 16 != 0) return TTS_ERR_UNSUPPORTED;   // rows start 16-byte aligned
  if (V > (1 << 30)) return TTS_ERR_UNSUPPORTED;                                        // column indices are int32
  if (reinterpret_cast<uintptr_t>(teacher) & 15u) return TTS_ERR_INVALID_ARG;

  DeviceSetup d;
  const int32_t st = setup_for_current_device(&d);
  if (st != TTS_OK) return st;

  // as tts_accept_mask: enough CTAs to fill the machine at small T, at most kSplitsMax slices, slices a multiple of 8
  int splits = (2 * d.sm_count + T - 1) / T;
  splits = max(1, min(splits, kSplitsMax));
  int chunk = (V + splits - 1) / splits;
  chunk = (chunk + 7) / 8 * 8;
  splits = (V + chunk - 1) / chunk;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  const dim3 grid(splits, T);
  if (bf)
    static_argmax_partial_kernel<true><<<grid, 256, 0, s>>>(teacher, V, chunk, d.scratch);
  else
    static_argmax_partial_kernel<false><<<grid, 256, 0, s>>>(teacher, V, chunk, d.scratch);
  static_mask_finalize_kernel<<<1, 256, 0, s>>>(d.scratch, splits, tok, T, seg_len, mask_out, tau_out, am_out);
  const cudaError_t e = cudaGetLastError();
  return e == cudaSuccess ? TTS_OK : fail(e);
}

}  // extern "C"
