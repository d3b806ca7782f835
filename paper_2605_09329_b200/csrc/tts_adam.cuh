// Low-precision moment storage of the AdamW update (include/tts.h TTS_MOMENT_BF16; R26): the counter-based
// draws of the stochastic rounding of v and the two fp32 -> bf16 conversions.  The fp64 oracle has its own
// implementation of the same generator (nothing is shared): both follow the definition written out here.
#pragma once

#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace tts {

// sqrt(v) of Adam's denominator as ONE MUFU instruction.  __fsqrt_rn expands to a reciprocal square root, a Newton
// step and a branch to a slow path per element; the branch keeps ptxas from interleaving the elements a thread
// updates, and the update kernels' epilogues (the per-SM bound of every variant that is not HBM-bound) then stall on
// fixed instruction latencies: ncu, round 2.  Relative error 2^-22 against tolerances of 2e-3 (R12, R13).  The
// non-ftz approximations (and __fdividef) wrap every MUFU in a subnormal test and two scalings: 6 more instructions
// per element for inputs that cannot change the result.
__device__ __forceinline__ float adam_sqrt(float x) {
  float y;
  asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));   // ftz: a subnormal v gives 0, i.e. den = eps (sqrt(v) < 1.1e-19 << eps)
  return y;
}
// 1 / den for den = sqrt(v) / sqrt(1 - b2^n) + eps >= eps: one MUFU, no subnormal scaling (den is normal whenever eps is)
__device__ __forceinline__ float adam_rcp(float x) {
  float y;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

// 32 pseudo-random bits for the PAIR of vertically adjacent elements (2k, j), (2k + 1, j) at Adam count n -- the even
// row rounds with the high half, the odd row with the low half (every thread of the update kernels owns such pairs, so
// one hash serves two elements: the hash was a third of the bf16-moment pass's instructions):
//   pidx = (v >> 1) * d + j
//   x = lo32(pidx) ^ (n * 0x9E3779B9) ^ (seed * 0x85EBCA6B) ^ (hi32(pidx) * 0xC2B2AE35)
//   x ^= x >> 16;  x *= 0x7FEB352D;  x ^= x >> 15;  x *= 0x846CA68B;  x ^= x >> 16
// `key` = (n * 0x9E3779B9) ^ (seed * 0x85EBCA6B) is formed once per thread.
__device__ __forceinline__ uint32_t sr_key(uint32_t n, uint32_t seed) { return (n * 0x9E3779B9u) ^ (seed * 0x85EBCA6Bu); }
__device__ __forceinline__ uint32_t sr_bits32(unsigned long long pidx, uint32_t key) {
  uint32_t x = static_cast<uint32_t>(pidx) ^ key ^ (static_cast<uint32_t>(pidx >> 32) * 0xC2B2AE35u);
  x ^= x >> 16; x *= 0x7FEB352Du; x ^= x >> 15; x *= 0x846CA68Bu; x ^= x >> 16;
  return x;
}
// stochastic rounding: the 16 discarded bits f round away from zero iff f + r >= 65536, so E_r[result] = x
__device__ __forceinline__ uint16_t bf16_bits_sr(float x, uint32_t r16) {
  return static_cast<uint16_t>((__float_as_uint(x) + r16) >> 16);
}
__device__ __forceinline__ uint16_t bf16_bits_rn(float x) { return __bfloat16_as_ushort(__float2bfloat16_rn(x)); }
__device__ __forceinline__ float bf16_bits_widen(uint16_t b) { return __uint_as_float(static_cast<uint32_t>(b) << 16); }

}  // namespace tts
