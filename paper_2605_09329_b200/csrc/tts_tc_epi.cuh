// a3 fused into the epilogue of the a2 logits kernels (north_star (1)): while the z^T tile
// [128 vocabulary rows x T16 canvas rows] leaves tensor memory, the same epilogue warps take the online log-softmax
// statistics of teacher and draft rows from it -- per canvas row r the tuple of SURVEY 8(a) a3
//     m_t = max t,  s_t = sum e^{t - m_t},  a = sum e^{t - m_t} (t - z),  m_z = max z,  s_z = sum e^{z - m_z}
// -- next to the matching teacher tile, which TMA stages into shared memory (bf16 teachers; fp32 teachers are read
// with 128-bit loads).  No separate sweep over [T, V] reads z and the teacher again, and no probability tensor exists.
//
// Shape of the work.  A thread of the four epilogue warps owns one vocabulary row (a tensor-memory lane) and gets 16
// canvas rows per tcgen05.ld; the statistics reduce over the VOCABULARY, i.e. across lanes.  So each chunk of 16
// canvas rows goes through a [16 r][128 v] transposition tile in shared memory (padded: conflict-free both ways);
// afterwards thread (r = tid / 8, part = tid % 8) sweeps 16 consecutive vocabulary entries of canvas row r in
// registers (one rescale to the chunk maximum, then one exp per element), the 8 parts of a row are merged with warp
// shuffles, and the row's first lane folds the result into the CTA's running tuple of that row (shared memory, one
// owner thread per row: no races).  When the CTA has finished its tiles it writes one tuple per row, and the merge
// kernel of tts_stats.cu (double precision) turns all CTAs' tuples into lse_t, lse_z, KL_r and the loss.
#pragma once

#include <cuda_runtime.h>
#include <math_constants.h>
#include <stdint.h>

#include "tts_tc_ptx.cuh"

namespace tts {
namespace epi {

constexpr int kRows = 16;                       // canvas rows per chunk (one tcgen05.ld.x16)
constexpr int kZtPitch = 132;                   // floats per canvas row of the transposition tile: 4 x (32 + 1)
constexpr int kZtBytes = kRows * kZtPitch * 4;  // 8448
constexpr int kTBufBytes = kRows * 128 * 2;     // 4096: one [16 r x 128 v] bf16 teacher box
constexpr int kFields = 5;
constexpr int kBarA = 1, kBarB = 2;             // named barriers of the four epilogue warps

struct Params {
  const void* teacher;   // [T, V] (direct loads: fp32 teachers)
  float* part;           // [T][n_split][8] tuples; this CTA writes split blockIdx.x
  int n_split;
  int T, V;
  int enabled;           // 0: plain z store (z_ref / shard paths that need the 8-field sweep of tts_stats.cu)
};

// bytes of shared memory the epilogue needs behind the pipeline stages
__host__ __device__ inline int smem_bytes(int T16) { return kZtBytes + 2 * kTBufBytes + T16 * kFields * 4 + 32; }

struct Shared {
  float* zt;        // [16][132]
  uint8_t* tbuf;    // [2][4096]
  float* run;       // [T16][5]
  uint64_t* t_full; // [2]
  __device__ Shared(uint8_t* base, int T16)
      : zt(reinterpret_cast<float*>(base)), tbuf(base + kZtBytes),
        run(reinterpret_cast<float*>(base + kZtBytes + 2 * kTBufBytes)),
        t_full(reinterpret_cast<uint64_t*>(base + kZtBytes + 2 * kTBufBytes + T16 * kFields * 4 + 8)) {}
};

// once per CTA, by the epilogue threads (tid_e = 0..127), before the first tile
__device__ __forceinline__ void init(const Shared& sh, int T16, int tid_e) {
  for (int r = tid_e; r < T16; r += 128) {
    float* o = sh.run + r * kFields;
    o[0] = -CUDART_INF_F; o[1] = 0.f; o[2] = 0.f; o[3] = -CUDART_INF_F; o[4] = 0.f;
  }
  if (tid_e == 0) {
    ptx::mbar_init(&sh.t_full[0], 1);
    ptx::mbar_init(&sh.t_full[1], 1);
    ptx::fence_barrier_init();
  }
  ptx::named_barrier_sync(kBarA, 128);
}

// One [128 v x T16 r] accumulator tile: stores z (rows < T) and folds the tile into the running statistics.
//   tmem_tile: TMEM address of the tile's first column, lane bits of this warp's quarter included
//   v0:        first vocabulary row of the tile (all 128 rows valid: V % 128 == 0 on this path)
//   g:         chunks processed so far by this CTA (parity of the teacher double buffer), advanced here
// `release` is called once, after the tile's last tcgen05.ld has completed (the accumulator may be overwritten).
template <bool BF16, typename Release>
__device__ __forceinline__ void tile(const Params& p, const Shared& sh, const void* tm_teacher, uint32_t tmem_tile,
                                     int v0, int T16, float* z, int z_ld, int tid_e, uint32_t& g, Release release) {
  const int q = tid_e >> 5, lane = tid_e & 31;
  const int rr = tid_e >> 3, part = tid_e & 7;
  const int n_chunks = T16 / kRows;
  float* zc = z + v0 + tid_e;
  float* zt_w = sh.zt + q * 33 + lane;                                 // + i * kZtPitch
  const float* zt_r = sh.zt + rr * kZtPitch + (part >> 1) * 33 + (part & 1) * 16;
  if (BF16 && tid_e == 0) {                                            // chunk 0's teacher box: under the MMA wait
    ptx::mbar_expect_tx(&sh.t_full[g & 1], kTBufBytes);
    ptx::tma_load_2d(sh.tbuf + (g & 1) * kTBufBytes, tm_teacher, &sh.t_full[g & 1], v0, 0);
  }
  for (int c = 0; c < n_chunks; ++c, ++g) {
    const int c0 = c * kRows;
    if (BF16 && tid_e == 0 && c + 1 < n_chunks) {                      // next chunk's box into the other buffer
      ptx::mbar_expect_tx(&sh.t_full[(g + 1) & 1], kTBufBytes);
      ptx::tma_load_2d(sh.tbuf + ((g + 1) & 1) * kTBufBytes, tm_teacher, &sh.t_full[(g + 1) & 1], v0, c0 + kRows);
    }
    uint32_t r[16];
    ptx::tmem_ld_32x32b_x16(tmem_tile + c0, r);
    ptx::tmem_ld_wait();
    if (c + 1 == n_chunks) release();
    if (c0 + 16 <= p.T) {
#pragma unroll
      for (int i = 0; i < 16; ++i) zc[(size_t)(c0 + i) * z_ld] = __uint_as_float(r[i]);
    } else {                                                           // rows T .. T16 are MMA padding: never stored
#pragma unroll
      for (int i = 0; i < 16; ++i)
        if (c0 + i < p.T) zc[(size_t)(c0 + i) * z_ld] = __uint_as_float(r[i]);
    }
#pragma unroll
    for (int i = 0; i < 16; ++i) zt_w[i * kZtPitch] = __uint_as_float(r[i]);
    ptx::named_barrier_sync(kBarA, 128);
    // ---- thread (rr, part): 16 vocabulary entries of canvas row c0 + rr.  Rows >= T (padding: z = 0, teacher box
    // zero-filled) run through the same instructions, so that the warp stays converged for the shuffles; only the
    // fold into the running tuple is guarded.
    const int row = c0 + rr;
    float zz[16], tt[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) zz[k] = zt_r[k];
    if (BF16) {
      ptx::mbar_wait(&sh.t_full[g & 1], (g >> 1) & 1);
      const uint4* src = reinterpret_cast<const uint4*>(sh.tbuf + (g & 1) * kTBufBytes + rr * 256 + part * 32);
      const uint4 a = src[0], b = src[1];
      const uint32_t w[8] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w};
#pragma unroll
      for (int k = 0; k < 8; ++k) {
        tt[2 * k] = __uint_as_float(w[k] << 16);
        tt[2 * k + 1] = __uint_as_float(w[k] & 0xFFFF0000u);
      }
    } else {
      const float4* src = reinterpret_cast<const float4*>(
          static_cast<const float*>(p.teacher) + (size_t)(row < p.T ? row : 0) * p.V + v0 + part * 16);
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const float4 x = __ldg(src + k);
        tt[4 * k] = x.x; tt[4 * k + 1] = x.y; tt[4 * k + 2] = x.z; tt[4 * k + 3] = x.w;
      }
    }
    // the row's maxima over this tile: 16 local entries, then the row's 8 parts (lanes 8 (lane / 8) .. + 7)
    float mt = -CUDART_INF_F, mz = -CUDART_INF_F;
#pragma unroll
    for (int k = 0; k < 16; ++k) { mt = fmaxf(mt, tt[k]); mz = fmaxf(mz, zz[k]); }
#pragma unroll
    for (int o = 1; o < 8; o <<= 1) {
      mt = fmaxf(mt, __shfl_xor_sync(0xffffffffu, mt, o));
      mz = fmaxf(mz, __shfl_xor_sync(0xffffffffu, mz, o));
    }
    // one exp per element against the tile maxima (teacher entries at -inf carry p = 0 and are dropped)
    float st = 0.f, a = 0.f, sz = 0.f;
    const float mt_s = mt == -CUDART_INF_F ? 0.f : mt;                   // all -inf: every e is 0, avoid inf - inf
#pragma unroll
    for (int k = 0; k < 16; ++k) {
      const float e = __expf(tt[k] - mt_s);
      st += e;
      a += tt[k] == -CUDART_INF_F ? 0.f : e * (tt[k] - zz[k]);
      sz += __expf(zz[k] - mz);
    }
#pragma unroll
    for (int o = 1; o < 8; o <<= 1) {
      st += __shfl_xor_sync(0xffffffffu, st, o);
      a += __shfl_xor_sync(0xffffffffu, a, o);
      sz += __shfl_xor_sync(0xffffffffu, sz, o);
    }
    if (part == 0 && row < p.T) {                                      // the row's owner folds the tile's tuple in
      float* o = sh.run + row * kFields;
      const float Mt = fmaxf(o[0], mt), Mz = fmaxf(o[3], mz);
      const float eo = o[0] == -CUDART_INF_F ? 0.f : __expf(o[0] - Mt);
      const float en = mt == -CUDART_INF_F ? 0.f : __expf(mt - Mt);
      o[1] = o[1] * eo + st * en;
      o[2] = o[2] * eo + a * en;
      o[0] = Mt;
      const float fo = o[3] == -CUDART_INF_F ? 0.f : __expf(o[3] - Mz);
      o[4] = o[4] * fo + sz * __expf(mz - Mz);
      o[3] = Mz;
    }
    ptx::named_barrier_sync(kBarB, 128);                               // zt and this teacher buffer may be reused
  }
}

// after the CTA's last tile: one tuple per canvas row into split `split` of the partial-statistics buffer
__device__ __forceinline__ void flush(const Params& p, const Shared& sh, int split, int tid_e) {
  ptx::named_barrier_sync(kBarA, 128);                                 // the owners' last folds are visible
  for (int r = tid_e; r < p.T; r += 128) {
    const float* s = sh.run + r * kFields;
    float* o = p.part + ((size_t)r * p.n_split + split) * 8;
    o[0] = s[0]; o[1] = s[1]; o[2] = s[2]; o[3] = s[3]; o[4] = s[4];
    o[5] = -CUDART_INF_F; o[6] = 0.f; o[7] = 0.f;                      // no reference distribution on this path
  }
}

}  // namespace epi
}  // namespace tts
