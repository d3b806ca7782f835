// Pass B of the distillation step for one canvas (T <= 16 rows): ONE persistent kernel per step that streams the
// optimiser state exactly once and does, per tile of [16 vocabulary rows x 1024 hidden columns],
//
//   a6  gW^T tile = h^T . dl            tcgen05, accumulators in TMEM (gW never exists in HBM)
//   a7  SGD / AdamW on the fp32 master  epilogue straight out of TMEM; the master / m / v sub-tiles arrive by TMA, are
//       + bf16 working-copy write-back  updated IN PLACE in shared memory and leave by TMA stores
//   a5  gh^T[j, r] += W_in[v, j] dl[r, v]   tcgen05 as well: the bf16 tile of W_in is RE-DERIVED from the fp32
//                                       master values the epilogue holds in registers (precondition
//                                       W_in == rn_bf16(W_master), include/tts.h) and written to shared memory as
//                                       the A operand, so bf16 W is not read from HBM again.  gh == NULL skips a5.
//
// Why this tile shape.  The pass is HBM-bound (26 bytes per parameter, 12 flop); what the memory system sees is
// seven concurrent streams, three read and four written.  Measured on B200 with the same ring of TMA loads and
// TMA stores and real (non-zero) data, only the shape of the sub-tile moved per pipeline stage changed:
//     [128 cols x 16 rows] 5.65 TB/s   [256 x 8] 5.9   [512 x 4] 6.0   [1024 x 2] 6.7 (7 stages) / 6.4 (6 stages)
// and per-thread 4-byte stores instead of TMA stores: 5.6 TB/s.  Long row segments (4 KB per tensor row) keep DRAM
// pages open across the read and write streams.  So a pipeline stage is [2 rows x 1024 columns] of master, m
// and v (24 KB), a tile is 8 stages, and a CTA owns ONE 1024-column stripe of the parameter matrix for the whole
// kernel: its h^T operand (8 blocks of [128 j x 16 k]) is loaded once, and its gh accumulators (8 blocks of
// [128 j x 16 r], 128 TMEM columns) persist in TMEM and are flushed once, with fp32 atomics, at the end.
//
// Operands, both pre-tiled by the a4 kernels in the canonical no-swizzle core-matrix order ([8 rows][16 bytes]
// contiguous), so a tile is one contiguous bulk copy:
//   hTc [d][16 k]                                        A of gW: copied once per CTA into TENSOR MEMORY (lane = hidden
//       column, 8 columns = 16 canvas rows packed in pairs); tcgen05.mma reads A from there, shared memory keeps a
//       seventh state stage instead (ring depth is what the pass's bandwidth scales with)
//   dlC [V / 16][2 planes][T16 / 8][2][8 r][8 v]          dl = hi + lo (bf16 split).  One shared-memory copy serves
//       both contractions: core matrices [8 r][8 v] are the MN-major B of gW (N = v, K = r) and the K-major B
//       of gh (N = r, K = v); only the roles of the two descriptor strides swap.
#include <string.h>

#include "tts_adam.cuh"
#include "tts_common.cuh"
#include "tts_tc_ptx.cuh"
#include "tts_tc_state.h"

namespace tts {
namespace {

constexpr int kMJ = 128;         // hidden columns per MMA block = MMA M = TMEM lanes
constexpr int kJB = 8;           // MMA blocks per stripe
constexpr int kSW = kMJ * kJB;   // stripe width: 1024 hidden columns
constexpr int kTV = 16;          // vocabulary rows per tile = MMA N of gW = MMA K of gh
constexpr int kSV = 2;           // vocabulary rows per pipeline stage
constexpr int kSubs = kTV / kSV; // 8 stages per tile
constexpr int kBoxW = 256;       // TMA box width (elements): 4 boxes per tensor per stage
constexpr int kBoxes = kSW / kBoxW;
constexpr int kT16 = 16;         // canvas rows (padded)
constexpr int kMaxStages = 10;   // state ring depth: 7 x 24 KB with fp32 moments, 10 x 16 KB with bf16 moments (h^T lives in
                                 // tensor memory, not shared memory)
constexpr int kOpStages = 2;     // dl tile ring depth
constexpr int kTensorBytes = kSV * kSW * 4;          // 8 KB per fp32 tensor per stage
constexpr int kStageBytes = 3 * kTensorBytes;        // 24 KB (fp32 moments)
constexpr int kMomBytesLp = kSV * kSW * 2;           // 4 KB per bf16 moment tensor per stage
constexpr int kStageBytesLp = kTensorBytes + 2 * kMomBytesLp;   // 16 KB (bf16 moments)
constexpr int kWoBytes = kSV * kSW * 2;              // 4 KB: bf16 W_out staging of one sub-tile (one per group)
constexpr int kWtBytes = kSW * kTV * 2;              // 32 KB: re-derived bf16 W^T tile (A operand of gh)
constexpr int kDlBytes = 2 * kT16 * kTV * 2;         // 1 KB: dl tile, both planes
constexpr int kThreads = 384;    // warp 0 state TMA, 1 MMA, 2 TMEM alloc, 3 operand loads, 4-11 epilogue
constexpr int kGhCol0 = 2 * kJB * kTV;               // 256: first TMEM column of the gh accumulators
constexpr int kHtCol0 = kGhCol0 + kJB * kT16;        // 384: h^T of the stripe, 8 blocks x 8 columns (16 k packed in pairs)
constexpr int kTmemCols = 512;

struct FusedParams {
  float* master;
  float* gW_debug;
  float* gh;                  // NULL: a5 is skipped
  const __nv_bfloat16* hTc;
  const __nv_bfloat16* dlC;
  int V, d, T;
  int n_stripes;              // d / 1024
  int stages;
  const float* step_scalars;  // device {1 / (1 - b1^n), 1 / sqrt(1 - b2^n)} of this step
  const unsigned long long* step_count;   // device: Adam's count n of this step (keys the stochastic rounding of v)
  uint32_t sr_seed;
  float lr, b1, b2, eps, decay;   // decay = 1 - lr wd
};

__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
  const __nv_bfloat162 p = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<const uint32_t*>(&p);
}

// The bands of this CTA, as at most two segments (stripe, first band, step, count).
//   grid % n_stripes == 0 (configs 2, 3: 148 = 4 x 37): CTA b owns stripe b % n_stripes and every peers-th band of it.
//   otherwise (d = 5120: 5 stripes over 148 CTAs would be 30 / 29 peers; any SM budget): the n_stripes x n_bands units,
//   stripe-major, are cut into gridDim equal contiguous ranges; grid >= n_stripes, so a range spans at most two
//   stripes.  A CTA that crosses re-loads h^T into tensor memory and flushes its gh accumulators once more.
struct Seg {
  int stripe, first, step, n;
};
struct Walk {
  Seg s0, s1;      // scalars, selected with seg(): an indexed array would live in local memory
  int n_seg, n_my;
  __device__ Walk(int b, int grid, int n_stripes, int n_bands) : s0{0, 0, 1, 0}, s1{0, 0, 1, 0}, n_seg(0), n_my(0) {
    if (grid % n_stripes == 0) {
      const int peers = grid / n_stripes, first = b / n_stripes;
      const int n = first < n_bands ? (n_bands - first + peers - 1) / peers : 0;
      if (n > 0) { s0 = Seg{b % n_stripes, first, peers, n}; n_seg = 1; n_my = n; }
    } else {
      const long U = (long)n_stripes * n_bands;
      const long u0 = U * b / grid, u1 = U * (b + 1) / grid;
      if (u0 < u1) {
        const int st = (int)(u0 / n_bands);
        const long end = u1 < (long)(st + 1) * n_bands ? u1 : (long)(st + 1) * n_bands;
        s0 = Seg{st, (int)(u0 - (long)st * n_bands), 1, (int)(end - u0)};
        n_seg = 1;
        if (end < u1) { s1 = Seg{st + 1, 0, 1, (int)(u1 - end)}; n_seg = 2; }
        n_my = (int)(u1 - u0);
      }
    }
  }
  template <bool SK>
  __device__ __forceinline__ Seg seg(int sg) const { return (!SK || sg == 0) ? s0 : s1; }
  template <bool SK>
  __device__ __forceinline__ int segs() const { return SK ? n_seg : (n_seg > 0 ? 1 : 0); }
};

// SK: the stream-K walk (up to two segments); false: one segment, known at compile time (grid % n_stripes == 0)
// MOM: 1 = Adam's moments are stored as bf16 (TTS_MOMENT_BF16: a stage is 16 KB, the ring 10 deep; m is written back
// round-to-nearest-even, v with stochastic rounding keyed by (element index, Adam count, seed): tts_adam.cuh)
template <bool ADAM, bool SK, int MOM>
__global__ void __launch_bounds__(kThreads, 1)
tc_update_gh_kernel(const __grid_constant__ CUtensorMap tm_master, const __grid_constant__ CUtensorMap tm_m,
                    const __grid_constant__ CUtensorMap tm_v, const __grid_constant__ CUtensorMap tm_wout,
                    const FusedParams p) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = ptx::align_smem_1024(smem_raw);
  const int kStages = p.stages;
  constexpr int kStageB = MOM ? kStageBytesLp : kStageBytes;
  constexpr int kMomB = MOM ? kMomBytesLp : kTensorBytes;            // bytes of one moment tensor in a stage
  constexpr int kMomE = MOM ? 2 : 4;                                  // bytes per moment element
  uint8_t* st = smem;                                   // [kStages]{master [4 boxes][2 v][256] fp32, m, v likewise}
  uint8_t* wt = st + kStages * kStageB;                             // [8 jb][2 v-groups][16 j-groups][8 j][8 v] bf16
  uint8_t* wo = wt + kWtBytes;                          // [2 groups][4 boxes][2 v][256] bf16
  uint8_t* dl = wo + 2 * kWoBytes;                      // [kOpStages][2 planes][2 r-groups][2 v-groups][8 r][8 v] bf16
  uint64_t* bars = reinterpret_cast<uint64_t*>(dl + kOpStages * kDlBytes);
  uint64_t* st_full = bars;                    // [kMaxStages]
  uint64_t* st_empty = st_full + kMaxStages;   // [kMaxStages]
  uint64_t* op_full = st_empty + kMaxStages;   // [kOpStages]
  uint64_t* op_empty = op_full + kOpStages;    // [kOpStages]
  uint64_t* acc_full = op_empty + kOpStages;   // [2]
  uint64_t* acc_empty = acc_full + 2;          // [2]
  uint64_t* h_full = acc_empty + 2;            // [1]
  uint64_t* wt_full = h_full + 1;              // [1]
  uint64_t* wt_empty = wt_full + 1;            // [1]
  uint64_t* gh_full = wt_empty + 1;            // [1]
  uint64_t* gh_empty = gh_full + 1;            // [1]
  uint64_t* done_bar = gh_empty + 1;           // [1] epilogue warps finished (watchdog)
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(done_bar + 1);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const bool do_gh = p.gh != nullptr;
  const Walk w(blockIdx.x, gridDim.x, p.n_stripes, p.V / kTV);

  if (warp == 0 && lane == 0) {
    ptx::prefetch_tensormap(&tm_master);
    if (ADAM) { ptx::prefetch_tensormap(&tm_m); ptx::prefetch_tensormap(&tm_v); }
    ptx::prefetch_tensormap(&tm_wout);
  }
  if (warp == 1 && lane == 0) {
    for (int i = 0; i < kStages; ++i) { ptx::mbar_init(&st_full[i], 1); ptx::mbar_init(&st_empty[i], 1); }
    for (int i = 0; i < kOpStages; ++i) { ptx::mbar_init(&op_full[i], 1); ptx::mbar_init(&op_empty[i], 1); }
    for (int i = 0; i < 2; ++i) { ptx::mbar_init(&acc_full[i], 1); ptx::mbar_init(&acc_empty[i], 8); }
    ptx::mbar_init(h_full, 8);
    ptx::mbar_init(wt_full, 8);
    ptx::mbar_init(wt_empty, 1);
    ptx::mbar_init(gh_full, 1);
    ptx::mbar_init(gh_empty, 4);
    ptx::mbar_init(done_bar, 8);
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
    // ===== optimiser-state producer: [2 v x 1024 j] of master / m / v per stage, 4 boxes of [256 x 2] each =====
    if (lane == 0) {
      uint32_t n = 0;
      for (int sg = 0; sg < w.template segs<SK>(); ++sg) {
      const Seg cs = w.template seg<SK>(sg);
      const int j_stripe = cs.stripe * kSW;
      for (int k = 0; k < cs.n; ++k) {
        const int v0 = (cs.first + k * cs.step) * kTV;
        for (int sub = 0; sub < kSubs; ++sub, ++n) {
          const int s = n % kStages;
          ptx::mbar_wait(&st_empty[s], ((n / kStages) & 1) ^ 1);
          uint8_t* dst = st + s * kStageB;
          ptx::mbar_expect_tx(&st_full[s], ADAM ? kTensorBytes + 2 * kMomB : kTensorBytes);
          const int r0 = v0 + sub * kSV;
#pragma unroll
          for (int b = 0; b < kBoxes; ++b) {
            const int c0 = j_stripe + b * kBoxW, off = b * kSV * kBoxW * 4, off_m = b * kSV * kBoxW * kMomE;
            ptx::tma_load_2d(dst + off, &tm_master, &st_full[s], c0, r0);
            if (ADAM) {
              ptx::tma_load_2d(dst + kTensorBytes + off_m, &tm_m, &st_full[s], c0, r0);
              ptx::tma_load_2d(dst + kTensorBytes + kMomB + off_m, &tm_v, &st_full[s], c0, r0);
            }
          }
        }
      }
      }   // segments
    }
  } else if (warp == 3) {
    // ===== operand loads: one 1 KB dl tile per band =====
    if (lane == 0 && w.n_my > 0) {
      int i = 0;
      for (int sg = 0; sg < w.template segs<SK>(); ++sg) {
      const Seg cs = w.template seg<SK>(sg);
      for (int k = 0; k < cs.n; ++k, ++i) {
        const int band = cs.first + k * cs.step;
        const int s = i % kOpStages;
        ptx::mbar_wait(&op_empty[s], ((i / kOpStages) & 1) ^ 1);
        ptx::mbar_expect_tx(&op_full[s], kDlBytes);
        ptx::bulk_load_1d(dl + s * kDlBytes, p.dlC + (size_t)band * (kDlBytes / 2), kDlBytes, &op_full[s]);
      }
      }   // segments
    }
  } else if (warp == 1) {
    // ===== MMA issuer =====
    if (lane == 0 && w.n_my > 0) {
      constexpr uint32_t idesc_gw = ptx::make_idesc_bf16(kMJ, kTV, 0, 1);    // A = h^T K-major, B = dl MN-major
      constexpr uint32_t idesc_gh = ptx::make_idesc_bf16(kMJ, kT16, 0, 0);   // A = W^T K-major, B = dl K-major
      // acc[jb][j, v] = sum_r h^T[j, r] (dl_hi + dl_lo)[r, v]
      auto issue_gw = [&](int i) {
        const int ab = i & 1, s = i % kOpStages;
        ptx::mbar_wait(&acc_empty[ab], ((i >> 1) & 1) ^ 1);
        ptx::mbar_wait(&op_full[s], (i / kOpStages) & 1);
        ptx::tc_fence_after();
        const uint32_t b0 = ptx::smem_u32(dl + s * kDlBytes);
        for (int jb = 0; jb < kJB; ++jb) {
          for (int pl = 0; pl < 2; ++pl) {
            // B: MN-major, no swizzle: core matrices [8 r x 8 v]; v-groups 128 B apart (SBO), r-groups 256 B (LBO)
            const uint64_t bd = ptx::make_smem_desc(b0 + pl * 512, 256, 128, 0);
            // A = the block's h^T rows from tensor memory (lane = hidden column, 8 columns = 16 canvas rows)
            ptx::mma_f16_ts(tmem_base + ab * (kJB * kTV) + jb * kTV, tmem_base + kHtCol0 + jb * 8, bd, idesc_gw, pl);
          }
        }
        ptx::mma_commit(&acc_full[ab]);
      };
      int i = 0;   // bands issued so far (ring and accumulator phases run on over the segments)
      for (int sg = 0; sg < w.template segs<SK>(); ++sg) {
        const int n = w.template seg<SK>(sg).n;
        ptx::mbar_wait(h_full, sg & 1);          // this segment's h^T is in tensor memory
        ptx::tc_fence_after();
        if (!do_gh) {
          for (int k = 0; k < n; ++k, ++i) {
            issue_gw(i);
            ptx::mma_commit(&op_empty[i % kOpStages]);
          }
          continue;
        }
        if (sg > 0) {                            // the previous segment's gh accumulators have been flushed
          ptx::mbar_wait(gh_empty, (sg - 1) & 1);
          ptx::tc_fence_after();
        }
        issue_gw(i);
        for (int k = 0; k < n; ++k, ++i) {
          if (k + 1 < n) issue_gw(i + 1);
          // the epilogue has re-derived the whole [16 v x 1024 j] bf16 tile of W_in
          ptx::mbar_wait(wt_full, i & 1);
          ptx::tc_fence_after();
          const uint32_t b0 = ptx::smem_u32(dl + (i % kOpStages) * kDlBytes);
          for (int jb = 0; jb < kJB; ++jb) {
            // A: K-major, no swizzle: core matrices [8 j x 8 v]; j-groups 128 B apart (SBO), v-groups 2 KB (LBO)
            const uint64_t ad = ptx::make_smem_desc(ptx::smem_u32(wt + jb * 4096), 2048, 128, 0);
            for (int pl = 0; pl < 2; ++pl) {
              // B: K-major, no swizzle: the same core matrices; v-groups 128 B apart (LBO), r-groups 256 B (SBO)
              const uint64_t bd = ptx::make_smem_desc(b0 + pl * 512, 128, 256, 0);
              ptx::mma_f16_ss(tmem_base + kGhCol0 + jb * kT16, ad, bd, idesc_gh, (k > 0) | pl);
            }
          }
          ptx::mma_commit(wt_empty);
          ptx::mma_commit(&op_empty[i % kOpStages]);
        }
        ptx::mma_commit(gh_full);
      }
    }
  } else if (warp >= 4) {
    // ===== epilogue: 2 groups x 4 warps; group g takes sub-tiles sub % 2 == g; warp quarter q owns TMEM lanes 32q.. =====
    // thread (q, lane) <-> jj = 32 q + lane: hidden columns jb * 128 + jj of the stripe, jb = 0..7, both rows of a stage
    const int q = warp & 3, g = (warp - 4) >> 2;
    const int jj = q * 32 + lane;
    const bool leader = jj == 0;               // issues the group's TMA stores and releases its state stages
    const float c1 = ADAM ? p.lr * p.step_scalars[0] : 0.f, inv_sqrt_bc2 = ADAM ? p.step_scalars[1] : 0.f;
    const uint32_t key = MOM ? sr_key(static_cast<uint32_t>(*p.step_count), p.sr_seed) : 0u;
    // element (v, jb) of a stage tensor sits in box jb / 2, row v, column (jb % 2) * 128 + jj
    uint8_t* wt_thr = wt + (jj >> 3) * 128 + (jj & 7) * 16;   // + jb * 4096 + (v >> 3) * 2048 + (v & 7) * 2
    __nv_bfloat16* wo_g = reinterpret_cast<__nv_bfloat16*>(wo + g * kWoBytes);
    int prev_s = -1;                           // stage whose stores this group issued last
    int i = 0;   // bands processed so far
    for (int sg = 0; sg < w.template segs<SK>(); ++sg) {
    const Seg cs = w.template seg<SK>(sg);
    const int j_stripe = cs.stripe * kSW;
    {
      // the segment's h^T operand -> tensor memory: hTc row j holds h[0..16, j] (32 bytes); this group writes four of
      // the eight 128-column blocks.  (Every gW MMA of the previous segment is complete: its accumulators were read.)
      for (int jb = 4 * g; jb < 4 * g + 4; ++jb) {
        const uint4* row = reinterpret_cast<const uint4*>(p.hTc + (size_t)(j_stripe + jb * kMJ + jj) * kT16);
        const uint4 lo = __ldg(row), hi = __ldg(row + 1);
        const uint32_t r[8] = {lo.x, lo.y, lo.z, lo.w, hi.x, hi.y, hi.z, hi.w};
        ptx::tmem_st_32x32b_x8(tmem_base + kHtCol0 + jb * 8 + (static_cast<uint32_t>(q * 32) << 16), r);
      }
      ptx::tmem_st_wait();
      ptx::tc_fence_before();
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive(h_full);
    }
    for (int k = 0; k < cs.n; ++k, ++i) {
      const int v0 = (cs.first + k * cs.step) * kTV;
      const int ab = i & 1;
      ptx::mbar_wait(&acc_full[ab], (i >> 1) & 1);
      ptx::tc_fence_after();
      for (int sub = g; sub < kSubs; sub += 2) {
        const uint32_t n = (uint32_t)i * kSubs + sub;
        const int s = n % kStages;
        // gradients: columns (2 sub, 2 sub + 1) of each of the 8 accumulator blocks
        uint32_t gr[kJB][2];
#pragma unroll
        for (int jb = 0; jb < kJB; ++jb)
          ptx::tmem_ld_32x32b_x2(tmem_base + ab * (kJB * kTV) + jb * kTV + sub * kSV +
                                     (static_cast<uint32_t>(q * 32) << 16), gr[jb]);
        ptx::mbar_wait(&st_full[s], (n / kStages) & 1);
        float* sM = reinterpret_cast<float*>(st + s * kStageB) + jj;
        uint16_t* sLm = reinterpret_cast<uint16_t*>(st + s * kStageB + kTensorBytes) + jj;   // MOM: bf16 m, then v
        uint16_t* sLv = reinterpret_cast<uint16_t*>(st + s * kStageB + kTensorBytes + kMomB) + jj;
        float M[kJB][2], mm[kJB][2], vv[kJB][2];
#pragma unroll
        for (int jb = 0; jb < kJB; ++jb)
#pragma unroll
          for (int v = 0; v < 2; ++v) {
            const int e = (jb >> 1) * 512 + v * 256 + (jb & 1) * 128;
            M[jb][v] = sM[e];
            if (ADAM) {
              if (MOM) { mm[jb][v] = bf16_bits_widen(sLm[e]); vv[jb][v] = bf16_bits_widen(sLv[e]); }
              else { mm[jb][v] = sM[kSV * kSW + e]; vv[jb][v] = sM[2 * kSV * kSW + e]; }
            }
          }
        if (do_gh) {
          // a5 operand: W_in[v, j] = rn_bf16(master[v, j]); rows (2 sub, 2 sub + 1) of this thread's 8 columns
          if (sub < 2) ptx::mbar_wait(wt_empty, (i & 1) ^ 1);   // gh MMAs of the previous tile have read wt
          uint8_t* dst = wt_thr + (sub >> 2) * 2048 + (sub & 3) * 4;
#pragma unroll
          for (int jb = 0; jb < kJB; ++jb) *reinterpret_cast<uint32_t*>(dst + jb * 4096) = pack_bf16(M[jb][0], M[jb][1]);
          if (sub >= kSubs - 2) {               // the group's last sub-tile of this tile
            ptx::fence_proxy_async_smem();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(wt_full);
          }
        }
        ptx::tmem_ld_wait();
        // a7 in place: the thread rewrites exactly the shared-memory words it read
#pragma unroll
        for (int jb = 0; jb < kJB; ++jb) {
          // MOM: one hash for the two rows (even, odd) of this column (tts_adam.cuh)
          const uint32_t rnd = MOM ? sr_bits32((unsigned long long)((v0 + sub * kSV) >> 1) * (unsigned long long)p.d +
                                                   (j_stripe + jb * kMJ + jj), key) : 0u;
#pragma unroll
          for (int v = 0; v < 2; ++v) {
            const int e = (jb >> 1) * 512 + v * 256 + (jb & 1) * 128;
            const float gg = __uint_as_float(gr[jb][v]);
            if (ADAM) {
              const float m1 = p.b1 * mm[jb][v] + (1.f - p.b1) * gg;
              const float v1 = p.b2 * vv[jb][v] + (1.f - p.b2) * gg * gg;
              const float den = adam_sqrt(v1) * inv_sqrt_bc2 + p.eps;
              M[jb][v] = fmaf(-(c1 * m1), adam_rcp(den), M[jb][v] * p.decay);     // the step uses the unrounded moments
              if (MOM) {
                sLm[e] = bf16_bits_rn(m1);
                sLv[e] = bf16_bits_sr(v1, v == 0 ? rnd >> 16 : rnd & 0xFFFFu);
              } else {
                sM[kSV * kSW + e] = m1;
                sM[2 * kSV * kSW + e] = v1;
              }
            } else {
              M[jb][v] = M[jb][v] - p.lr * gg;
            }
            sM[e] = M[jb][v];
          }
        }
        if (p.gW_debug) {
#pragma unroll
          for (int jb = 0; jb < kJB; ++jb)
#pragma unroll
            for (int v = 0; v < 2; ++v)
              p.gW_debug[(size_t)(v0 + sub * kSV + v) * p.d + j_stripe + jb * kMJ + jj] = __uint_as_float(gr[jb][v]);
        }
        // the group's previous stores have read their shared memory: release that stage, reuse the bf16 staging
        if (leader) {
          ptx::bulk_wait_group_read<0>();
          if (prev_s >= 0) ptx::mbar_arrive(&st_empty[prev_s]);
        }
        ptx::named_barrier_sync(1 + g, 128);
#pragma unroll
        for (int jb = 0; jb < kJB; ++jb)
#pragma unroll
          for (int v = 0; v < 2; ++v)
            wo_g[(jb >> 1) * 512 + v * 256 + (jb & 1) * 128 + jj] = __float2bfloat16_rn(M[jb][v]);
        ptx::fence_proxy_async_smem();
        ptx::named_barrier_sync(1 + g, 128);
        if (leader) {
          const int r0 = v0 + sub * kSV;
          const uint8_t* sT = st + s * kStageB;
#pragma unroll
          for (int b = 0; b < kBoxes; ++b) {
            const int c0 = j_stripe + b * kBoxW, off = b * kSV * kBoxW;
            ptx::tma_store_2d(&tm_master, sT + off * 4, c0, r0);
            if (ADAM) {
              ptx::tma_store_2d(&tm_m, sT + kTensorBytes + off * kMomE, c0, r0);
              ptx::tma_store_2d(&tm_v, sT + kTensorBytes + kMomB + off * kMomE, c0, r0);
            }
            ptx::tma_store_2d(&tm_wout, wo_g + off, c0, r0);
          }
          ptx::bulk_commit_group();
        }
        prev_s = s;
      }
      ptx::tc_fence_before();
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive(&acc_empty[ab]);
    }
    // ===== gh flush: the segment's accumulators -> fp32 atomics (group 0: one warp per lane quarter) =====
    if (do_gh && g == 0) {
      ptx::mbar_wait(gh_full, sg & 1);
      ptx::tc_fence_after();
      for (int jb = 0; jb < kJB; ++jb) {
        float* gc = p.gh + j_stripe + jb * kMJ + jj;
        uint32_t r[16];
        ptx::tmem_ld_32x32b_x16(tmem_base + kGhCol0 + jb * kT16 + (static_cast<uint32_t>(q * 32) << 16), r);
        ptx::tmem_ld_wait();
#pragma unroll
        for (int kk = 0; kk < 16; ++kk)
          if (kk < p.T) atomicAdd(gc + (size_t)kk * p.d, __uint_as_float(r[kk]));
      }
      ptx::tc_fence_before();
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive(gh_empty);   // the next segment may overwrite the accumulators
    }
    }   // segments
    if (leader) ptx::bulk_wait_group_read<0>();   // shared memory must outlive the last stores' reads
    if (lane == 0) ptx::watchdog_arrive(done_bar);
  } else if (warp == 2) {
    ptx::watchdog_wait(done_bar);
  }
  ptx::tc_fence_before();
  __syncthreads();
  if (warp == 2) {
    ptx::tc_fence_after();
    ptx::tmem_dealloc(tmem_base, kTmemCols);
  }
}

constexpr int kStagesF32 = 6, kStagesLp = 6;
size_t fused_smem(bool lowp) {
  return 1024 + (lowp ? (size_t)kStagesLp * kStageBytesLp : (size_t)kStagesF32 * kStageBytes) + kWtBytes +
         2 * (size_t)kWoBytes + (size_t)kOpStages * kDlBytes + 512;
}

// hTc[j][k] = h[k, j] for k < 16 (rows k >= T are zero): 32 bytes per hidden column, the order in which the epilogue
// warps of the fused pass copy a stripe's h^T into tensor memory.  One thread per hidden column j.
__global__ void __launch_bounds__(256) tc_prep_hc_kernel(const __nv_bfloat16* __restrict__ h, int d, int T,
                                                         __nv_bfloat16* __restrict__ hTc) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= d) return;
  __nv_bfloat16* row = hTc + (size_t)j * kT16;
  for (int k = 0; k < kT16; ++k) row[k] = k < T ? h[(size_t)k * d + j] : __float2bfloat16_rn(0.f);
}

// a4 for this pass: dl = coef_r (q - p) from z, teacher and the row normalisers, split into two bf16 (dl = hi + lo
// to 2^-16 relative) and written pre-tiled: dlC[v / 16][plane][r / 8][(v % 16) / 8][r % 8][v % 8].
// One thread per vocabulary row v (loads coalesced over v for every canvas row r).
template <bool BF16>
__global__ void __launch_bounds__(256) tc_prep_dlc_kernel(const void* __restrict__ teacher, const float* __restrict__ z,
                                                          const float* __restrict__ z_ref, float lam,
                                                          int V, int z_ld, int T, int T_max,
                                                          const float* __restrict__ row_stats,
                                                          __nv_bfloat16* __restrict__ dlC) {
  __shared__ float sh[4 * kT16];   // lse_t, lse_z, coef, lse_ref
  if (threadIdx.x < kT16) {
    const int r = threadIdx.x;
    sh[r] = r < T ? row_stats[0 * T_max + r] : 0.f;
    sh[kT16 + r] = r < T ? row_stats[1 * T_max + r] : 0.f;
    sh[2 * kT16 + r] = r < T ? row_stats[3 * T_max + r] : 0.f;
    sh[3 * kT16 + r] = r < T ? row_stats[4 * T_max + r] : 0.f;
  }
  __syncthreads();
  const int v = blockIdx.x * blockDim.x + threadIdx.x;
  if (v >= V) return;
  __nv_bfloat16* tile = dlC + (size_t)(v / kTV) * (kDlBytes / 2) + ((v % kTV) >> 3) * 64 + (v & 7);
#pragma unroll
  for (int r = 0; r < kT16; ++r) {
    float dl = 0.f;
    if (r < T) {
      const float t = BF16 ? __bfloat162float(static_cast<const __nv_bfloat16*>(teacher)[(size_t)r * V + v])
                           : static_cast<const float*>(teacher)[(size_t)r * V + v];
      const float qv = expf(z[(size_t)r * z_ld + v] - sh[kT16 + r]);
      const float pv = expf(t - sh[r]);   // t = -inf -> 0
      float g = qv - pv;
      if (z_ref) g += lam * (qv - expf(z_ref[(size_t)r * z_ld + v] - sh[3 * kT16 + r]));
      dl = sh[2 * kT16 + r] * g;
    }
    const __nv_bfloat16 hi = __float2bfloat16_rn(dl);
    const __nv_bfloat16 lo = __float2bfloat16_rn(dl - __bfloat162float(hi));
    const int e = (r >> 3) * 128 + (r & 7) * 8;
    tile[e] = hi;
    tile[256 + e] = lo;
  }
}

}  // namespace

cudaError_t tc_fused_init(tts_ctx* c) {
  if (cudaError_t w = ptx::set_watchdog_cycles(c->watchdog_cycles)) return w;
  cudaError_t e;
  TcState* st = static_cast<TcState*>(c->tc_state);
  if ((e = cudaMalloc(&st->hTc, (size_t)c->cfg.d * kT16 * 2)) != cudaSuccess) return e;
  if ((e = cudaMalloc(&st->dlC, (size_t)c->cfg.V * 2 * kT16 * 2)) != cudaSuccess) return e;
  const int smem = (int)fused_smem(false), smem_lp = (int)fused_smem(true);
  const auto attr = cudaFuncAttributeMaxDynamicSharedMemorySize;
  if ((e = cudaFuncSetAttribute(tc_update_gh_kernel<true, false, 0>, attr, smem)) != cudaSuccess) return e;
  if ((e = cudaFuncSetAttribute(tc_update_gh_kernel<true, true, 0>, attr, smem)) != cudaSuccess) return e;
  if ((e = cudaFuncSetAttribute(tc_update_gh_kernel<false, true, 0>, attr, smem)) != cudaSuccess) return e;
  if ((e = cudaFuncSetAttribute(tc_update_gh_kernel<false, false, 0>, attr, smem)) != cudaSuccess) return e;
  if ((e = cudaFuncSetAttribute(tc_update_gh_kernel<true, false, 1>, attr, smem_lp)) != cudaSuccess) return e;
  return cudaFuncSetAttribute(tc_update_gh_kernel<true, true, 1>, attr, smem_lp);
}

// Grid of the fused pass, 0 when the shape does not qualify (T > 16 rows, d or V not a multiple of the tile, or an
// SM budget below one CTA per 1024-column stripe: a CTA owns exactly one stripe, so the wide kernel (tts_tc_wide.cu), which
// walks any grid, serves that case).
int tc_fused_grid(const tts_ctx* c, int T16) {
  if (T16 > kT16 || c->cfg.d % kSW != 0 || c->cfg.V % kTV != 0) return 0;
  const int n_stripes = c->cfg.d / kSW;
  const long n_tiles = (long)(c->cfg.V / kTV) * n_stripes;
  const bool lowp = c->cfg.optimizer == TTS_ADAMW && c->cfg.moment_dtype == TTS_MOMENT_BF16;
  int grid = tc_update_ctas(c, lowp);
  if (grid < n_stripes) return 0;
  if (grid > n_tiles) grid = (int)n_tiles;
  // A grid that is a multiple of the stripe count lets every CTA own ONE stripe for the whole pass (no second h^T load,
  // one gh flush, the walk known at compile time): d = 4096 runs 132 = 4 x 33 CTAs, d = 5120 130 = 5 x 26 (measured
  // 3.11 ms; 135, 140 and 145 CTAs 3.36-3.38 ms, the stream-K walk over all 148 3.21 ms).
  const int whole = grid - grid % n_stripes;
  if (whole >= n_stripes && 10 * whole >= 9 * grid) grid = whole;
  return grid;
}

// a4: the operands of the fused pass (h^T tiles and the pre-tiled dl planes)
cudaError_t tc_launch_prep_fused(tts_ctx* c, const StepArgs& a, const float* z, cudaStream_t s, int* launches) {
  TcState* st = static_cast<TcState*>(c->tc_state);
  const int V = c->cfg.V, d = c->cfg.d;
  tc_prep_hc_kernel<<<(d + 255) / 256, 256, 0, s>>>(static_cast<const __nv_bfloat16*>(a.h), d, a.T, st->hTc);
  if (c->cfg.logits_dtype == TTS_BF16)
    tc_prep_dlc_kernel<true><<<(V + 255) / 256, 256, 0, s>>>(a.teacher, z, a.z_ref, a.lambda, V, V, a.T, c->cfg.T_max,
                                                              c->row_stats, st->dlC);
  else
    tc_prep_dlc_kernel<false><<<(V + 255) / 256, 256, 0, s>>>(a.teacher, z, a.z_ref, a.lambda, V, V, a.T, c->cfg.T_max,
                                                               c->row_stats, st->dlC);
  *launches += 2;
  return cudaGetLastError();
}

cudaError_t tc_launch_update_fused(tts_ctx* c, const StepArgs& a, int grid, cudaStream_t s, int* launches) {
  TcState* st = static_cast<TcState*>(c->tc_state);
  const int V = c->cfg.V, d = c->cfg.d, T = a.T;
  const bool adam = c->cfg.optimizer == TTS_ADAMW;
  cudaError_t e;
  if (a.gh_out && (e = cudaMemsetAsync(a.gh_out, 0, (size_t)T * d * sizeof(float), s)) != cudaSuccess) return e;
  CUtensorMap tm_master, tm_m, tm_v, tm_wout;
  if (make_map_2d(st, &tm_master, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, a.master, d, V, kBoxW, kSV,
                  CU_TENSOR_MAP_SWIZZLE_NONE) != CUDA_SUCCESS)
    return cudaErrorInvalidValue;
  if (make_map_2d(st, &tm_wout, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, a.W_out, d, V, kBoxW, kSV,
                  CU_TENSOR_MAP_SWIZZLE_NONE) != CUDA_SUCCESS)
    return cudaErrorInvalidValue;
  tm_m = tm_master;
  tm_v = tm_master;
  const bool lowp = adam && c->cfg.moment_dtype == TTS_MOMENT_BF16;
  if (adam) {
    const CUtensorMapDataType mdt = lowp ? CU_TENSOR_MAP_DATA_TYPE_BFLOAT16 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32;
    const int msz = lowp ? 2 : 4;
    if (make_map_2d(st, &tm_m, mdt, msz, a.adam_m, d, V, kBoxW, kSV, CU_TENSOR_MAP_SWIZZLE_NONE) != CUDA_SUCCESS)
      return cudaErrorInvalidValue;
    if (make_map_2d(st, &tm_v, mdt, msz, a.adam_v, d, V, kBoxW, kSV, CU_TENSOR_MAP_SWIZZLE_NONE) != CUDA_SUCCESS)
      return cudaErrorInvalidValue;
  }
  FusedParams p;
  p.master = a.master;
  p.gW_debug = a.gW_debug; p.gh = a.gh_out; p.hTc = st->hTc; p.dlC = st->dlC;
  p.V = V; p.d = d; p.T = T;
  p.n_stripes = d / kSW;
  p.stages = lowp ? kStagesLp : kStagesF32;
  p.lr = a.lr; p.b1 = a.beta1; p.b2 = a.beta2; p.eps = a.eps;
  p.decay = 1.f - a.lr * a.wd;
  p.step_scalars = a.step_scalars;
  p.step_count = c->step_count_dev;
  p.sr_seed = static_cast<uint32_t>(c->cfg.sr_seed);
  const size_t smem = fused_smem(lowp);
  const bool sk = grid % p.n_stripes != 0;
  if (lowp) {
    if (sk) tc_update_gh_kernel<true, true, 1><<<grid, kThreads, smem, s>>>(tm_master, tm_m, tm_v, tm_wout, p);
    else tc_update_gh_kernel<true, false, 1><<<grid, kThreads, smem, s>>>(tm_master, tm_m, tm_v, tm_wout, p);
  } else if (adam) {
    if (sk) tc_update_gh_kernel<true, true, 0><<<grid, kThreads, smem, s>>>(tm_master, tm_m, tm_v, tm_wout, p);
    else tc_update_gh_kernel<true, false, 0><<<grid, kThreads, smem, s>>>(tm_master, tm_m, tm_v, tm_wout, p);
  } else {
    if (sk) tc_update_gh_kernel<false, true, 0><<<grid, kThreads, smem, s>>>(tm_master, tm_m, tm_v, tm_wout, p);
    else tc_update_gh_kernel<false, false, 0><<<grid, kThreads, smem, s>>>(tm_master, tm_m, tm_v, tm_wout, p);
  }
  *launches += 1;
  return cudaGetLastError();
}

}  // namespace tts
