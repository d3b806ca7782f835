// The two W-streaming contractions of the distillation step on tcgen05 (sm_100a).  Both are strictly
// W-bandwidth-bound at small T (16 flop per byte of W at T = 16): the kernels are persistent, one CTA per
// SM, with a TMA producer warp keeping a deep ring of W tiles in flight, one MMA-issuing thread, and four
// epilogue warps draining the TMEM accumulator of tile i while the ring already streams tile i + 1.
//
//   logits (a2)  z^T[v, r] = sum_j W_in[v, j] h[r, j]          M = 128 vocabulary rows, N = T16, K = d
//                A = W_in tile, K-major (rows of W are contiguous in j);  B = h, K-major
//   gh     (a5)  gh^T[j, r] = sum_v W_in[v, j] dl[r, v]        M = 128 hidden columns, N = T16 rows, K = vocabulary
//                A = W_in tile, MN-major (the same row-major W: j is contiguous, K = v strides by a row);
//                B = the fp16 plane S dl [r, v] of tts_tc_wide.cu, K-major; the W tile is rewritten as fp16 in
//                shared memory (see the kernel); the epilogue multiplies by 1 / (16 S).  The vocabulary is split
//                over CTAs; partial tiles are reduced with fp32 atomics into gh (zeroed first).  (One canvas with
//                d % 1024 == 0 never comes here: tts_tc_fused.cu forms gh inside the update pass.  Beyond 256 rows
//                the logits pass is served by the CTA-pair kernel of tts_tc_pair.cu.)
#include <cuda_fp16.h>
#include <string.h>

#include "tts_common.cuh"
#include "tts_tc_epi.cuh"
#include "tts_tc_ptx.cuh"
#include "tts_tc_state.h"

namespace tts {
namespace {

constexpr int kGemmThreads = 256;   // warp 0 TMA producer, 1 MMA issuer, 2 TMEM allocator, 3 idle, 4-7 epilogue
constexpr int kGhThreads = 384;     // gh: warps 8-11 convert the bf16 W tile of a stage to fp16 in place
constexpr float kGhWScale = 16.f;   // bf16 -> fp16 scale of W: exact for 2^-18 <= |W| < 4094
constexpr int kATile = kTileMN * kKC * 2;   // 16 KB: [128 x 64] bf16 (K-major) or 2 x [64 k x 64 mn] (MN-major)
constexpr int kMaxStages = 8;
constexpr int kSmemBudget = 200 * 1024;
constexpr int kSmemLimit = 232448;  // 227 KB: the most dynamic shared memory a CTA can have on sm_100
constexpr int kNMax = 256;          // largest MMA N

__host__ __device__ inline int pow2_cols(int n) {
  int c = 32;
  while (c < n) c <<= 1;
  return c;
}

struct Bars {
  uint64_t full[kMaxStages];
  uint64_t empty[kMaxStages];
  uint64_t acc_full[2];
  uint64_t acc_empty[2];
  uint64_t conv[kMaxStages];   // gh: the stage's W tile is fp16 now
  uint64_t done;               // epilogue warps finished (watchdog)
  uint32_t tmem_slot;
};

// ------------------------------------------------------------------ a2: draft logits
struct LogitsParams {
  float* z;
  int z_ld;
  int n_vt;        // V / 128
  int k_chunks;    // d / 64
  int T16, T;      // padded rows (MMA N) and the caller's rows: rows >= T are computed but never stored
  int box_rows;    // rows per h box (<= 256)
  int n_boxes;     // h boxes per stage
  int stages;
  int n_acc;       // TMEM accumulators (2 when 2 * T16 <= 512)
  int tmem_cols;
  int stream_k;    // 1: every CTA owns an equal, contiguous range of (tile, K chunk) units; tiles cut by a range
                   // boundary are accumulated into the zeroed z with fp32 RED (exactly two addends: order-free)
};

// Work of CTA b: units [u_beg, u_end) of the n_vt * k_chunks (tile, chunk) units, walked tile by tile.
struct LogitsWalk {
  long u, u_end;
  int k_chunks;
  __device__ LogitsWalk(const LogitsParams& p) : k_chunks(p.k_chunks) {
    if (p.stream_k) {
      const long total = (long)p.n_vt * p.k_chunks;
      u = total * blockIdx.x / gridDim.x;
      u_end = total * (blockIdx.x + 1) / gridDim.x;
    } else {   // whole tiles, round robin
      u = (long)blockIdx.x * p.k_chunks;
      u_end = (long)p.n_vt * p.k_chunks;
    }
  }
  __device__ bool done() const { return u >= u_end; }
  // current piece: tile vt, chunks [c_beg, c_end)
  __device__ void piece(int& vt, int& c_beg, int& c_end) const {
    vt = (int)(u / k_chunks);
    c_beg = (int)(u - (long)vt * k_chunks);
    const long rest = u_end - u;
    c_end = rest < k_chunks - c_beg ? c_beg + (int)rest : k_chunks;
  }
  __device__ void next(const LogitsParams& p, int c_beg, int c_end) {
    u += c_end - c_beg;
    if (!p.stream_k) u += (long)(gridDim.x - 1) * k_chunks;
  }
};

// Upper 32 bits of a K-major, 128-byte-swizzled operand descriptor: SBO = 1024 B, version 1, swizzle mode 2;
// the lower 32 bits are (address >> 4) | LBO (16 B >> 4) << 16, so stepping 16 K elements (32 B) adds 2.
constexpr uint32_t kDescHiSw128 = (1024u >> 4) | (1u << 14) | (ptx::kSwizzle128B << 29);
__device__ __forceinline__ uint32_t desc_lo_sw128(uint32_t smem_addr) { return ((smem_addr >> 4) & 0x3FFFu) | (1u << 16); }
__device__ __forceinline__ uint64_t desc64(uint32_t hi, uint32_t lo) { return (static_cast<uint64_t>(hi) << 32) | lo; }

// WIDE = false: T16 <= 256, one MMA per 16-element K step.  The single issuing thread is the pipeline's narrowest
// point at T = 16 (a [128 x 16 x 16] MMA finishes in a few cycles): with descriptors rebuilt per instruction the
// kernel ran at 3.7 TB/s, MMA-issue-bound; the loop below is 2 integer adds per MMA.
// TB: the teacher is bf16 (its tiles are staged by TMA for the fused a3 statistics; fp32 teachers use vector loads)
template <bool WIDE, bool TB>
__global__ void __launch_bounds__(kGemmThreads, 1)
tc_logits_kernel(const __grid_constant__ CUtensorMap tm_W, const __grid_constant__ CUtensorMap tm_h,
                 const __grid_constant__ CUtensorMap tm_teacher, const LogitsParams p, const epi::Params ep) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = ptx::align_smem_1024(smem_raw);
  const int b_bytes = p.n_boxes * p.box_rows * kKC * 2;
  const int stage_bytes = kATile + b_bytes;
  Bars* bars = reinterpret_cast<Bars*>(smem + p.stages * stage_bytes);
  uint8_t* epi_base = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(bars + 1) + 127) & ~uintptr_t(127));
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  if (warp == 0 && lane == 0) {
    ptx::prefetch_tensormap(&tm_W);
    ptx::prefetch_tensormap(&tm_h);
    if (TB && ep.enabled) ptx::prefetch_tensormap(&tm_teacher);
  }
  if (warp == 1 && lane == 0) {
    for (int i = 0; i < p.stages; ++i) { ptx::mbar_init(&bars->full[i], 1); ptx::mbar_init(&bars->empty[i], 1); }
    for (int i = 0; i < 2; ++i) { ptx::mbar_init(&bars->acc_full[i], 1); ptx::mbar_init(&bars->acc_empty[i], 4); }
    ptx::mbar_init(&bars->done, 4);
    ptx::fence_barrier_init();
  }
  if (warp == 2) {
    ptx::tmem_alloc(&bars->tmem_slot, p.tmem_cols);
    ptx::tmem_relinquish();
  }
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  const uint32_t tmem_base = bars->tmem_slot;

  if (warp == 0) {
    // ===== TMA producer: one [128 v x 64 k] W tile (two 64-row boxes) + the matching h chunk per stage =====
    if (lane == 0) {
      uint32_t n = 0;
      int vt, c_beg, c_end;
      for (LogitsWalk w(p); !w.done(); w.next(p, c_beg, c_end)) {
        w.piece(vt, c_beg, c_end);
        for (int kc = c_beg; kc < c_end; ++kc, ++n) {
          const int s = n % p.stages;
          ptx::mbar_wait(&bars->empty[s], ((n / p.stages) & 1) ^ 1);
          uint8_t* A = smem + s * stage_bytes;
          ptx::mbar_expect_tx(&bars->full[s], stage_bytes);
          ptx::tma_load_2d(A, &tm_W, &bars->full[s], kc * kKC, vt * kTileMN);
          ptx::tma_load_2d(A + kATile / 2, &tm_W, &bars->full[s], kc * kKC, vt * kTileMN + 64);
          for (int b = 0; b < p.n_boxes; ++b)
            ptx::tma_load_2d(A + kATile + b * p.box_rows * kKC * 2, &tm_h, &bars->full[s], kc * kKC, b * p.box_rows);
        }
      }
    }
  } else if (warp == 1) {
    // ===== MMA issuer: the whole warp walks the pipeline, one elected lane issues =====
    const uint32_t idesc = ptx::make_idesc_bf16(kTileMN, WIDE ? kNMax : p.T16, 0, 0);
    const uint32_t smem0 = ptx::smem_u32(smem);
    uint32_t n = 0, it = 0;
    int vt, c_beg, c_end;
    for (LogitsWalk w(p); !w.done(); w.next(p, c_beg, c_end), ++it) {
      w.piece(vt, c_beg, c_end);
      const int ab = it % p.n_acc;
      ptx::mbar_wait(&bars->acc_empty[ab], ((it / p.n_acc) & 1) ^ 1);
      ptx::tc_fence_after();
      const uint32_t d_tmem = tmem_base + ab * p.T16;
      for (int kc = c_beg; kc < c_end; ++kc, ++n) {
        const int s = n % p.stages;
        ptx::mbar_wait(&bars->full[s], (n / p.stages) & 1);
        ptx::tc_fence_after();
        if (ptx::elect_one()) {
          const uint32_t a_lo = desc_lo_sw128(smem0 + s * stage_bytes);
          const uint32_t b_lo = desc_lo_sw128(smem0 + s * stage_bytes + kATile);
#pragma unroll
          for (int ks = 0; ks < kKC / 16; ++ks) {
            if (!WIDE) {
              ptx::mma_f16_ss(d_tmem, desc64(kDescHiSw128, a_lo + 2 * ks), desc64(kDescHiSw128, b_lo + 2 * ks), idesc,
                              (kc != c_beg) | ks);
            } else {
              for (int c0 = 0; c0 < p.T16; c0 += kNMax) {
                const int nn = min(kNMax, p.T16 - c0);
                ptx::mma_f16_ss(d_tmem + c0, desc64(kDescHiSw128, a_lo + 2 * ks),
                                desc64(kDescHiSw128, b_lo + (c0 * kKC * 2 >> 4) + 2 * ks),
                                ptx::make_idesc_bf16(kTileMN, nn, 0, 0), (kc != c_beg) | ks);
              }
            }
          }
          ptx::mma_commit(&bars->empty[s]);
        }
        __syncwarp();
      }
      if (ptx::elect_one()) ptx::mma_commit(&bars->acc_full[ab]);
      __syncwarp();
    }
  } else if (warp >= 4) {
    // ===== epilogue: thread = one vocabulary row (TMEM lane); a warp's access to one canvas row is 128 contiguous bytes.
    // Whole tiles also feed the fused a3 statistics (tts_tc_epi.cuh); a tile cut by a stream-K range boundary is only
    // accumulated into z here (its statistics come from the small fix-up sweep of tts_stats.cu) =====
    const int q = warp & 3;
    const int tid_e = threadIdx.x - 128;
    const epi::Shared esh(epi_base, p.T16);
    if (ep.enabled) epi::init(esh, p.T16, tid_e);
    uint32_t it = 0, g = 0;
    int vt, c_beg, c_end;
    for (LogitsWalk w(p); !w.done(); w.next(p, c_beg, c_end), ++it) {
      w.piece(vt, c_beg, c_end);
      const bool partial = c_end - c_beg < p.k_chunks;
      const int ab = it % p.n_acc;
      ptx::mbar_wait(&bars->acc_full[ab], (it / p.n_acc) & 1);
      ptx::tc_fence_after();
      const uint32_t tmem_tile = tmem_base + ab * p.T16 + (static_cast<uint32_t>(q * 32) << 16);
      auto release = [&]() {
        ptx::tc_fence_before();
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(&bars->acc_empty[ab]);
      };
      if (ep.enabled && !partial) {
        epi::tile<TB>(ep, esh, &tm_teacher, tmem_tile, vt * kTileMN, p.T16, p.z, p.z_ld, tid_e, g, release);
        continue;
      }
      float* zc = p.z + vt * kTileMN + q * 32 + lane;
      for (int c0 = 0; c0 < p.T16; c0 += 16) {
        uint32_t r[16];
        ptx::tmem_ld_32x32b_x16(tmem_tile + c0, r);
        ptx::tmem_ld_wait();
        // rows T .. T16 exist only as MMA padding: a caller's draft_logits_out has exactly T rows
        if (c0 + 16 <= p.T) {
          if (partial) {
#pragma unroll
            for (int i = 0; i < 16; ++i) atomicAdd(zc + (size_t)(c0 + i) * p.z_ld, __uint_as_float(r[i]));
          } else {
#pragma unroll
            for (int i = 0; i < 16; ++i) zc[(size_t)(c0 + i) * p.z_ld] = __uint_as_float(r[i]);
          }
        } else {
#pragma unroll
          for (int i = 0; i < 16; ++i)
            if (c0 + i < p.T) {
              if (partial) atomicAdd(zc + (size_t)(c0 + i) * p.z_ld, __uint_as_float(r[i]));
              else zc[(size_t)(c0 + i) * p.z_ld] = __uint_as_float(r[i]);
            }
        }
      }
      release();
    }
    if (ep.enabled) epi::flush(ep, esh, blockIdx.x, tid_e);
    if (lane == 0) ptx::watchdog_arrive(&bars->done);
  } else if (warp == 2) {
    ptx::watchdog_wait(&bars->done);
  }
  ptx::tc_fence_before();
  __syncthreads();
  if (warp == 2) {
    ptx::tc_fence_after();
    ptx::tmem_dealloc(tmem_base, p.tmem_cols);
  }
}

// ------------------------------------------------------------------ a5: gh
struct GhParams {
  float* gh;
  float* part;             // TTS_FLAG_DETERMINISTIC: [slots][T16][128] per-unit parts instead of fp32 RED into gh
  const float* dl_scale;   // {S, 1 / S} of the fp16 dl plane
  int T, d, T16;
  int planes;        // dl planes stacked along N (2: rows T16 .. 2 T16 hold the lo plane)
  int N;             // planes * T16: accumulator columns
  int n_jt;          // d / 128
  int n_ju;          // units along j: n_jt, or ceil(n_jt / 2) cluster units with MC
  int n_split;       // vocabulary splits
  int chunks_split;  // K chunks (of 64 vocabulary rows) per split
  int chunks_total;  // V / 64
  int box_rows;      // rows per dl box (<= 256)
  int n_boxes;       // dl boxes per stage
  int n_acc;         // TMEM accumulators (2 when 2 * T16 <= 512)
  int stages;
  int tmem_cols;
};

// One accumulator [128 j x T16 r] per unit (j tile, vocabulary split): the W tile of a K chunk is read once and
// multiplied with all canvas rows (MMA pieces of N <= 256), so bf16 W streams from HBM exactly once per step.
// Operand formats: dl needs more than bf16's 8 significant bits (a row with one dominant entry would miss the
// 2e-3 max|gh| bar), kind::f16 wants A and B in one format, and W arrives as bf16 from the caller's memory: so four
// otherwise idle warps rewrite each W tile in shared memory as fp16(16 W) (element-wise, so the swizzle is
// untouched; exact for 2^-18 <= |W| < 4094, values beyond are clamped) before the MMAs of that stage are issued.
// MC (T16 > 256): a cluster of two CTAs takes two adjacent j tiles of the same vocabulary split; each CTA loads ONE of
// the two 256-row dl boxes of a stage and TMA multicasts it to both, so a dl chunk leaves L2 once per two j tiles
// (this kernel runs at the L2 slice throughput: 6.2 GB at 8.5 TB/s without it).  Everything else stays per CTA; a
// stage is reused when BOTH CTAs' MMAs have read it (empty[s] collects both commits, each multicast to both CTAs).
template <bool MC>
__global__ void __launch_bounds__(kGhThreads, 1)
tc_gh_kernel(const __grid_constant__ CUtensorMap tm_W, const __grid_constant__ CUtensorMap tm_dl, const GhParams p) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = ptx::align_smem_1024(smem_raw);
  const int b_bytes = p.n_boxes * p.box_rows * kKC * 2;
  const int stage_bytes = kATile + b_bytes;
  Bars* bars = reinterpret_cast<Bars*>(smem + p.stages * stage_bytes);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int n_units = p.n_ju * p.n_split;
  const int cta = MC ? (int)ptx::cluster_ctarank() : 0;
  const int u_first = MC ? (int)(blockIdx.x >> 1) : (int)blockIdx.x, u_step = MC ? (int)(gridDim.x >> 1) : (int)gridDim.x;
  // unit u -> first hidden column of this CTA's tile (beyond d with MC and an odd tile count: zero fill, nothing flushed)
  auto unit_j0 = [&](int u) { return ((u % p.n_ju) * (MC ? 2 : 1) + cta) * kTileMN; };

  if (warp == 0 && lane == 0) {
    ptx::prefetch_tensormap(&tm_W);
    ptx::prefetch_tensormap(&tm_dl);
  }
  if (warp == 1 && lane == 0) {
    for (int i = 0; i < p.stages; ++i) {
      ptx::mbar_init(&bars->full[i], 1); ptx::mbar_init(&bars->empty[i], MC ? 2 : 1); ptx::mbar_init(&bars->conv[i], 128);
    }
    for (int i = 0; i < 2; ++i) { ptx::mbar_init(&bars->acc_full[i], 1); ptx::mbar_init(&bars->acc_empty[i], 4); }
    ptx::mbar_init(&bars->done, 4);
    ptx::fence_barrier_init();
  }
  if (warp == 2) {
    ptx::tmem_alloc(&bars->tmem_slot, p.tmem_cols);
    ptx::tmem_relinquish();
  }
  ptx::tc_fence_before();
  if (MC) ptx::cluster_sync(); else __syncthreads();
  ptx::tc_fence_after();
  const uint32_t tmem_base = bars->tmem_slot;

  if (warp >= 8) {
    // ===== W tile bf16 -> fp16(16 W), in place: 16 KB per stage, 8 x 16 bytes per thread =====
    const int t = threadIdx.x - 256;
    uint32_t n = 0;
    for (int u = u_first; u < n_units; u += u_step) {
      const int sp = u / p.n_ju;
      const int c_beg = sp * p.chunks_split, c_end = min(p.chunks_total, c_beg + p.chunks_split);
      for (int kc = c_beg; kc < c_end; ++kc, ++n) {
        const int s = n % p.stages;
        ptx::mbar_wait(&bars->full[s], (n / p.stages) & 1);
        uint4* A = reinterpret_cast<uint4*>(smem + s * stage_bytes);
#pragma unroll
        for (int k = 0; k < kATile / 16 / 128; ++k) {
          uint4 x = A[k * 128 + t];
          uint32_t* w = reinterpret_cast<uint32_t*>(&x);
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            const float lo = fminf(fmaxf(__uint_as_float(w[e] << 16) * kGhWScale, -65504.f), 65504.f);
            const float hi = fminf(fmaxf(__uint_as_float(w[e] & 0xFFFF0000u) * kGhWScale, -65504.f), 65504.f);
            const __half2 h2 = __floats2half2_rn(lo, hi);
            w[e] = *reinterpret_cast<const uint32_t*>(&h2);
          }
          A[k * 128 + t] = x;
        }
        ptx::fence_proxy_async_smem();
        ptx::mbar_arrive(&bars->conv[s]);
      }
    }
  } else if (warp == 0) {
    if (lane == 0) {
      uint32_t n = 0;
      for (int u = u_first; u < n_units; u += u_step) {
        const int j0 = unit_j0(u), sp = u / p.n_ju;
        const int c_beg = sp * p.chunks_split, c_end = min(p.chunks_total, c_beg + p.chunks_split);
        for (int kc = c_beg; kc < c_end; ++kc, ++n) {
          const int s = n % p.stages;
          ptx::mbar_wait(&bars->empty[s], ((n / p.stages) & 1) ^ 1);
          uint8_t* A = smem + s * stage_bytes;
          ptx::mbar_expect_tx(&bars->full[s], stage_bytes);
          // W rows kc*64 .. +63 (K), columns j0 .. j0+127 (M) as two [64 k x 64 m] boxes
          ptx::tma_load_2d(A, &tm_W, &bars->full[s], j0, kc * kKC);
          ptx::tma_load_2d(A + kATile / 2, &tm_W, &bars->full[s], j0 + 64, kc * kKC);
          if (MC) {   // this CTA's one of the two dl boxes, to both CTAs
            ptx::tma_load_2d_multicast(A + kATile + cta * p.box_rows * kKC * 2, &tm_dl, &bars->full[s], kc * kKC,
                                       cta * p.box_rows, 3);
          } else {
            for (int b = 0; b < p.n_boxes; ++b)   // rows beyond the scratch are out of bounds: zero fill
              ptx::tma_load_2d(A + kATile + b * p.box_rows * kKC * 2, &tm_dl, &bars->full[s], kc * kKC, b * p.box_rows);
          }
        }
      }
    }
  } else if (warp == 1) {
    if (lane == 0) {
      uint32_t n = 0, it = 0;
      for (int u = u_first; u < n_units; u += u_step, ++it) {
        const int sp = u / p.n_ju;
        const int c_beg = sp * p.chunks_split, c_end = min(p.chunks_total, c_beg + p.chunks_split);
        const int ab = it % p.n_acc;
        ptx::mbar_wait(&bars->acc_empty[ab], ((it / p.n_acc) & 1) ^ 1);
        ptx::tc_fence_after();
        const uint32_t d_tmem = tmem_base + ab * p.N;
        for (int kc = c_beg; kc < c_end; ++kc, ++n) {
          const int s = n % p.stages;
          ptx::mbar_wait(&bars->full[s], (n / p.stages) & 1);
          ptx::mbar_wait(&bars->conv[s], (n / p.stages) & 1);
          ptx::tc_fence_after();
          const uint32_t a0 = ptx::smem_u32(smem + s * stage_bytes), b0 = a0 + kATile;
#pragma unroll
          for (int ks = 0; ks < kKC / 16; ++ks) {
            // A (fp16 16 W, MN-major, 128-byte swizzle): 64 m per 128-byte row, one row per k; 8-row groups 1 KB apart
            // (SBO), the second 64-m block kATile/2 further (LBO); 16 k per instruction = 2 KB
            const uint64_t ad = ptx::make_smem_desc(a0 + ks * 2048, kATile / 2, 1024, ptx::kSwizzle128B);
            for (int c0 = 0; c0 < p.N; c0 += kNMax) {
              const int nn = min(kNMax, p.N - c0);
              // B (fp16 S dl, K-major): rows r, 64 v per 128-byte row
              const uint64_t bd = ptx::make_smem_desc(b0 + c0 * kKC * 2 + ks * 32, 16, 1024, ptx::kSwizzle128B);
              ptx::mma_f16_ss(d_tmem + c0, ad, bd,
                              ptx::make_idesc_f16(kTileMN, nn, ptx::kFmtF16, ptx::kFmtF16, 1, 0),
                              (kc != c_beg) || ks != 0);
            }
          }
          if (MC) ptx::mma_commit_multicast(&bars->empty[s], 3); else ptx::mma_commit(&bars->empty[s]);
        }
        ptx::mma_commit(&bars->acc_full[ab]);
      }
    }
  } else if (warp >= 4) {
    const int q = warp & 3;
    const float inv_s = p.dl_scale[1] * (1.f / kGhWScale);
    uint32_t it = 0;
    for (int u = u_first; u < n_units; u += u_step, ++it) {
      const int j0 = unit_j0(u);
      const int ab = it % p.n_acc;
      ptx::mbar_wait(&bars->acc_full[ab], (it / p.n_acc) & 1);
      ptx::tc_fence_after();
      float* gc = p.gh + j0 + q * 32 + lane;
      for (int c0 = 0; c0 < p.T16; c0 += 16) {
        if (c0 >= p.T) break;
        uint32_t r[16], r2[16];
        ptx::tmem_ld_32x32b_x16(tmem_base + ab * p.N + c0 + (static_cast<uint32_t>(q * 32) << 16), r);
        if (p.planes == 2)
          ptx::tmem_ld_32x32b_x16(tmem_base + ab * p.N + p.T16 + c0 + (static_cast<uint32_t>(q * 32) << 16), r2);
        ptx::tmem_ld_wait();
        // deterministic mode: this unit's part goes to its own slot (a warp stores 128 contiguous bytes per canvas
        // row); tc_gh_reduce_kernel adds the slots of a j tile in split order
        float* pc = p.part ? p.part + ((size_t)(MC ? 2 * u + cta : u) * p.T16 + c0) * kTileMN + q * 32 + lane : nullptr;
#pragma unroll
        for (int i = 0; i < 16; ++i) {
          float x = __uint_as_float(r[i]);
          if (p.planes == 2) x += __uint_as_float(r2[i]);
          if (c0 + i < p.T && j0 < p.d) {
            if (pc) pc[(size_t)i * kTileMN] = x * inv_s;
            else atomicAdd(gc + (size_t)(c0 + i) * p.d, x * inv_s);
          }
        }
      }
      ptx::tc_fence_before();
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive(&bars->acc_empty[ab]);
    }
    if (lane == 0) ptx::watchdog_arrive(&bars->done);
  } else if (warp == 2) {
    ptx::watchdog_wait(&bars->done);
  }
  ptx::tc_fence_before();
  if (MC) ptx::cluster_sync(); else __syncthreads();
  if (warp == 2) {
    ptx::tc_fence_after();
    ptx::tmem_dealloc(tmem_base, p.tmem_cols);
  }
}

// gh[r, j] = sum over the vocabulary splits of the j tile's parts, in split order (fixed: bit-reproducible)
__global__ void __launch_bounds__(128) tc_gh_reduce_kernel(const float* __restrict__ part, int n_ju, int n_split, int mc,
                                                           int T16, int d, float* __restrict__ gh) {
  const int jt = blockIdx.x, r = blockIdx.y, jj = threadIdx.x;
  float acc = 0.f;
  for (int sp = 0; sp < n_split; ++sp) {
    const int slot = mc ? 2 * (sp * n_ju + (jt >> 1)) + (jt & 1) : sp * n_ju + jt;
    acc += part[((size_t)slot * T16 + r) * kTileMN + jj];
  }
  gh[(size_t)r * d + jt * kTileMN + jj] = acc;
}

// Work split of the gh kernel (shared by the launch and by the sizing of the deterministic-mode scratch).
struct GhPlan {
  bool mc;
  int grid, n_ju, n_split, chunks_split, planes, N, box_rows, n_boxes;
};
GhPlan gh_plan(const tts_ctx* c, int T16) {
  GhPlan g;
  const int n_jt = c->cfg.d / kTileMN, chunks_total = c->cfg.V / kKC;
  g.grid = (c->cfg.max_ctas > 0 && c->cfg.max_ctas < c->sm_count) ? c->cfg.max_ctas : c->sm_count;
  g.planes = tc_wide_planes(T16);
  g.N = g.planes * T16;
  g.box_rows = g.N <= kNMax ? g.N : kNMax;
  g.n_boxes = (g.N + g.box_rows - 1) / g.box_rows;
  // MC: clusters of two CTAs on adjacent j tiles share every dl box by TMA multicast (two boxes: 256 < T16 <= 512)
  g.mc = g.n_boxes == 2 && g.grid >= 2;
  if (g.mc) g.grid &= ~1;
  const int n_cl = g.mc ? g.grid / 2 : g.grid;
  g.n_ju = g.mc ? (n_jt + 1) / 2 : n_jt;
  // About two units per CTA (cluster): each is a contiguous run of vocabulary chunks for one 128-column tile of gh,
  // flushed with fp32 RED (256 KB per unit at T = 512: more units would make the flush the bottleneck).  Units of
  // one vocabulary split run side by side on consecutive CTAs, so a dl chunk is fetched into L2 once for all j tiles.
  int n_split = (2 * n_cl) / g.n_ju;
  if (n_split < 1) n_split = 1;
  if (n_split > chunks_total) n_split = chunks_total;
  g.chunks_split = (chunks_total + n_split - 1) / n_split;
  g.n_split = (chunks_total + g.chunks_split - 1) / g.chunks_split;
  return g;
}

int pick_stages(int stage_bytes, int extra = 0) {
  int s = ((extra ? kSmemLimit : kSmemBudget) - (int)sizeof(Bars) - 1024 - extra) / stage_bytes;
  return s < 1 ? 1 : (s > kMaxStages ? kMaxStages : s);
}

}  // namespace

cudaError_t tc_gemm_init(tts_ctx* c) {
  if (cudaError_t w = ptx::set_watchdog_cycles(c->watchdog_cycles)) return w;
  cudaError_t e;
  const auto attr = cudaFuncAttributeMaxDynamicSharedMemorySize;
  if ((e = cudaFuncSetAttribute(tc_logits_kernel<false, true>, attr, kSmemLimit)) != cudaSuccess) return e;
  if ((e = cudaFuncSetAttribute(tc_logits_kernel<false, false>, attr, kSmemLimit)) != cudaSuccess) return e;
  if ((e = cudaFuncSetAttribute(tc_logits_kernel<true, true>, attr, kSmemLimit)) != cudaSuccess) return e;
  if ((e = cudaFuncSetAttribute(tc_logits_kernel<true, false>, attr, kSmemLimit)) != cudaSuccess) return e;
  const int smem_max = kSmemBudget + 16 * 1024;
  if ((e = cudaFuncSetAttribute(tc_gh_kernel<false>, attr, smem_max)) != cudaSuccess) return e;
  return cudaFuncSetAttribute(tc_gh_kernel<true>, attr, smem_max);
}

// a2 (+ a3 when `fuse_stats`).  *n_split_out = number of per-row tuples the fused epilogue (plus the fix-up sweep over
// tiles cut by the stream-K walk) left in c->stat_part, 0 when the statistics were not fused.
cudaError_t tc_launch_logits(tts_ctx* c, const StepArgs& a, float* z_out, bool fuse_stats, cudaStream_t s, int* launches,
                             int* n_split_out) {
  TcState* st = static_cast<TcState*>(c->tc_state);
  const int V = c->cfg.V, d = c->cfg.d, T = a.T;
  const int T16 = (T + 15) / 16 * 16;
  const bool tb = c->cfg.logits_dtype == TTS_BF16;
  *n_split_out = 0;
  LogitsParams p;
  p.z = z_out; p.z_ld = V;
  p.n_vt = V / kTileMN; p.k_chunks = d / kKC; p.T16 = T16; p.T = T;
  p.box_rows = T16 <= kNMax ? T16 : kNMax;
  p.n_boxes = (T16 + p.box_rows - 1) / p.box_rows;
  const int stage_bytes = kATile + p.n_boxes * p.box_rows * kKC * 2;
  const int epi_bytes = fuse_stats ? 128 + epi::smem_bytes(T16) : 0;
  p.stages = pick_stages(stage_bytes, epi_bytes);
  p.n_acc = 2 * T16 <= 512 ? 2 : 1;
  p.tmem_cols = pow2_cols(p.n_acc * T16);
  CUtensorMap tm_W, tm_h, tm_t;
  if (make_map_2d(st, &tm_W, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, a.W_in, d, V, kKC, 64,
                  CU_TENSOR_MAP_SWIZZLE_128B) != CUDA_SUCCESS)
    return cudaErrorInvalidValue;
  // rows >= T of a box are out of bounds: TMA fills them with zeros
  if (make_map_2d(st, &tm_h, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, a.h, d, T, kKC, p.box_rows,
                  CU_TENSOR_MAP_SWIZZLE_128B) != CUDA_SUCCESS)
    return cudaErrorInvalidValue;
  tm_t = tm_h;
  if (fuse_stats && tb &&
      make_map_2d(st, &tm_t, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, a.teacher, V, T, kTileMN, epi::kRows,
                  CU_TENSOR_MAP_SWIZZLE_NONE) != CUDA_SUCCESS)
    return cudaErrorInvalidValue;
  int grid = tc_logits_ctas(c);
  if (grid > p.n_vt) grid = p.n_vt;
  // Stream-K for one canvas: 1187 tiles over 148 CTAs would quantise to 9 waves of 8.02; equal contiguous unit
  // ranges keep every SM busy to the end.  A range spans >= k_chunks units (grid <= n_vt), so a tile is cut at most
  // once: it receives exactly two partial sums (or one store), and 0 + a + b does not depend on the order.
  p.stream_k = T16 <= 32 && p.n_vt % grid != 0;
  // tiles cut by a range boundary: z by fp32 RED in the kernel, statistics by the fix-up sweep afterwards
  int cut[kStatFixMax], n_cut = 0;
  if (p.stream_k) {
    cudaError_t e = cudaMemsetAsync(z_out, 0, (size_t)T * V * sizeof(float), s);
    if (e != cudaSuccess) return e;
    const long total = (long)p.n_vt * p.k_chunks;
    for (int b = 1; b < grid; ++b) {
      const long u = total * b / grid;
      if (u % p.k_chunks == 0) continue;
      if (n_cut == kStatFixMax) return cudaErrorInvalidConfiguration;   // unreachable: grid <= kStatFixMax (tc_logits_ctas)
      cut[n_cut++] = (int)(u / p.k_chunks) * kTileMN;
    }
  }
  epi::Params ep;
  ep.teacher = a.teacher; ep.part = c->stat_part; ep.n_split = grid + n_cut; ep.T = T; ep.V = V;
  ep.enabled = fuse_stats ? 1 : 0;
  const size_t smem = 1024 + (size_t)p.stages * stage_bytes + sizeof(Bars) + epi_bytes;
  if (T16 <= kNMax) {
    if (tb) tc_logits_kernel<false, true><<<grid, kGemmThreads, smem, s>>>(tm_W, tm_h, tm_t, p, ep);
    else tc_logits_kernel<false, false><<<grid, kGemmThreads, smem, s>>>(tm_W, tm_h, tm_t, p, ep);
  } else {
    if (tb) tc_logits_kernel<true, true><<<grid, kGemmThreads, smem, s>>>(tm_W, tm_h, tm_t, p, ep);
    else tc_logits_kernel<true, false><<<grid, kGemmThreads, smem, s>>>(tm_W, tm_h, tm_t, p, ep);
  }
  *launches += 1;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess || !fuse_stats) return e;
  if (n_cut > 0) e = launch_row_stats_tiles(c, a, z_out, V, cut, n_cut, grid, ep.n_split, s, launches);
  *n_split_out = ep.n_split;
  return e;
}

// slots of the deterministic-mode scratch for steps of up to T16 rows ([slots][T16][128] fp32)
size_t tc_gh_part_floats(const tts_ctx* c, int T16) {
  const GhPlan g = gh_plan(c, T16);
  return (size_t)g.n_ju * g.n_split * (g.mc ? 2 : 1) * T16 * kTileMN;
}

cudaError_t tc_launch_gh(tts_ctx* c, const StepArgs& a, cudaStream_t s, int* launches) {
  TcState* st = static_cast<TcState*>(c->tc_state);
  const int V = c->cfg.V, d = c->cfg.d, T = a.T;
  const int T16 = (T + 15) / 16 * 16;
  cudaError_t e;
  const bool det = (c->cfg.flags & TTS_FLAG_DETERMINISTIC) != 0 && c->gh_part != nullptr;
  if (!det && (e = cudaMemsetAsync(a.gh_out, 0, (size_t)T * d * sizeof(float), s)) != cudaSuccess) return e;
  const GhPlan g = gh_plan(c, T16);
  int grid = g.grid;
  const bool mc = g.mc;
  GhParams p;
  p.gh = a.gh_out; p.part = det ? c->gh_part : nullptr;
  p.dl_scale = st->dl_scale; p.T = T; p.d = d; p.T16 = T16;
  p.n_jt = d / kTileMN;
  p.chunks_total = V / kKC;
  p.planes = g.planes;
  p.N = g.N;
  p.box_rows = g.box_rows;
  p.n_boxes = g.n_boxes;
  p.n_acc = 2 * p.N <= 512 ? 2 : 1;
  p.tmem_cols = pow2_cols(p.n_acc * p.N);
  p.n_ju = g.n_ju;
  p.chunks_split = g.chunks_split;
  p.n_split = g.n_split;
  const int stage_bytes = kATile + p.n_boxes * p.box_rows * kKC * 2;
  p.stages = pick_stages(stage_bytes);
  CUtensorMap tm_W, tm_dl;
  if (make_map_2d(st, &tm_W, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, a.W_in, d, V, 64, kKC,
                  CU_TENSOR_MAP_SWIZZLE_128B) != CUDA_SUCCESS)
    return cudaErrorInvalidValue;
  if (make_map_2d(st, &tm_dl, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 2, st->dlR, V, (uint64_t)st->P, kKC, p.box_rows,
                  CU_TENSOR_MAP_SWIZZLE_128B) != CUDA_SUCCESS)
    return cudaErrorInvalidValue;
  const int n_units = p.n_ju * p.n_split;
  const size_t smem = 1024 + (size_t)p.stages * stage_bytes + sizeof(Bars);
  if (!mc) {
    if (grid > n_units) grid = n_units;
    tc_gh_kernel<false><<<grid, kGhThreads, smem, s>>>(tm_W, tm_dl, p);
  } else {
    if (grid > 2 * n_units) grid = 2 * n_units;
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(kGhThreads);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = s;
    cudaLaunchAttribute attr;
    attr.id = cudaLaunchAttributeClusterDimension;
    attr.val.clusterDim.x = 2; attr.val.clusterDim.y = 1; attr.val.clusterDim.z = 1;
    cfg.attrs = &attr;
    cfg.numAttrs = 1;
    if ((e = cudaLaunchKernelEx(&cfg, tc_gh_kernel<true>, tm_W, tm_dl, p)) != cudaSuccess) return e;
  }
  *launches += 1;
  if (det) {
    tc_gh_reduce_kernel<<<dim3(p.n_jt, T), kTileMN, 0, s>>>(c->gh_part, p.n_ju, p.n_split, mc ? 1 : 0, T16, d, a.gh_out);
    *launches += 1;
  }
  return cudaGetLastError();
}

}  // namespace tts
