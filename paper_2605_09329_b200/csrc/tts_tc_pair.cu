// CTA-pair (cta_group::2) variants of the W-streaming contractions for SEVERAL canvases (256 < T16 <= 512).
//
// Why.  With one CTA per [128 x T16] output tile every tile pulls the whole other operand through the L2 -> SM
// crossbar: the T = 512 logits and gh kernels of tts_tc_gemm.cu move 6.2 GB each at 8.0 .. 8.4 TB/s (the L2 slice
// throughput every operand-heavy kernel here saturates at) with the tensor pipe a third busy.  A pair of CTAs on the
// two SMs of a TPC computes a [256 x T16] tile with ONE tcgen05.mma.cta_group::2 stream: each CTA stages its own 128
// rows of the A operand and only HALF of the B operand's rows, the tensor cores of both SMs read both halves.  Operand
// bytes per output drop from (128 + 512) to (256 + 512) per 256 rows: 6.2 -> 3.7 GB, and the logits pass goes from
// 0.78 to 0.59 ms (tensor pipe 31% -> 41% busy; what remains is bytes in flight over latency: 4 stages x 48 KB of
// shared memory against a ~4 us load-to-free loop).  The same treatment of the gh contraction (M = 256 hidden columns
// per pair) was built and measured: L2 -> SM bytes 6.2 -> 3.7 GB as predicted, time unchanged (0.76 ms: its loop is
// latency-bound through TMA -> in-smem fp16 conversion -> MMA, not crossbar-bound), so gh stays on tts_tc_gemm.cu.
//
//   logits (a2)  z^T[v, r] = sum_j W_in[v, j] h[r, j]   M = 256 vocabulary rows (128 per CTA), N = T16 in pieces
//                of <= 256, K = d.  CTA c of the pair holds W rows [256 t + 128 c, +128) and, of every N piece, the h
//                rows [piece + 128 c, +128).  Accumulator rows 128 c .. 128 c + 127 live in CTA c's tensor memory;
//                each CTA's epilogue writes its own rows of z.
//
// Protocol (cluster of 2; "leader" = CTA 0 issues the MMAs and owns the barriers the issuer waits on):
//   full[s]      in the leader, 1 arrival (its producer's expect_tx of BOTH CTAs' bytes); both CTAs' TMA loads count
//                their bytes on it (cp.async.bulk.tensor.cta_group::2 with the peer bit of the barrier address cleared)
//   empty[s]     in each CTA, signalled by the leader's tcgen05.commit multicast to both: both producers reuse stage s
//   acc_full     in each CTA, commit multicast; acc_empty in the leader, 8 arrivals (4 epilogue warps x 2 CTAs)
#include <cuda_fp16.h>
#include <string.h>

#include "tts_common.cuh"
#include "tts_tc_epi.cuh"
#include "tts_tc_ptx.cuh"
#include "tts_tc_state.h"

namespace tts {
namespace {

constexpr int kPThreads = 256;      // warp 0 TMA producer, 1 MMA issuer (leader), 2 TMEM allocator, 4-7 epilogue
constexpr int kPATile = 128 * kKC * 2;   // 16 KB: this CTA's [128 x 64] K-major A tile
constexpr int kPMaxStages = 6;
constexpr int kPNMax = 256;
constexpr int kPSmemBudget = 208 * 1024;
constexpr int kPSmemLimit = 232448;   // 227 KB

struct PairBars {
  uint64_t full[kPMaxStages];
  uint64_t empty[kPMaxStages];
  uint64_t acc_full;
  uint64_t acc_empty;
  uint64_t done;       // epilogue warps finished (watchdog)
  uint32_t tmem_slot;
};

struct PairLogitsParams {
  float* z;
  int z_ld, V;
  int n_pt;        // pair tiles: ceil(V / 256)
  int k_chunks;    // d / 64
  int T16, T;      // padded rows (MMA N) and the caller's rows: rows >= T are computed but never stored
  int n_pieces;    // ceil(T16 / 256)
  int stages;
  // work split: `n_rounds` rounds of whole tiles (tile = pair + round * n_pairs, below n_main), then the `n_left`
  // tiles from n_main on are cut along K into two halves each (594 tiles over 74 pairs would otherwise be 8.03 waves
  // rounding to 9); the two partial sums are accumulated into the zeroed z columns with fp32 RED (order-free)
  int n_rounds, n_main, n_left;
};

struct PairItem {
  int pt, c_beg, c_end;
  bool partial;
};

struct PairWalk {
  int pair, n_pairs, round;
  long u, u_end;
  __device__ PairWalk(const PairLogitsParams& p, int pair_, int n_pairs_) : pair(pair_), n_pairs(n_pairs_), round(0) {
    // every leftover tile is cut ONCE, in the middle of K: 2 n_left <= n_pairs halves, one per pair.  A z entry then
    // receives exactly two partial sums, and 0 + a + b does not depend on their order: z, hence the loss and the
    // weights, are bit-reproducible run to run.  (Cutting the leftovers over all pairs gave ~n_pairs / n_left
    // unordered fp32 addends per entry for 0.03 ms.)
    const long U = (long)p.n_left * p.k_chunks;
    const int n_cut = 2 * p.n_left;
    u = pair < n_cut ? U * pair / n_cut : 0;
    u_end = pair < n_cut ? U * (pair + 1) / n_cut : 0;
  }
  __device__ bool next(const PairLogitsParams& p, PairItem& w) {
    while (round < p.n_rounds) {
      const int pt = pair + round * n_pairs;
      ++round;
      if (pt < p.n_main) { w.pt = pt; w.c_beg = 0; w.c_end = p.k_chunks; w.partial = false; return true; }
    }
    if (u >= u_end) return false;
    const int t = (int)(u / p.k_chunks);
    w.c_beg = (int)(u - (long)t * p.k_chunks);
    const long rest = u_end - u;
    w.c_end = rest < p.k_chunks - w.c_beg ? w.c_beg + (int)rest : p.k_chunks;
    w.pt = p.n_main + t;
    w.partial = true;
    u += w.c_end - w.c_beg;
    return true;
  }
};

constexpr uint32_t kDescHiSw128 = (1024u >> 4) | (1u << 14) | (ptx::kSwizzle128B << 29);
__device__ __forceinline__ uint32_t desc_lo_sw128(uint32_t smem_addr) { return ((smem_addr >> 4) & 0x3FFFu) | (1u << 16); }
__device__ __forceinline__ uint64_t desc64(uint32_t hi, uint32_t lo) { return (static_cast<uint64_t>(hi) << 32) | lo; }

// TB: bf16 teacher (TMA-staged tiles for the fused a3 statistics of tts_tc_epi.cuh; fp32 teachers use vector loads)
template <bool TB>
__global__ void __launch_bounds__(kPThreads, 1)
tc_logits_pair_kernel(const __grid_constant__ CUtensorMap tm_W, const __grid_constant__ CUtensorMap tm_h,
                      const __grid_constant__ CUtensorMap tm_teacher, const PairLogitsParams p, const epi::Params ep) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = ptx::align_smem_1024(smem_raw);
  const int piece_bytes = 128 * kKC * 2;                      // this CTA's 128 rows of one N piece: 16 KB
  const int stage_bytes = kPATile + p.n_pieces * piece_bytes;
  PairBars* bars = reinterpret_cast<PairBars*>(smem + p.stages * stage_bytes);
  uint8_t* epi_base = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(bars + 1) + 127) & ~uintptr_t(127));
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t cta = ptx::cluster_ctarank();
  const int pair = blockIdx.x >> 1, n_pairs = gridDim.x >> 1;

  if (warp == 0 && lane == 0) {
    ptx::prefetch_tensormap(&tm_W);
    ptx::prefetch_tensormap(&tm_h);
  }
  if (warp == 1 && lane == 0) {
    for (int i = 0; i < p.stages; ++i) { ptx::mbar_init(&bars->full[i], 1); ptx::mbar_init(&bars->empty[i], 1); }
    ptx::mbar_init(&bars->acc_full, 1);
    ptx::mbar_init(&bars->acc_empty, 8);
    ptx::mbar_init(&bars->done, 4);
    ptx::fence_barrier_init();
  }
  if (warp == 2) {
    ptx::tmem_alloc_pair(&bars->tmem_slot, 512);
    ptx::tmem_relinquish_pair();
  }
  ptx::tc_fence_before();
  ptx::cluster_sync();
  ptx::tc_fence_after();
  const uint32_t tmem_base = bars->tmem_slot;

  if (warp == 0) {
    // ===== TMA producer (both CTAs): own W rows + own half of every h piece; bytes counted on the leader's barrier =====
    if (lane == 0) {
      uint32_t n = 0;
      PairWalk walk(p, pair, n_pairs);
      PairItem w;
      while (walk.next(p, w)) {
        const int v0 = w.pt * 256 + (int)cta * 128;           // rows beyond V: zero fill
        for (int kc = w.c_beg; kc < w.c_end; ++kc, ++n) {
          const int s = n % p.stages;
          ptx::mbar_wait(&bars->empty[s], ((n / p.stages) & 1) ^ 1);
          uint8_t* A = smem + s * stage_bytes;
          if (cta == 0) ptx::mbar_expect_tx(&bars->full[s], 2 * stage_bytes);
          ptx::tma_load_2d_pair(A, &tm_W, &bars->full[s], kc * kKC, v0);
          ptx::tma_load_2d_pair(A + kPATile / 2, &tm_W, &bars->full[s], kc * kKC, v0 + 64);
          for (int q = 0; q < p.n_pieces; ++q) {
            const int nn = min(kPNMax, p.T16 - q * kPNMax);   // this CTA supplies rows [nn / 2 * cta, + nn / 2) of the piece
            ptx::tma_load_2d_pair(A + kPATile + q * piece_bytes, &tm_h, &bars->full[s], kc * kKC,
                                  q * kPNMax + (int)cta * (nn / 2));
          }
        }
      }
    }
  } else if (warp == 1) {
    // ===== MMA issuer: leader only =====
    if (cta == 0 && lane == 0) {
      const uint32_t smem0 = ptx::smem_u32(smem);
      uint32_t n = 0, it = 0;
      PairWalk walk(p, pair, n_pairs);
      PairItem w;
      for (; walk.next(p, w); ++it) {
        ptx::mbar_wait_cluster(&bars->acc_empty, (it & 1) ^ 1);
        ptx::tc_fence_after();
        for (int kc = w.c_beg; kc < w.c_end; ++kc, ++n) {
          const int s = n % p.stages;
          ptx::mbar_wait(&bars->full[s], (n / p.stages) & 1);
          ptx::tc_fence_after();
          const uint32_t a_lo = desc_lo_sw128(smem0 + s * stage_bytes);
#pragma unroll
          for (int ks = 0; ks < kKC / 16; ++ks) {
            for (int q = 0; q < p.n_pieces; ++q) {
              const int nn = min(kPNMax, p.T16 - q * kPNMax);
              const uint32_t b_lo = desc_lo_sw128(smem0 + s * stage_bytes + kPATile + q * piece_bytes);
              ptx::mma_f16_ss_pair(tmem_base + q * kPNMax, desc64(kDescHiSw128, a_lo + 2 * ks),
                                   desc64(kDescHiSw128, b_lo + 2 * ks), ptx::make_idesc_bf16(256, nn, 0, 0),
                                   (kc != w.c_beg) | ks);
            }
          }
          ptx::mma_commit_pair(&bars->empty[s]);
        }
        ptx::mma_commit_pair(&bars->acc_full);
      }
    }
  } else if (warp >= 4) {
    // ===== epilogue (both CTAs): thread = one vocabulary row of this CTA's half of the tile.  Whole tiles also feed
    // the fused a3 statistics; the K-split leftover tiles are only accumulated into z (fix-up sweep of tts_stats.cu) =====
    const int q4 = warp & 3;
    const int tid_e = threadIdx.x - 128;
    const epi::Shared esh(epi_base, p.T16);
    if (ep.enabled) epi::init(esh, p.T16, tid_e);
    uint32_t it = 0, g = 0;
    PairWalk walk(p, pair, n_pairs);
    PairItem w;
    for (; walk.next(p, w); ++it) {
      ptx::mbar_wait(&bars->acc_full, it & 1);
      ptx::tc_fence_after();
      const int v0 = w.pt * 256 + (int)cta * 128;
      const uint32_t tmem_tile = tmem_base + (static_cast<uint32_t>(q4 * 32) << 16);
      auto release = [&]() {
        ptx::tc_fence_before();
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive_cta0(&bars->acc_empty);
      };
      if (ep.enabled && !w.partial && v0 < p.V) {
        epi::tile<TB>(ep, esh, &tm_teacher, tmem_tile, v0, p.T16, p.z, p.z_ld, tid_e, g, release);
        continue;
      }
      const int v = v0 + q4 * 32 + lane;
      float* zc = p.z + v;
      for (int c0 = 0; c0 < p.T16; c0 += 16) {
        uint32_t r[16];
        ptx::tmem_ld_32x32b_x16(tmem_tile + c0, r);
        ptx::tmem_ld_wait();
        if (v < p.V) {
          if (w.partial) {
#pragma unroll
            for (int i = 0; i < 16; ++i)
              if (c0 + i < p.T) atomicAdd(zc + (size_t)(c0 + i) * p.z_ld, __uint_as_float(r[i]));
          } else {
#pragma unroll
            for (int i = 0; i < 16; ++i)
              if (c0 + i < p.T) zc[(size_t)(c0 + i) * p.z_ld] = __uint_as_float(r[i]);
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
  ptx::cluster_sync();
  if (warp == 2) {
    ptx::tc_fence_after();
    ptx::tmem_dealloc_pair(tmem_base, 512);
  }
}

}  // namespace

cudaError_t tc_pair_init(tts_ctx* c) {
  if (cudaError_t w = ptx::set_watchdog_cycles(c->watchdog_cycles)) return w;
  cudaError_t e = cudaFuncSetAttribute(tc_logits_pair_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kPSmemLimit);
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(tc_logits_pair_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, kPSmemLimit);
}

// 1 when the pair kernels serve this step: several canvases beyond one MMA's N, an even grid of at least one pair
int tc_pair_eligible(const tts_ctx* c, int T16) {
  if (T16 <= kPNMax || T16 > 512) return 0;
  const int grid = c->cfg.max_ctas > 0 ? c->cfg.max_ctas : c->sm_count;
  return grid >= 2;
}

cudaError_t tc_launch_logits_pair(tts_ctx* c, const StepArgs& a, float* z_out, bool fuse_stats, cudaStream_t s,
                                  int* launches, int* n_split_out) {
  TcState* st = static_cast<TcState*>(c->tc_state);
  const int V = c->cfg.V, d = c->cfg.d, T = a.T;
  const int T16 = (T + 15) / 16 * 16;
  const bool tb = c->cfg.logits_dtype == TTS_BF16;
  *n_split_out = 0;
  PairLogitsParams p;
  p.z = z_out; p.z_ld = V; p.V = V;
  p.n_pt = (V + 255) / 256;
  p.k_chunks = d / kKC;
  p.T16 = T16; p.T = T;
  p.n_pieces = (T16 + kPNMax - 1) / kPNMax;
  const int stage_bytes = kPATile + p.n_pieces * 128 * kKC * 2;
  const int epi_bytes = fuse_stats ? 128 + epi::smem_bytes(T16) : 0;
  p.stages = ((fuse_stats ? kPSmemLimit : kPSmemBudget) - (int)sizeof(PairBars) - 1024 - epi_bytes) / stage_bytes;
  if (p.stages > kPMaxStages) p.stages = kPMaxStages;
  if (p.stages < 2) return cudaErrorInvalidConfiguration;
  CUtensorMap tm_W, tm_h, tm_t;
  if (make_map_2d(st, &tm_W, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, a.W_in, d, V, kKC, 64,
                  CU_TENSOR_MAP_SWIZZLE_128B) != CUDA_SUCCESS)
    return cudaErrorInvalidValue;
  // rows >= T of a box are out of bounds: TMA fills them with zeros
  if (make_map_2d(st, &tm_h, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, a.h, d, T, kKC, 128,
                  CU_TENSOR_MAP_SWIZZLE_128B) != CUDA_SUCCESS)
    return cudaErrorInvalidValue;
  tm_t = tm_h;
  if (fuse_stats && tb &&
      make_map_2d(st, &tm_t, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, a.teacher, V, T, 128, epi::kRows,
                  CU_TENSOR_MAP_SWIZZLE_NONE) != CUDA_SUCCESS)
    return cudaErrorInvalidValue;
  int grid = tc_logits_ctas(c);
  grid &= ~1;
  if (grid > 2 * p.n_pt) grid = 2 * p.n_pt;
  const int n_pairs = grid / 2;
  p.n_rounds = p.n_pt / n_pairs;
  p.n_left = p.n_pt % n_pairs;
  if (p.n_left > n_pairs / 2) { p.n_rounds += 1; p.n_left = 0; }   // a nearly full last round: whole tiles
  p.n_main = p.n_pt - p.n_left;
  int cut[kStatFixMax], n_cut = 0;
  if (p.n_left > 0) {
    // the K-split tiles accumulate into zeroed columns [256 n_main, V) of z; their statistics come from the fix-up sweep
    const size_t v_left = (size_t)p.n_main * 256;
    cudaError_t e = cudaMemset2DAsync(z_out + v_left, (size_t)V * sizeof(float), 0, (V - v_left) * sizeof(float), T, s);
    if (e != cudaSuccess) return e;
    for (size_t v = v_left; v < (size_t)V; v += 128) {
      if (n_cut == kStatFixMax) return cudaErrorInvalidConfiguration;   // unreachable: <= grid / 2 tiles, grid <= kStatFixMax
      cut[n_cut++] = (int)v;
    }
  }
  epi::Params ep;
  ep.teacher = a.teacher; ep.part = c->stat_part; ep.n_split = grid + n_cut; ep.T = T; ep.V = V;
  ep.enabled = fuse_stats ? 1 : 0;
  cudaLaunchConfig_t cfg;
  memset(&cfg, 0, sizeof(cfg));
  cfg.gridDim = dim3(grid);
  cfg.blockDim = dim3(kPThreads);
  cfg.dynamicSmemBytes = 1024 + (size_t)p.stages * stage_bytes + sizeof(PairBars) + epi_bytes;
  cfg.stream = s;
  cudaLaunchAttribute attr;
  attr.id = cudaLaunchAttributeClusterDimension;
  attr.val.clusterDim.x = 2; attr.val.clusterDim.y = 1; attr.val.clusterDim.z = 1;
  cfg.attrs = &attr;
  cfg.numAttrs = 1;
  cudaError_t e = tb ? cudaLaunchKernelEx(&cfg, tc_logits_pair_kernel<true>, tm_W, tm_h, tm_t, p, ep)
                     : cudaLaunchKernelEx(&cfg, tc_logits_pair_kernel<false>, tm_W, tm_h, tm_t, p, ep);
  *launches += 1;
  if (e != cudaSuccess || !fuse_stats) return e;
  if (n_cut > 0) e = launch_row_stats_tiles(c, a, z_out, V, cut, n_cut, grid, ep.n_split, s, launches);
  *n_split_out = ep.n_split;
  return e;
}

}  // namespace tts
