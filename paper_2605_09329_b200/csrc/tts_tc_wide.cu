// Pass B of the distillation step for MORE than one canvas (16 < T <= 512 rows, SURVEY 8(a) a4 + a6 + a7), and for
// one-canvas shapes whose hidden size is not a multiple of the fused kernel's 1024-column stripe.
//
// Why it differs from tts_tc_fused.cu.  gW = dl^T h is a rank-T update: at T = 512 every [128 j x N v] tile of gW
// needs (128 + N) x 512 operand values, and an operand that is re-fetched per tile costs as much L2 -> SM traffic as
// the optimiser state itself costs HBM traffic (the first version of this kernel re-read 512 KB of operands per
// 426 KB of state and ran at 4.1 TB/s).  So here
//   * a CTA owns one 128-column stripe of the parameter matrix at a time and keeps the stripe's h^T operand
//     [128 j x Kp] RESIDENT in tensor memory (tcgen05.mma with A from TMEM; 256 of the 512 columns at T = 512), which
//     leaves all of shared memory to the state ring (resident in shared memory instead, the ring shrinks to two
//     stages: measured 4.35 ms against 3.07);
//   * dl is ONE 16-bit plane: fp16 with a power-of-two scale chosen from the row coefficients (|dl S| <= 2^14), i.e.
//     11 significant bits against bf16's 8 (one bf16 plane misses the 2e-3 max|gW| bar on rows with a dominant
//     entry; the hi/lo bf16 split of the one-canvas kernel would double K).  kind::f16 wants A and B in the same
//     format (a bf16 x fp16 MMA traps as an illegal instruction on sm_100a), so h^T is converted to fp16 as well:
//     exact for bf16 inputs after a power-of-two scale S_h from max|h| (|h S_h| <= 2^14; only values below
//     2^-28 max|h| lose bits).  The epilogue multiplies the accumulator by 1 / (S S_h) (exact);
//   * per band of NV vocabulary rows the only operand traffic is the band's dl rows [NV x Kp] (8 B per parameter
//     at T = 512 against 26 B of state);
//   * work is cut in one of two ways (tc_launch_update_wide): a FIXED-STRIPE walk when the grid is (nearly) a multiple of
//     the stripe count -- every CTA keeps one stripe for the whole pass and takes every (grid / n_stripes)-th band, so
//     the CTAs of a phase sweep the same vocabulary rows and their 512-byte row segments add up to whole rows at the
//     memory controllers --, else windowed stream-K: the vocabulary is cut into windows whose dl rows (<= 12 MB) stay in L2
//     (evict_last) while every stripe passes over them; inside a window the (stripe, band) units, stripe-major, are
//     split into gridDim equal contiguous ranges, so the grid is balanced to one band for any SM budget and a CTA
//     changes stripe (reloads A) at most twice per window.
// The state moves as in the fused kernel: TMA loads of [16 v x 128 j] sub-tiles of master / m / v into a ring,
// AdamW applied in place in shared memory (a thread updates its column of a sub-tile in two halves of 8 rows, so that one
// barrier round and one set of TMA stores serve 16 rows: the bf16-moment pass, which is bound by these warps, gains 3%),
// TMA stores of the three tensors and the bf16 working copy.
#include <cuda_fp16.h>
#include <string.h>

#include "tts_adam.cuh"
#include "tts_common.cuh"
#include "tts_tc_ptx.cuh"
#include "tts_tc_state.h"

namespace tts {
namespace {

constexpr int kWJ = 128;                 // stripe width = MMA M = TMEM lanes
constexpr int kWSV = 16;                 // vocabulary rows per state stage (= sub-tile: one barrier round, one set of TMA stores)
constexpr int kWH = 8;                   // rows a thread holds at a time: a sub-tile is updated in two halves
constexpr int kWTensorBytes = kWSV * kWJ * 4;   // 8 KB per tensor per stage
constexpr int kWStageBytes = 3 * kWTensorBytes; // 24 KB (fp32 moments)
constexpr int kWMomBytesLp = kWSV * kWJ * 2;    // 4 KB per bf16 moment tensor per stage
constexpr int kWStageBytesLp = kWTensorBytes + 2 * kWMomBytesLp;   // 16 KB (bf16 moments, TTS_MOMENT_BF16)
constexpr int kWWoBytes = kWSV * kWJ * 2;       // 4 KB: bf16 staging of one sub-tile (one per epilogue group)
constexpr int kWThreads = 384;           // warp 0 state TMA, 1 MMA, 2 TMEM alloc, 3 operand TMA, 4-11 epilogue
constexpr int kWMaxStages = 24;
constexpr int kWOpStagesMax = 4;         // dl band ring (depth chosen per launch)
constexpr int kWSmemBudget = 225 * 1024;
constexpr int kWAccCols = 64;            // TMEM columns reserved for the two gW accumulators (NV <= 32)
constexpr long kWWindowBytes = 12l << 20;
constexpr int kWGhCol0 = 192;            // GH: first TMEM column of the gh accumulators (h^T ends at 64 + 128 = 192)
constexpr int kWGhMaxN = 256;            // GH: most canvas rows (x dl planes) whose gh accumulators fit next to h^T
constexpr int kWWtBytes = kWJ * 32 * 2;  // GH: the band's W^T tile [128 j x 32 v] fp16 (A operand of gh), 8 KB

struct WideParams {
  float* gW_debug;
  const uint16_t* hTT;        // [d, Kp] fp16 bits
  const float* dl_scale;      // {S, 1 / S, S_h, 1 / S_h}
  float* gh;                  // GH: [T, d] fp32, zeroed; this kernel adds its parts with fp32 RED
  int T, T16, planes;         // GH: rows, padded rows, dl planes stacked along K (the gh accumulators have planes * T16 columns)
  int V, d, Kp;
  int n_stripes, n_bands, n_win, stages, op_stages;
  int fixed;                  // 1: every CTA keeps ONE stripe (grid % n_stripes == 0) and takes every (grid / n_stripes)-th band
  const float* step_scalars;  // device {1 / (1 - b1^n), 1 / sqrt(1 - b2^n)} of this step
  const unsigned long long* step_count;   // device: Adam's count n of this step (keys the stochastic rounding of v)
  uint32_t sr_seed;
  float lr, b1, b2, eps, decay;   // decay = 1 - lr wd
};

struct WideBars {
  uint64_t st_full[kWMaxStages];
  uint64_t st_empty[kWMaxStages];
  uint64_t op_full[kWOpStagesMax];
  uint64_t op_empty[kWOpStagesMax];
  uint64_t acc_full[2];
  uint64_t acc_empty[2];
  uint64_t a_full;
  uint64_t wt_full, wt_empty, gh_full, gh_empty;   // GH
  uint64_t done;       // epilogue warps finished (watchdog)
  uint32_t tmem_slot;
};

// The sequence of (stripe, band) units of this CTA: window by window, a contiguous range of each window's units --
// the SAME relative range in every window, walked forwards in even windows and backwards in odd ones, so that a
// window ends in the stripe the next one starts in and h^T is reloaded only where a range crosses a stripe boundary.
struct WideWalk {
  int n_stripes, n_bands, n_win;
  int win, wb0, wbn;
  int left;            // units of the current window still to hand out
  int cs, cb, dir;     // next unit: stripe, band within the window, direction (+1 even windows, -1 odd ones)
  int fixed, fstep;    // fixed-stripe walk: cs = the CTA's stripe, cb = its next band, fstep = CTAs per stripe
  __device__ WideWalk(const WideParams& p) : n_stripes(p.n_stripes), n_bands(p.n_bands), n_win(p.n_win), win(-1),
                                             wb0(0), wbn(1), left(0), cs(0), cb(0), dir(1), fixed(p.fixed), fstep(1) {
    if (fixed) {
      cs = blockIdx.x % n_stripes;
      cb = blockIdx.x / n_stripes;
      fstep = gridDim.x / n_stripes;
    }
  }
  // one 64-bit division per window; inside a window the walk is increments only (every role calls this once per band,
  // the epilogue threads included)
  __device__ bool get(int& stripe, int& band) {
    if (fixed) {
      if (cb >= n_bands) return false;
      stripe = cs;
      band = cb;
      cb += fstep;
      return true;
    }
    while (left == 0) {
      if (++win >= n_win) return false;
      wb0 = (int)((long)n_bands * win / n_win);
      wbn = (int)((long)n_bands * (win + 1) / n_win) - wb0;
      const long units = (long)n_stripes * wbn;
      const long u_lo = units * blockIdx.x / gridDim.x, u_hi = units * (blockIdx.x + 1) / gridDim.x;
      left = (int)(u_hi - u_lo);
      dir = (win & 1) ? -1 : 1;
      const long u = dir > 0 ? u_lo : u_hi - 1;
      cs = (int)(u / wbn);
      cb = (int)(u - (long)cs * wbn);
    }
    stripe = cs;
    band = wb0 + cb;
    cb += dir;
    if (cb == wbn) { cb = 0; ++cs; }
    else if (cb < 0) { cb = wbn - 1; --cs; }
    --left;
    return true;
  }
};

constexpr uint32_t kDescHiSw128 = (1024u >> 4) | (1u << 14) | (ptx::kSwizzle128B << 29);
__device__ __forceinline__ uint32_t desc_lo_sw128(uint32_t smem_addr) { return ((smem_addr >> 4) & 0x3FFFu) | (1u << 16); }
__device__ __forceinline__ uint64_t desc64(uint32_t hi, uint32_t lo) { return (static_cast<uint64_t>(hi) << 32) | lo; }

// GH (planes * T16 <= 256): gh^T[j, r] += W_in[v, j] dl[r, v] is formed here as well, as in the one-canvas kernel: the
// band's W_in tile is re-derived from the master values the epilogue holds (precondition W_in == rn_bf16(W_master)),
// written to shared memory as fp16(16 W) (the A operand), the dl band already in shared memory is read a second
// time as the MN-major B operand, and the stripe's accumulators [128 j x planes T16] persist in tensor memory until
// the CTA leaves the stripe.  No gh kernel, no second pass over W.
// MOM: 1 = bf16 moments (TTS_MOMENT_BF16; stages of 8 KB; m nearest-even, v stochastic rounding: tts_adam.cuh)
template <bool ADAM, int NV, bool GH, int MOM>
__global__ void __launch_bounds__(kWThreads, 1)
tc_update_wide_kernel(const __grid_constant__ CUtensorMap tm_dlT,
                      const __grid_constant__ CUtensorMap tm_master, const __grid_constant__ CUtensorMap tm_m,
                      const __grid_constant__ CUtensorMap tm_v, const __grid_constant__ CUtensorMap tm_wout,
                      const WideParams p) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = ptx::align_smem_1024(smem_raw);
  constexpr int kSubs = NV / kWSV;
  constexpr int kStageB = MOM ? kWStageBytesLp : kWStageBytes;
  constexpr int kMomB = MOM ? kWMomBytesLp : kWTensorBytes;
  const int b_bytes = NV * p.Kp * 2;                   // [Kp / 64][NV v][64 k] fp16, 128-byte swizzle
  uint8_t* sB = smem;
  const int kWOpStages = p.op_stages;
  uint8_t* st = sB + kWOpStages * b_bytes;             // [stages][3][16 v][128 j] fp32
  uint8_t* wo = st + p.stages * kStageB;               // [2 groups][16 v][128 j] bf16
  uint8_t* wt = wo + 2 * kWWoBytes;                    // GH: [4 v-groups][16 j-groups][8 j][8 v] fp16, K-major core matrices
  WideBars* bars = reinterpret_cast<WideBars*>(wt + (GH ? kWWtBytes : 0));

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int nks = p.Kp / 16;                           // MMA K steps per band

  if (warp == 0 && lane == 0) {
    ptx::prefetch_tensormap(&tm_master);
    if (ADAM) { ptx::prefetch_tensormap(&tm_m); ptx::prefetch_tensormap(&tm_v); }
    ptx::prefetch_tensormap(&tm_wout);
  }
  if (warp == 3 && lane == 0) {
    ptx::prefetch_tensormap(&tm_dlT);
  }
  if (warp == 1 && lane == 0) {
    for (int i = 0; i < p.stages; ++i) { ptx::mbar_init(&bars->st_full[i], 1); ptx::mbar_init(&bars->st_empty[i], 1); }
    for (int i = 0; i < kWOpStages; ++i) { ptx::mbar_init(&bars->op_full[i], 1); ptx::mbar_init(&bars->op_empty[i], 1); }
    for (int i = 0; i < 2; ++i) { ptx::mbar_init(&bars->acc_full[i], 1); ptx::mbar_init(&bars->acc_empty[i], 8); }
    ptx::mbar_init(&bars->a_full, 8);
    ptx::mbar_init(&bars->wt_full, 8);
    ptx::mbar_init(&bars->wt_empty, 1);
    ptx::mbar_init(&bars->gh_full, 1);
    ptx::mbar_init(&bars->gh_empty, 4);
    ptx::mbar_init(&bars->done, 8);
    ptx::fence_barrier_init();
  }
  if (warp == 2) {
    ptx::tmem_alloc(&bars->tmem_slot, 512);
    ptx::tmem_relinquish();
  }
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  const uint32_t tmem_base = bars->tmem_slot;
  const uint32_t tmem_A = tmem_base + kWAccCols;       // Kp / 2 columns: h^T of the stripe, K packed in pairs

  if (warp == 0) {
    // ===== optimiser-state producer: [16 v x 128 j] of master / m / v per stage =====
    if (lane == 0) {
      const uint64_t pol = ptx::policy_evict_first();
      WideWalk w(p);
      int ps = 0;
      uint32_t pph = 0, n = 0;
      int stripe, band;
      while (w.get(stripe, band)) {
        const int j0 = stripe * kWJ, v0 = band * NV;
        for (int sub = 0; sub < kSubs; ++sub, ++n) {
          int s;
          uint32_t ph;
          if (GH) { s = ps; ph = pph; if (++ps == p.stages) { ps = 0; pph ^= 1; } }
          else { s = n % p.stages; ph = (n / p.stages) & 1; }   // see the epilogue for why the two instances differ
          ptx::mbar_wait(&bars->st_empty[s], ph ^ 1);
          uint8_t* dst = st + s * kStageB;
          ptx::mbar_expect_tx(&bars->st_full[s], ADAM ? kWTensorBytes + 2 * kMomB : kWTensorBytes);
          const int r0 = v0 + sub * kWSV;
          ptx::tma_load_2d_hint(dst, &tm_master, &bars->st_full[s], j0, r0, pol);
          if (ADAM) {
            ptx::tma_load_2d_hint(dst + kWTensorBytes, &tm_m, &bars->st_full[s], j0, r0, pol);
            ptx::tma_load_2d_hint(dst + kWTensorBytes + kMomB, &tm_v, &bars->st_full[s], j0, r0, pol);
          }
        }
      }
    }
  } else if (warp == 3) {
    // ===== operand producer: the band's dl rows [NV v x Kp] =====
    if (lane == 0) {
      const uint64_t pol = ptx::policy_evict_last();
      WideWalk w(p);
      uint32_t i = 0;
      int stripe, band;
      while (w.get(stripe, band)) {
        const int s = i % kWOpStages;
        ptx::mbar_wait(&bars->op_empty[s], ((i / kWOpStages) & 1) ^ 1);
        ptx::mbar_expect_tx(&bars->op_full[s], b_bytes);
        for (int c = 0; c < p.Kp / kKC; ++c)
          ptx::tma_load_2d_hint(sB + s * b_bytes + c * (NV * 128), &tm_dlT, &bars->op_full[s], c * kKC, band * NV, pol);
        ++i;
      }
    }
  } else if (warp == 1) {
    // ===== MMA issuer: acc[j, v] = sum_r h^T[j, r] (S dl)[r, v]   (M = 128, N = NV, K = 16 per instruction) =====
    if (lane == 0) {
      constexpr uint32_t idesc = ptx::make_idesc_f16(kWJ, NV, ptx::kFmtF16, ptx::kFmtF16, 0, 0);
      const uint32_t sB0 = ptx::smem_u32(sB);
      WideWalk w(p);
      uint32_t i = 0, a_n = 0;
      int stripe, band, cur = -1;
      // GH: gh MMAs of band i are issued after the gW MMAs of band i + 1 (the epilogue produces their A operand while
      // it drains band i's accumulator), and before the CTA leaves a stripe
      const int n_gh = p.planes * p.T16;
      const uint32_t idesc_gh = ptx::make_idesc_f16(kWJ, n_gh, ptx::kFmtF16, ptx::kFmtF16, 0, 1);   // A K-major, B MN-major
      const uint32_t wt0 = ptx::smem_u32(wt);
      bool pending = false, first_gh = true;
      uint32_t i_prev = 0;
      auto issue_gh = [&]() {
        ptx::mbar_wait(&bars->wt_full, i_prev & 1);
        ptx::tc_fence_after();
        const uint32_t b_base = sB0 + (i_prev % kWOpStages) * b_bytes;
#pragma unroll
        for (int ks = 0; ks < NV / 16; ++ks) {
          // A: W^T tile, K-major, no swizzle: core matrices [8 j x 8 v]; j-groups 128 B apart (SBO), v-groups 2 KB (LBO)
          const uint64_t ad = ptx::make_smem_desc(wt0 + ks * 4096, 2048, 128, 0);
          // B: the dl band read MN-major (N = canvas row, contiguous in the 128-byte rows; K = vocabulary row):
          // 16 k rows = 2 KB per step, 8-row groups 1 KB apart (SBO), 64-row blocks of N one K chunk apart (LBO)
          const uint64_t bd = ptx::make_smem_desc(b_base + ks * 2048, NV * 128, 1024, ptx::kSwizzle128B);
          ptx::mma_f16_ss(tmem_base + kWGhCol0, ad, bd, idesc_gh, (first_gh ? 0u : 1u) | ks);
        }
        first_gh = false;
        ptx::mma_commit(&bars->wt_empty);
        ptx::mma_commit(&bars->op_empty[i_prev % kWOpStages]);
        pending = false;
      };
      while (w.get(stripe, band)) {
        if (stripe != cur) {
          if (GH && cur >= 0) {
            if (pending) issue_gh();
            ptx::mma_commit(&bars->gh_full);             // the old stripe's accumulators are complete
          }
          ptx::mbar_wait(&bars->a_full, a_n & 1);
          ptx::tc_fence_after();
          if (GH && cur >= 0) {                          // ... and flushed: the new stripe starts from zero
            ptx::mbar_wait(&bars->gh_empty, (a_n - 1) & 1);
            ptx::tc_fence_after();
            first_gh = true;
          }
          ++a_n;
          cur = stripe;
        }
        const int ab = i & 1, s = i % kWOpStages;
        ptx::mbar_wait(&bars->acc_empty[ab], ((i >> 1) & 1) ^ 1);
        ptx::mbar_wait(&bars->op_full[s], (i / kWOpStages) & 1);
        ptx::tc_fence_after();
        const uint32_t d_tmem = tmem_base + ab * NV;
        const uint32_t b_base = sB0 + s * b_bytes;
        for (int ks = 0; ks < nks; ++ks) {
          const uint32_t b_lo = desc_lo_sw128(b_base + (ks >> 2) * (NV * 128)) + 2 * (ks & 3);
          ptx::mma_f16_ts(d_tmem, tmem_A + ks * 8, desc64(kDescHiSw128, b_lo), idesc, ks);
        }
        if (!GH) ptx::mma_commit(&bars->op_empty[s]);
        ptx::mma_commit(&bars->acc_full[ab]);
        if (GH) {
          if (pending) issue_gh();
          i_prev = i;
          pending = true;
        }
        ++i;
      }
      if (GH && cur >= 0) {
        if (pending) issue_gh();
        ptx::mma_commit(&bars->gh_full);
      }
    }
  } else if (warp >= 4) {
    // ===== epilogue: 2 groups x 4 warps; group g takes sub-tiles sub % 2 == g; warp quarter q owns TMEM lanes 32q.. =====
    const int q = warp & 3, g = (warp - 4) >> 2;
    const int jj = q * 32 + lane;              // hidden column of the stripe = TMEM lane
    const bool leader = jj == 0;               // issues the group's TMA stores and releases its state stages
    const uint32_t lane_bits = static_cast<uint32_t>(q * 32) << 16;
    __nv_bfloat16* wo_g = reinterpret_cast<__nv_bfloat16*>(wo + g * kWWoBytes);
    const float inv_s = p.dl_scale[1] * p.dl_scale[3];
    const float c1 = ADAM ? p.lr * p.step_scalars[0] : 0.f, inv_sqrt_bc2 = ADAM ? p.step_scalars[1] : 0.f;
    const uint32_t key = MOM ? sr_key(static_cast<uint32_t>(*p.step_count), p.sr_seed) : 0u;
    WideWalk w(p);
    uint32_t i = 0, n_flush = 0;
    int stripe, band, cur = -1, prev_s = -1;
    int st_s = g;                 // p.stages >= 2 > g
    uint32_t st_ph = 0;           // no division by the runtime ring depth in the per-sub-tile path
    uint8_t* wt_thr = wt + (jj >> 3) * 128 + (jj & 7) * 16;   // + (v >> 3) * 2048: this thread's 16-byte chunk of 8 v
    // GH: the stripe's gh accumulators -> fp32 RED (group 0: one warp per lane quarter), then the issuer may reuse them
    auto flush_gh = [&](int stripe_done) {
      if (g != 0) return;
      ptx::mbar_wait(&bars->gh_full, n_flush & 1);
      ptx::tc_fence_after();
      const float inv_gh = p.dl_scale[1] * (1.f / 16.f);
      float* gc = p.gh + stripe_done * kWJ + jj;
      for (int c0 = 0; c0 < p.T16; c0 += 16) {
        if (c0 >= p.T) break;
        uint32_t r[16], r2[16];
        ptx::tmem_ld_32x32b_x16(tmem_base + kWGhCol0 + c0 + lane_bits, r);
        if (p.planes == 2) ptx::tmem_ld_32x32b_x16(tmem_base + kWGhCol0 + p.T16 + c0 + lane_bits, r2);
        ptx::tmem_ld_wait();
#pragma unroll
        for (int k = 0; k < 16; ++k) {
          float x = __uint_as_float(r[k]);
          if (p.planes == 2) x += __uint_as_float(r2[k]);
          if (c0 + k < p.T) atomicAdd(gc + (size_t)(c0 + k) * p.d, x * inv_gh);
        }
      }
      ptx::tc_fence_before();
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive(&bars->gh_empty);
      ++n_flush;
    };
    while (w.get(stripe, band)) {
      const int j0 = stripe * kWJ, v0 = band * NV;
      if (stripe != cur) {
        if (GH && cur >= 0) flush_gh(cur);
        // every MMA that read the old stripe is complete: this warp has waited on the previous band's acc_full.
        // hTT is tiled [stripe][K step][128 j][16 k]: a warp reads 1 KB contiguous per K step; this group writes
        // half of the K steps.
        const uint4* tile = reinterpret_cast<const uint4*>(p.hTT + ((size_t)stripe * nks * kWJ + jj) * 16);
        const int ks_end = (g + 1) * (nks / 2);
        for (int ks0 = g * (nks / 2); ks0 < ks_end; ks0 += 4) {     // four K steps of loads in flight per thread
          uint4 lo[4], hi[4];
#pragma unroll
          for (int u = 0; u < 4; ++u)
            if (ks0 + u < ks_end) {
              lo[u] = __ldg(tile + (size_t)(ks0 + u) * kWJ * 2);
              hi[u] = __ldg(tile + (size_t)(ks0 + u) * kWJ * 2 + 1);
            }
#pragma unroll
          for (int u = 0; u < 4; ++u)
            if (ks0 + u < ks_end) {
              const uint32_t r[8] = {lo[u].x, lo[u].y, lo[u].z, lo[u].w, hi[u].x, hi[u].y, hi[u].z, hi[u].w};
              ptx::tmem_st_32x32b_x8(tmem_A + (ks0 + u) * 8 + lane_bits, r);
            }
        }
        ptx::tmem_st_wait();
        ptx::tc_fence_before();
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(&bars->a_full);
        cur = stripe;
      }
      const int ab = i & 1;
      ptx::mbar_wait(&bars->acc_full[ab], (i >> 1) & 1);
      ptx::tc_fence_after();
      for (int sub = g; sub < kSubs; sub += 2) {
        // stage and phase of sub-tile n = i * kSubs + sub.  The gh-forming instance steps them (the group's stages
        // advance by 2); the other one divides by the runtime ring depth.  Measured, same box, both ways round: stepping
        // takes the gh-forming update from 2.90 to 2.77 ms at 64 rows and the plain one from 2.97 to 3.18 ms at 512
        // (an explicit delay only slows the kernels, so it is ptxas' schedule of the two codings, not pacing; the same
        // change slows the one-canvas kernel by 6%).
        int s;
        uint32_t st_par;
        if (GH) {
          s = st_s; st_par = st_ph;
          st_s += 2;
          if (st_s >= p.stages) { st_s -= p.stages; st_ph ^= 1; }
        } else {
          const uint32_t n = i * kSubs + sub;
          s = n % p.stages; st_par = (n / p.stages) & 1;
        }
        uint32_t wpk[kWSV / 2];                                  // the updated rows as bf16 pairs, for the working copy
#pragma unroll
        for (int hf = 0; hf < kWSV / kWH; ++hf) {
        uint32_t gr[kWH];
        ptx::tmem_ld_32x32b_x8(tmem_base + ab * NV + sub * kWSV + hf * kWH + lane_bits, gr);
        if (hf == 0) ptx::mbar_wait(&bars->st_full[s], st_par);
        float* sM = reinterpret_cast<float*>(st + s * kStageB) + hf * kWH * kWJ + jj;
        uint16_t* sLm = reinterpret_cast<uint16_t*>(st + s * kStageB + kWTensorBytes) + hf * kWH * kWJ + jj;   // MOM: bf16 m, then v
        uint16_t* sLv = reinterpret_cast<uint16_t*>(st + s * kStageB + kWTensorBytes + kMomB) + hf * kWH * kWJ + jj;
        float M[kWH], mm[kWH], vv[kWH];
#pragma unroll
        for (int r = 0; r < kWH; ++r) {
          M[r] = sM[r * kWJ];
          if (ADAM) {
            if (MOM) { mm[r] = bf16_bits_widen(sLm[r * kWJ]); vv[r] = bf16_bits_widen(sLv[r * kWJ]); }
            else { mm[r] = sM[kWSV * kWJ + r * kWJ]; vv[r] = sM[2 * kWSV * kWJ + r * kWJ]; }
          }
        }
        if (GH) {
          // a5 operand: W_in[v, j] = rn_bf16(master[v, j]), as fp16(16 W): eight rows of this thread's column
          if (hf == 0) ptx::mbar_wait(&bars->wt_empty, (i & 1) ^ 1);   // the gh MMAs of the previous band have read wt
          uint32_t pk[4];
#pragma unroll
          for (int r = 0; r < 4; ++r) {
            const __nv_bfloat162 b2 = __floats2bfloat162_rn(M[2 * r], M[2 * r + 1]);       // W_in = rn_bf16(master)
            const uint32_t bb = *reinterpret_cast<const uint32_t*>(&b2);
            const float lo = __uint_as_float(bb << 16) * 16.f, hi = __uint_as_float(bb & 0xFFFF0000u) * 16.f;
            // fp16(16 W), saturating (|W| >= 4094 clamps, as in tts_tc_gemm.cu)
            asm("cvt.rn.satfinite.f16x2.f32 %0, %1, %2;" : "=r"(pk[r]) : "f"(hi), "f"(lo));
          }
          *reinterpret_cast<uint4*>(wt_thr + (sub * (kWSV / kWH) + hf) * 2048) = make_uint4(pk[0], pk[1], pk[2], pk[3]);
          if (hf == kWSV / kWH - 1) {                            // both groups' sub-tiles make up the band (kSubs == 2)
            ptx::fence_proxy_async_smem();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(&bars->wt_full);
          }
        }
        ptx::tmem_ld_wait();
        // a7 in place: the thread rewrites exactly the shared-memory words it read
        uint32_t rnd = 0u;
        const int row0 = v0 + sub * kWSV + hf * kWH;
#pragma unroll
        for (int r = 0; r < kWH; ++r) {
          const float gg = __uint_as_float(gr[r]) * inv_s;
          gr[r] = __float_as_uint(gg);
          // MOM: one hash for the two rows (even, odd) of this column (tts_adam.cuh)
          if (MOM && (r & 1) == 0)
            rnd = sr_bits32((unsigned long long)((row0 + r) >> 1) * (unsigned long long)p.d + (j0 + jj), key);
          if (ADAM) {
            const float m1 = p.b1 * mm[r] + (1.f - p.b1) * gg;
            const float v1 = p.b2 * vv[r] + (1.f - p.b2) * gg * gg;
            const float den = adam_sqrt(v1) * inv_sqrt_bc2 + p.eps;
            M[r] = fmaf(-(c1 * m1), adam_rcp(den), M[r] * p.decay);     // the step uses the unrounded moments
            if (MOM) {
              sLm[r * kWJ] = bf16_bits_rn(m1);
              sLv[r * kWJ] = bf16_bits_sr(v1, (r & 1) == 0 ? rnd >> 16 : rnd & 0xFFFFu);
            } else {
              sM[kWSV * kWJ + r * kWJ] = m1;
              sM[2 * kWSV * kWJ + r * kWJ] = v1;
            }
          } else {
            M[r] = M[r] - p.lr * gg;
          }
          sM[r * kWJ] = M[r];
        }
        if (p.gW_debug) {
#pragma unroll
          for (int r = 0; r < kWH; ++r) p.gW_debug[(size_t)(row0 + r) * p.d + j0 + jj] = __uint_as_float(gr[r]);
        }
#pragma unroll
        for (int r = 0; r < kWH / 2; ++r) {
          const __nv_bfloat162 b2 = __floats2bfloat162_rn(M[2 * r], M[2 * r + 1]);
          wpk[hf * (kWH / 2) + r] = *reinterpret_cast<const uint32_t*>(&b2);
        }
        }   // halves
        // the group's previous stores have read their shared memory: release that stage, reuse the bf16 staging
        if (leader) {
          ptx::bulk_wait_group_read<0>();
          if (prev_s >= 0) ptx::mbar_arrive(&bars->st_empty[prev_s]);
        }
        ptx::named_barrier_sync(1 + g, 128);
        {
          uint16_t* wo16 = reinterpret_cast<uint16_t*>(wo_g) + jj;
#pragma unroll
          for (int r = 0; r < kWSV / 2; ++r) {
            wo16[(2 * r) * kWJ] = static_cast<uint16_t>(wpk[r] & 0xFFFFu);
            wo16[(2 * r + 1) * kWJ] = static_cast<uint16_t>(wpk[r] >> 16);
          }
        }
        ptx::fence_proxy_async_smem();
        ptx::named_barrier_sync(1 + g, 128);
        if (leader) {
          const int r0 = v0 + sub * kWSV;
          const uint8_t* sT = st + s * kStageB;
          ptx::tma_store_2d(&tm_master, sT, j0, r0);
          if (ADAM) {
            ptx::tma_store_2d(&tm_m, sT + kWTensorBytes, j0, r0);
            ptx::tma_store_2d(&tm_v, sT + kWTensorBytes + kMomB, j0, r0);
          }
          ptx::tma_store_2d(&tm_wout, wo_g, j0, r0);
          ptx::bulk_commit_group();
        }
        prev_s = s;
      }
      ptx::tc_fence_before();
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive(&bars->acc_empty[ab]);
      ++i;
    }
    if (GH && cur >= 0) flush_gh(cur);
    if (leader) ptx::bulk_wait_group_read<0>();   // shared memory must outlive the last stores' reads
    if (lane == 0) ptx::watchdog_arrive(&bars->done);
  } else if (warp == 2) {
    ptx::watchdog_wait(&bars->done);
  }
  ptx::tc_fence_before();
  __syncthreads();
  if (warp == 2) {
    ptx::tc_fence_after();
    ptx::tmem_dealloc(tmem_base, 512);
  }
}

// ------------------------------------------------------------------ a4: operands
// Power-of-two scale of a 16-bit fp16 plane whose entries are bounded by `bound`: S = 2^(14 - e) with bound <= 2^e.
__device__ __forceinline__ float pow2_scale_from_bound(float bound) {
  if (!(bound > 0.f) || !isfinite(bound)) return 1.f;
  int e;
  frexpf(bound, &e);          // bound = m 2^e, m in [0.5, 1)
  int k = 14 - e;
  k = k > 100 ? 100 : (k < -100 ? -100 : k);
  return ldexpf(1.f, k);
}

// max |h| over the T x d hidden states, as the bit pattern of a non-negative float (atomicMax on the zeroed slot)
__global__ void __launch_bounds__(256) tc_h_absmax_kernel(const __nv_bfloat16* __restrict__ h, size_t n,
                                                          unsigned int* __restrict__ out_bits) {
  __shared__ float red[32];
  float m = 0.f;
  const size_t nvec = n / 8;                     // rows of h start 16-byte aligned (d % 128 == 0 on this path)
  const uint4* hv = reinterpret_cast<const uint4*>(h);
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += (size_t)gridDim.x * blockDim.x) {
    float f[8];
    unpack_bf16x8(__ldg(hv + i), f);
#pragma unroll
    for (int k = 0; k < 8; ++k) m = fmaxf(m, fabsf(f[k]));
  }
  for (size_t i = nvec * 8 + (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
    m = fmaxf(m, fabsf(__bfloat162float(h[i])));
  m = block_max(m, red);
  if (threadIdx.x == 0) atomicMax(out_bits, __float_as_uint(m));
}

// hTT = fp16(S_h h[k, j]) for k < T (and again at k + T16 with two dl planes), 0 elsewhere up to Kp, tiled
// [j / 128][k / 16][j % 128][k % 16]: the order in which a stripe's rows go to tensor memory.  32 x 32 transpose tiles through shared memory.
__global__ void __launch_bounds__(256) tc_prep_hT_kernel(const __nv_bfloat16* __restrict__ h, int d, int T, int T16,
                                                         int planes, int Kp,
                                                         const unsigned int* __restrict__ absmax_bits,
                                                         uint16_t* __restrict__ hTT, float* __restrict__ dl_scale) {
  __shared__ uint16_t tile[32][33];
  const float Sh = pow2_scale_from_bound(__uint_as_float(*absmax_bits));
  if (blockIdx.x == 0 && blockIdx.y == 0 && threadIdx.x == 0) { dl_scale[2] = Sh; dl_scale[3] = 1.f / Sh; }
  const int j0 = blockIdx.x * 32, k0 = blockIdx.y * 32;
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
  for (int k = ty; k < 32; k += 8) {
    const int kk = k0 + k;
    const int r = (planes == 2 && kk >= T16) ? kk - T16 : kk;       // the lo plane of dl meets the same rows of h
    const float x = (r < T && kk < planes * T16 && j0 + tx < d) ? __bfloat162float(h[(size_t)r * d + j0 + tx]) : 0.f;
    tile[k][tx] = __half_as_ushort(__float2half_rn(x * Sh));
  }
  __syncthreads();
  for (int j = ty; j < 32; j += 8)
    if (j0 + j < d && k0 + tx < Kp) {
      const int jg = j0 + j, kg = k0 + tx;
      hTT[(((size_t)(jg / 128) * (Kp / 16) + kg / 16) * 128 + jg % 128) * 16 + kg % 16] = tile[tx][j];
    }
}

// dl = coef_r ((q - p) + lambda (q - q_ref)) from z, teacher and the row normalisers, scaled by S and rounded to fp16;
// one [128 v x 64 k] tile per block, two adjacent vocabulary rows per thread.  Up to 32 rows the 64-wide K chunk has room for a second plane, so dl S is
// split hi + lo (two fp16, 2^-22) at no cost in operand bytes or MMAs and the h^T operand repeats its rows.  Written twice, both coalesced: dlT[v, r] (r contiguous: the K-major B operand
// of gW; transposed through shared memory, 128-byte row segments) and dlR[r, v] (the K-major B operand of gh).
// FAST (one fp16 plane, 2^-12): ex2.approx-based __expf, error ~|x| 1e-7, far inside the plane's rounding.
template <bool BF16, bool FAST>
__global__ void __launch_bounds__(256) tc_prep_dl_wide_kernel(const void* __restrict__ teacher, const float* __restrict__ z,
                                                              const float* __restrict__ z_ref, float lam, int V,
                                                              int z_ld, int T, int T16, int planes, int Kp, int T_max,
                                                              const float* __restrict__ row_stats,
                                                              uint16_t* __restrict__ dlT, uint16_t* __restrict__ dlR,
                                                              float* __restrict__ dl_scale) {
  constexpr int kTileV = 128;                     // vocabulary rows per block: two adjacent ones per thread
  constexpr int kPitch = 66;                      // halves: 33 words per row (phase-1 stores 2-way conflicted at most)
  __shared__ __align__(16) uint16_t tile[kTileV * kPitch];
  __shared__ float sh[4 * 64];                    // lse_t, lse_z, coef, lse_ref of the tile's rows
  __shared__ float red[32];
  const int v0 = blockIdx.x * kTileV, r0 = blockIdx.y * 64;
  float cmax = 0.f;
  for (int r = threadIdx.x; r < T; r += blockDim.x) cmax = fmaxf(cmax, fabsf(row_stats[3 * T_max + r]));
  cmax = block_max(cmax, red);
  const float S = pow2_scale_from_bound(cmax * (1.f + (z_ref ? lam : 0.f)));
  if (blockIdx.x == 0 && blockIdx.y == 0 && threadIdx.x == 0) { dl_scale[0] = S; dl_scale[1] = 1.f / S; }
  // K index k of the operand -> canvas row: k < T16 is the (hi) plane of row k; with two planes (2 T16 <= 64) k in
  // [T16, 2 T16) is the lo plane of row k - T16
  if (threadIdx.x < 64) {
    const int k = r0 + threadIdx.x;
    const int r = (planes == 2 && k >= T16) ? k - T16 : k;
    const bool ok = r < T && k < planes * T16;
    sh[threadIdx.x] = ok ? row_stats[0 * T_max + r] : 0.f;
    sh[64 + threadIdx.x] = ok ? row_stats[1 * T_max + r] : 0.f;
    sh[128 + threadIdx.x] = ok ? row_stats[3 * T_max + r] : 0.f;
    sh[192 + threadIdx.x] = ok ? row_stats[4 * T_max + r] : 0.f;
  }
  __syncthreads();
  const int vv = 2 * (threadIdx.x & 63);          // V % 128 == 0 on this path: v, v + 1 < V, 8-byte aligned pairs
  const int v = v0 + vv;
  for (int rr = threadIdx.x >> 6; rr < 64; rr += 4) {
    const int k = r0 + rr;
    const bool lo_plane = planes == 2 && k >= T16;
    const int r = lo_plane ? k - T16 : k;
    float dl[2] = {0.f, 0.f};
    if (r < T && k < planes * T16) {
      float t[2];
      if (BF16) {
        const uint32_t tb = *reinterpret_cast<const uint32_t*>(static_cast<const __nv_bfloat16*>(teacher) + (size_t)r * V + v);
        t[0] = __uint_as_float(tb << 16); t[1] = __uint_as_float(tb & 0xFFFF0000u);
      } else {
        const float2 tf = *reinterpret_cast<const float2*>(static_cast<const float*>(teacher) + (size_t)r * V + v);
        t[0] = tf.x; t[1] = tf.y;
      }
      const float2 zz = *reinterpret_cast<const float2*>(z + (size_t)r * z_ld + v);
      float2 zr = make_float2(0.f, 0.f);
      if (z_ref) zr = *reinterpret_cast<const float2*>(z_ref + (size_t)r * z_ld + v);
      const float zv[2] = {zz.x, zz.y}, zrv[2] = {zr.x, zr.y};
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        const float az = zv[e] - sh[64 + rr], at = t[e] - sh[rr];
        const float qv = FAST ? __expf(az) : expf(az);
        const float pv = FAST ? __expf(at) : expf(at);   // t = -inf -> 0
        float g = qv - pv;
        if (z_ref) {
          const float ar = zrv[e] - sh[192 + rr];
          g += lam * (qv - (FAST ? __expf(ar) : expf(ar)));
        }
        dl[e] = sh[128 + rr] * g * S;
      }
    }
    uint16_t hv[2];
#pragma unroll
    for (int e = 0; e < 2; ++e) {
      __half hq = __float2half_rn(dl[e]);
      if (lo_plane) hq = __float2half_rn(dl[e] - __half2float(hq));   // dl S = hi + lo to 2^-22
      hv[e] = __half_as_ushort(hq);
      tile[(vv + e) * kPitch + rr] = hv[e];
    }
    if (dlR && k < planes * T16)   // rows T .. T16 of a plane are zero
      *reinterpret_cast<uint32_t*>(dlR + (size_t)k * V + v) = (uint32_t)hv[0] | ((uint32_t)hv[1] << 16);
  }
  __syncthreads();
  // 8 threads per vocabulary row: 16 bytes each -> one 128-byte segment of dlT per row
  const int seg = threadIdx.x & 7;
  for (int row = threadIdx.x >> 3; row < kTileV; row += 32) {
    const uint32_t* src = reinterpret_cast<const uint32_t*>(tile + row * kPitch + seg * 8);
    *reinterpret_cast<uint4*>(dlT + (size_t)(v0 + row) * Kp + r0 + seg * 8) = make_uint4(src[0], src[1], src[2], src[3]);
  }
}

template <bool ADAM, int NV, bool GH, int MOM>
cudaError_t launch_wide(int grid, size_t smem, cudaStream_t s, const CUtensorMap& tm_dlT,
                        const CUtensorMap& tm_master, const CUtensorMap& tm_m, const CUtensorMap& tm_v,
                        const CUtensorMap& tm_wout, const WideParams& p) {
  tc_update_wide_kernel<ADAM, NV, GH, MOM><<<grid, kWThreads, smem, s>>>(tm_dlT, tm_master, tm_m, tm_v, tm_wout, p);
  return cudaGetLastError();
}


template <bool ADAM, int NV, bool GH, int MOM>
cudaError_t wide_attr() {
  return cudaFuncSetAttribute(tc_update_wide_kernel<ADAM, NV, GH, MOM>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                              kWSmemBudget + 2048);
}

}  // namespace

cudaError_t tc_wide_init(tts_ctx* c) {
  if (cudaError_t w = ptx::set_watchdog_cycles(c->watchdog_cycles)) return w;
  cudaError_t e;
  if ((e = wide_attr<true, 32, false, 0>()) != cudaSuccess) return e;
  if ((e = wide_attr<false, 32, false, 0>()) != cudaSuccess) return e;
  if ((e = wide_attr<true, 32, true, 0>()) != cudaSuccess) return e;
  if ((e = wide_attr<false, 32, true, 0>()) != cudaSuccess) return e;
  if ((e = wide_attr<true, 32, false, 1>()) != cudaSuccess) return e;
  return wide_attr<true, 32, true, 1>();
}

// dl planes of the wide path: hi + lo while both fit the 64-wide K chunk (T16 <= 32), one plane beyond
int tc_wide_planes(int T16) { return 2 * T16 <= kKC ? 2 : 1; }

// 1 when the wide update kernel forms gh itself (its accumulators fit next to h^T in tensor memory)
int tc_wide_fuses_gh(const tts_ctx* c, int T16) {
  if (c->cfg.flags & (TTS_FLAG_SEPARATE_GH | TTS_FLAG_DETERMINISTIC)) return 0;
  return tc_wide_planes(T16) * T16 <= kWGhMaxN;
}

// a4 of the wide path: h^T rows and the fp16 dl planes
cudaError_t tc_launch_prep_wide(tts_ctx* c, const StepArgs& a, const float* z, cudaStream_t s, int* launches) {
  TcState* st = static_cast<TcState*>(c->tc_state);
  const int V = c->cfg.V, d = c->cfg.d, T = a.T;
  const int T16 = (T + 15) / 16 * 16;
  const int Kp = (T16 + kKC - 1) / kKC * kKC;
  unsigned int* absmax = reinterpret_cast<unsigned int*>(st->dl_scale + 4);
  cudaError_t e = cudaMemsetAsync(absmax, 0, sizeof(unsigned int), s);
  if (e != cudaSuccess) return e;
  const __nv_bfloat16* h = static_cast<const __nv_bfloat16*>(a.h);
  const size_t n_h = (size_t)T * d;
  int ab_grid = (int)((n_h / 8 + 255) / 256);
  ab_grid = ab_grid < 1 ? 1 : (ab_grid > 4 * c->sm_count ? 4 * c->sm_count : ab_grid);
  tc_h_absmax_kernel<<<ab_grid, 256, 0, s>>>(h, n_h, absmax);
  const int planes = tc_wide_planes(T16);
  tc_prep_hT_kernel<<<dim3((d + 31) / 32, Kp / 32), 256, 0, s>>>(h, d, T, T16, planes, Kp, absmax,
                                                                  static_cast<uint16_t*>(st->hTT), st->dl_scale);
  uint16_t* dlT = static_cast<uint16_t*>(st->dlT);
  // the row-major plane is the gh KERNEL's operand: not needed when the update kernel forms gh itself
  uint16_t* dlR = (a.gh_out && !tc_wide_fuses_gh(c, T16)) ? static_cast<uint16_t*>(st->dlR) : nullptr;
  const dim3 grid(V / 128, Kp / 64);
  const bool bf = c->cfg.logits_dtype == TTS_BF16, fast = planes == 1;
  auto kern = bf ? (fast ? tc_prep_dl_wide_kernel<true, true> : tc_prep_dl_wide_kernel<true, false>)
                 : (fast ? tc_prep_dl_wide_kernel<false, true> : tc_prep_dl_wide_kernel<false, false>);
  kern<<<grid, 256, 0, s>>>(a.teacher, z, a.z_ref, a.lambda, V, V, T, T16, planes, Kp, c->cfg.T_max, c->row_stats, dlT,
                            dlR, st->dl_scale);
  *launches += 3;
  return cudaGetLastError();
}

// a6 + a7 of the wide path
cudaError_t tc_launch_update_wide(tts_ctx* c, const StepArgs& a, cudaStream_t s, int* launches) {
  TcState* st = static_cast<TcState*>(c->tc_state);
  const int V = c->cfg.V, d = c->cfg.d, T = a.T;
  const int T16 = (T + 15) / 16 * 16;
  const int Kp = (T16 + kKC - 1) / kKC * kKC;
  const bool adam = c->cfg.optimizer == TTS_ADAMW;
  constexpr int NV = 32;
  CUtensorMap tm_dlT, tm_master, tm_m, tm_v, tm_wout;
  // the operand map depends on this step's Kp (row pitch of the scratch)
  if (make_map_2d(st, &tm_dlT, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 2, st->dlT, Kp, V, kKC, NV,
                  CU_TENSOR_MAP_SWIZZLE_128B) != CUDA_SUCCESS)
    return cudaErrorInvalidValue;
  if (make_map_2d(st, &tm_master, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, a.master, d, V, kWJ, kWSV,
                  CU_TENSOR_MAP_SWIZZLE_NONE) != CUDA_SUCCESS)
    return cudaErrorInvalidValue;
  if (make_map_2d(st, &tm_wout, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, a.W_out, d, V, kWJ, kWSV,
                  CU_TENSOR_MAP_SWIZZLE_NONE) != CUDA_SUCCESS)
    return cudaErrorInvalidValue;
  tm_m = tm_master;
  tm_v = tm_master;
  const bool lowp = adam && c->cfg.moment_dtype == TTS_MOMENT_BF16;
  if (adam) {
    const CUtensorMapDataType mdt = lowp ? CU_TENSOR_MAP_DATA_TYPE_BFLOAT16 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32;
    const int msz = lowp ? 2 : 4;
    if (make_map_2d(st, &tm_m, mdt, msz, a.adam_m, d, V, kWJ, kWSV, CU_TENSOR_MAP_SWIZZLE_NONE) != CUDA_SUCCESS)
      return cudaErrorInvalidValue;
    if (make_map_2d(st, &tm_v, mdt, msz, a.adam_v, d, V, kWJ, kWSV, CU_TENSOR_MAP_SWIZZLE_NONE) != CUDA_SUCCESS)
      return cudaErrorInvalidValue;
  }
  WideParams p;
  p.gW_debug = a.gW_debug;
  p.hTT = static_cast<const uint16_t*>(st->hTT);
  p.dl_scale = st->dl_scale;
  p.V = V; p.d = d; p.Kp = Kp;
  p.n_stripes = d / kWJ;
  p.n_bands = V / NV;
  const long dl_bytes = (long)V * Kp * 2;
  p.n_win = (int)((dl_bytes + kWWindowBytes - 1) / kWWindowBytes);
  if (p.n_win < 1) p.n_win = 1;
  if (p.n_win > p.n_bands) p.n_win = p.n_bands;
  cudaError_t e;
  const bool gh_here = a.gh_out != nullptr && tc_wide_fuses_gh(c, T16);
  p.gh = gh_here ? a.gh_out : nullptr;
  p.T = T; p.T16 = T16; p.planes = tc_wide_planes(T16);
  if (gh_here && (e = cudaMemsetAsync(a.gh_out, 0, (size_t)T * d * sizeof(float), s)) != cudaSuccess) return e;
  p.op_stages = gh_here ? 3 : 2;   // with gh a band's dl rows stay until the gh MMAs issued one band later have read them
  const int fixed = 1024 + p.op_stages * NV * Kp * 2 + 2 * kWWoBytes + (gh_here ? kWWtBytes : 0) + (int)sizeof(WideBars);
  const int stage_bytes = lowp ? kWStageBytesLp : kWStageBytes;
  p.stages = (kWSmemBudget - fixed) / stage_bytes;
  // ring depth: with 12 KB stages the pass's speed was flat from 7 stages (84 KB) up at the grid tc_update_ctas picks
  // (8: 2.68 ms at 64 rows, 2.78 at 256, 2.83 at 512; 6: 3.04 / 3.13 / 3.12); the 24 KB stages of today give 6 (512 rows)
  // to 8 of them: 144-192 KB in flight, deeper rings only take shared memory
  if (p.stages > (lowp ? kWMaxStages : 8)) p.stages = lowp ? kWMaxStages : 8;
  if (p.stages < 2) return cudaErrorInvalidConfiguration;
  p.lr = a.lr; p.b1 = a.beta1; p.b2 = a.beta2; p.eps = a.eps;
  p.decay = 1.f - a.lr * a.wd;
  p.step_scalars = a.step_scalars;
  p.step_count = c->step_count_dev;
  p.sr_seed = static_cast<uint32_t>(c->cfg.sr_seed);
  const long units = (long)p.n_stripes * (p.n_bands / p.n_win);
  int grid = tc_update_ctas(c, lowp);
  if (grid > units) grid = (int)units;
  // Fixed-stripe walk when the grid is (nearly) a multiple of the stripe count: a CTA keeps ONE stripe for the whole pass
  // (h^T goes to tensor memory once, gh is flushed once) and takes every (grid / n_stripes)-th band, so the CTAs of one
  // phase sweep the same vocabulary rows across all stripes at about the same time: the 512-byte row segments of their
  // boxes add up to whole rows at the memory controllers, and a band's dl rows are fetched once and hit L2 for the other
  // stripes without any window.  d = 4096: 128 = 32 x 4 CTAs; 512 rows 2.83 -> 2.62 ms, 256 rows 2.78 -> 2.68, 64 rows
  // 2.69 -> 2.66 (same box).  Other grids (an SM budget, few stripes) keep the windowed stream-K walk.
  p.fixed = 0;
  {
    const int whole = grid - grid % p.n_stripes;
    // (the bf16-moment pass is bound by its epilogue warps and wants every SM: 64 rows 2.17 ms on 148 CTAs with the
    // stream-K walk against 2.45 on 128 with this one, so it takes the fixed walk only when nothing is given up)
    if (whole >= p.n_stripes && (lowp ? whole == grid : 100 * whole >= 85 * grid)) { p.fixed = 1; grid = whole; }
  }
  const size_t smem = (size_t)fixed + (size_t)p.stages * stage_bytes;
  if (lowp)
    e = gh_here ? launch_wide<true, NV, true, 1>(grid, smem, s, tm_dlT, tm_master, tm_m, tm_v, tm_wout, p)
                : launch_wide<true, NV, false, 1>(grid, smem, s, tm_dlT, tm_master, tm_m, tm_v, tm_wout, p);
  else if (gh_here)
    e = adam ? launch_wide<true, NV, true, 0>(grid, smem, s, tm_dlT, tm_master, tm_m, tm_v, tm_wout, p)
             : launch_wide<false, NV, true, 0>(grid, smem, s, tm_dlT, tm_master, tm_m, tm_v, tm_wout, p);
  else
    e = adam ? launch_wide<true, NV, false, 0>(grid, smem, s, tm_dlT, tm_master, tm_m, tm_v, tm_wout, p)
             : launch_wide<false, NV, false, 0>(grid, smem, s, tm_dlT, tm_master, tm_m, tm_v, tm_wout, p);
  *launches += 1;
  return e;
}

}  // namespace tts
