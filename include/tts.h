/*
 * tts.h -- C ABI of the B200-native online-distillation step of Test-Time
 * Speculation (TTS), arxiv/paper_2605_09329.  Citations are lines of
 * /root/reference/PAPER.md ("PAPER.md:<line>") and readings R<n> of DESIGN.md.
 *
 * What the library does.  After a speculative-decoding round the caller holds
 * the target's (teacher's) logits over the C canvas positions, the canvas
 * tokens and the draft's state.  It wants
 *   (i)  tau, the accepted-prefix length            (PAPER.md:115 step c, 152), and
 *   (ii) the draft updated by ONE optimisation step on
 *            L_t(q) = sum_k w_k KL(p_k || q_k) [+ lambda sum_k w_k KL(q_t,k || q_k)]
 *        evaluated at q = q_t                        (Alg. 1 154-158),
 *        off the critical path on a side stream.
 * The trained parameters are the draft LM head W[V,d] (bf16 working copy + fp32
 * master + optimiser state); the gradient w.r.t. the draft hidden states h is
 * returned for whatever sits upstream.  At one step per round the lambda term is
 * identically zero in loss and gradient (q = q_t), so it is not computed (R3).
 *
 * Conventions
 *   - Plain C, no C++ exceptions cross the ABI.  Every function returns a status
 *     (TTS_OK = 0) unless stated otherwise.
 *   - Unless a parameter says "host", every data pointer is a DEVICE pointer on
 *     the ctx's device, 16-byte aligned, row-major contiguous.  The caller owns
 *     every tensor; the library owns only the scratch inside tts_ctx (allocated
 *     in tts_ctx_create, never in a step).
 *   - `stream` parameters are cudaStream_t handles passed as void* (so that this
 *     header needs no CUDA include).  Step and mask calls only ENQUEUE work; they
 *     never synchronise the host.  Device outputs are valid once the stream has
 *     reached the step's done-event (tts_wait_step / tts_sync_step).
 *   - One ctx per side stream.  Calls on one ctx are not thread-safe; distinct
 *     ctxs are independent.
 *   - There is no CPU fallback: on a machine without an sm_100 device
 *     tts_ctx_create fails with TTS_ERR_ARCH / TTS_ERR_CUDA.
 */
#ifndef TTS_H_
#define TTS_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* status codes */
enum {
  TTS_OK = 0,
  TTS_ERR_INVALID_ARG = 1, /* NULL where data is required, T out of range, misaligned pointer */
  TTS_ERR_UNSUPPORTED = 2, /* dtype / shape combination outside the supported set */
  TTS_ERR_CUDA = 3,        /* a CUDA call failed; see tts_last_cuda_error */
  TTS_ERR_ARCH = 4         /* device is not compute capability 10.x */
};

/* dtypes */
enum { TTS_F32 = 0, TTS_BF16 = 1 };
/* optimisers: Alg. 1 writes plain gradient descent; App. C.1 names Adam */
enum { TTS_SGD = 0, TTS_ADAMW = 1 };
/* which canvas rows enter the loss (R2).  The paper sums over all k = 1..C. */
enum { TTS_ROWS_ALL = 0, TTS_ROWS_ACCEPTED = 1, TTS_ROWS_ACCEPTED_PLUS_ONE = 2 };
/* kernel family.  AUTO: tcgen05/TMA kernels when param_dtype is bf16 and the shape
 * qualifies (V % 128 == 0, d % 128 == 0, T_max <= 512), CUDA-core kernels otherwise
 * (fp32 parameters, e.g. BASELINE config 1; other shapes).  SIMT forces the CUDA-core kernels. */
enum { TTS_PATH_AUTO = 0, TTS_PATH_SIMT = 1 };
/* precision of Adam's moments m, v (the paper fixes only "Adam"; R6, R26).  F32 is the default and what
 * every BASELINE.json configuration uses.  BF16 is an opt-in variant that cuts the step's bytes (tensor path, AdamW
 * only); its layout and rounding rules are given at tts_distill_step.  (Value 2 was TTS_MOMENT_Q8 up to version 0.2.0:
 * declared, never implemented; it is gone and tts_ctx_create refuses the value like any other unknown one.) */
enum { TTS_MOMENT_F32 = 0, TTS_MOMENT_BF16 = 1 };
/* tts_config.flags */
enum {
  TTS_FLAG_CHECK_PRECONDITIONS = 1, /* every step also runs the checks behind tts_last_device_status (debug mode)  */
  TTS_FLAG_DETERMINISTIC = 2,       /* gh is reduced in a fixed order (two-stage: per-CTA parts, then one sum) so    */
                                    /* that a step is bit-reproducible run to run; costs one small kernel + scratch  */
  TTS_FLAG_SEPARATE_GH = 4          /* gh is contracted against the W_in BUFFER by its own kernel instead of being   */
                                    /* re-derived from the master inside the update pass: for callers who cannot     */
                                    /* guarantee W_in == rn_bf16(W_master); costs a second read of W_in              */
};
/* bits of tts_last_device_status */
enum {
  TTS_DEV_W_MISMATCH = 1,        /* W_in != rn_bf16(W_master) somewhere (precondition 1 of tts_distill_step)       */
  TTS_DEV_NONFINITE_TEACHER = 2, /* a teacher logit is NaN or +inf (-inf is legal: a masked vocabulary entry, R23) */
  TTS_DEV_NONFINITE_H = 4,       /* a hidden state is NaN or +-inf                                                 */
  TTS_DEV_BAD_TOKEN = 8,         /* tts_accept_stochastic saw a draft token outside [0, V) (treated as rejected)   */
  TTS_DEV_NONFINITE_LOSS = 16    /* the step's loss came out NaN / inf                                             */
};

typedef struct tts_ctx tts_ctx;

typedef struct {
  int32_t V;            /* vocabulary size                                                    */
  int32_t d;            /* draft hidden size                                                  */
  int32_t T_max;        /* max rows (canvas positions x sequences) per step, <= 4096          */
  int32_t seg_len;      /* C: rows per sequence; the prefix logic restarts every seg_len rows */
  int32_t param_dtype;  /* TTS_BF16: bf16 working copy + fp32 master | TTS_F32: fp32 only     */
  int32_t logits_dtype; /* teacher logits: TTS_BF16 | TTS_F32                                 */
  int32_t optimizer;    /* TTS_SGD | TTS_ADAMW                                                */
  float lr, beta1, beta2, eps, weight_decay; /* R5: eps outside the sqrt, bias correction on, */
                                             /* decoupled decay M <- M (1 - lr wd)            */
  int32_t mask_mode;    /* TTS_ROWS_*                                                         */
  int32_t max_ctas;     /* 0 = one CTA per SM; else cap the persistent kernels' grids so the  */
                        /* main stream keeps SMs while the step overlaps it    */
  int32_t kernel_path;  /* TTS_PATH_*                                                         */
  int32_t moment_dtype; /* TTS_MOMENT_*: storage format of adam_m / adam_v (0 = fp32)                 */
  int32_t max_inner_steps; /* largest K of tts_distill_inner_steps; > 1 reserves its z_ref scratch    */
                        /* (T_max x V fp32) in tts_ctx_create so that no step call ever allocates     */
  int32_t flags;        /* TTS_FLAG_* (0 = none)                                                      */
  int32_t sr_seed;      /* TTS_MOMENT_BF16: seed of the stochastic-rounding draws of v                */
} tts_config;

const char* tts_status_string(int32_t status);
/* library version, major*10000 + minor*100 + patch */
int32_t tts_version(void);

/* Creates a context on `device` (a CUDA ordinal) and allocates all scratch.
 * Errors: INVALID_ARG (NULL, non-positive sizes, T_max % seg_len != 0), UNSUPPORTED,
 * ARCH (not sm_10x), CUDA. */
int32_t tts_ctx_create(const tts_config* cfg, int32_t device, tts_ctx** out);
int32_t tts_ctx_destroy(tts_ctx* ctx);

/* Hyper-parameters may change between steps. */
int32_t tts_set_lr(tts_ctx* ctx, float lr);
/* Adam's bias-correction step count n lives in DEVICE memory of the ctx: 0 after create, incremented by the first
 * kernel of every tts_distill_step on the step's stream (so the first step uses n = 1, and a replayed CUDA graph of
 * the step keeps counting).  Set it to resume a stream or after restoring a snapshot (the paper resets the
 * speculator between requests).  Both calls synchronise the WHOLE DEVICE (every stream of every
 * process on it, a co-resident target model's included): set-up and debugging only.  A running service uses the
 * stream-ordered forms below. */
int32_t tts_set_step_count(tts_ctx* ctx, int64_t n);
int64_t tts_get_step_count(const tts_ctx* ctx);   /* returns the count (-1 on error), not a status */
/* Stream-ordered forms that do NOT synchronise the device: the set is enqueued on `stream` (put it on the step's side
 * stream between two steps); the get enqueues a copy on `stream` and blocks the host on THAT stream only. */
int32_t tts_set_step_count_async(tts_ctx* ctx, int64_t n, void* stream);
int64_t tts_get_step_count_on(tts_ctx* ctx, void* stream);
/* Device status word (bits TTS_DEV_*), accumulated by the kernels since the last read.  Which checks run:
 *   always                       TTS_DEV_BAD_TOKEN, TTS_DEV_NONFINITE_LOSS
 *   TTS_FLAG_CHECK_PRECONDITIONS TTS_DEV_W_MISMATCH (every element of W_in against rn_bf16(W_master)),
 *                                TTS_DEV_NONFINITE_TEACHER, TTS_DEV_NONFINITE_H (complete scans); +0.6 ms at the
 *                                Qwen3-8B head: a debug mode.  tts_check_preconditions runs the same checks once.
 * tts_last_device_status blocks the host until the last step on this ctx is done (as tts_sync_step) AND until the last
 * tts_check_preconditions / tts_accept_stochastic call is done, whatever stream each was enqueued on (non-blocking
 * streams included); it then takes the word (one atomic exchange with 0, on a stream of the ctx's own -- no other
 * stream of the process is touched) and returns the bits, -1 on error.  Checks enqueued on a THIRD stream before those
 * two calls are covered only if that stream was ordered before one of them.
 * tts_device_status_on is the stream-ordered form for a serving loop: the exchange is enqueued on `stream`, behind
 * whatever the caller enqueued there, and the host blocks on that stream only.  Not inside a stream capture (-1). */
int32_t tts_last_device_status(tts_ctx* ctx);
int32_t tts_device_status_on(tts_ctx* ctx, void* stream);
int32_t tts_check_preconditions(tts_ctx* ctx, const void* teacher_logits, const void* h, const void* W_in,
                                const float* W_master, int32_t T, void* stream);
/* A tensor-path kernel whose internal pipeline stalls (a protocol error, never a legal state) does not hang the GPU:
 * a watchdog warp in every persistent kernel traps once the kernel has been running for more than a limit, the launch
 * fails with cudaErrorLaunchFailed and the next call that synchronises (tts_sync_step, tts_round_host,
 * tts_last_device_status, ...) returns TTS_ERR_CUDA.  A trap ends the PROCESS's CUDA context on that GPU -- everything
 * the process holds there, a co-resident target model included.
 *   what is measured  SM cycles since the kernel's own launch, NOT since its last progress: a healthy kernel that is
 *                     stretched past the limit trips it too (cuda-gdb, compute-sanitizer, time-slicing with another
 *                     process; a step takes milliseconds, so this needs a slowdown of three orders of magnitude).
 *   the limit         2^34 cycles (8.7 s at 1.965 GHz) by default.  The environment variable TTS_WATCHDOG_CYCLES, read
 *                     by tts_ctx_create, replaces it: a decimal cycle count, 0 = never trap (use that under a debugger
 *                     or sanitizer); anything else that does not parse makes tts_ctx_create return INVALID_ARG.  The
 *                     value is stored once per GPU for the whole process: the last ctx created on a GPU decides.
 * tts_debug_trip_watchdog proves the mechanism: it launches a deliberately stalled pipeline on `stream`, blocks until
 * the launch has failed and returns TTS_ERR_CUDA; the process's CUDA context is unusable afterwards (run it in a process
 * of its own). */
int32_t tts_debug_trip_watchdog(tts_ctx* ctx, void* stream);
/* CUDA error code (cudaError_t as int) of the last failed CUDA call on this ctx, 0 if none. */
int32_t tts_last_cuda_error(const tts_ctx* ctx);
/* 1 if the last tts_distill_step on this ctx ran the tcgen05/TMA kernels, 0 if CUDA-core. */
int32_t tts_last_step_used_tensor_path(const tts_ctx* ctx);
/* number of kernels the last tts_distill_step / tts_accept_mask enqueued (for bench.py's gpu_launches) */
int32_t tts_last_launch_count(const tts_ctx* ctx);

/*
 * a1.  Greedy accepted-prefix mask: the accept loop of PAPER.md:97-101 / Alg. 1 "Accept"
 * with the greedy rule "teacher argmax == draft token" in place of the
 * stochastic min{1,p/q} test (north_star (4); R8).
 *   am[r]   = argmax_v teacher_logits[r,v], LOWEST index on ties (R11), raw values compared
 *   mask[r] = 1 iff rows s*C .. r of r's segment all have am == draft_tokens
 *   tau[s]  = number of matched draft positions in segment s, 0..C.  The paper's acceptance
 *             length (which counts the target's bonus token) is tau + 1 (R9).
 * Row r of teacher_logits is the distribution that judges draft_tokens[r]; no shift is
 * applied inside the library (R10).  Logits must be finite or -inf; NaN gives undefined
 * results.  Integer/compare only: bit-exact.
 */
int32_t tts_accept_mask(tts_ctx* ctx,
                        const void* teacher_logits,  /* [T,V] logits_dtype                     */
                        const int32_t* draft_tokens, /* [T]   canvas tokens                    */
                        int32_t T,                   /* multiple of seg_len, 1..T_max          */
                        uint8_t* mask_out,           /* [T]   1 = inside the accepted prefix   */
                        int32_t* tau_out,            /* [T/seg_len]                            */
                        int32_t* teacher_argmax_out, /* [T] or NULL                            */
                        void* stream);

/*
 * a1 without a ctx and without any allocation.  Same operation, same readings and same outputs as tts_accept_mask
 * (R8, R9, R11), for callers that cannot allocate device memory when they need the mask: a
 * serving process whose own pool already holds the whole GPU, code inside a region where cudaMalloc is off limits
 * because it synchronises the device and would stall the decode stream, or an embedder that routes every GPU byte
 * through its own allocator.  Such a caller cannot use tts_ctx_create (it cudaMallocs the ctx's scratch), so this call
 * takes the shapes directly and keeps the per-(row, slice) argmax candidates in a fixed array of
 * TTS_STATIC_SCRATCH_BYTES that is part of the library image: every GPU on which the library's code is loaded holds
 * one copy until the process exits, whether or not this call is ever made.
 *   limits     T <= TTS_STATIC_T_MAX; a larger T returns TTS_ERR_INVALID_ARG and enqueues nothing.  V <= 2^30, rows
 *              16-byte aligned (V % 8 == 0 for bf16, V % 4 == 0 for fp32), T % seg_len == 0, as tts_accept_mask.
 *   device     the calling thread's CURRENT device; `stream` and every pointer must belong to it (device pointers).
 *   first call on each device also resolves the array's address on that device (cudaGetSymbolAddress, under a lock)
 *              and reads two device attributes; make that first call outside any stream capture.  Later calls only
 *              launch two kernels on `stream`.  No call here uses cudaMalloc, cudaFree or an allocating library routine.
 *   sharing    all calls on one device use the same array.  Nothing in it has to start at zero (each call writes every
 *              slot it later reads), and it keeps the last call's candidates afterwards.  Two calls whose kernels can
 *              run at the same time on one GPU (different streams without an ordering between them, or two host
 *              threads) race on it and may both return wrong masks: order them, e.g. keep them on one stream.
 *   errors     INVALID_ARG (NULL, sizes, T over the limit, misaligned teacher), UNSUPPORTED (dtype, row alignment,
 *              device ordinal >= 64), ARCH (current device is not sm_10x), CUDA (code in tts_static_last_cuda_error).
 */
#define TTS_STATIC_T_MAX 512
#define TTS_STATIC_SCRATCH_BYTES 264192 /* 512 rows x 64 slices x (fp32 value + int32 index) + 512 x int32 */
int32_t tts_accept_mask_static(const void* teacher_logits,  /* [T,V] logits_dtype, device                      */
                               int32_t logits_dtype,        /* TTS_BF16 | TTS_F32                              */
                               int32_t V, int32_t seg_len,
                               const int32_t* draft_tokens, /* [T]                                             */
                               int32_t T,                   /* multiple of seg_len, 1..TTS_STATIC_T_MAX        */
                               uint8_t* mask_out,           /* [T]                                             */
                               int32_t* tau_out,            /* [T/seg_len]                                     */
                               int32_t* teacher_argmax_out, /* [T] or NULL                                     */
                               void* stream);
/* cudaError_t (as int) of the last failed CUDA call that tts_accept_mask_static made on the calling thread, 0 if none */
int32_t tts_static_last_cuda_error(void);

/*
 * f2.  The paper's own accept rule, "standard speculative rejection sampling" (Alg. 1):
 * canvas tokens are considered left to right, x_{t+k} is accepted with probability min{1, p(x_{t+k}) / q(x_{t+k})},
 * and the loop breaks at the first rejection.  p = softmax(teacher_logits[r]), q =
 * softmax(draft_logits[r]) -- after a round both are at hand.  Randomness is the caller's:
 *   uniforms[r]           U[0,1): row r is accepted iff every earlier row of its sequence was and
 *                         uniforms[r] * q_r(tok_r) <= p_r(tok_r)            (fp32 products of fp64-normalised p, q)
 *   uniforms_resample[s]  U[0,1): at the first rejected row of sequence s the replacement token is drawn from the
 *                         residual distribution norm(max(0, p - q)) by inverse CDF over the vocabulary order: the
 *                         smallest v with sum_{v' <= v} max(0, p - q) >= u * sum_v max(0, p - q)
 *   next_token_out[s]     that token; -1 when the whole canvas was accepted (the bonus token needs the target's
 *                         distribution at position C + 1, which this call does not see)
 *   draft tokens outside [0, cfg.V) are rejected (never dereferenced) and set TTS_DEV_BAD_TOKEN: the call takes the
 *                         WHOLE vocabulary, it is not shard-aware (a shard holds cfg.V local rows, tokens are global)
 *   diag_out [T,4] or NULL: the diagnostics of the paper's section 3 (Fig. 4), free by-products of
 *                         the same vocabulary sweep:  H(p_r) in nats,  -log q_r(argmax_v p_r),  p_r(tok_r),  q_r(tok_r)
 * tau_out / mask_out as in tts_accept_mask.  draft_logits: [T,V] fp32, row stride V (V % 4 == 0).
 */
int32_t tts_accept_stochastic(tts_ctx* ctx,
                              const void* teacher_logits,     /* [T,V] logits_dtype                  */
                              const float* draft_logits,      /* [T,V] fp32                          */
                              const int32_t* draft_tokens,    /* [T]                                 */
                              const float* uniforms,          /* [T]                                 */
                              const float* uniforms_resample, /* [T/seg_len]                         */
                              int32_t T, uint8_t* mask_out, int32_t* tau_out, int32_t* next_token_out,
                              float* diag_out, void* stream);

/*
 * a2-a8.  One TTS update (Alg. 1 "Loss" + "Update"):
 *   z      = h W_in^T                                   draft logits at q = q_t
 *   KL_r   = KL(softmax(teacher_r) || softmax(z_r)), -inf teacher entries = p 0
 *   omega_r= pos_weight[r] * maskfactor_r               (w_k of PAPER.md:123-127; R1, R2)
 *   loss   = loss_scale * sum_r omega_r KL_r            a SUM, not a mean (R3')
 *   dl     = loss_scale * omega_r (softmax(z_r) - softmax(teacher_r))
 *   gW     = dl^T h,  gh = dl W_in
 *   SGD    : M <- M - lr gW
 *   AdamW  : M <- M (1 - lr wd); m <- b1 m + (1-b1) g; v <- b2 v + (1-b2) g^2;
 *            M <- M - lr (m / (1-b1^n)) / (sqrt(v / (1-b2^n)) + eps)      (R5)
 *   W_out  = rn_bf16(M)   (TTS_BF16)   |   W_out = M   (TTS_F32, W_master == NULL)
 *   TTS_MOMENT_BF16 (opt-in, R26): adam_m / adam_v hold bf16 [V,d] (18 instead of 26 bytes per parameter in the update
 *            pass; with a2's read of W_in, 20 instead of 28 per step).  Per element: widen m, v exactly; update as above with the UNROUNDED new moments; store
 *            m = rn_bf16(m_new) and v = bf16 by STOCHASTIC rounding of v_new (beta2 = 0.999 decays v by 0.1% per
 *            step, below half a bf16 ulp: nearest rounding would freeze it): the 16 discarded fp32 bits f round
 *            away from zero iff f + r >= 65536, r = 16 bits of a counter-based generator keyed by the element's
 *            position (v, j) (LOCAL rows on a vocabulary shard), Adam's count n and cfg.sr_seed.  One 32-bit hash
 *            serves the two vertically adjacent elements (2k, j) and (2k + 1, j):
 *              pidx = (v >> 1) * d + j
 *              x = lo32(pidx) ^ (n * 0x9E3779B9) ^ (sr_seed * 0x85EBCA6B) ^ (hi32(pidx) * 0xC2B2AE35)
 *              x ^= x >> 16; x *= 0x7FEB352D; x ^= x >> 15; x *= 0x846CA68B; x ^= x >> 16
 *              r = x >> 16 for even v, x & 0xFFFF for odd v
 *
 * Preconditions: for TTS_BF16, W_in == rn_bf16(W_master) element-wise at entry; teacher_logits
 * and h must stay untouched until the done-event (the step consumes the buffers captured at
 * dispatch time; R17); W_out may alias W_in, but when draft rounds keep reading
 * W_in during the update pass distinct buffers and swap them at the barrier (R18).
 * All kernels are enqueued on side_stream; a done-event is recorded after the last one.
 */
int32_t tts_distill_step(tts_ctx* ctx,
                         const void* teacher_logits, /* [T,V] logits_dtype                                   */
                         const void* h,              /* [T,d] param_dtype: draft hidden states               */
                         const void* W_in,           /* [V,d] param_dtype: weights that produced q_t         */
                         void* W_out,                /* [V,d] param_dtype: updated weights; may alias W_in   */
                         float* W_master,            /* [V,d] fp32 in place; NULL iff TTS_F32                */
                         void* adam_m,               /* [V,d] moment_dtype in place; NULL iff TTS_SGD        */
                         void* adam_v,               /* [V,d] moment_dtype in place; NULL iff TTS_SGD        */
                         const float* pos_weight,    /* [T]   w_k already expanded per row                   */
                         const uint8_t* mask,        /* [T]   from tts_accept_mask; may be NULL for ROWS_ALL */
                         int32_t T,                  /* multiple of seg_len, 1..T_max                        */
                         float loss_scale,           /* multiplies the loss and every gradient               */
                         float* loss_out,            /* [1]                                                  */
                         float* kl_rows_out,         /* [T] unweighted KL_r, or NULL                         */
                         float* gh_out,              /* [T,d] fp32, or NULL (then gh is not computed)        */
                         float* gW_debug_out,        /* [V,d] fp32, or NULL (parity mode: extra 4 V d bytes) */
                         void* side_stream);

/*
 * f1.  The same step with optional extras (host struct, read during the call; NULL = tts_distill_step):
 *   draft_logits      [T,V] fp32 device, row stride V, or NULL.  "each time a draft canvas is generated, we naturally
 *                     have access to both the drafter's probabilities q and the target's probabilities p"
 *                     (PAPER.md:109): the drafter's logits z of the canvas rows are taken as given and pass a2 (one
 *                     read of the bf16 W, 7% of the step's bytes) is skipped.  They must be the logits of (h, W_in).
 *   draft_logits_out  [T,V] fp32 device or NULL: a2 writes z here instead of the ctx scratch, so that the caller can
 *                     pass it back as ref_logits of later inner steps.  Exclusive with draft_logits.
 *   ref_logits, lambda  the regulariser  lambda * K~L(q_t || q)  of PAPER.md:119-121 with q_t = softmax(ref_logits):
 *                       loss += loss_scale * lambda * sum_r omega_r KL(q_t,r || q_r)
 *                       dl    = loss_scale * omega_r [(q - p) + lambda (q - q_t)]
 *                     At q = q_t (one step per round, the paper's default) both vanish for every
 *                     lambda (R3); the term matters for K > 1 inner steps.  ref_logits NULL or lambda 0 skips it.
 *   kl_rows_out stays KL(p_r || q_r), the first term only.
 */
typedef struct {
  const float* draft_logits;
  float* draft_logits_out;
  const float* ref_logits;
  float lambda;
} tts_step_extras;

int32_t tts_distill_step_ex(tts_ctx* ctx, const void* teacher_logits, const void* h, const void* W_in, void* W_out,
                            float* W_master, void* adam_m, void* adam_v, const float* pos_weight,
                            const uint8_t* mask, int32_t T, float loss_scale, float* loss_out, float* kl_rows_out,
                            float* gh_out, float* gW_debug_out,
                            const tts_step_extras* extras, /* host, may be NULL */
                            void* side_stream);

/*
 * K optimisation steps on the same round's signal (section 6.5; the paper's default and best is K = 1).
 * Step 1 is tts_distill_step (q = q_t: the lambda term is inert) and keeps its draft logits as z_ref; steps 2..K
 * recompute z from the weights step k-1 wrote and add lambda * K~L(q_t || q).  Step 1 reads W_in and writes W_out,
 * later steps update W_out in place; master / m / v advance K times and Adam's count by K.
 *   draft_logits  [T,V] fp32 device or NULL: the drafter's own logits for step 1 (and z_ref), as in tts_distill_step_ex
 *   loss_out      [K] device: the loss of every inner step;  kl_rows_out [T] or NULL: step 1's KL rows;
 *   gh_out        [T,d] or NULL: the LAST step's gradient w.r.t. h
 * K > 1 without caller-supplied draft_logits needs the z_ref scratch: create the ctx with max_inner_steps >= K
 * (else TTS_ERR_INVALID_ARG); no step call allocates.
 */
int32_t tts_distill_inner_steps(tts_ctx* ctx, const void* teacher_logits, const void* h, const void* W_in, void* W_out,
                                float* W_master, void* adam_m, void* adam_v, const float* pos_weight,
                                const uint8_t* mask, int32_t T, float loss_scale, int32_t K, float lambda,
                                const float* draft_logits, float* loss_out, float* kl_rows_out, float* gh_out,
                                void* side_stream);

/*
 * Per-phase device timing (for bench.py's roofline line).  When enabled, tts_distill_step records
 * CUDA events on side_stream between its phases (no host synchronisation is added).  Phases:
 *   0 = a2 draft logits, 1 = a3 row statistics + loss, 2 = a4 dlogits / operand preparation,
 *   3 = a5 gh (0 when fused into phase 4), 4 = a6 + a7 gW contraction fused with the update.
 * tts_profile_read synchronises with the last profiled step, writes the MEAN milliseconds per phase
 * over the steps recorded since the last read (at most 256 are kept) into ms_out (HOST, [5]), stores
 * the number of steps averaged in *n_steps_out (HOST, may be NULL) and resets the accumulation.
 */
enum { TTS_NUM_PHASES = 5 };
int32_t tts_profile_enable(tts_ctx* ctx, int32_t enable);
int32_t tts_profile_read(tts_ctx* ctx, float* ms_out, int32_t* n_steps_out);

/*
 * f3: CUDA-graph capture.  tts_accept_mask and tts_distill_step[_ex] may be called while their stream
 * is being captured (cudaStreamBeginCapture .. EndCapture): they allocate nothing, never synchronise, and every
 * step-dependent scalar (Adam's count and bias corrections) is read from device memory.  What is baked into the
 * captured graph: all pointer arguments (so a W_in / W_out double buffer needs one graph per parity, or W_out ==
 * W_in), T, loss_scale and the ctx's hyper-parameters at capture time (re-capture after tts_set_lr).  Inside a
 * capture no done-event is recorded and the phase profile is off; after cudaGraphLaunch on a stream call
 * tts_record_done on that stream, then tts_wait_step / tts_sync_step as usual (graph replay ignores
 * cross-stream events recorded elsewhere, hence the paper's CPU-side barrier = tts_sync_step).
 */
int32_t tts_record_done(tts_ctx* ctx, void* stream);

/* The paper's barrier after S-1 rounds: main_stream waits (on the device) for the
 * last step's done-event. */
int32_t tts_wait_step(tts_ctx* ctx, void* main_stream);
/* Host blocks until the last step is done: the CPU-side barrier the paper needed in front of
 * CUDA-graph replay. */
int32_t tts_sync_step(tts_ctx* ctx);

/*
 * One whole round through HOST buffers (used for end-to-end timing): copies the round's inputs
 * from (preferably pinned) host memory into ctx-owned staging buffers (two slots of T_max x (V + d) inputs, allocated
 * by the FIRST tts_round_host / tts_round_host_begin call on the ctx -- the one exception to "only tts_ctx_create
 * allocates", so that callers who never use these calls do not hold 311 MB at T_max = 512), runs tts_accept_mask and
 * tts_distill_step on `stream`, copies loss / tau / mask back and synchronises the stream.
 * The persistent draft state (W, master, m, v) stays resident on the device: device pointers.
 * The teacher logits (the bulk of the bytes: 160 MB at 512 rows) travel on a copy stream owned by the ctx while pass
 * a2, which needs only h and W_in, already runs on `stream` (tensor path); a1 and a3 wait for the copy.
 *
 * tts_round_host_begin / tts_round_host_end are the same round split into "enqueue" and "wait for the results": begin
 * returns at once; the ctx has two staging slots, so a second round may be begun before the first is ended, and its
 * teacher logits then travel while the first round's step still runs (the updates are asynchronous by design,
 * round n + 1's verification does not wait for round n's update).  At most two rounds may be pending
 * (else TTS_ERR_INVALID_ARG); rounds end in the order they were begun; the host buffers of a round -- inputs and
 * outputs -- must stay untouched until its end call returns; every pending round must use the same `stream`.
 * tts_round_host == begin + end and refuses to run while begun rounds are pending.
 *
 * Ordering of the inputs: the teacher copy does NOT wait for `stream` (that is what lets it run under the previous
 * round's step), so the host input buffers must be complete ON THE HOST when begin is called; a caller that fills them
 * with work enqueued on `stream` (a D2H of the verifier's logits, say) synchronises that work first.
 * Errors: every argument the step could refuse (NULL or misaligned parameter tensors, T, a master / moment pointer that
 * does not fit the ctx's dtype and optimiser) is refused before anything is enqueued.  If a CUDA call fails after that,
 * the call blocks until whatever it had already enqueued on `stream` and on the copy stream has drained, returns
 * TTS_ERR_CUDA, and the round does not count as begun: the host buffers are free again and the slot is reusable.
 */
int32_t tts_round_host(tts_ctx* ctx,
                       const void* teacher_logits_host, /* host [T,V] logits_dtype */
                       const void* h_host,              /* host [T,d] param_dtype  */
                       const int32_t* draft_tokens_host,/* host [T]                */
                       const float* pos_weight_host,    /* host [T]                */
                       int32_t T, float loss_scale,
                       const void* W_in, void* W_out, float* W_master, void* adam_m, void* adam_v, /* device */
                       float* gh_dev,                   /* device [T,d] or NULL    */
                       float* loss_host,                /* host [1]                */
                       int32_t* tau_host,               /* host [T/seg_len]        */
                       uint8_t* mask_host,              /* host [T] or NULL        */
                       void* stream);
int32_t tts_round_host_begin(tts_ctx* ctx, const void* teacher_logits_host, const void* h_host,
                             const int32_t* draft_tokens_host, const float* pos_weight_host, int32_t T, float loss_scale,
                             const void* W_in, void* W_out, float* W_master, void* adam_m, void* adam_v, float* gh_dev,
                             float* loss_host, int32_t* tau_host, uint8_t* mask_host, void* stream);
int32_t tts_round_host_end(tts_ctx* ctx);

/*
 * f4.  The step sharded over the VOCABULARY across n_shards GPUs, one process per GPU.  Shard g owns
 * cfg.V consecutive rows [v_offset, v_offset + cfg.V) of W / master / m / v (each process creates its ctx with its
 * own local V) and the matching columns of the teacher logits as a contiguous [T, cfg.V] tensor -- the way a
 * tensor-parallel target delivers them.  h, pos_weight, mask and the draft tokens are replicated.  The paper's TTS
 * runs on one GPU; the shard axis follows from the step's algebra: every quantity that couples
 * vocabulary rows is a per-canvas-row reduction, so the exchange is tiny and the 28 bytes per parameter stay local.
 *   1. tts_shard_begin_step   a2 + this shard's a3 sweep; stats_out [T, 8] fp32 = per row the online tuple
 *                             (m_t, s_t, a, m_z, s_z, m_ref, s_ref, b) of SURVEY 8(a) a3 over the shard's columns
 *   2. the caller all-gathers the tuples -> stats_all [n_shards, T, 8]           (32 T bytes per rank)
 *   3. tts_shard_finish_step  merges the tuples (associative: same rule as between CTAs) into the GLOBAL lse_t,
 *                             lse_z, KL_r and loss -- identical on every shard -- then a4 .. a7 on the shard's rows
 *                             with no further communication; gh_partial_out [T, d] = this shard's sum over its rows
 *   4. the caller all-reduces (sum) gh_partial_out                               (4 T d bytes)
 * Between 1 and 3 the ctx keeps the shard's draft logits: call them in pairs, with the same T and extras, on the
 * same stream.  Adam's step count advances in tts_shard_finish_step.  With n_shards = 1 the pair equals
 * tts_distill_step_ex.  For the mask, tts_shard_argmax gives this shard's (max value, GLOBAL index = local index +
 * v_offset; 0x7fffffff for an all -inf slice) per row, the caller all-gathers both [T] arrays, and
 * tts_shard_accept_mask applies the lowest-global-index rule (R11) and the prefix logic of tts_accept_mask.
 */
enum { TTS_SHARD_STAT_FIELDS = 8 };
int32_t tts_shard_begin_step(tts_ctx* ctx,
                             const void* teacher_logits_local, /* [T, cfg.V] logits_dtype                   */
                             const void* h,                    /* [T, d]                                   */
                             const void* W_in_local,           /* [cfg.V, d]                               */
                             int32_t T,
                             const tts_step_extras* extras,    /* host, may be NULL; logits pointers are local [T, cfg.V] */
                             float* stats_out,                 /* [T, 8]                                   */
                             void* side_stream);
int32_t tts_shard_finish_step(tts_ctx* ctx,
                              const float* stats_all,          /* [n_shards, T, 8], own shard included     */
                              int32_t n_shards,                /* 1..1024                                  */
                              const void* teacher_logits_local, const void* h, const void* W_in_local,
                              void* W_out_local, float* W_master_local, void* adam_m_local, void* adam_v_local,
                              const float* pos_weight, const uint8_t* mask, int32_t T, float loss_scale,
                              float* loss_out,                 /* [1] the GLOBAL loss                      */
                              float* kl_rows_out,              /* [T] global KL_r, or NULL                 */
                              float* gh_partial_out,           /* [T, d] this shard's part of gh, or NULL  */
                              float* gW_debug_out,             /* [cfg.V, d] or NULL                       */
                              const tts_step_extras* extras, void* side_stream);
int32_t tts_shard_argmax(tts_ctx* ctx, const void* teacher_logits_local, int32_t T, int32_t v_offset,
                         float* val_out /* [T] */, int32_t* idx_out /* [T] */, void* stream);
int32_t tts_shard_accept_mask(tts_ctx* ctx, const float* val_all /* [n_shards, T] */,
                              const int32_t* idx_all /* [n_shards, T] */, int32_t n_shards,
                              const int32_t* draft_tokens, int32_t T, uint8_t* mask_out, int32_t* tau_out,
                              int32_t* teacher_argmax_out /* [T] or NULL */, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* TTS_H_ */
