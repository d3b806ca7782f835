"""fp64 CPU oracle for the Test-Time Speculation (TTS) distillation step.

TEST INFRASTRUCTURE ONLY.  Only ``tests/``, ``__graft_entry__.smoke()`` and
``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import this
file.  It shares no code with the CUDA path (``paper_2605_09329_b200/``) and
neither imports the other.  It is deliberately plain and slow: numpy in fp64,
the formulas of the paper written out in the paper's order, no blocking or
fusion beyond an optional split of the vocabulary into slabs (used only so
that the 150K-row configurations fit in host memory; the arithmetic per
element is unchanged).

What it computes, with the passage each step follows
(PAPER.md = /root/reference/PAPER.md, arxiv/paper_2605_09329):

  * ``accept_mask``       greedy longest matching prefix; loop structure of the
                          accept step, PAPER.md:97-101 (§4 step 2) and Alg. 1
                          "Accept" PAPER.md:152.  Greedy variant per north_star
                          (reading R8).
  * ``accept_stochastic`` the paper's own rule min{1, p/q} with the residual resample and the
                          section-3 diagnostics.
  * ``row_weights``       w_k of PAPER.md:123-127 expanded per row, times the
                          mask factor chosen by ``mask_mode`` (R2).
  * ``loss_and_grads``    L_t = K~L(p||q) + lambda K~L(q_t||q), PAPER.md:119-125,
                          Alg. 1; gradient evaluated at q = q_t
                          (PAPER.md:158).
  * ``sgd_update``        q <- q - eta grad L, Alg. 1 "Update" PAPER.md:158.
  * ``adamw_update``      "an optimizer (Adam) step", PAPER.md:393 (App. C.1);
                          hyper-parameter conventions per DESIGN.md R5.
  * ``distill_step``      the whole step (dense, small shapes); optionally with the drafter's
                          own logits taken as given and the lambda term.
  * ``distill_inner_steps`` K steps on one round's signal (section 6.5).
  * ``distill_step_rows`` the same step restricted to a subset of vocabulary
                          rows, given the full-vocabulary normalisers, so that a
                          full-size configuration can be checked on samples.

  * ``adamw_update_lowp`` the same Adam step with the moments STORED in bf16 (f4, an opt-in variant; the paper fixes
                          only "Adam"): dequantise -> update in full precision -> requantise, m by
                          round-to-nearest-even, v by stochastic rounding with the counter-based bits of
                          ``sr_bits16`` (R26).

  * ``shard_row_stats`` / ``merge_shard_stats``  the per-row online tuple (m_t, s_t, a, m_z, s_z) over a slice of
                          the vocabulary and its associative merge: what vocabulary shards exchange;
                          pinned against the plain logsumexp / KL of the whole row.

Pins (tests/test_oracle_pins.py): brute-force enumeration through the softmax
Jacobian, central finite differences, closed forms (V=2, uniform draft,
one-hot teacher, teacher == draft), invariants, and reduction to fp64
torch autograd / torch.optim.  No function here is "parity unpinned".
"""

from __future__ import annotations

import numpy as np

# mask_mode values (R2)
ROWS_ALL = 0
ROWS_ACCEPTED = 1
ROWS_ACCEPTED_PLUS_ONE = 2


# ----------------------------------------------------------------------------
# bf16 <-> fp32/fp64 bit conversions (the oracle's own; the CUDA path and the
# input generators each have theirs)
# ----------------------------------------------------------------------------

def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """Round-to-nearest-even fp32 -> bf16, returned as uint16 bit patterns."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    u = x.view(np.uint32).astype(np.uint64)
    lsb = (u >> 16) & 1
    r = (u + 0x7FFF + lsb) >> 16
    out = r.astype(np.uint16)
    nan = np.isnan(x)
    if nan.any():
        out = np.where(nan, np.uint16(0x7FC0), out)
    return out


def bf16_bits_to_f64(b: np.ndarray) -> np.ndarray:
    """Exact widening of bf16 bit patterns to fp64."""
    b = np.ascontiguousarray(b, dtype=np.uint16)
    return (b.astype(np.uint32) << 16).view(np.float32).astype(np.float64)


def widen(x: np.ndarray) -> np.ndarray:
    """Inputs arrive as the exact bits the GPU receives: uint16 = bf16 bits,
    float32 or float64 arrays are widened exactly."""
    if x.dtype == np.uint16:
        return bf16_bits_to_f64(x)
    return np.asarray(x, dtype=np.float64)


# ----------------------------------------------------------------------------
# a1: accepted-prefix mask (greedy variant)
# ----------------------------------------------------------------------------

def accept_mask(teacher_logits, draft_tokens, seg_len):
    """Row k of ``teacher_logits`` judges ``draft_tokens[k]`` (R10).

    am[r]   = argmax_v t[r, v], lowest index on ties (R11)
    mask[r] = 1 while every earlier row of the same segment matched, else 0
    tau[s]  = number of matched draft positions in segment s (0..seg_len) (R9)
    """
    t = widen(teacher_logits)
    tok = np.asarray(draft_tokens, dtype=np.int64)
    T = t.shape[0]
    assert T % seg_len == 0 and tok.shape == (T,)
    am = np.zeros(T, dtype=np.int32)
    mask = np.zeros(T, dtype=np.uint8)
    tau = np.zeros(T // seg_len, dtype=np.int32)
    for s in range(T // seg_len):
        alive = True                      # "if x_{t+k} rejected then break"
        for k in range(seg_len):
            r = s * seg_len + k
            row = t[r]
            # lowest index among the maxima, written out (not np.argmax) so the
            # tie rule is visible
            best_v = int(np.flatnonzero(row == row.max())[0])
            am[r] = best_v
            if alive and best_v == tok[r]:
                mask[r] = 1
                tau[s] += 1
            else:
                alive = False
    return mask, tau, am


# ----------------------------------------------------------------------------
# f2: the paper's own accept rule and its section-3 diagnostics
# ----------------------------------------------------------------------------

def accept_stochastic(teacher_logits, draft_logits, draft_tokens, uniforms, uniforms_resample, seg_len):
    """Standard speculative rejection sampling (Alg. 1 "Accept"), step by step as PAPER.md:97-101:

        k <- 1; while k <= C: accept x_{t+k} with probability min{1, p(x_{t+k}) / q(x_{t+k})};
                              if rejected: break;  k <- k + 1

    with p = softmax(teacher row), q = softmax(draft row), "accept with probability a" realised as u <= a for the
    caller's uniform u.  At the first rejected position the replacement token is drawn from the residual
    distribution norm(max(0, p - q)) by inverse CDF in vocabulary order with the caller's second uniform.
    Diagnostics per row: H(p_r), -log q_r(argmax_v p_r), p_r(tok_r), q_r(tok_r).

    Returns dict(mask, tau, next_token (-1: whole canvas accepted), diag [T,4], ratio [T], rej_row [S],
    resid_cdf {s: cumulative residual of the rejected row}) -- the last three let a test judge near-ties.
    """
    t = widen(teacher_logits)
    z = np.asarray(draft_logits, dtype=np.float64)
    tok = np.asarray(draft_tokens, dtype=np.int64)
    u = np.asarray(uniforms, dtype=np.float64)
    u2 = np.asarray(uniforms_resample, dtype=np.float64)
    T, V = t.shape
    S = T // seg_len
    lp = t - logsumexp_rows(t)[:, None]
    lq = z - logsumexp_rows(z)[:, None]
    p, q = np.exp(lp), np.exp(lq)
    diag = np.zeros((T, 4))
    ratio = np.zeros(T)
    for r in range(T):
        with np.errstate(invalid="ignore"):
            diag[r, 0] = -np.where(p[r] > 0.0, p[r] * lp[r], 0.0).sum()
        top = int(np.flatnonzero(t[r] == t[r].max())[0])
        diag[r, 1] = -lq[r, top]
        diag[r, 2] = p[r, tok[r]]
        diag[r, 3] = q[r, tok[r]]
        ratio[r] = np.inf if q[r, tok[r]] == 0.0 else p[r, tok[r]] / q[r, tok[r]]
    mask = np.zeros(T, dtype=np.uint8)
    tau = np.zeros(S, dtype=np.int32)
    nxt = np.full(S, -1, dtype=np.int32)
    rej = np.full(S, -1, dtype=np.int32)
    cdfs = {}
    for s in range(S):
        for k in range(seg_len):
            r = s * seg_len + k
            if u[r] <= min(1.0, ratio[r]):
                mask[r] = 1
                tau[s] += 1
            else:
                rej[s] = r
                resid = np.maximum(0.0, p[r] - q[r])
                cdf = np.cumsum(resid)
                cdfs[s] = cdf
                target = u2[s] * cdf[-1]
                hit = np.flatnonzero((cdf >= target) & (resid > 0.0))
                nxt[s] = int(hit[0]) if hit.size else -1
                break
    return dict(mask=mask, tau=tau, next_token=nxt, diag=diag, ratio=ratio, rej_row=rej, resid_cdf=cdfs)


# ----------------------------------------------------------------------------
# a8 weights
# ----------------------------------------------------------------------------

def row_weights(pos_weight, mask, mask_mode, seg_len):
    """omega_r = w_k times the mask factor.  ROWS_ALL: factor 1 (PAPER.md:123 sums
    over every k = 1..C).  ROWS_ACCEPTED: factor mask[r].  ROWS_ACCEPTED_PLUS_ONE:
    also the first rejected row of each segment."""
    w = np.asarray(pos_weight, dtype=np.float64).copy()
    if mask_mode == ROWS_ALL or mask is None:
        return w
    m = np.asarray(mask, dtype=np.float64).copy()
    if mask_mode == ROWS_ACCEPTED_PLUS_ONE:
        T = m.shape[0]
        for s in range(T // seg_len):
            seg = m[s * seg_len:(s + 1) * seg_len]
            n = int(seg.sum())
            if n < seg_len:
                seg[n] = 1.0
    return w * m


# ----------------------------------------------------------------------------
# a2-a6: loss and gradients
# ----------------------------------------------------------------------------

def logsumexp_rows(x):
    m = x.max(axis=1, keepdims=True)
    return (m + np.log(np.exp(x - m).sum(axis=1, keepdims=True)))[:, 0]


def kl_rows_from_logits(a_logits, b_logits):
    """KL(softmax(a) || softmax(b)) per row; terms with softmax(a)=0 dropped."""
    la = a_logits - logsumexp_rows(a_logits)[:, None]
    lb = b_logits - logsumexp_rows(b_logits)[:, None]
    pa = np.exp(la)
    with np.errstate(invalid="ignore"):
        term = np.where(pa > 0.0, pa * (la - lb), 0.0)
    return term.sum(axis=1)


def loss_and_grads(teacher_logits, h, W, omega, loss_scale=1.0, lam=0.0, z_ref=None, z=None):
    """Dense evaluation.  Returns dict(loss, kl_rows, z, lse_t, lse_z, dl, gW, gh).

    1. z[r,v] = sum_j h[r,j] W[v,j]                      (q = q_t)
       or, when ``z`` is given, the drafter's own logits of the canvas rows: after a round "we naturally have
       access to both the drafter's probabilities q and the target's probabilities p"
    2. log p = t - lse(t), log q = z - lse(z)
    3. KL_r = sum_v p (log p - log q)
    4. loss = loss_scale * sum_r omega_r KL_r            (a sum)
       + loss_scale * lam * sum_r omega_r KL(q_ref||q)_r
    5. dl = loss_scale * omega_r [(q - p) + lam (q - q_ref)]
    6. gW = dl^T h, gh = dl W
    """
    t = widen(teacher_logits)
    hh = widen(h)
    WW = widen(W)
    om = np.asarray(omega, dtype=np.float64)
    z = hh @ WW.T if z is None else np.asarray(z, dtype=np.float64)
    lse_t = logsumexp_rows(t)
    lse_z = logsumexp_rows(z)
    p = np.exp(t - lse_t[:, None])
    q = np.exp(z - lse_z[:, None])
    kl = kl_rows_from_logits(t, z)
    loss = loss_scale * float((om * kl).sum())
    dl = (q - p)
    if lam != 0.0:
        zr = z if z_ref is None else np.asarray(z_ref, dtype=np.float64)
        q_ref = np.exp(zr - logsumexp_rows(zr)[:, None])
        kl_reg = kl_rows_from_logits(zr, z)
        loss += loss_scale * lam * float((om * kl_reg).sum())
        dl = dl + lam * (q - q_ref)
    dl = loss_scale * om[:, None] * dl
    gW = dl.T @ hh
    gh = dl @ WW
    return dict(loss=loss, kl_rows=kl, z=z, lse_t=lse_t, lse_z=lse_z, dl=dl, gW=gW, gh=gh)


# ----------------------------------------------------------------------------
# a7: updates
# ----------------------------------------------------------------------------

def sgd_update(M, g, lr):
    """Alg. 1 'Update': M <- M - lr g."""
    return np.asarray(M, dtype=np.float64) - lr * g


def adamw_update(M, m, v, g, step, lr, beta1, beta2, eps, weight_decay):
    """Adam with decoupled weight decay, bias correction on,
    step counted from 1, eps outside the square root (R5)."""
    M = np.asarray(M, dtype=np.float64)
    m = np.asarray(m, dtype=np.float64)
    v = np.asarray(v, dtype=np.float64)
    M = M * (1.0 - lr * weight_decay)
    m_new = beta1 * m + (1.0 - beta1) * g
    v_new = beta2 * v + (1.0 - beta2) * g * g
    m_hat = m_new / (1.0 - beta1 ** step)
    v_hat = v_new / (1.0 - beta2 ** step)
    M_new = M - lr * m_hat / (np.sqrt(v_hat) + eps)
    return M_new, m_new, v_new


# ----------------------------------------------------------------------------
# f4: Adam with low-precision moment storage (R26; PAPER.md:393 names only "Adam")
# ----------------------------------------------------------------------------

def sr_bits16(idx, step, seed, d):
    """16 pseudo-random bits per element for stochastic rounding: a counter-based generator, so that the GPU and the
    oracle draw the same bits without exchanging them (each side implements it on its own).  Key: the element's
    position (v, j) in the [V, d] matrix (given as the linear index idx = v * d + j, 64-bit, and the row length d),
    Adam's count n of the step being taken, a caller seed.  ONE 32-bit hash serves the two vertically adjacent
    elements (2k, j) and (2k + 1, j) -- the even row takes its high half, the odd row its low half (R26: the
    hash is a third of the bf16-moment kernel's instructions, and every thread of the update kernels owns such pairs):

        pidx = (v >> 1) * d + j                                                                     (64-bit)
        x = lo32(pidx) ^ (n * 0x9E3779B9) ^ (seed * 0x85EBCA6B) ^ (hi32(pidx) * 0xC2B2AE35)       (mod 2^32)
        x ^= x >> 16;  x *= 0x7FEB352D;  x ^= x >> 15;  x *= 0x846CA68B;  x ^= x >> 16            (an integer mixer)
        bits = x >> 16 if v is even else x & 0xFFFF
    """
    idx = np.asarray(idx, dtype=np.uint64)
    d64 = np.uint64(d)
    v = idx // d64
    j = idx - v * d64
    pidx = (v >> np.uint64(1)) * d64 + j
    m32 = np.uint64(0xFFFFFFFF)
    lo = pidx & m32
    hi = pidx >> np.uint64(32)
    x = lo ^ ((np.uint64(step) * np.uint64(0x9E3779B9)) & m32) ^ ((np.uint64(seed) * np.uint64(0x85EBCA6B)) & m32) \
        ^ ((hi * np.uint64(0xC2B2AE35)) & m32)
    x ^= x >> np.uint64(16)
    x = (x * np.uint64(0x7FEB352D)) & m32
    x ^= x >> np.uint64(15)
    x = (x * np.uint64(0x846CA68B)) & m32
    x ^= x >> np.uint64(16)
    odd = (v & np.uint64(1)).astype(bool)
    return np.where(odd, x & np.uint64(0xFFFF), x >> np.uint64(16)).astype(np.uint32)


def f32_to_bf16_bits_sr(x, r16):
    """Stochastic rounding fp32 -> bf16 with 16 random bits r per element: the 16 discarded mantissa bits f of x
    round up with probability f / 65536 (up iff f + r >= 65536), so that E_r[result] = x exactly for uniform r."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    u = x.view(np.uint32).astype(np.uint64)
    return ((u + np.asarray(r16, dtype=np.uint64)) >> np.uint64(16)).astype(np.uint16)


def adamw_update_lowp(M, m_bits, v_bits, g, step, lr, beta1, beta2, eps, weight_decay, *, idx, seed, d):
    """Adam (conventions of ``adamw_update``, R5) with m and v STORED as bf16 (R26):

      1. dequantise        m = widen(m_bits), v = widen(v_bits)                      (exact)
      2. update            M, m_new, v_new exactly as adamw_update: the parameter step uses the UNROUNDED m_new, v_new
      3. requantise        m_bits' = rn_bf16(rn_fp32(m_new))                         round to nearest even
                           v_bits' = sr_bf16(rn_fp32(v_new), sr_bits16(idx, step, seed, d))   stochastic rounding:
                           beta2 = 0.999 decays v by 0.1% per step, below half a bf16 ulp (0.2-0.4%), so nearest
                           rounding would freeze v whenever g^2 << v; stochastic rounding keeps E[v] exact.
    The quantisation decisions are taken on the fp32 value (the precision the kernel computes in).
    Returns (M_new fp64, m_bits' uint16, v_bits' uint16, m_new fp64, v_new fp64)."""
    m = bf16_bits_to_f64(m_bits)
    v = bf16_bits_to_f64(v_bits)
    M_new, m_new, v_new = adamw_update(M, m, v, g, step, lr, beta1, beta2, eps, weight_decay)
    m_q = f32_to_bf16_bits(m_new.astype(np.float32))
    v_q = f32_to_bf16_bits_sr(v_new.astype(np.float32), sr_bits16(idx, step, seed, d))
    return M_new, m_q, v_q, m_new, v_new


def working_copy_bits(M_new):
    """bf16 working copy = rn_bf16(rn_fp32(M_new)): the GPU's master is fp32."""
    return f32_to_bf16_bits(np.asarray(M_new, dtype=np.float64).astype(np.float32))


# ----------------------------------------------------------------------------
# whole step
# ----------------------------------------------------------------------------

def distill_step(teacher_logits, h, W_in, W_master, adam_m, adam_v, pos_weight, mask,
                 *, seg_len, mask_mode=ROWS_ALL, loss_scale=1.0, optimizer="adamw",
                 lr=1e-5, beta1=0.9, beta2=0.999, eps=1e-8, weight_decay=0.0, step=1,
                 draft_logits=None, lam=0.0, z_ref=None, moments="f32", sr_seed=0):
    """One TTS update (Alg. 1 lines 'Loss' + 'Update'), dense.

    moments      : "f32" (default) or "bf16": adam_m / adam_v are uint16 bf16 bit patterns, updated by
                   ``adamw_update_lowp`` (the element index of W[v, j] is v * d + j); the result then also carries
                   ``m_bits`` / ``v_bits`` (what is stored) next to the unrounded ``m`` / ``v``

    draft_logits : the drafter's logits z, taken as given instead of h W_in^T
    lam, z_ref   : the regulariser lam * K~L(q_t || q) with q_t = softmax(z_ref)

    W_in     : working weights that produced q_t (bf16 bits or fp32)
    W_master : fp32 master (None when the parameters are fp32: W_in is the parameter)
    Returns dict with loss, kl_rows, gW, gh, master, m, v (fp64) and W_out
    (bf16 bits when a master exists, else fp32).
    """
    omega = row_weights(pos_weight, mask, mask_mode, seg_len)
    r = loss_and_grads(teacher_logits, h, W_in, omega, loss_scale, lam=lam, z_ref=z_ref, z=draft_logits)
    M = widen(W_master) if W_master is not None else widen(W_in)
    if optimizer == "sgd":
        M_new = sgd_update(M, r["gW"], lr)
        m_new = v_new = None
    elif moments == "bf16":
        V_, d_ = M.shape
        idx = np.arange(V_, dtype=np.uint64)[:, None] * np.uint64(d_) + np.arange(d_, dtype=np.uint64)[None, :]
        M_new, m_q, v_q, m_new, v_new = adamw_update_lowp(M, adam_m, adam_v, r["gW"], step, lr, beta1, beta2, eps,
                                                          weight_decay, idx=idx, seed=sr_seed, d=d_)
    else:
        M_new, m_new, v_new = adamw_update(M, widen(adam_m), widen(adam_v), r["gW"], step,
                                           lr, beta1, beta2, eps, weight_decay)
    out = dict(r)
    out.update(omega=omega, master=M_new, m=m_new, v=v_new)
    if optimizer != "sgd" and moments == "bf16":
        out.update(m_bits=m_q, v_bits=v_q)
    if W_master is not None:
        out["W_out"] = working_copy_bits(M_new)
    else:
        out["W_out"] = M_new.astype(np.float32)
    return out


def distill_inner_steps(teacher_logits, h, W_in, W_master, adam_m, adam_v, pos_weight, mask, *, K, lam,
                        step=1, draft_logits=None, **kw):
    """K optimisation steps on the same round's training signal (section 6.5).  q_t is the drafter
    that produced the canvas: z_ref = the logits of step 1 (h W_in^T, or the drafter's own ``draft_logits``).
    Step 1 is evaluated at q = q_t, where the lam term and its gradient vanish; steps 2..K recompute z from the
    weights the previous step wrote and add lam * K~L(q_t || q).  With a master, the working
    copy of step k is rn_bf16(rn_fp32(master_k)) and the GPU's master is fp32, so the master is rounded to fp32
    between steps.  Returns the last step's dict plus ``losses`` (all K)."""
    W, M, m, v = W_in, W_master, adam_m, adam_v
    z_ref, losses, out, kl1 = None, [], None, None
    for k in range(K):
        if k == 0:
            out = distill_step(teacher_logits, h, W, M, m, v, pos_weight, mask, step=step, draft_logits=draft_logits,
                               **kw)
            z_ref, kl1 = out["z"], out["kl_rows"]
        else:
            out = distill_step(teacher_logits, h, W, M, m, v, pos_weight, mask, step=step + k, lam=lam, z_ref=z_ref,
                               **kw)
        losses.append(out["loss"])
        W = out["W_out"]
        M = out["master"].astype(np.float32) if W_master is not None else None
        m, v = out["m"], out["v"]
    out = dict(out)
    out.update(losses=np.array(losses), kl_rows_step1=kl1)
    return out


def row_normalisers(teacher_logits, h, W_in, slab=8192):
    """Full-vocabulary z, lse_t, lse_z, KL_r computed slab by slab over V (same
    arithmetic as ``loss_and_grads`` steps 1-3; only the matmul is split)."""
    t = widen(teacher_logits)
    hh = widen(h)
    V = W_in.shape[0]
    z = np.empty((hh.shape[0], V), dtype=np.float64)
    for v0 in range(0, V, slab):
        z[:, v0:v0 + slab] = hh @ widen(W_in[v0:v0 + slab]).T
    lse_t = logsumexp_rows(t)
    lse_z = logsumexp_rows(z)
    kl = kl_rows_from_logits(t, z)
    return z, lse_t, lse_z, kl


def distill_step_rows(rows, z, lse_t, lse_z, teacher_logits, h, W_in_rows, W_master_rows,
                      adam_m_rows, adam_v_rows, omega, *, loss_scale=1.0, optimizer="adamw",
                      lr=1e-5, beta1=0.9, beta2=0.999, eps=1e-8, weight_decay=0.0, step=1, moments="f32", sr_seed=0):
    """The step for the vocabulary rows ``rows`` only (gW rows, updated state),
    given the full-vocabulary normalisers from ``row_normalisers``."""
    t = widen(teacher_logits)[:, rows]
    hh = widen(h)
    om = np.asarray(omega, dtype=np.float64)
    p = np.exp(t - lse_t[:, None])
    q = np.exp(z[:, rows] - lse_z[:, None])
    dl = loss_scale * om[:, None] * (q - p)
    gW = dl.T @ hh
    M = widen(W_master_rows) if W_master_rows is not None else widen(W_in_rows)
    out = {}
    if optimizer == "sgd":
        M_new, m_new, v_new = sgd_update(M, gW, lr), None, None
    elif moments == "bf16":
        d_ = M.shape[1]
        idx = np.asarray(rows, dtype=np.uint64)[:, None] * np.uint64(d_) + np.arange(d_, dtype=np.uint64)[None, :]
        M_new, m_q, v_q, m_new, v_new = adamw_update_lowp(M, adam_m_rows, adam_v_rows, gW, step, lr, beta1, beta2, eps,
                                                          weight_decay, idx=idx, seed=sr_seed, d=d_)
        out.update(m_bits=m_q, v_bits=v_q)
    else:
        M_new, m_new, v_new = adamw_update(M, widen(adam_m_rows), widen(adam_v_rows), gW, step,
                                           lr, beta1, beta2, eps, weight_decay)
    out.update(dl=dl, gW=gW, master=M_new, m=m_new, v=v_new)
    return out


def gh_full(z, lse_t, lse_z, teacher_logits, W_in, omega, loss_scale=1.0, slab=8192):
    """gh = dl W accumulated slab by slab over V (a5)."""
    t = widen(teacher_logits)
    om = np.asarray(omega, dtype=np.float64)
    V = W_in.shape[0]
    gh = np.zeros((t.shape[0], W_in.shape[1]), dtype=np.float64)
    for v0 in range(0, V, slab):
        sl = slice(v0, min(V, v0 + slab))
        dl = loss_scale * om[:, None] * (np.exp(z[:, sl] - lse_z[:, None]) - np.exp(t[:, sl] - lse_t[:, None]))
        gh += dl @ widen(W_in[sl])
    return gh


# ----------------------------------------------------------------------------
# what vocabulary shards exchange
# ----------------------------------------------------------------------------

def shard_row_stats(teacher_cols, z_cols):
    """Per row, over the columns of one vocabulary slice:
        m_t = max t,  s_t = sum e^{t - m_t},  a = sum e^{t - m_t} (t - z),  m_z = max z,  s_z = sum e^{z - m_z}
    Teacher entries equal to -inf have p = 0 and are dropped (0 log 0 := 0); a slice whose teacher entries are all
    -inf gives (m_t, s_t, a) = (-inf, 0, 0).  Returns [T, 5] fp64."""
    t = widen(teacher_cols)
    z = np.asarray(z_cols, dtype=np.float64)
    T = t.shape[0]
    out = np.zeros((T, 5), dtype=np.float64)
    for r in range(T):
        keep = t[r] != -np.inf
        if keep.any():
            mt = t[r][keep].max()
            e = np.exp(t[r][keep] - mt)
            out[r, 0], out[r, 1], out[r, 2] = mt, e.sum(), (e * (t[r][keep] - z[r][keep])).sum()
        else:
            out[r, 0] = -np.inf
        mz = z[r].max()
        out[r, 3], out[r, 4] = mz, np.exp(z[r] - mz).sum()
    return out


def merge_shard_stats(stats_all):
    """stats_all [G, T, 5] -> (lse_t, lse_z, KL_r) of the whole rows: rescale every slice to the common maximum,
    add, then  lse_t = m_t + log s_t,  lse_z = m_z + log s_z,  KL_r = a / s_t - lse_t + lse_z."""
    st = np.asarray(stats_all, dtype=np.float64)
    mt = st[:, :, 0].max(axis=0)
    mz = st[:, :, 3].max(axis=0)
    with np.errstate(invalid="ignore"):
        et = np.where(st[:, :, 0] == -np.inf, 0.0, np.exp(st[:, :, 0] - mt[None, :]))
    ez = np.exp(st[:, :, 3] - mz[None, :])
    s_t = (st[:, :, 1] * et).sum(axis=0)
    a = (st[:, :, 2] * et).sum(axis=0)
    s_z = (st[:, :, 4] * ez).sum(axis=0)
    lse_t = mt + np.log(s_t)
    lse_z = mz + np.log(s_z)
    return lse_t, lse_z, a / s_t - lse_t + lse_z
