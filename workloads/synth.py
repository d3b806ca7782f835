"""Seeded synthetic inputs for the TTS distillation step.

This module serves BOTH the CUDA path's tests/bench and the oracle's tests; it
holds none of the method's arithmetic (no softmax, KL, gradient or optimiser):
only random draws, the draft-logit product that the recipes need to build
"teacher = draft logits + perturbation", bf16 rounding, and the planting of an
accepted prefix.  It imports neither the oracle nor the CUDA binding.

The arrays stand in for the paper's benchmark workloads (AIME, MATH-500,
OlympiadBench, GPQA-diamond, TheoremQA, LiveCodeBench), which are
not available here: only the shapes (T, V, d), the structure "teacher = draft +
perturbation", an acceptance-length distribution with mean near the paper's
2.4-4.9 (Tables 1-3) and drift over thousands of rounds are reproduced.

bf16 tensors are returned as uint16 bit patterns (round-to-nearest-even) so that
the oracle and the GPU consume identical bits.
"""

from __future__ import annotations

import numpy as np

# dtype / optimiser / mask-mode codes: numerically equal to include/tts.h
F32, BF16 = 0, 1
SGD, ADAMW = 0, 1
ROWS_ALL, ROWS_ACCEPTED, ROWS_ACCEPTED_PLUS_ONE = 0, 1, 2

CONFIGS = {
    # BASELINE.json configs[0]
    1: dict(name="tiny_fp32", V=1024, d=64, T=8, seg_len=8, n_seq=1, param=F32, logits=F32,
            optimizer=SGD, lr=1e-3, seed=0, sigma=("const", 1.5), weights="ones",
            plant=False, loss_scale=1.0),
    # configs[1]
    2: dict(name="llama31_8b_head", V=128256, d=4096, T=16, seg_len=16, n_seq=1, param=BF16,
            logits=BF16, optimizer=ADAMW, lr=1e-5, seed=1, sigma=("const", 1.0), weights="ones",
            plant=False, loss_scale=1.0),
    # configs[2]  (headline)
    3: dict(name="qwen3_8b_head", V=151936, d=4096, T=16, seg_len=16, n_seq=1, param=BF16,
            logits=BF16, optimizer=ADAMW, lr=1e-5, seed=2, sigma=("uniform", 0.5, 3.0),
            weights="exp7", plant=True, loss_scale=1.0),
    # configs[3]
    4: dict(name="batched_32x16", V=151936, d=4096, T=512, seg_len=16, n_seq=32, param=BF16,
            logits=BF16, optimizer=ADAMW, lr=1e-5, seed=3000, sigma=("uniform", 0.5, 3.0),
            weights="exp7", plant=True, loss_scale=1.0 / 32.0),
    # configs[4]  (stream; per-round teacher is built by the harness, see stream_round())
    5: dict(name="qwen3_32b_head_stream", V=151936, d=5120, T=16, seg_len=16, n_seq=1, param=BF16,
            logits=BF16, optimizer=ADAMW, lr=1e-5, seed=4, sigma=("const", 1.5), weights="exp7",
            plant=False, loss_scale=1.0, rounds=4000, mu_max=3.0),
}
ADAM_DEFAULTS = dict(beta1=0.9, beta2=0.999, eps=1e-8, weight_decay=0.0)


def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    x = np.ascontiguousarray(x, dtype=np.float32)
    u = x.view(np.uint32)
    r = (u + (np.uint32(0x7FFF) + ((u >> np.uint32(16)) & np.uint32(1)))) >> np.uint32(16)
    return r.astype(np.uint16)


def bf16_bits_to_f32(b: np.ndarray) -> np.ndarray:
    return (np.ascontiguousarray(b, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32)


def position_weights(kind: str, seg_len: int, n_seq: int) -> np.ndarray:
    """w_k expanded per row.  'ones': w_k = 1 (the standard
    distillation loss).  'exp7': w_k = exp(-(k-1)/7), k = 1..C, a decreasing
    profile as PAPER.md:127 describes (the authors' values are not in the paper)."""
    k = np.arange(seg_len, dtype=np.float64)
    w = np.ones(seg_len) if kind == "ones" else np.exp(-k / 7.0)
    return np.tile(w, n_seq).astype(np.float32)


def _draft_logits_f32(h_f32: np.ndarray, W_f32_rows, V: int, slab: int = 16384) -> np.ndarray:
    """h . W^T in fp32, slab by slab (generator only: shapes the teacher)."""
    z = np.empty((h_f32.shape[0], V), dtype=np.float32)
    for v0 in range(0, V, slab):
        z[:, v0:v0 + slab] = h_f32 @ W_f32_rows(v0, min(V, v0 + slab)).T
    return z


def _plant_prefix(t: np.ndarray, tok: np.ndarray, tau_star: int) -> None:
    """Make exactly the first tau_star rows of this segment match (in place)."""
    C = t.shape[0]
    for k in range(min(tau_star, C)):
        t[k, tok[k]] = t[k].max() + 1.0
    if tau_star < C:
        k = tau_star
        if int(np.argmax(t[k])) == int(tok[k]):
            second = np.partition(t[k], -2)[-2]
            t[k, tok[k]] = second - 1.0


def make_case(cfg_id: int, *, V: int | None = None, d: int | None = None, n_seq: int | None = None,
              seg_len: int | None = None, seed: int | None = None, nonzero_state: bool = False,
              step: int = 1):
    """Build one step's inputs for BASELINE.json config ``cfg_id`` (1-4), optionally
    scaled down (V, d, n_seq, seg_len overrides keep the recipe).  Returns a dict of
    numpy arrays (bf16 as uint16 bits) plus the hyper-parameters.

    nonzero_state: draw Adam moments as if earlier steps had happened instead of the configs' m = v = 0, to exercise
    the general update.  Every recipe stays inside the set an optimiser run can reach: moments that are exponential
    averages of ONE gradient sequence satisfy m^2 <= (1-b1)^2 / ((1-b2) (1 - b1^2/b2)) v = 52.8 v (Cauchy-Schwarz,
    b = 0.9 / 0.999), i.e. |m| / sqrt(v) <= 7.27 (R12); independent draws of m and v do not.
        True / "mix"   element (v, j) takes recipe (v + j) % 4 of: "uniform", "const2", "const10", "const1000"
        "uniform"      v ~ 1e-10 chi^2,  m = sqrt(v) U(-7.2, 7.2): the whole reachable band of |m| / sqrt(v)
        "const<n>"     the state after n steps of a CONSTANT gradient g0 ~ 1e-5 N(0,1) (the most ordinary Adam
                       state): m = g0 (1 - b1^n), v = g0^2 (1 - b2^n); |m| / sqrt(v) = 4.25 / 6.52 / 1.26 at
                       n = 2 / 10 / 1000.  Pass step = n + 1 for the matching bias corrections.
    """
    c = dict(CONFIGS[cfg_id])
    c.update(ADAM_DEFAULTS)
    if V is not None: c["V"] = V
    if d is not None: c["d"] = d
    if seg_len is not None: c["seg_len"] = seg_len
    if n_seq is not None: c["n_seq"] = n_seq
    if seed is not None: c["seed"] = seed
    V, d, C, S = c["V"], c["d"], c["seg_len"], c["n_seq"]
    T = C * S
    c["T"] = T
    bf = c["param"] == BF16

    rng_w = np.random.Generator(np.random.PCG64(c["seed"] if cfg_id != 4 else 2999))
    master = rng_w.standard_normal((V, d), dtype=np.float32)
    master *= np.float32(0.02)
    if bf:
        W_bits = f32_to_bf16_bits(master)
        rows = lambda a, b: bf16_bits_to_f32(W_bits[a:b])
    else:
        W_bits = None
        rows = lambda a, b: master[a:b]

    h_all = np.empty((T, d), dtype=np.float32)
    t_all = np.empty((T, V), dtype=np.float32)
    tok_all = np.empty(T, dtype=np.int32)
    tau_star = np.zeros(S, dtype=np.int32)
    for s in range(S):
        rng = rng_w if cfg_id != 4 else np.random.Generator(np.random.PCG64(c["seed"] + s))
        h = rng.standard_normal((C, d), dtype=np.float32)
        if bf:
            h = bf16_bits_to_f32(f32_to_bf16_bits(h))
        z = _draft_logits_f32(h, rows, V)
        kind = c["sigma"]
        if kind[0] == "const":
            sig = np.full(C, kind[1], dtype=np.float32)
        else:
            sig = rng.uniform(kind[1], kind[2], size=C).astype(np.float32)
        t = z + sig[:, None] * rng.standard_normal((C, V), dtype=np.float32)
        tok = np.argmax(z, axis=1).astype(np.int32)
        if c["plant"]:
            g = int(rng.geometric(0.4))
            tau_star[s] = min(g, C)
            _plant_prefix(t, tok, int(tau_star[s]))
        if c["logits"] == BF16:
            t = bf16_bits_to_f32(f32_to_bf16_bits(t))
        if c["plant"]:  # re-verify after rounding
            am = np.argmax(t, axis=1)
            ts = int(tau_star[s])
            assert (am[:ts] == tok[:ts]).all() and (ts == C or am[ts] != tok[ts])
        h_all[s * C:(s + 1) * C] = h
        t_all[s * C:(s + 1) * C] = t
        tok_all[s * C:(s + 1) * C] = tok

    out = dict(cfg=c, V=V, d=d, T=T, seg_len=C, tau_star=tau_star if c["plant"] else None,
               draft_tokens=tok_all, pos_weight=position_weights(c["weights"], C, S),
               loss_scale=float(c["loss_scale"]), step=step)
    out["teacher"] = f32_to_bf16_bits(t_all) if c["logits"] == BF16 else t_all
    out["h"] = f32_to_bf16_bits(h_all) if bf else h_all
    if bf:
        out["W"] = W_bits
        out["master"] = master
    else:
        out["W"] = master
        out["master"] = None
    if c["optimizer"] == ADAMW:
        if nonzero_state:
            out["m"], out["v"] = adam_state(V, d, "mix" if nonzero_state is True else nonzero_state, c["seed"] + 77,
                                            c["beta1"], c["beta2"])
        else:
            out["m"] = np.zeros((V, d), dtype=np.float32)
            out["v"] = np.zeros((V, d), dtype=np.float32)
    else:
        out["m"] = out["v"] = None
    return out


def adam_state(V: int, d: int, kind: str, seed: int, beta1: float = 0.9, beta2: float = 0.999):
    """Non-zero Adam moments (m, v) of the recipes documented at make_case (all inside |m| / sqrt(v) <= 7.27)."""
    rs = np.random.Generator(np.random.PCG64(seed))

    def uniform():
        v = (1e-10 * rs.standard_normal((V, d), dtype=np.float32) ** 2).astype(np.float32)
        m = (np.sqrt(v) * rs.uniform(-7.2, 7.2, (V, d)).astype(np.float32)).astype(np.float32)
        return m, v

    def const(n):
        g0 = (1e-5 * rs.standard_normal((V, d), dtype=np.float32)).astype(np.float64)
        return ((g0 * (1.0 - beta1 ** n)).astype(np.float32), (g0 * g0 * (1.0 - beta2 ** n)).astype(np.float32))

    if kind == "uniform":
        return uniform()
    if kind.startswith("const"):
        return const(int(kind[5:]))
    assert kind == "mix", kind
    parts = [uniform(), const(2), const(10), const(1000)]
    sel = (np.arange(V)[:, None] + np.arange(d)[None, :]) % 4
    m = np.empty((V, d), dtype=np.float32)
    v = np.empty((V, d), dtype=np.float32)
    for k, (pm, pv) in enumerate(parts):
        m[sel == k] = pm[sel == k]
        v[sel == k] = pv[sel == k]
    return m, v


def stream_direction(V: int, seed: int = 4) -> np.ndarray:
    """Config 5: the fixed drift direction u in R^V (R16): a scalar mean
    added to every logit cancels in the softmax, so the drift is mu_t * u."""
    return np.random.Generator(np.random.PCG64(seed * 1000003 + 1)).standard_normal(V, dtype=np.float32)


def stream_mu(t: int, rounds: int = 4000, mu_max: float = 3.0) -> float:
    return mu_max * t / rounds


def make_stream(*, V: int, d: int, rounds: int, seg_len: int = 16, seed: int = 4, mu_max: float = 3.0,
                sigma: float = 1.5, total_rounds: int | None = None):
    """Config 5 scaled down, on the host, for the round-by-round parity test (R16): a fixed initial head
    (master ~ N(0,0.02), W0 = rn_bf16(master)), the drift direction u, and per round t
        h_t ~ N(0,1) (bf16),  teacher_t = rn_bf16(h_t . W0^T + mu_t u + sigma eps_t),  tokens_t = argmax h_t . W0^T.
    The teacher is built from the INITIAL weights so that the GPU path and the oracle, whose weights evolve
    separately, consume identical bits at every round.  (bench.py's full-size stream builds it from the current
    weights on the device instead, which is what a verifier would see; that run is timed, not compared.)
    Returns (case0, rounds_list): case0 has cfg / W / master / m / v / pos_weight; rounds_list[t] = dict(teacher, h,
    draft_tokens)."""
    c = dict(CONFIGS[5])
    c.update(ADAM_DEFAULTS)
    c.update(V=V, d=d, seg_len=seg_len, T=seg_len, n_seq=1, seed=seed)
    total = total_rounds or rounds
    rng = np.random.Generator(np.random.PCG64(seed))
    master = rng.standard_normal((V, d), dtype=np.float32) * np.float32(0.02)
    W_bits = f32_to_bf16_bits(master)
    W0 = bf16_bits_to_f32(W_bits)
    u = stream_direction(V, seed)
    out = []
    for t in range(rounds):
        r = np.random.Generator(np.random.PCG64([seed, t]))
        h = bf16_bits_to_f32(f32_to_bf16_bits(r.standard_normal((seg_len, d), dtype=np.float32)))
        z = h @ W0.T
        tl = z + np.float32(stream_mu(t, total, mu_max)) * u[None, :] + np.float32(sigma) * r.standard_normal(
            (seg_len, V), dtype=np.float32)
        out.append(dict(teacher=f32_to_bf16_bits(tl), h=f32_to_bf16_bits(h),
                        draft_tokens=np.argmax(z, axis=1).astype(np.int32)))
    case0 = dict(cfg=c, V=V, d=d, T=seg_len, seg_len=seg_len, W=W_bits, master=master,
                 m=np.zeros((V, d), dtype=np.float32), v=np.zeros((V, d), dtype=np.float32),
                 pos_weight=position_weights(c["weights"], seg_len, 1), loss_scale=1.0)
    return case0, out


def planted_mask_cases(V: int, seg_len: int, seed: int = 11, dtype=BF16):
    """Teacher logits / tokens with planted tau in {0, 1, 3, seg_len}, ties at the
    maximum (lowest index must win) and -inf entries; one segment per case."""
    rng = np.random.Generator(np.random.PCG64(seed))
    taus = [0, 1, min(3, seg_len), seg_len]
    S = len(taus) + 2
    t = (2.0 * rng.standard_normal((S * seg_len, V), dtype=np.float32)).astype(np.float32)
    if dtype == BF16:
        t = bf16_bits_to_f32(f32_to_bf16_bits(t))
    tok = rng.integers(0, V, size=S * seg_len).astype(np.int32)
    expect_tau = []
    for s, ta in enumerate(taus):
        seg = t[s * seg_len:(s + 1) * seg_len]
        _plant_prefix(seg, tok[s * seg_len:(s + 1) * seg_len], ta)
        expect_tau.append(ta)
    # ties: two equal maxima, token = the lower index on rows 0..1, the higher on row 2
    s = len(taus)
    seg = t[s * seg_len:(s + 1) * seg_len]
    for k in range(min(3, seg_len)):
        lo, hi = sorted(rng.choice(V, size=2, replace=False).tolist())
        top = np.float32(64.0)
        seg[k, lo] = top
        seg[k, hi] = top
        tok[s * seg_len + k] = lo if k < 2 else hi
    expect_tau.append(min(2, seg_len))
    # -inf entries everywhere except a few finite ones; also row maximum at v = V-1
    s += 1
    seg = t[s * seg_len:(s + 1) * seg_len]
    seg[:, ::2] = -np.inf
    seg[0, V - 1] = np.float32(100.0)
    tok[s * seg_len] = V - 1
    if seg_len > 1:
        tok[s * seg_len + 1] = (int(np.argmax(seg[1])) + 1) % V  # mismatch at k = 1
    expect_tau.append(1 if seg_len > 1 else 1)
    out_t = f32_to_bf16_bits(t) if dtype == BF16 else t
    return out_t, tok, np.array(expect_tau, dtype=np.int32)


# ----------------------------------------------------------------------------
# Full-size cases built ON THE DEVICE (bench.py and the full-size parity tests).
# Same recipe as make_case, with torch's seeded device generator in place of numpy's
# (the full-size host recipe needs minutes and ~10 GB of host memory per case).  Only
# random draws, the draft-logit product the recipe needs, bf16 rounding, argmax for the
# canvas tokens and the prefix planting: none of the method's arithmetic.
# ----------------------------------------------------------------------------

def make_case_device(cfg_id: int, device="cuda:0", *, seed_offset: int = 0, n_seq: int | None = None,
                     V: int | None = None, d: int | None = None, shared_h: bool = False):
    """Returns a dict of torch tensors on ``device``: teacher [T,V], h [T,d], W [V,d] (bf16),
    master/m/v [V,d] fp32, draft_tokens [T] i32, pos_weight [T] f32, plus cfg, tau_star (host
    numpy) and loss_scale.  ``seed_offset`` gives independent replicas (multi-GPU ranks); with ``shared_h`` the hidden
    states do not depend on it (vocabulary shards: every rank holds the same h and its own rows of W)."""
    import torch

    c = dict(CONFIGS[cfg_id])
    c.update(ADAM_DEFAULTS)
    if n_seq is not None: c["n_seq"] = n_seq
    if V is not None: c["V"] = V
    if d is not None: c["d"] = d
    V, d, C, S = c["V"], c["d"], c["seg_len"], c["n_seq"]
    T = C * S
    c["T"] = T
    assert c["param"] == BF16 and c["logits"] == BF16
    dev = torch.device(device)
    g = torch.Generator(device=dev)
    g.manual_seed(1000003 * (c["seed"] + 1) + seed_offset)
    rng = np.random.Generator(np.random.PCG64(c["seed"] + 7919 * seed_offset))

    master = torch.empty((V, d), dtype=torch.float32, device=dev)
    master.normal_(0.0, 0.02, generator=g)
    W = master.to(torch.bfloat16)
    gh_ = g
    if shared_h:
        gh_ = torch.Generator(device=dev)
        gh_.manual_seed(1000003 * (c["seed"] + 1) + 999983)
    h = torch.empty((T, d), dtype=torch.float32, device=dev).normal_(0.0, 1.0, generator=gh_).to(torch.bfloat16)
    z = (h.float() @ W.float().T) if T * V <= (1 << 24) else torch.cat(
        [h[i:i + 64].float() @ W.float().T for i in range(0, T, 64)], 0)
    kind = c["sigma"]
    if kind[0] == "const":
        sig = np.full(T, kind[1], dtype=np.float32)
    else:
        sig = rng.uniform(kind[1], kind[2], size=T).astype(np.float32)
    noise = torch.empty((T, V), dtype=torch.float32, device=dev).normal_(0.0, 1.0, generator=g)
    t = z + torch.from_numpy(sig).to(dev)[:, None] * noise
    del noise
    tok = torch.argmax(z, dim=1).to(torch.int32)
    tau_star = None
    if c["plant"]:
        tau_star = np.minimum(rng.geometric(0.4, size=S), C).astype(np.int32)
        rmax = t.max(dim=1).values
        for s in range(S):
            for k in range(C):
                r = s * C + k
                if k < tau_star[s]:
                    t[r, tok[r]] = rmax[r] + 1.0
                elif k == tau_star[s]:
                    if int(torch.argmax(t[r])) == int(tok[r]):
                        t[r, tok[r]] = torch.topk(t[r], 2).values[1] - 1.0
    teacher = t.to(torch.bfloat16)
    del t, z
    pw = torch.from_numpy(position_weights(c["weights"], C, S)).to(dev)
    out = dict(cfg=c, V=V, d=d, T=T, seg_len=C, tau_star=tau_star, teacher=teacher, h=h, W=W, master=master,
               m=torch.zeros_like(master), v=torch.zeros_like(master), draft_tokens=tok, pos_weight=pw,
               loss_scale=float(c["loss_scale"]), step=1)
    return out
