"""Pins for the fp64 oracle (oracle/tts_oracle.py): every function is checked
against something other than itself -- brute-force enumeration through the
softmax Jacobian in plain Python floats, central finite differences, closed
forms, invariants, and fp64 torch autograd / torch.optim (the paper's own
implementation is "a sequence of standard pytorch kernels").
The paper prints no worked numeric example for this path, so
there are no printed values to hit.
"""
import math

import numpy as np
import pytest
import torch

from oracle import tts_oracle as O


def _rng(seed):
    return np.random.Generator(np.random.PCG64(seed))


def _small(seed, T=3, V=5, d=3):
    r = _rng(seed)
    h = r.standard_normal((T, d))
    W = 0.5 * r.standard_normal((V, d))
    t = r.standard_normal((T, V)) * 1.3
    om = r.uniform(0.2, 1.0, size=T)
    return t, h, W, om


# ---------------------------------------------------------------- 1. brute force
def _brute(t, h, W, om, scale):
    """Literal definitions, plain Python floats, no max-subtraction, no (q-p)
    shortcut: dL/dz_v = sum_u (-p_u/q_u) * q_u (delta_uv - q_v)."""
    T, V = len(t), len(t[0])
    d = len(h[0])
    loss = 0.0
    dz = [[0.0] * V for _ in range(T)]
    kls = []
    for r in range(T):
        z = [sum(h[r][j] * W[v][j] for j in range(d)) for v in range(V)]
        se_t = sum(math.exp(x) for x in t[r])
        se_z = sum(math.exp(x) for x in z)
        p = [math.exp(x) / se_t for x in t[r]]
        q = [math.exp(x) / se_z for x in z]
        kl = sum(p[u] * math.log(p[u] / q[u]) for u in range(V))
        kls.append(kl)
        loss += scale * om[r] * kl
        for v in range(V):
            acc = 0.0
            for u in range(V):
                dq_u_dz_v = q[u] * ((1.0 if u == v else 0.0) - q[v])
                acc += (-p[u] / q[u]) * dq_u_dz_v
            dz[r][v] = scale * om[r] * acc
    gW = [[sum(dz[r][v] * h[r][j] for r in range(T)) for j in range(d)] for v in range(V)]
    gh = [[sum(dz[r][v] * W[v][j] for v in range(V)) for j in range(d)] for r in range(T)]
    return loss, kls, dz, gW, gh


@pytest.mark.parametrize("T,V,d,seed", [(1, 2, 1, 0), (2, 3, 2, 1), (3, 5, 3, 2), (3, 2, 3, 3)])
def test_brute_force_enumeration(T, V, d, seed):
    t, h, W, om = _small(seed, T, V, d)
    scale = 0.7
    loss, kls, dz, gW, gh = _brute(t.tolist(), h.tolist(), W.tolist(), om.tolist(), scale)
    r = O.loss_and_grads(t, h, W, om, loss_scale=scale)
    assert r["loss"] == pytest.approx(loss, rel=1e-12, abs=1e-14)
    np.testing.assert_allclose(r["kl_rows"], kls, rtol=1e-11, atol=1e-14)
    np.testing.assert_allclose(r["dl"], dz, rtol=1e-10, atol=1e-14)
    np.testing.assert_allclose(r["gW"], gW, rtol=1e-10, atol=1e-14)
    np.testing.assert_allclose(r["gh"], gh, rtol=1e-10, atol=1e-14)


# ---------------------------------------------------------------- 2. finite differences
@pytest.mark.parametrize("lam", [0.0, 0.3])
def test_finite_differences(lam):
    T, V, d = 3, 16, 4
    t, h, W, om = _small(7, T, V, d)
    z_ref = (h @ W.T) + 0.2 * _rng(8).standard_normal((T, V)) if lam else None
    f = lambda hh, WW: O.loss_and_grads(t, hh, WW, om, 1.3, lam, z_ref)["loss"]
    r = O.loss_and_grads(t, h, W, om, 1.3, lam, z_ref)
    eps = 1e-6
    gW_fd = np.zeros_like(W)
    for v in range(V):
        for j in range(d):
            Wp, Wm = W.copy(), W.copy()
            Wp[v, j] += eps
            Wm[v, j] -= eps
            gW_fd[v, j] = (f(h, Wp) - f(h, Wm)) / (2 * eps)
    gh_fd = np.zeros_like(h)
    for rr in range(T):
        for j in range(d):
            hp, hm = h.copy(), h.copy()
            hp[rr, j] += eps
            hm[rr, j] -= eps
            gh_fd[rr, j] = (f(hp, W) - f(hm, W)) / (2 * eps)
    np.testing.assert_allclose(r["gW"], gW_fd, rtol=2e-7, atol=2e-9)
    np.testing.assert_allclose(r["gh"], gh_fd, rtol=2e-7, atol=2e-9)


# ---------------------------------------------------------------- 3. closed forms
def test_teacher_equals_draft_gives_zero():
    _, h, W, om = _small(3, 4, 9, 3)
    t = h @ W.T
    r = O.loss_and_grads(t, h, W, om)
    assert r["loss"] == 0.0
    assert np.all(r["kl_rows"] == 0.0)
    assert np.all(r["dl"] == 0.0) and np.all(r["gW"] == 0.0) and np.all(r["gh"] == 0.0)


def test_binary_vocab_closed_form():
    t = np.array([[0.3, -1.1], [2.0, 0.5]])
    h = np.array([[1.0, 0.5], [-0.3, 2.0]])
    W = np.array([[0.2, -0.4], [0.7, 0.1]])
    z = h @ W.T
    sig = lambda x: 1.0 / (1.0 + np.exp(-x))
    p = sig(t[:, 0] - t[:, 1])
    q = sig(z[:, 0] - z[:, 1])
    kl = p * np.log(p / q) + (1 - p) * np.log((1 - p) / (1 - q))
    r = O.loss_and_grads(t, h, W, np.ones(2))
    np.testing.assert_allclose(r["kl_rows"], kl, rtol=1e-13)
    np.testing.assert_allclose(r["dl"][:, 0], q - p, rtol=1e-12)
    np.testing.assert_allclose(r["dl"][:, 1], p - q, rtol=1e-12)


def test_uniform_draft_closed_form():
    t, h, _, om = _small(4, 3, 11, 4)
    W = np.zeros((11, 4))
    r = O.loss_and_grads(t, h, W, np.ones(3))
    p = np.exp(t) / np.exp(t).sum(1, keepdims=True)
    H = -(p * np.log(p)).sum(1)
    np.testing.assert_allclose(r["kl_rows"], np.log(11) - H, rtol=1e-12)


def test_one_hot_teacher_is_cross_entropy():
    t, h, W, _ = _small(5, 3, 7, 3)
    t = np.zeros_like(t)
    hot = [2, 0, 6]
    for r_, j in enumerate(hot):
        t[r_, j] = 800.0  # exactly one-hot in fp64
    r = O.loss_and_grads(t, h, W, np.ones(3))
    z = h @ W.T
    q = np.exp(z) / np.exp(z).sum(1, keepdims=True)
    np.testing.assert_allclose(r["kl_rows"], [-np.log(q[i, j]) for i, j in enumerate(hot)], rtol=1e-12)
    e = np.zeros_like(q)
    for i, j in enumerate(hot):
        e[i, j] = 1.0
    np.testing.assert_allclose(r["dl"], q - e, rtol=1e-12, atol=1e-15)


def test_sgd_and_adam_first_step_closed_forms():
    r = _rng(6)
    M = r.standard_normal((6, 4))
    g = r.standard_normal((6, 4)) * 1e-3
    g[0, 0] = 0.0
    np.testing.assert_array_equal(O.sgd_update(M, g, 0.01), M - 0.01 * g)
    lr, eps = 1e-3, 1e-8
    Mn, m, v = O.adamw_update(M, np.zeros_like(M), np.zeros_like(M), g, 1, lr, 0.9, 0.999, eps, 0.0)
    np.testing.assert_allclose(m, 0.1 * g, rtol=1e-14)
    np.testing.assert_allclose(v, 0.001 * g * g, rtol=1e-12)
    np.testing.assert_allclose(Mn - M, -lr * g / (np.abs(g) + eps), rtol=1e-9, atol=1e-18)
    assert np.all(np.abs(Mn - M) < lr) and (Mn - M)[0, 0] == 0.0
    # decoupled decay acts on the weights only
    Mn2, m2, v2 = O.adamw_update(M, np.zeros_like(M), np.zeros_like(M), np.zeros_like(g), 1, lr, 0.9, 0.999, eps, 0.1)
    np.testing.assert_allclose(Mn2, M * (1 - lr * 0.1), rtol=1e-15)
    assert not m2.any() and not v2.any()


# ---------------------------------------------------------------- 4. invariants
def test_invariants():
    T, V, d = 4, 23, 5
    t, h, W, om = _small(9, T, V, d)
    r = O.loss_and_grads(t, h, W, om, 0.8)
    assert np.all(r["kl_rows"] >= 0)
    np.testing.assert_allclose(r["dl"].sum(1), 0, atol=1e-15)
    np.testing.assert_allclose(r["gW"].sum(0), 0, atol=1e-14)
    # rank(gW) <= T: gW x = 0 for x orthogonal to span(h)
    qh, _ = np.linalg.qr(h.T, mode="complete")
    x = qh[:, T:] if d > T else None
    if x is not None and x.size:
        np.testing.assert_allclose(r["gW"] @ x, 0, atol=1e-14)
    # gh_r = scale * omega_r (E_q[W] - E_p[W])
    z = h @ W.T
    q = np.exp(z) / np.exp(z).sum(1, keepdims=True)
    p = np.exp(t) / np.exp(t).sum(1, keepdims=True)
    np.testing.assert_allclose(r["gh"], 0.8 * om[:, None] * (q @ W - p @ W), rtol=1e-11, atol=1e-15)
    # shift invariance of teacher rows
    r2 = O.loss_and_grads(t + np.arange(T)[:, None] * 3.7, h, W, om, 0.8)
    np.testing.assert_allclose(r2["loss"], r["loss"], rtol=1e-12)
    np.testing.assert_allclose(r2["gW"], r["gW"], rtol=1e-9, atol=1e-14)
    # linearity in loss_scale and in each omega_r; omega_r = 0 rows contribute nothing
    r3 = O.loss_and_grads(t, h, W, om, 1.6)
    np.testing.assert_allclose(r3["gW"], 2 * r["gW"], rtol=1e-12)
    om0 = om.copy()
    om0[1] = 0.0
    r4 = O.loss_and_grads(t, h, W, om0, 0.8)
    keep = [0, 2, 3]
    r5 = O.loss_and_grads(t[keep], h[keep], W, om[keep], 0.8)
    np.testing.assert_allclose(r4["gW"], r5["gW"], rtol=1e-12, atol=1e-16)
    np.testing.assert_allclose(r4["loss"], r5["loss"], rtol=1e-13)
    assert not r4["gh"][1].any()
    # vocabulary permutation
    perm = _rng(10).permutation(V)
    r6 = O.loss_and_grads(t[:, perm], h, W[perm], om, 0.8)
    np.testing.assert_allclose(r6["gW"], r["gW"][perm], rtol=1e-10, atol=1e-15)
    np.testing.assert_allclose(r6["gh"], r["gh"], rtol=1e-10, atol=1e-15)
    np.testing.assert_allclose(r6["loss"], r["loss"], rtol=1e-13)


def test_lambda_inert_at_one_step():
    """at q = q_t (z_ref = z) the regulariser changes nothing."""
    t, h, W, om = _small(12, 3, 13, 4)
    a = O.loss_and_grads(t, h, W, om, 1.0, 0.0)
    b = O.loss_and_grads(t, h, W, om, 1.0, 5.0, z_ref=None)
    c = O.loss_and_grads(t, h, W, om, 1.0, 5.0, z_ref=h @ W.T)
    for k in ("loss", "dl", "gW", "gh"):
        np.testing.assert_array_equal(np.asarray(a[k]), np.asarray(b[k]))
        np.testing.assert_array_equal(np.asarray(a[k]), np.asarray(c[k]))


def test_minus_inf_teacher_entries():
    t, h, W, om = _small(13, 2, 9, 3)
    t[:, [1, 4]] = -np.inf
    r = O.loss_and_grads(t, h, W, om)
    keep = [0, 2, 3, 5, 6, 7, 8]
    z = h @ W.T
    p = np.exp(t[:, keep]) / np.exp(t[:, keep]).sum(1, keepdims=True)
    lq = z - np.log(np.exp(z).sum(1, keepdims=True))
    kl = (p * (np.log(p) - lq[:, keep])).sum(1)
    np.testing.assert_allclose(r["kl_rows"], kl, rtol=1e-12)
    assert np.isfinite(r["gW"]).all()


# ---------------------------------------------------------------- 5. library routines
def test_reduces_to_torch_kl_div_autograd():
    T, V, d = 5, 37, 6
    t, h, W, _ = _small(14, T, V, d)
    ht = torch.tensor(h, dtype=torch.float64, requires_grad=True)
    Wt = torch.tensor(W, dtype=torch.float64, requires_grad=True)
    z = ht @ Wt.T
    loss = torch.nn.functional.kl_div(torch.log_softmax(z, -1), torch.softmax(torch.tensor(t), -1), reduction="sum")
    loss.backward()
    r = O.loss_and_grads(t, h, W, np.ones(T))
    assert r["loss"] == pytest.approx(loss.item(), rel=1e-12)
    np.testing.assert_allclose(r["gW"], Wt.grad.numpy(), rtol=1e-10, atol=1e-15)
    np.testing.assert_allclose(r["gh"], ht.grad.numpy(), rtol=1e-10, atol=1e-15)


def test_weighted_loss_matches_torch_autograd():
    T, V, d = 4, 19, 5
    t, h, W, om = _small(15, T, V, d)
    ht = torch.tensor(h, requires_grad=True)
    Wt = torch.tensor(W, requires_grad=True)
    z = ht @ Wt.T
    kl = torch.nn.functional.kl_div(torch.log_softmax(z, -1), torch.softmax(torch.tensor(t), -1), reduction="none").sum(-1)
    loss = 0.25 * (torch.tensor(om) * kl).sum()
    loss.backward()
    r = O.loss_and_grads(t, h, W, om, 0.25)
    assert r["loss"] == pytest.approx(loss.item(), rel=1e-12)
    np.testing.assert_allclose(r["gW"], Wt.grad.numpy(), rtol=1e-10, atol=1e-15)


@pytest.mark.parametrize("wd", [0.0, 0.05])
def test_adamw_matches_torch_optim(wd):
    r = _rng(16)
    M = r.standard_normal((7, 5))
    Mt = torch.tensor(M, dtype=torch.float64, requires_grad=True)
    opt = torch.optim.AdamW([Mt], lr=3e-3, betas=(0.9, 0.999), eps=1e-8, weight_decay=wd)
    m = np.zeros_like(M)
    v = np.zeros_like(M)
    Mo = M.copy()
    for step in range(1, 5):
        g = r.standard_normal((7, 5)) * 10.0 ** r.integers(-6, 0)
        Mt.grad = torch.tensor(g)
        opt.step()
        Mo, m, v = O.adamw_update(Mo, m, v, g, step, 3e-3, 0.9, 0.999, 1e-8, wd)
        np.testing.assert_allclose(Mo, Mt.detach().numpy(), rtol=1e-12, atol=1e-15)
    st = opt.state[Mt]
    np.testing.assert_allclose(m, st["exp_avg"].numpy(), rtol=1e-12)
    np.testing.assert_allclose(v, st["exp_avg_sq"].numpy(), rtol=1e-12)


def test_sgd_matches_torch_optim():
    r = _rng(17)
    M = r.standard_normal((4, 3))
    g = r.standard_normal((4, 3))
    Mt = torch.tensor(M, requires_grad=True)
    opt = torch.optim.SGD([Mt], lr=1e-3)
    Mt.grad = torch.tensor(g)
    opt.step()
    np.testing.assert_allclose(O.sgd_update(M, g, 1e-3), Mt.detach().numpy(), rtol=1e-15)


def test_inner_steps_match_torch_autograd_adamw_loop():
    """K steps with the lambda term against an fp64 torch loop: autograd on
    sum_r w_r [KL(p||q) + lam KL(q_t||q)] + torch.optim.AdamW (the paper's own implementation is standard
    PyTorch kernels).  fp32 parameters (no master) so no rounding sits between steps."""
    T, V, d, K, lam = 4, 23, 6, 3, 0.7
    t, h, W, om = _small(21, T, V, d)
    W32, h32 = W.astype(np.float32), h.astype(np.float32)
    Wt = torch.tensor(W32.astype(np.float64), requires_grad=True)
    ht = torch.tensor(h32.astype(np.float64))
    tt, omt = torch.tensor(t), torch.tensor(om)
    opt = torch.optim.AdamW([Wt], lr=2e-3, betas=(0.9, 0.999), eps=1e-8, weight_decay=0.01)
    with torch.no_grad():
        q_t = torch.softmax(ht @ Wt.T, -1)
    losses = []
    for k in range(K):
        opt.zero_grad()
        logq = torch.log_softmax(ht @ Wt.T, -1)
        kl = torch.nn.functional.kl_div(logq, torch.softmax(tt, -1), reduction="none").sum(-1)
        reg = torch.nn.functional.kl_div(logq, q_t, reduction="none").sum(-1)
        loss = 0.5 * (omt * (kl + lam * reg)).sum()
        loss.backward()
        opt.step()
        losses.append(loss.item())
    r = O.distill_inner_steps(t, h32, W32, None, np.zeros((V, d)), np.zeros((V, d)), om, None, K=K, lam=lam,
                              seg_len=T, loss_scale=0.5, optimizer="adamw", lr=2e-3, weight_decay=0.01)
    np.testing.assert_allclose(r["losses"], losses, rtol=1e-6)   # W_out is fp32-rounded between steps, torch is not
    # W_out is fp32-rounded every step (the parameters ARE fp32 here): agreement to fp32 rounding of three steps
    np.testing.assert_allclose(r["W_out"], Wt.detach().numpy(), rtol=0, atol=3e-7)
    assert r["losses"][1] < r["losses"][0]            # the same signal again: the loss falls


def test_given_draft_logits_replace_the_product():
    """draft_logits given: identical to the computed path when they ARE h W^T; otherwise gW, gh
    follow dl of the given logits (pinned through the chain rule: gW = dl^T h with dl from softmax(z_given))."""
    T, V, d = 3, 11, 4
    t, h, W, om = _small(22, T, V, d)
    a = O.loss_and_grads(t, h, W, om)
    b = O.loss_and_grads(t, h, W, om, z=h @ W.T)
    for k in ("loss", "gW", "gh", "dl"):
        np.testing.assert_allclose(b[k], a[k], rtol=1e-13, atol=1e-16)
    zg = h @ W.T + 0.1 * _rng(5).standard_normal((T, V))
    c = O.loss_and_grads(t, h, W, om, z=zg)
    q = np.exp(zg - zg.max(1, keepdims=True)); q /= q.sum(1, keepdims=True)
    p = np.exp(t - t.max(1, keepdims=True)); p /= p.sum(1, keepdims=True)
    np.testing.assert_allclose(c["dl"], om[:, None] * (q - p), rtol=1e-12, atol=1e-15)
    np.testing.assert_allclose(c["gW"], (om[:, None] * (q - p)).T @ h, rtol=1e-12, atol=1e-15)
    assert c["loss"] == pytest.approx(float((om * (p * (np.log(p) - np.log(q))).sum(1)).sum()), rel=1e-12)


def test_bf16_rounding_matches_torch():
    r = _rng(18)
    x = np.concatenate([r.standard_normal(20000).astype(np.float32) * 10.0 ** r.integers(-8, 4),
                        np.array([0.0, -0.0, 1.0, 1.00390625, 1.01171875, 3.3895314e38, 1e-40, np.inf, -np.inf],
                                 dtype=np.float32)])
    # exact ties: odd/even mantissa with the low half = 0x8000
    ties = (np.array([0x3F808000, 0x3F818000, 0xBF808000, 0x00008000, 0x00018000], dtype=np.uint32)).view(np.float32)
    x = np.concatenate([x, ties]).astype(np.float32)
    ref = torch.tensor(x).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    np.testing.assert_array_equal(O.f32_to_bf16_bits(x), ref)
    np.testing.assert_array_equal(O.bf16_bits_to_f64(ref), torch.tensor(x).to(torch.bfloat16).double().numpy())


# ---------------------------------------------------------------- 6. statistical sanity
def test_expected_kl_near_half_sigma_squared():
    r = _rng(19)
    V = 20000
    z = 1.28 * r.standard_normal((4, V))
    for sigma in (0.5, 1.0):
        t = z + sigma * r.standard_normal((4, V))
        kl = O.kl_rows_from_logits(t, z)
        assert np.all(np.abs(kl / (sigma ** 2 / 2) - 1) < 0.1)


# ---------------------------------------------------------------- 7. mask
def _mask_ref(t, tok, C):
    T = len(tok)
    mask, tau = [0] * T, [0] * (T // C)
    am = []
    for r in range(T):
        best, bi = -math.inf, 0
        first = True
        for v, x in enumerate(t[r]):
            if first or x > best:
                best, bi, first = x, v, False
        am.append(bi)
    for s in range(T // C):
        for k in range(C):
            if am[s * C + k] != tok[s * C + k]:
                break
            mask[s * C + k] = 1
            tau[s] += 1
    return mask, tau, am


def test_accept_mask_against_python_reference_and_properties():
    from workloads import synth
    for dtype in (synth.F32, synth.BF16):
        t, tok, exp_tau = synth.planted_mask_cases(257, 8, seed=3, dtype=dtype)
        mask, tau, am = O.accept_mask(t, tok, 8)
        tw = O.widen(t)
        m2, tau2, am2 = _mask_ref(tw.tolist(), tok.tolist(), 8)
        np.testing.assert_array_equal(mask, m2)
        np.testing.assert_array_equal(tau, tau2)
        np.testing.assert_array_equal(am, am2)
        np.testing.assert_array_equal(tau, exp_tau)
        for s in range(len(tau)):
            seg = mask[s * 8:(s + 1) * 8]
            assert np.all(np.diff(seg.astype(int)) <= 0)          # a prefix
            assert seg.sum() == tau[s]                            # tau = popcount
            assert np.all(am[s * 8:(s + 1) * 8][seg == 1] == tok[s * 8:(s + 1) * 8][seg == 1])
            if tau[s] < 8:
                assert am[s * 8 + tau[s]] != tok[s * 8 + tau[s]]  # first 0 at the first mismatch


def test_stochastic_acceptance_preserves_the_target_distribution():
    """The defining property of speculative rejection sampling: with x ~ q, accept w.p. min{1, p/q}, else resample
    from norm(max(0, p - q)), the emitted token is distributed exactly as p.  Evaluated through the oracle on a fine
    midpoint grid of both uniforms (resolution 1/n), summed over x with weight q(x)."""
    r = _rng(31)
    V, n = 6, 150
    t = r.standard_normal((1, V)) * 1.5
    z = r.standard_normal((1, V)) * 1.5
    p = np.exp(t[0] - t[0].max()); p /= p.sum()
    q = np.exp(z[0] - z[0].max()); q /= q.sum()
    grid = (np.arange(n) + 0.5) / n
    out = np.zeros(V)
    for x in range(V):
        uu, vv = np.meshgrid(grid, grid, indexing="ij")
        N = n * n
        res = O.accept_stochastic(np.repeat(t, N, 0), np.repeat(z, N, 0), np.full(N, x), uu.ravel(), vv.ravel(), 1)
        emitted = np.where(res["mask"] == 1, x, res["next_token"])
        assert (emitted >= 0).all()
        out += q[x] * np.bincount(emitted, minlength=V) / N
    np.testing.assert_allclose(out, p, atol=2.5 / n)
    # and the accept probability itself: sum_x q min(1, p/q) = sum_x min(p, q)
    assert res["ratio"][0] == pytest.approx(p[V - 1] / q[V - 1], rel=1e-12)


def test_stochastic_acceptance_loop_and_diagnostics():
    r = _rng(32)
    C, S, V = 4, 3, 17
    t = r.standard_normal((C * S, V)) * 2.0
    z = r.standard_normal((C * S, V))
    t[5, 3] = -np.inf
    tok = r.integers(0, V, size=C * S)
    u = r.uniform(size=C * S)
    u[0:C] = 0.0                       # sequence 0: u = 0 accepts everything (ratio > 0)
    u2 = r.uniform(size=S)
    res = O.accept_stochastic(t, z, tok, u, u2, C)
    p = torch.softmax(torch.tensor(t), -1).numpy()
    q = torch.softmax(torch.tensor(z), -1).numpy()
    assert res["tau"][0] == C and res["next_token"][0] == -1
    for s in range(S):                 # pure-Python restatement of the loop
        n = 0
        for k in range(C):
            rr = s * C + k
            if u[rr] <= min(1.0, p[rr, tok[rr]] / q[rr, tok[rr]]):
                n += 1
            else:
                break
        assert res["tau"][s] == n
        np.testing.assert_array_equal(res["mask"][s * C:(s + 1) * C], [1] * n + [0] * (C - n))
        if n < C:
            rr = s * C + n
            nt = res["next_token"][s]
            assert p[rr, nt] > q[rr, nt]                       # inside the residual's support
            resid = np.maximum(0, p[rr] - q[rr])
            assert resid[:nt].sum() < u2[s] * resid.sum() <= resid[:nt + 1].sum() + 1e-15
    import scipy.stats
    for rr in range(C * S):
        assert res["diag"][rr, 0] == pytest.approx(scipy.stats.entropy(p[rr]), rel=1e-10)
        assert res["diag"][rr, 1] == pytest.approx(-math.log(q[rr, int(np.argmax(p[rr]))]), rel=1e-10)
        assert res["diag"][rr, 2] == pytest.approx(p[rr, tok[rr]], rel=1e-10)
        assert res["diag"][rr, 3] == pytest.approx(q[rr, tok[rr]], rel=1e-10)
    # p == q: ratio 1, everything accepted for any u < 1
    res = O.accept_stochastic(z, z, tok, np.full(C * S, 0.999999), u2, C)
    assert (res["tau"] == C).all()


def test_row_weights_modes():
    w = np.array([1.0, 0.9, 0.8, 0.7] * 2)
    mask = np.array([1, 1, 0, 0, 0, 0, 0, 0], dtype=np.uint8)
    np.testing.assert_array_equal(O.row_weights(w, mask, O.ROWS_ALL, 4), w)
    np.testing.assert_array_equal(O.row_weights(w, mask, O.ROWS_ACCEPTED, 4), [1, .9, 0, 0, 0, 0, 0, 0])
    np.testing.assert_array_equal(O.row_weights(w, mask, O.ROWS_ACCEPTED_PLUS_ONE, 4), [1, .9, .8, 0, 1.0, 0, 0, 0])
    full = np.ones(4, dtype=np.uint8)
    np.testing.assert_array_equal(O.row_weights(w[:4], full, O.ROWS_ACCEPTED_PLUS_ONE, 4), w[:4])


# ---------------------------------------------------------------- 8. whole step / slab pieces
def test_step_pieces_agree_with_dense_step():
    from workloads import synth
    c = synth.make_case(3, V=640, d=64, nonzero_state=True, step=3)
    mask, tau, _ = O.accept_mask(c["teacher"], c["draft_tokens"], c["seg_len"])
    np.testing.assert_array_equal(tau, c["tau_star"])
    kw = dict(lr=1e-3, beta1=0.9, beta2=0.999, eps=1e-8, weight_decay=0.01, step=3)
    full = O.distill_step(c["teacher"], c["h"], c["W"], c["master"], c["m"], c["v"], c["pos_weight"], mask,
                          seg_len=c["seg_len"], mask_mode=O.ROWS_ACCEPTED_PLUS_ONE, optimizer="adamw", **kw)
    z, lse_t, lse_z, kl = O.row_normalisers(c["teacher"], c["h"], c["W"], slab=100)
    np.testing.assert_allclose(kl, full["kl_rows"], rtol=1e-12)
    rows = np.array([0, 5, 127, 128, 300, 639])
    part = O.distill_step_rows(rows, z, lse_t, lse_z, c["teacher"], c["h"], c["W"][rows], c["master"][rows],
                               c["m"][rows], c["v"][rows], full["omega"], optimizer="adamw", **kw)
    np.testing.assert_allclose(part["gW"], full["gW"][rows], rtol=1e-12, atol=1e-18)
    np.testing.assert_allclose(part["master"], full["master"][rows], rtol=1e-14)
    gh = O.gh_full(z, lse_t, lse_z, c["teacher"], c["W"], full["omega"], slab=77)
    np.testing.assert_allclose(gh, full["gh"], rtol=1e-10, atol=1e-16)
    # the working copy is rn_bf16(rn_fp32(master))
    ref = torch.tensor(full["master"]).float().to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    np.testing.assert_array_equal(full["W_out"], ref)


def test_golden_config1_regression():
    """tests/golden/config1_tiny.txt was written by tests/golden/make_golden.py,
    which calls only oracle/ and the input recipe."""
    import os
    from workloads import synth
    path = os.path.join(os.path.dirname(__file__), "golden", "config1_tiny.txt")
    vals = {}
    for line in open(path):
        if line.startswith("#") or not line.strip():
            continue
        k, v = line.split("=", 1)
        vals[k.strip()] = v.strip()
    c = synth.make_case(1)
    mask, tau, _ = O.accept_mask(c["teacher"], c["draft_tokens"], c["seg_len"])
    r = O.distill_step(c["teacher"], c["h"], c["W"], None, None, None, c["pos_weight"], mask,
                       seg_len=c["seg_len"], optimizer="sgd", lr=c["cfg"]["lr"])
    assert r["loss"] == pytest.approx(float(vals["loss"]), rel=1e-12)
    np.testing.assert_allclose(r["kl_rows"], [float(x) for x in vals["kl_rows"].split()], rtol=1e-12)
    assert int(vals["tau"]) == int(tau[0])
    assert float(np.abs(r["gW"]).max()) == pytest.approx(float(vals["gW_absmax"]), rel=1e-12)
    assert float(np.abs(r["gh"]).max()) == pytest.approx(float(vals["gh_absmax"]), rel=1e-12)


def test_shard_tuples_merge_to_the_whole_row_normalisers():
    """the per-slice tuples (m_t, s_t, a, m_z, s_z), merged, give the plain logsumexp of the whole teacher
    and draft rows and the plain KL -- for uneven slices, -inf teacher entries and a slice that is all -inf."""
    rng = np.random.Generator(np.random.PCG64(21))
    T, V = 5, 97
    t = 3.0 * rng.standard_normal((T, V))
    z = 2.0 * rng.standard_normal((T, V))
    t[:, 7::11] = -np.inf
    t[2, 40:70] = -np.inf                          # row 2: the middle slice has no finite teacher entry
    want_t, want_z, want_kl = O.logsumexp_rows(t), O.logsumexp_rows(z), O.kl_rows_from_logits(t, z)
    for cuts in ([0, V], [0, 40, 70, V], [0, 1, 2, 50, V]):
        st = np.stack([O.shard_row_stats(t[:, a:b], z[:, a:b]) for a, b in zip(cuts[:-1], cuts[1:])])
        lse_t, lse_z, kl = O.merge_shard_stats(st)
        np.testing.assert_allclose(lse_t, want_t, rtol=1e-13)
        np.testing.assert_allclose(lse_z, want_z, rtol=1e-13)
        np.testing.assert_allclose(kl, want_kl, rtol=1e-11, atol=1e-13)
    # brute force on one row, literal definitions
    r = 1
    p = np.exp(t[r]) / np.exp(t[r]).sum()
    q = np.exp(z[r]) / np.exp(z[r]).sum()
    kl_lit = sum(p[v] * (np.log(p[v]) - np.log(q[v])) for v in range(V) if p[v] > 0)
    assert abs(kl[r] - kl_lit) < 1e-12


# ----------------------------------------------------------------------------
# f4: Adam with bf16 moment storage (R26).  Pins of adamw_update_lowp / sr_bits16 / f32_to_bf16_bits_sr
# ----------------------------------------------------------------------------

def _bf16_bits_py(x):
    """fp32 -> (bits of the bf16 at or below |x|, the 16 discarded bits), through struct: independent of numpy views."""
    import struct
    u = struct.unpack("<I", struct.pack("<f", x))[0]
    return u >> 16, u & 0xFFFF


def _bf16_val_py(b):
    import struct
    return struct.unpack("<f", struct.pack("<I", (b & 0xFFFF) << 16))[0]


def test_stochastic_rounding_is_exactly_unbiased_over_all_16_bit_draws():
    """E_r[sr(x, r)] = x EXACTLY when r runs over all 65536 values: the discarded fraction f rounds up for exactly f of
    them.  Also: every result is one of the two bf16 neighbours of x, and r = 0 truncates."""
    rs = np.arange(65536, dtype=np.uint32)
    for x in (1.2345678, 3.0e-11, 0.999, 65504.0, -0.3333333, 1.0, 7.0e-39):
        x32 = np.float32(x)
        q = O.f32_to_bf16_bits_sr(np.full(65536, x32, dtype=np.float32), rs)
        vals = O.bf16_bits_to_f64(q)
        lo_bits, f = _bf16_bits_py(float(x32))
        lo, hi = _bf16_val_py(lo_bits), _bf16_val_py(lo_bits + 1)
        assert set(np.unique(q).tolist()) <= {lo_bits, lo_bits + 1}
        assert int((q == lo_bits + 1).sum()) == f                     # rounds away from zero for exactly f draws
        assert q[0] == lo_bits
        assert vals.mean() == pytest.approx(float(x32), rel=1e-15, abs=0.0) or f == 0
        # mean = lo + (hi - lo) f / 65536 = x, term by term
        assert lo + (hi - lo) * f / 65536.0 == pytest.approx(float(x32), rel=1e-15)


def test_sr_bits_are_uniform_and_decorrelated():
    """The counter-based generator has no paper value to hit; what the method needs from it is uniform 16-bit draws that
    are independent across elements, steps and seeds."""
    n, d = 1 << 20, 1024
    idx = np.arange(n, dtype=np.uint64)
    a = O.sr_bits16(idx, 1, 0, d).astype(np.float64)
    assert a.min() >= 0 and a.max() <= 65535
    assert abs(a.mean() - 32767.5) < 4 * 18918.0 / np.sqrt(n)        # sd of U{0..65535} = 18918
    counts = np.bincount((a.astype(np.int64) >> 8), minlength=256)    # chi-square over the top byte
    chi2 = ((counts - n / 256.0) ** 2 / (n / 256.0)).sum()
    assert chi2 < 255 + 6 * np.sqrt(2 * 255)
    for bit in range(16):                                             # every bit is fair
        assert abs(((a.astype(np.int64) >> bit) & 1).mean() - 0.5) < 4 * 0.5 / np.sqrt(n)
    b = O.sr_bits16(idx, 2, 0, d).astype(np.float64)                  # next step, same elements
    c = O.sr_bits16(idx, 1, 1, d).astype(np.float64)                  # another seed
    e1 = O.sr_bits16(idx + np.uint64(1), 1, 0, d).astype(np.float64)  # neighbours along the row
    e2 = O.sr_bits16(idx + np.uint64(d), 1, 0, d).astype(np.float64)  # neighbours along the column: rows 2k and 2k + 1
    #                                                                 # share ONE hash and take different halves of it
    e3 = O.sr_bits16(idx + np.uint64(2 * d), 1, 0, d).astype(np.float64)   # the next pair of rows
    e4 = O.sr_bits16(idx + np.uint64(1 << 33), 1, 0, d).astype(np.float64)  # beyond 2^32 pairs: the high word counts
    for other in (b, c, e1, e2, e3, e4):
        assert abs(np.corrcoef(a, other)[0, 1]) < 5.0 / np.sqrt(n)
        assert (a == other).mean() < 4.0 / 65536
    # the definition, written out once more with Python integers on a few elements (a transposed v / j or a swapped
    # half fails here)
    def mix(x):
        x ^= x >> 16; x = (x * 0x7FEB352D) & 0xFFFFFFFF; x ^= x >> 15; x = (x * 0x846CA68B) & 0xFFFFFFFF; x ^= x >> 16
        return x
    for v, j, dd, step, seed in ((0, 0, 8, 1, 0), (1, 0, 8, 1, 0), (6, 5, 8, 3, 7), (7, 5, 8, 3, 7), (2 ** 31 + 1, 77, 4096, 9, 12345)):
        pidx = (v >> 1) * dd + j
        x = mix((pidx & 0xFFFFFFFF) ^ ((step * 0x9E3779B9) & 0xFFFFFFFF) ^ ((seed * 0x85EBCA6B) & 0xFFFFFFFF)
                ^ (((pidx >> 32) * 0xC2B2AE35) & 0xFFFFFFFF))
        want = (x & 0xFFFF) if (v & 1) else (x >> 16)
        assert int(O.sr_bits16(np.array([v * dd + j], dtype=np.uint64), step, seed, dd)[0]) == want


def test_lowp_adam_matches_a_scalar_loop_in_the_stated_order():
    """dequantise -> update with the unrounded moments -> requantise (m nearest-even, v stochastic), element by element
    in plain Python floats with struct-based bf16 conversions."""
    rng = np.random.Generator(np.random.PCG64(31))
    V, d = 7, 5
    M = rng.standard_normal((V, d)) * 0.02
    g = rng.standard_normal((V, d)) * 1e-3
    m_bits = O.f32_to_bf16_bits((rng.standard_normal((V, d)) * 1e-4).astype(np.float32))
    v_bits = O.f32_to_bf16_bits((rng.standard_normal((V, d)) ** 2 * 1e-8).astype(np.float32))
    idx = np.arange(V, dtype=np.uint64)[:, None] * np.uint64(d) + np.arange(d, dtype=np.uint64)[None, :]
    lr, b1, b2, eps, wd, n, seed = 1e-3, 0.9, 0.999, 1e-8, 0.01, 4, 9
    Mn, mq, vq, m_new, v_new = O.adamw_update_lowp(M, m_bits, v_bits, g, n, lr, b1, b2, eps, wd, idx=idx, seed=seed, d=d)
    bits = O.sr_bits16(idx, n, seed, d)
    for i in range(V):
        for j in range(d):
            m0, v0 = _bf16_val_py(int(m_bits[i, j])), _bf16_val_py(int(v_bits[i, j]))
            Mw = M[i, j] * (1.0 - lr * wd)
            m1 = b1 * m0 + (1.0 - b1) * g[i, j]
            v1 = b2 * v0 + (1.0 - b2) * g[i, j] * g[i, j]
            want = Mw - lr * (m1 / (1.0 - b1 ** n)) / ((v1 / (1.0 - b2 ** n)) ** 0.5 + eps)
            assert Mn[i, j] == pytest.approx(want, rel=1e-13)
            assert m_new[i, j] == pytest.approx(m1, rel=1e-14) and v_new[i, j] == pytest.approx(v1, rel=1e-14)
            # m: nearest even on the fp32 value
            lo_b, f = _bf16_bits_py(float(np.float32(m1)))
            up = f > 0x8000 or (f == 0x8000 and (lo_b & 1))
            assert int(mq[i, j]) == lo_b + (1 if up else 0)
            # v: up iff the discarded bits plus the element's draw carry
            lo_b, f = _bf16_bits_py(float(np.float32(v1)))
            assert int(vq[i, j]) == lo_b + (1 if f + int(bits[i, j]) >= 65536 else 0)


def test_lowp_v_decays_in_expectation_where_nearest_rounding_freezes():
    """Why v is rounded stochastically: with zero gradients v must decay as beta2^n.  Nearest rounding leaves a bf16 v
    unchanged for ever (0.1% per step is below half an ulp); the stochastic rule follows beta2^n in the mean."""
    nel, steps, b2 = 20000, 200, 0.999
    idx = np.arange(nel, dtype=np.uint64)[None, :]
    v0 = np.full((1, nel), 1.0e-6, dtype=np.float32)
    v_bits = O.f32_to_bf16_bits(v0)
    v_rne = v_bits.copy()
    m_bits = np.zeros((1, nel), dtype=np.uint16)
    M = np.zeros((1, nel))
    g = np.zeros((1, nel))
    start = O.bf16_bits_to_f64(v_bits).mean()
    for n in range(1, steps + 1):
        _, m_bits, v_bits, _, _ = O.adamw_update_lowp(M, m_bits, v_bits, g, n, 1e-5, 0.9, b2, 1e-8, 0.0, idx=idx, seed=3, d=nel)
        v_rne = O.f32_to_bf16_bits((b2 * O.bf16_bits_to_f64(v_rne)).astype(np.float32))
    got = O.bf16_bits_to_f64(v_bits).mean() / start
    assert got == pytest.approx(b2 ** steps, rel=5e-3)               # 0.8186
    assert O.bf16_bits_to_f64(v_rne).mean() / start == 1.0            # frozen


def test_lowp_step_uses_unrounded_moments_for_the_parameter_update():
    from workloads import synth
    c = synth.make_case(3, V=384, d=64, nonzero_state="mix", step=5)
    mask, _, _ = O.accept_mask(c["teacher"], c["draft_tokens"], c["seg_len"])
    mb, vb = O.f32_to_bf16_bits(c["m"]), O.f32_to_bf16_bits(c["v"])
    kw = dict(seg_len=c["seg_len"], lr=1e-5, step=5)
    lo = O.distill_step(c["teacher"], c["h"], c["W"], c["master"], mb, vb, c["pos_weight"], mask, moments="bf16",
                        sr_seed=1, **kw)
    hi = O.distill_step(c["teacher"], c["h"], c["W"], c["master"], O.bf16_bits_to_f64(mb), O.bf16_bits_to_f64(vb),
                        c["pos_weight"], mask, **kw)
    np.testing.assert_array_equal(lo["master"], hi["master"])          # same dequantised moments in, same step out
    np.testing.assert_array_equal(lo["m"], hi["m"])
    # what is stored lies within one bf16 ulp of the unrounded moments (half an ulp for m)
    m_err = np.abs(O.bf16_bits_to_f64(lo["m_bits"]) - lo["m"])
    v_err = np.abs(O.bf16_bits_to_f64(lo["v_bits"]) - lo["v"])
    assert np.all(m_err <= 2.0 ** -8 * np.abs(lo["m"]) + 1e-45)
    assert np.all(v_err <= 2.0 ** -7 * np.abs(lo["v"]) + 1e-45)
    rows = np.array([3, 100, 383])
    z, lse_t, lse_z, _ = O.row_normalisers(c["teacher"], c["h"], c["W"])
    part = O.distill_step_rows(rows, z, lse_t, lse_z, c["teacher"], c["h"], c["W"][rows], c["master"][rows], mb[rows],
                               vb[rows], lo["omega"], lr=1e-5, step=5, moments="bf16", sr_seed=1)
    np.testing.assert_array_equal(part["v_bits"], lo["v_bits"][rows])   # the draws are keyed by the GLOBAL element index
    np.testing.assert_array_equal(part["m_bits"], lo["m_bits"][rows])
