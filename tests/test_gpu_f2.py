"""f2: stochastic acceptance min{1, p/q} with the residual resample and the section-3 diagnostics
 against the oracle.  The accept decision and the inverse-CDF index are integers decided
by floating point: rows whose uniform sits within 1e-4 (relative) of the acceptance ratio, and resample targets within
1e-5 of a CDF step, admit either neighbour; everything else must match exactly."""
import numpy as np
import pytest
import torch

from oracle import tts_oracle as O
from paper_2605_09329_b200 import tts
from workloads import synth

from gpu_util import _dev

pytestmark = pytest.mark.gpu


def _case(V, d, n_seq, seg_len, dtype, seed):
    case = synth.make_case(4, V=V, d=d, n_seq=n_seq, seg_len=seg_len, seed=seed)
    W, h = O.widen(case["W"]), O.widen(case["h"])
    z = (h @ W.T).astype(np.float32)
    rng = np.random.Generator(np.random.PCG64(seed + 1))
    T = case["T"]
    # draft tokens SAMPLED from q (what a stochastic drafter does), so p/q spans both sides of 1
    q = np.exp(z - z.max(1, keepdims=True)); q /= q.sum(1, keepdims=True)
    tok = np.array([rng.choice(V, p=q[r] / q[r].sum()) for r in range(T)], dtype=np.int32)
    t = synth.bf16_bits_to_f32(case["teacher"])
    t[1, 7::5] = -np.inf
    teacher = synth.f32_to_bf16_bits(t) if dtype == synth.BF16 else t
    u = rng.uniform(size=T).astype(np.float32)
    u[:seg_len] = 0.0                                   # sequence 0 accepts its whole canvas
    u2 = rng.uniform(size=n_seq).astype(np.float32)
    return case, teacher, z, tok, u, u2


@pytest.mark.parametrize("V,d,n_seq,seg_len,dtype", [(4096, 64, 6, 8, synth.BF16), (151936, 32, 4, 16, synth.BF16),
                                                      (1000, 32, 5, 4, synth.F32), (8, 8, 3, 1, synth.F32)])
def test_accept_stochastic_matches_oracle(V, d, n_seq, seg_len, dtype):
    case, teacher, z, tok, u, u2 = _case(V, d, n_seq, seg_len, dtype, 40 + V % 97)
    T = case["T"]
    o = O.accept_stochastic(teacher, z, tok, u, u2, seg_len)
    cfg = tts.make_config(V, d, T, seg_len, tts.TTS_BF16, dtype, tts.TTS_ADAMW)
    ctx = tts.tts_ctx_create(cfg, 0)
    try:
        mask = torch.zeros(T, dtype=torch.uint8, device="cuda")
        tau = torch.zeros(n_seq, dtype=torch.int32, device="cuda")
        nxt = torch.full((n_seq,), -7, dtype=torch.int32, device="cuda")
        diag = torch.zeros(T, 4, device="cuda")
        tts.tts_accept_stochastic(ctx, _dev(teacher), _dev(z), _dev(tok), _dev(u), _dev(u2), T, mask, tau, nxt, diag)
        torch.cuda.synchronize()
        assert tts.tts_last_launch_count(ctx) == 4
        g_mask, g_tau, g_nxt, g_diag = mask.cpu().numpy(), tau.cpu().numpy(), nxt.cpu().numpy(), diag.cpu().numpy()
    finally:
        tts.tts_ctx_destroy(ctx)
    # diagnostics
    np.testing.assert_allclose(g_diag[:, 0], o["diag"][:, 0], rtol=1e-3, atol=1e-5)
    np.testing.assert_allclose(g_diag[:, 1], o["diag"][:, 1], rtol=1e-3, atol=1e-5)
    np.testing.assert_allclose(g_diag[:, 2:], o["diag"][:, 2:], rtol=1e-3, atol=1e-12)
    # decisions: unique wherever the uniform is clear of the ratio
    clear = np.abs(u.astype(np.float64) - np.minimum(1.0, o["ratio"])) > 1e-4 * np.maximum(u, 1e-3)
    assert clear.mean() > 0.9
    for s in range(n_seq):
        rows = slice(s * seg_len, (s + 1) * seg_len)
        if clear[rows].all():
            np.testing.assert_array_equal(g_mask[rows], o["mask"][rows])
            assert g_tau[s] == o["tau"][s]
            if o["tau"][s] == seg_len:
                assert g_nxt[s] == -1
            else:
                cdf = o["resid_cdf"][s]
                target = float(u2[s]) * cdf[-1]
                v = int(g_nxt[s])
                assert 0 <= v < V
                lo = cdf[v - 1] if v > 0 else 0.0
                tol = 1e-5 * cdf[-1]
                assert cdf[v] > lo                                   # inside the residual's support (p > q)
                assert lo - tol <= target <= cdf[v] + tol, (s, v, int(o["next_token"][s]))
        # a prefix in any case
        m = g_mask[rows]
        assert (np.diff(m.astype(np.int8)) <= 0).all() and m.sum() == g_tau[s]
    assert g_tau[0] == seg_len and g_nxt[0] == -1


def test_accept_stochastic_equal_distributions_accept_everything():
    V, T = 2048, 16
    rng = np.random.Generator(np.random.PCG64(3))
    z = rng.standard_normal((T, V)).astype(np.float32)
    tok = rng.integers(0, V, size=T).astype(np.int32)
    u = np.full(T, 0.99, dtype=np.float32)
    ctx = tts.tts_ctx_create(tts.make_config(V, 64, T, 16, tts.TTS_BF16, tts.TTS_F32), 0)
    try:
        mask = torch.zeros(T, dtype=torch.uint8, device="cuda")
        tau = torch.zeros(1, dtype=torch.int32, device="cuda")
        nxt = torch.zeros(1, dtype=torch.int32, device="cuda")
        tts.tts_accept_stochastic(ctx, _dev(z), _dev(z), _dev(tok), _dev(u), _dev(np.array([0.5], np.float32)), T, mask,
                                  tau, nxt, None)
        torch.cuda.synchronize()
        assert int(tau[0]) == 16 and int(nxt[0]) == -1 and bool(mask.all())
    finally:
        tts.tts_ctx_destroy(ctx)
