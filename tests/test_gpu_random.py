"""Randomised shapes: vocabulary, hidden size, row count, optimiser state and SM budget drawn from a seeded generator,
so that every kernel family (one-canvas fused, wide with and without the gh contraction, CTA-pair logits, the
multicast gh kernel, stream-K walks under a capped grid) meets shapes nobody hand-picked.  Each case is compared with
the fp64 oracle at gpu_util.check_step's tolerances."""
import random

import pytest

from workloads import synth

from gpu_util import check_step, run_gpu, run_oracle

pytestmark = pytest.mark.gpu


def _draw(i):
    rnd = random.Random(1000 + i)
    d = rnd.choice([128, 256, 384, 512, 1024, 2048])
    V = 128 * rnd.randint(2, 24)
    n_seq = rnd.choice([1, 1, 2, 3, 5, 8, 12, 16, 17, 24, 32])
    seg = rnd.choice([8, 16]) if n_seq == 1 else 16
    nz = rnd.random() < 0.4
    mc = rnd.choice([0, 0, 0, 5, 37, 100])
    return d, V, n_seq, seg, nz, mc


@pytest.mark.parametrize("i", range(16))
def test_random_shape_against_oracle(i):
    d, V, n_seq, seg, nz, mc = _draw(i)
    case = synth.make_case(3 if n_seq == 1 else 4, V=V, d=d, n_seq=n_seq, seg_len=seg, seed=500 + i, nonzero_state=nz,
                           step=3 if nz else 1)
    g = run_gpu(case, max_ctas=mc)
    o = run_oracle(case)
    check_step(g, o, case)
    assert g["used_tensor"] == 1
