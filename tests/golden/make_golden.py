"""Writes tests/golden/config1_tiny.txt: oracle results on BASELINE.json configs[0]
(V=1024, d=64, T=8, fp32, seed 0, one SGD step lr=1e-3).  Calls only oracle/ and
the input recipe (workloads.synth holds no method arithmetic); never
the CUDA path.  The paper prints no worked example for this path, so this is a
regression fixture of the pinned oracle, not a paper value.

    python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import tts_oracle as O  # noqa: E402
from workloads import synth  # noqa: E402

c = synth.make_case(1)
mask, tau, am = O.accept_mask(c["teacher"], c["draft_tokens"], c["seg_len"])
r = O.distill_step(c["teacher"], c["h"], c["W"], None, None, None, c["pos_weight"], mask,
                   seg_len=c["seg_len"], optimizer="sgd", lr=c["cfg"]["lr"])
with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "config1_tiny.txt"), "w") as f:
    f.write("# oracle/tts_oracle.py on BASELINE.json configs[0]; written by tests/golden/make_golden.py\n")
    f.write("# loss = sum_k w_k KL(p_k||q_k), PAPER.md:119-125 (w_k = 1); SGD step PAPER.md:158\n")
    f.write("loss = %.17g\n" % r["loss"])
    f.write("kl_rows = %s\n" % " ".join("%.17g" % x for x in r["kl_rows"]))
    f.write("tau = %d\n" % int(tau[0]))
    f.write("gW_absmax = %.17g\n" % float(np.abs(r["gW"]).max()))
    f.write("gh_absmax = %.17g\n" % float(np.abs(r["gh"]).max()))
