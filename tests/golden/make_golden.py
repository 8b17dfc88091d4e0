"""Writes tests/golden/tiny_step.txt: the oracle's results for one full step on a tiny seeded system.

The paper (arxiv 2003.09468) prints no worked numerical example for this path, so there is no paper
value to store; this fixture is a REGRESSION guard of the oracle itself: it calls only `oracle/` (and the seeded input
generator), and tests/test_oracle_pins.py checks that the oracle still reproduces it, so that a later change of the
oracle's arithmetic cannot go unnoticed (such a change has to regenerate this file and say why in its commit message).

    python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import afqmc_oracle as orc                      # noqa: E402
from paper_2003_09468_b200 import synth                    # noqa: E402

CFG = dict(mesh=(2, 3, 1), m=3, n=2, nchol=4, nw=2, seed=3)


def compute():
    cfg = synth.tiny_config(**CFG)
    pb = synth.make_problem(cfg)
    Lh, ht = orc.half_rotate(pb.L, pb.psi_t, pb.h1)
    phi_new, energy, logdet = orc.step(cfg.mesh, pb.L, Lh, ht, pb.psi_t, pb.phi, pb.x, cfg.dtau, cfg.order)
    rows = []
    for w in range(cfg.nw):
        th, ld0, _ = orc.green(pb.psi_t, pb.phi[w])
        vb = orc.force_bias(cfg.mesh, Lh, th)
        rows.append(("logdet0[%d]" % w, ld0))
        rows.append(("vbias_sum[%d]" % w, complex(np.sum(vb))))
        rows.append(("logdet1[%d]" % w, complex(logdet[w])))
        for c, name in enumerate(("E1", "EC", "EX")):
            rows.append(("%s[%d]" % (name, w), complex(energy[w, c])))
        rows.append(("phi_new_sum[%d]" % w, complex(np.sum(phi_new[w]))))
    return rows


if __name__ == "__main__":
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "tiny_step.txt")
    with open(out, "w") as f:
        f.write("# oracle/afqmc_oracle.py, one step (PAPER.md:87-107, :142-160, :306-319) on synth.tiny_config(%r)\n" % (CFG,))
        f.write("# written by tests/golden/make_golden.py (calls only oracle/ and the seeded generator); name re im\n")
        for name, z in compute():
            f.write("%s %.17g %.17g\n" % (name, z.real, z.imag))
    print("wrote", out)
