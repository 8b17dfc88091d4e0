"""afqmc_local_energy against the oracle for every k-step shape of the register-B exchange kernel (m = 1 ... 28 bands per
k-point: no full k-step at all, a real-embedded tail with and without full k-steps, no tail), so that each instantiation of
the phased accumulation (commit groups of the operand ring in the order of use, negated third B side, tail parts added
directly) is compared element by element.  Tolerance: 1e-10 relative per energy component (north_star)."""
import numpy as np
import pytest
import torch

from oracle import afqmc_oracle as orc
from paper_2003_09468_b200 import synth

pytestmark = pytest.mark.gpu

SHAPES = [(1, 1, 3, (2, 1, 1), 3), (2, 1, 5, (2, 2, 1), 5), (2, 2, 4, (3, 1, 1), 2), (3, 2, 4, (2, 1, 2), 4),
          (4, 4, 5, (2, 1, 1), 4), (5, 3, 7, (2, 1, 1), 6), (6, 4, 9, (1, 3, 1), 7), (9, 4, 6, (2, 1, 1), 9),
          (10, 3, 5, (1, 1, 2), 5), (13, 4, 8, (2, 1, 1), 3), (17, 2, 4, (1, 1, 2), 4), (22, 4, 5, (2, 1, 1), 5),
          (28, 4, 6, (1, 2, 1), 5)]


@pytest.mark.parametrize("m,n,nchol,mesh,nw", SHAPES)
def test_local_energy_for_every_kstep_shape(m, n, nchol, mesh, nw):
    from paper_2003_09468_b200 import binding
    cfg = synth.tiny_config(mesh=mesh, m=m, n=n, nchol=nchol, nw=nw, seed=31 + m)
    pb = synth.make_problem(cfg)
    ctx = binding.from_problem(pb)
    try:
        Lh, ht = orc.half_rotate(pb.L, pb.psi_t, pb.h1)
        theta, _, info = ctx.green(torch.from_numpy(pb.phi).cuda())
        assert int(info.abs().sum()) == 0
        e = ctx.local_energy(theta).cpu().numpy()
        th = theta.cpu().numpy()
        for w in range(nw):
            eo = np.array(orc.local_energy(cfg.mesh, Lh, ht, th[w]))
            err = np.abs(e[w] - eo) / np.maximum(np.abs(eo), 1e-300)
            assert float(err.max()) < 1e-10, (w, e[w], eo)
    finally:
        ctx.close()
