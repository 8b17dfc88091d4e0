"""Run-to-run reproducibility: the library uses no atomics and fixed summation orders, so repeated calls on the same inputs must
agree BIT FOR BIT.  This is also the cheapest detector of a data race inside a kernel (a ring stage refilled before it was read
showed up exactly like this: whole warp slices of vHS changed from call to call)."""
import numpy as np
import pytest
import torch

from paper_2003_09468_b200 import synth

pytestmark = pytest.mark.gpu

CASES = [
    ("C1", dict(), 0),
    ("C2", dict(), 0),
    ("C3", dict(), 0),
    ("G1", dict(real_orbitals=True), 0),
    ("G1", dict(), 0),
    ("C2", dict(), 1),                     # precision = 1: complex64 storage + tcgen05 exchange
]


@pytest.mark.parametrize("name,kw,prec", CASES, ids=["C1", "C2", "C3", "G1_real", "G1", "C2_complex64"])
def test_step_is_bitwise_reproducible(name, kw, prec):
    from paper_2003_09468_b200 import binding
    cfg = synth.CONFIGS[name]
    pb = synth.make_problem(cfg, **kw)
    ctx = binding.from_problem(pb, precision=prec)
    try:
        cd = torch.complex64 if prec else torch.complex128
        phi0 = torch.from_numpy(pb.phi).cuda().to(cd)
        x = torch.from_numpy(pb.x).cuda().to(torch.float32 if prec else torch.float64)
        ref = None
        for rep in range(6):
            phi = phi0.clone()
            e, ld, info = ctx.step(phi, x, cfg.dtau, cfg.order)
            theta, _, _ = ctx.green(phi)
            vb = ctx.force_bias(theta)
            vhs = ctx.vhs(x, vb, cfg.dtau)
            out = [t.clone() for t in (phi, e, ld, theta, vb, vhs)]
            if ref is None:
                ref = out
            else:
                for a, b, what in zip(out, ref, ("phi", "energy", "logdet", "theta", "vbias", "vhs")):
                    assert torch.equal(a, b), (name, what, rep)
            del vhs
    finally:
        ctx.close()


def test_mixed_precision_exchange_is_bitwise_reproducible():
    from paper_2003_09468_b200 import binding
    cfg = synth.CONFIGS["C2"]
    pb = synth.make_problem(cfg)
    ctx = binding.from_problem(pb)
    try:
        theta, _, _ = ctx.green(torch.from_numpy(pb.phi).cuda())
        for mode in (1, 2):
            for tc in (1, 0):
                ctx.set_option("exchange_precision", mode)
                ctx.set_option("exchange_tc", tc)
                ref = ctx.local_energy(theta).clone()
                for _ in range(5):
                    assert torch.equal(ctx.local_energy(theta), ref), (mode, tc)
        ctx.set_option("exchange_precision", 0)
        ctx.set_option("exchange_tc", 1)
    finally:
        ctx.close()
