"""Real orbitals (second half; the dense Gamma-point supercell representation
with real orbitals): when h1, L and psi_t are real the half-rotated tensor is real, and force bias, vHS and exchange need two
real products per complex product instead of three.  The library detects exactly-zero imaginary parts in afqmc_create and
switches to the two-product variants of its kernels; walkers, Green's functions and every result stay complex.

Checked here: every call against the oracle (the same oracle functions: real inputs are a special case of the definitions),
and against the library's own complex kernels on the same inputs (option real_orbitals = 0)."""
import numpy as np
import pytest

from oracle import afqmc_oracle as orc
from paper_2003_09468_b200 import synth
from tests.test_gpu_parity import Case, _to_dev, relerr, run_chain_and_compare

pytestmark = pytest.mark.gpu

SHAPES = [
    dict(mesh=(1, 1, 1), m=12, n=5, nchol=19, nw=5),     # Gamma point, two a-groups, ragged everything
    dict(mesh=(1, 1, 1), m=33, n=4, nchol=9, nw=18),     # m > 28, two n-tiles per warp in force bias / vHS
    dict(mesh=(2, 1, 1), m=7, n=3, nchol=10, nw=3),      # real L on a two-point mesh: (Q,-Q) pairs with real blocks
    dict(mesh=(1, 1, 1), m=104, n=10, nchol=6, nw=3),    # theta blocks too large for one CTA: large-block exchange kernel
]


def _flops_flags(ctx, cfg):
    """The two-product kernels report 4 (force bias) real flops per complex multiply-add instead of 6."""
    return ctx.force_bias_flops(1) / (cfg.nk ** 2 * cfg.n * cfg.m * cfg.nchol)


@pytest.mark.parametrize("kw", SHAPES, ids=lambda k: "x".join(map(str, k["mesh"])) + "_m%d_n%d_c%d_w%d" % (k["m"], k["n"], k["nchol"], k["nw"]))
def test_real_orbitals_every_call_against_the_oracle_and_the_complex_kernels(kw):
    case = Case(synth.tiny_config(seed=41, **kw), real_orbitals=True)
    try:
        cfg, ctx, pb = case.cfg, case.ctx, case.pb
        assert np.all(pb.L.imag == 0) and np.all(pb.psi_t.imag == 0) and np.abs(pb.phi.imag).max() > 0
        assert _flops_flags(ctx, cfg) == 4.0                      # detected: the two-product variants run
        e_real = run_chain_and_compare(case)                      # every call, every walker, against the oracle
        # the same inputs through the complex (three-product) kernels
        theta_d, _, _ = ctx.green(_to_dev(pb.phi))
        x_d = _to_dev(pb.x)
        vb_r = ctx.force_bias(theta_d)
        vhs_r = ctx.vhs(x_d, vb_r, cfg.dtau)
        en_r = ctx.local_energy(theta_d)
        ctx.set_option("real_orbitals", 0)
        try:
            assert _flops_flags(ctx, cfg) == 6.0
            vb_c = ctx.force_bias(theta_d)
            vhs_c = ctx.vhs(x_d, vb_c, cfg.dtau)
            en_c = ctx.local_energy(theta_d)
            e_cplx = run_chain_and_compare(case)
        finally:
            ctx.set_option("real_orbitals", 1)
        assert relerr(vb_r.cpu().numpy(), vb_c.cpu().numpy()) < 1e-13
        assert relerr(vhs_r.cpu().numpy(), vhs_c.cpu().numpy()) < 1e-12
        assert np.max(np.abs(en_r.cpu().numpy() - en_c.cpu().numpy()) / np.abs(en_c.cpu().numpy())) < 1e-12
        assert np.max(np.abs(e_real - e_cplx) / np.abs(e_cplx)) < 1e-11
    finally:
        case.close()


def test_complex_inputs_are_not_mistaken_for_real():
    case = Case(synth.tiny_config(seed=41, mesh=(1, 1, 1), m=12, n=5, nchol=19, nw=2))
    try:
        assert _flops_flags(case.ctx, case.cfg) == 6.0
    finally:
        case.close()


def test_gamma_point_supercell_real_orbitals_full_size():
    """Synth config G1 (one k-point, m = 208, n = 32, nchol = 1040, 16 walkers) with real orbitals, every call and every
    walker against the oracle (as the complex G1 test: the 4M cross-check kernel cannot hold these theta blocks)."""
    case = Case(synth.CONFIGS["G1"], real_orbitals=True)
    try:
        assert _flops_flags(case.ctx, case.cfg) == 4.0
        run_chain_and_compare(case)
    finally:
        case.close()
