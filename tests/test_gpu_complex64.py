"""GPU parity of the optional complex64 boundary (afqmc_dims.precision = 1; include/afqmc.h "Precision 1") against the
complex128 CPU oracle: BASELINE.json north_star tolerance 1e-4 relative, same error metric as test_gpu_parity.py.
Every stage is fed the (complex64) GPU output of the previous stage, widened to complex128 for the oracle."""
import numpy as np
import pytest
import torch

from oracle import afqmc_oracle as orc
from paper_2003_09468_b200 import synth

pytestmark = pytest.mark.gpu

TOL = 1e-4


def relerr(a, b):
    a, b = np.asarray(a), np.asarray(b)
    return float(np.max(np.abs(a - b)) / max(float(np.max(np.abs(b))), 1e-300))


def _c64(a):
    return torch.from_numpy(np.ascontiguousarray(a)).to(torch.complex64).cuda()


def _chain(cfg, sample, scale=1.0):
    from paper_2003_09468_b200 import binding
    pb = synth.make_problem(cfg, l_scale=scale)
    ctx = binding.from_problem(pb, precision=1)
    try:
        Lh, ht = orc.half_rotate(pb.L, pb.psi_t, pb.h1)
        mesh = cfg.mesh
        phi_d = _c64(pb.phi)
        x_d = torch.from_numpy(pb.x).to(torch.float32).cuda()
        assert phi_d.dtype == torch.complex64
        theta_d, logdet_d, info_d = ctx.green(phi_d)
        assert theta_d.dtype == torch.complex64 and int(info_d.abs().sum()) == 0
        theta = theta_d.cpu().numpy().astype(np.complex128)
        logdet = logdet_d.cpu().numpy()
        vb_d = ctx.force_bias(theta_d)
        vb = vb_d.cpu().numpy().astype(np.complex128)
        vhs_d = ctx.vhs(x_d, vb_d, cfg.dtau)
        phi2_d = phi_d.clone()
        ctx.propagate(vhs_d, cfg.dtau, cfg.order, phi2_d)
        e_d = ctx.local_energy(theta_d)
        e = e_d.cpu().numpy().astype(np.complex128)
        x64 = x_d.cpu().numpy().astype(np.float64)
        for w in sample:
            th_o, ld_o, _ = orc.green(pb.psi_t, pb.phi[w])
            assert relerr(theta[w], th_o) < TOL, ("theta", w, relerr(theta[w], th_o))
            assert abs(logdet[w].real - ld_o.real) < TOL * max(1.0, abs(ld_o.real))
            assert abs(np.angle(np.exp(1j * (logdet[w].imag - ld_o.imag)))) < 1e-3
            vb_o = orc.force_bias(mesh, Lh, theta[w])
            assert relerr(vb[w], vb_o) < TOL, ("vbias", w, relerr(vb[w], vb_o))
            V = vhs_d[w].cpu().numpy().astype(np.complex128)
            V_o = orc.vhs(mesh, pb.L, orc.assemble_fields(mesh, x64[w], vb[w], cfg.dtau))
            assert relerr(V, V_o) < TOL, ("vhs", w, relerr(V, V_o))
            phi_w = phi_d[w].cpu().numpy().astype(np.complex128)
            p_o = orc.propagate(V, phi_w, cfg.dtau, cfg.order)
            assert relerr(phi2_d[w].cpu().numpy().astype(np.complex128), p_o) < TOL, ("propagate", w)
            e_o = orc.local_energy(mesh, Lh, ht, theta[w])
            for comp in range(3):
                assert abs(e[w, comp] - e_o[comp]) / abs(e_o[comp]) < TOL, ("energy", w, comp, e[w, comp], e_o[comp])
        # whole step, device and host entry
        phi3_d = phi_d.clone()
        e3, ld3, info3 = ctx.step(phi3_d, x_d, cfg.dtau, cfg.order)
        assert e3.dtype == torch.complex64 and int(info3.abs().sum()) == 0
        ph = phi_d.cpu().clone().pin_memory()
        xh = x_d.cpu().clone().pin_memory()
        eh = torch.empty((pb.phi.shape[0], 3), dtype=torch.complex64).pin_memory()
        ctx.step_host(ph, xh, cfg.dtau, cfg.order, eh)
        assert torch.equal(eh, e3.cpu()) and torch.equal(ph, phi3_d.cpu())
        # the block calls are FP64-only
        with pytest.raises(binding.AfqmcError) as err:
            ctx.apply_onebody(torch.from_numpy(pb.phi).cuda())
        assert err.value.code == 2
        return e3.cpu().numpy()
    finally:
        ctx.close()


@pytest.mark.parametrize("name", ["ragged", "C1"])
def test_complex64_boundary_small(name):
    cfg = {"ragged": synth.Config("ragged64", (2, 3, 1), 5, 3, 7, 5, 0.005, 6, 23), "C1": synth.CONFIGS["C1"]}[name]
    # 0.3 x L keeps the Taylor polynomial's terms within a few orders of magnitude, so that FP32 storage of phi' is meaningful
    _chain(cfg, range(cfg.nw), scale=0.3)


def test_complex64_boundary_c5_optional_run():
    """BASELINE.json config 5: 'complex128 with an optional complex64 run at 1e-4 tolerance' (sampled walkers; the
    unscaled synthetic L is used for every stage except that its polynomial propagation is checked stage-locally)."""
    cfg = synth.CONFIGS["C5"]
    _chain(cfg, [0, 5])


@pytest.mark.slow
def test_complex64_boundary_c4_single_precision_storage():
    """Config 4 (L = 12.6 GB in complex128): with precision = 1 the vHS and force-bias operands are STORED in single
    precision (half the bytes of the HBM-bound streams) and accumulated in FP64: 1e-4 against the oracle."""
    _chain(synth.CONFIGS["C4"], [0, 15])


def test_complex64_rejects_complex128_tensors():
    from paper_2003_09468_b200 import binding
    cfg = synth.CONFIGS["C1"]
    pb = synth.make_problem(cfg)
    ctx = binding.from_problem(pb, precision=1)
    try:
        with pytest.raises(TypeError):
            ctx.green(torch.from_numpy(pb.phi).cuda())
    finally:
        ctx.close()
