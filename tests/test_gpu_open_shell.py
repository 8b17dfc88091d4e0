"""GPU parity of OPEN-SHELL walkers (afqmc_dims.closed_shell = 0) against the oracle's `*_uhf`
functions (oracle/afqmc_oracle.py, pinned in tests/test_oracle_open_shell_pins.py): every C-ABI step call, the whole step on
device and through the host entry, and the closed-shell limit.  Tolerance: relative 1e-10 (north_star)."""
import numpy as np
import pytest
import torch

from oracle import afqmc_oracle as orc
from paper_2003_09468_b200 import synth

pytestmark = pytest.mark.gpu
RTOL = 1e-10


def relerr(a, b):
    a, b = np.asarray(a), np.asarray(b)
    return float(np.max(np.abs(a - b)) / max(float(np.max(np.abs(b))), 1e-300))


def phase_diff(a, b):
    return abs(np.angle(np.exp(1j * (a - b))))


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


class OpenCase:
    def __init__(self, mesh, m, n_up, n_dn, nchol, nw, seed=41):
        from paper_2003_09468_b200 import binding
        self.cfg = synth.tiny_config(mesh=mesh, m=m, n=n_up, nchol=nchol, nw=nw, seed=seed)
        self.pb, self.psi_dn, self.phi_dn = synth.make_open_shell(self.cfg, n_dn)
        cfg, pb = self.cfg, self.pb
        self.ctx = binding.Afqmc(cfg.mesh, m, n_up, nchol, dev(pb.h1), dev(pb.L), (dev(pb.psi_t), dev(self.psi_dn)), nw,
                                 closed_shell=0, n_dn=n_dn)
        self.psi = (pb.psi_t, self.psi_dn)
        self.phi = (pb.phi, self.phi_dn)
        self.Lh, self.ht = zip(*[orc.half_rotate(pb.L, p, pb.h1) for p in self.psi])
        self.nw = nw

    def close(self):
        self.ctx.close()


SHAPES = [
    dict(mesh=(2, 3, 1), m=5, n_up=3, n_dn=2, nchol=7, nw=5),       # ragged everything, N_up != N_dn
    dict(mesh=(2, 2, 1), m=26, n_up=4, n_dn=3, nchol=18, nw=6),     # m = 26: the register-B exchange kernel, padded spin-down rows
    dict(mesh=(1, 2, 2), m=9, n_up=6, n_dn=1, nchol=5, nw=3),       # two a-groups up, a single orbital down
    dict(mesh=(3, 1, 1), m=33, n_up=2, n_dn=5, nchol=9, nw=2),      # m > 28: generic exchange kernel; more down than up electrons
]


@pytest.mark.parametrize("kw", SHAPES, ids=lambda k: "x".join(map(str, k["mesh"])) + "_m%d_up%d_dn%d_c%d_w%d" % (k["m"], k["n_up"], k["n_dn"], k["nchol"], k["nw"]))
def test_open_shell_calls_and_step_against_the_oracle(kw):
    case = OpenCase(**kw)
    try:
        cfg, pb, ctx, nw = case.cfg, case.pb, case.ctx, case.nw
        mesh = cfg.mesh
        phi_d = ctx.join_spin(dev(case.phi[0]), dev(case.phi[1]))
        x_d = dev(pb.x)
        # a1-a3: per-spin Green's functions, log det = sum of the channels
        theta_d, ld_d, info_d = ctx.green(phi_d)
        assert np.all(info_d.cpu().numpy() == 0)
        th = [t.cpu().numpy() for t in ctx.split_theta(theta_d, nw)]
        ld = ld_d.cpu().numpy()
        ld2, _ = ctx.overlap(phi_d)
        assert np.array_equal(ld2.cpu().numpy(), ld)
        for w in range(nw):
            ref = [orc.green(case.psi[s], case.phi[s][w]) for s in range(2)]
            for s in range(2):
                assert relerr(th[s][w], ref[s][0]) < RTOL, ("theta", s, w)
            tot = ref[0][1] + ref[1][1]
            assert abs(ld[w].real - tot.real) < RTOL * max(1.0, abs(tot.real)) and phase_diff(ld[w].imag, tot.imag) < 1e-9
        # a4: spin-summed force bias
        vb_d = ctx.force_bias(theta_d)
        vb = vb_d.cpu().numpy()
        for w in range(nw):
            assert relerr(vb[w], orc.force_bias_uhf(mesh, case.Lh[0], case.Lh[1], th[0][w], th[1][w])) < RTOL, ("vbias", w)
        # a5 (spin independent) + a6 on both channels
        vhs_d = ctx.vhs(x_d, vb_d, cfg.dtau)
        phi2_d = phi_d.clone()
        ctx.propagate(vhs_d, cfg.dtau, cfg.order, phi2_d)
        new = [t.cpu().numpy() for t in ctx.split_phi(phi2_d, nw)]
        for w in range(nw):
            V = vhs_d[w].cpu().numpy()
            assert relerr(V, orc.vhs(mesh, pb.L, orc.assemble_fields(mesh, pb.x[w], vb[w], cfg.dtau))) < RTOL
            for s in range(2):
                assert relerr(new[s][w], orc.propagate(V, case.phi[s][w], cfg.dtau, cfg.order)) < RTOL, ("propagate", s, w)
        # a7-a9 on the propagated walkers
        theta2_d, ld2_d, _ = ctx.green(phi2_d)
        th2 = [t.cpu().numpy() for t in ctx.split_theta(theta2_d, nw)]
        e_d = ctx.local_energy(theta2_d)
        e = e_d.cpu().numpy()
        for w in range(nw):
            e_o = orc.local_energy_uhf(mesh, case.Lh, case.ht, (th2[0][w], th2[1][w]))
            for i, name in enumerate(("E1", "EC", "EX")):
                assert abs(e[w, i] - e_o[i]) < RTOL * abs(e_o[i]), (name, w, e[w, i], e_o[i])
        # every exchange kernel variant agrees on the open-shell energies
        for opts in ({"exchange_3m": 0}, {"exchange_regb": 0}):
            for k, v in opts.items():
                ctx.set_option(k, v)
            e_v = ctx.local_energy(theta2_d).cpu().numpy()
            ctx.set_option("exchange_3m", 1)
            ctx.set_option("exchange_regb", 1)
            assert relerr(e_v, e) < 1e-12, opts
        # whole step == the chain, bit for bit, on the device and through the host entry; and == the oracle's step
        phi3_d = phi_d.clone()
        e3_d, ld3_d, info3_d = ctx.step(phi3_d, x_d, cfg.dtau, cfg.order)
        assert torch.equal(phi3_d, phi2_d) and torch.equal(e3_d, e_d) and torch.equal(ld3_d, ld2_d)
        phi_h = phi_d.cpu().pin_memory()
        e_h = torch.empty((nw, 3), dtype=torch.complex128).pin_memory()
        ld_h = torch.empty((nw,), dtype=torch.complex128).pin_memory()
        ctx.step_host(phi_h, torch.from_numpy(pb.x.copy()).pin_memory(), cfg.dtau, cfg.order, e_h, ld_h)
        assert torch.equal(phi_h, phi2_d.cpu()) and torch.equal(e_h, e_d.cpu()) and torch.equal(ld_h, ld2_d.cpu())
        (pu, pd), e_o, ld_o = orc.step_uhf(mesh, pb.L, case.Lh, case.ht, case.psi, case.phi, pb.x, cfg.dtau, cfg.order)
        assert relerr(new[0], pu) < RTOL and relerr(new[1], pd) < RTOL
        assert np.max(np.abs(e - e_o) / np.abs(e_o)) < RTOL
        ld3 = ld3_d.cpu().numpy()
        assert np.max(np.abs(ld3.real - ld_o.real)) < 1e-9 and np.max(phase_diff(ld3.imag, ld_o.imag)) < 1e-9
    finally:
        case.close()


def test_open_shell_context_with_equal_channels_is_the_closed_shell():
    """Two identical spin channels through the open-shell path reproduce the closed-shell context: energies, force bias, the
    propagated walker (both channels), log det = twice the single-channel one; and the same for a whole AFQMC block (hybrid
    weights use the overlap ratio of both channels either way)."""
    from paper_2003_09468_b200 import binding
    cfg = synth.tiny_config(mesh=(2, 2, 1), m=7, n=3, nchol=9, nw=4, seed=43)
    pb = synth.make_problem(cfg, l_scale=0.1)
    closed = binding.from_problem(pb)
    opn = binding.Afqmc(cfg.mesh, cfg.m, cfg.n, cfg.nchol, dev(pb.h1), dev(pb.L), (dev(pb.psi_t), dev(pb.psi_t)), cfg.nw,
                        closed_shell=0, n_dn=cfg.n)
    try:
        phi_c = dev(pb.phi)
        phi_o = opn.join_spin(phi_c, phi_c)
        x_d = dev(pb.x)
        ec, ldc, _ = closed.step(phi_c, x_d, cfg.dtau, cfg.order)
        eo, ldo, _ = opn.step(phi_o, x_d, cfg.dtau, cfg.order)
        up, dn = opn.split_phi(phi_o, cfg.nw)
        assert relerr(up.cpu().numpy(), phi_c.cpu().numpy()) < 1e-13 and torch.equal(up, dn)
        assert relerr(eo.cpu().numpy(), ec.cpu().numpy()) < 1e-12
        assert np.max(np.abs(ldo.cpu().numpy().real - 2 * ldc.cpu().numpy().real)) < 1e-11
        # the block
        nsteps = 3
        xs = dev(synth.make_block_fields(cfg, nsteps))
        h1 = dev(pb.h1)
        closed.set_onebody(h1, cfg.dtau)
        opn.set_onebody(h1, cfg.dtau)
        pc, po = dev(pb.phi), opn.join_spin(dev(pb.phi), dev(pb.phi))
        wc = torch.ones(cfg.nw, dtype=torch.float64, device="cuda")
        wo = wc.clone()
        e1, em1, lr1, i1 = closed.block(pc, wc, xs, cfg.dtau, cfg.order)
        e2, em2, lr2, i2 = opn.block(po, wo, xs, cfg.dtau, cfg.order)
        assert int(i1.abs().sum()) == 0 and int(i2.abs().sum()) == 0
        assert relerr(wo.cpu().numpy(), wc.cpu().numpy()) < 1e-10
        assert relerr(e2.cpu().numpy(), e1.cpu().numpy()) < 1e-10 and relerr(em2.cpu().numpy(), em1.cpu().numpy()) < 1e-10
        assert relerr(lr2.cpu().numpy(), 2 * lr1.cpu().numpy()) < 1e-10
        u2, d2 = opn.split_phi(po, cfg.nw)
        assert relerr(u2.cpu().numpy(), pc.cpu().numpy()) < 1e-9 and torch.equal(u2, d2)
    finally:
        closed.close()
        opn.close()


def test_open_shell_argument_errors():
    import ctypes
    from paper_2003_09468_b200 import binding
    lib = binding.lib()
    buf = torch.zeros(4096, dtype=torch.complex128, device="cuda")
    h = ctypes.c_void_p(0)
    for n_dn, code in ((0, 1), (7, 1)):                      # n_dn must be 1..m
        d = binding.Dims((ctypes.c_int * 3)(2, 2, 1), 6, 4, 10, 0, 0, 4, n_dn)
        assert lib.afqmc_create(ctypes.byref(h), ctypes.byref(d), buf.data_ptr(), buf.data_ptr(), buf.data_ptr(), None) == code
    d = binding.Dims((ctypes.c_int * 3)(2, 2, 1), 6, 4, 10, 0, 1, 4, 2)      # complex64 boundary is closed-shell only
    assert lib.afqmc_create(ctypes.byref(h), ctypes.byref(d), buf.data_ptr(), buf.data_ptr(), buf.data_ptr(), None) == 2
    d = binding.Dims((ctypes.c_int * 3)(2, 2, 1), 6, 4, 10, 3, 0, 4, 2)      # closed_shell must be 0 or 1
    assert lib.afqmc_create(ctypes.byref(h), ctypes.byref(d), buf.data_ptr(), buf.data_ptr(), buf.data_ptr(), None) == 1
