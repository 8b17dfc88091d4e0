"""GPU parity of the AFQMC-block calls (include/afqmc.h "The AFQMC block") against the
CPU oracle on the same seeded inputs.  Same metric and 1e-10 tolerance as test_gpu_parity.py for single calls;
the multi-step block is held to 1e-8 on the walkers (errors pass through several overlap inversions)."""
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


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


SHAPES = {
    "ragged": synth.Config("ragged", (2, 3, 1), 5, 3, 7, 5, 0.005, 6, 21),
    "gamma": synth.Config("gamma", (1, 1, 1), 9, 2, 11, 3, 0.005, 4, 22),
    "C1": synth.CONFIGS["C1"],
}


@pytest.fixture(scope="module", params=list(SHAPES))
def case(request):
    from paper_2003_09468_b200 import binding
    cfg = SHAPES[request.param]
    pb = synth.make_problem(cfg, l_scale=0.1)
    ctx = binding.from_problem(pb)
    Lh, ht = orc.half_rotate(pb.L, pb.psi_t, pb.h1)
    yield dict(cfg=cfg, pb=pb, ctx=ctx, Lh=Lh, ht=ht)
    ctx.close()


def test_onebody_propagator_and_application(case):
    cfg, pb, ctx = case["cfg"], case["pb"], case["ctx"]
    for dtau in (cfg.dtau, 0.3, 4.0):                              # 4.0 needs several squarings
        b1 = ctx.set_onebody(_dev(pb.h1), dtau).cpu().numpy()
        b1_o = orc.onebody_half_propagator(pb.h1, dtau)
        for k in range(cfg.nk):
            assert relerr(b1[k], b1_o[k]) < 1e-12, (dtau, k, relerr(b1[k], b1_o[k]))
    b1 = ctx.set_onebody(_dev(pb.h1), cfg.dtau).cpu().numpy()
    phi_d = _dev(pb.phi)
    ctx.apply_onebody(phi_d)
    out = phi_d.cpu().numpy()
    for w in range(pb.phi.shape[0]):
        assert relerr(out[w], orc.apply_onebody(b1, pb.phi[w])) < RTOL


def test_apply_onebody_needs_a_propagator():
    from paper_2003_09468_b200 import binding
    cfg = SHAPES["gamma"]
    pb = synth.make_problem(cfg)
    ctx = binding.from_problem(pb)
    with pytest.raises(binding.AfqmcError) as e:
        ctx.apply_onebody(_dev(pb.phi))
    assert e.value.code == 1
    ctx.close()


def test_hybrid_weight(case):
    cfg, pb, ctx = case["cfg"], case["pb"], case["ctx"]
    nw = pb.phi.shape[0]
    phi_d, x_d = _dev(pb.phi), _dev(pb.x)
    theta_d, ld_old_d, _ = ctx.green(phi_d)
    vb_d = ctx.force_bias(theta_d)
    rng = np.random.default_rng(3)
    # any pair of overlaps exercises the formula; include a killed walker (phase change > pi/2) and a wrap
    ld_old = ld_old_d.cpu().numpy()
    ld_new = ld_old + 0.05 * (rng.standard_normal(nw) + 1j * rng.standard_normal(nw))
    ld_new[0] = ld_old[0] + 0.1 + 1.0j           # dtheta = 2.0 > pi/2: killed
    if nw > 1:
        ld_new[1] = ld_old[1] - 0.2 + 3.1j       # dtheta = 6.2 - 2 pi = -0.083: wraps, survives
    w0 = rng.random(nw) + 0.5
    w_d = _dev(w0.copy())
    _, logi_d = ctx.hybrid_weight(x_d, vb_d, cfg.dtau, ld_old_d, _dev(ld_new), w_d)
    w_g, logi = w_d.cpu().numpy(), logi_d.cpu().numpy()
    vb = vb_d.cpu().numpy()
    for w in range(nw):
        logI, dth, fac = orc.hybrid_weight(cfg.mesh, pb.x[w], vb[w], cfg.dtau, ld_old[w], ld_new[w])
        assert abs(logi[w] - logI) < RTOL * max(1.0, abs(logI)), (w, logi[w], logI)
        assert abs(w_g[w] - w0[w] * fac) <= RTOL * max(w0[w] * fac, 1e-3), (w, w_g[w], w0[w] * fac)
    assert w_g[0] == 0.0
    if nw > 1:
        assert w_g[1] > 0.0


def test_orthogonalize(case):
    cfg, pb, ctx = case["cfg"], case["pb"], case["ctx"]
    nw = pb.phi.shape[0]
    rng = np.random.default_rng(8)
    phi = np.empty_like(pb.phi)
    for w in range(nw):
        R0 = rng.standard_normal((cfg.N, cfg.N)) + 1j * rng.standard_normal((cfg.N, cfg.N))
        phi[w] = pb.phi[w] @ R0 * (10.0 ** (w - 1))               # non-orthonormal, different scales
    phi_d = _dev(phi)
    _, ldr_d, info_d = ctx.orthogonalize(phi_d)
    q, ldr, info = phi_d.cpu().numpy(), ldr_d.cpu().numpy(), info_d.cpu().numpy()
    assert np.all(info == 0)
    for w in range(nw):
        q_o, ldr_o = orc.orthogonalize(phi[w])
        assert relerr(np.conj(q[w].T) @ q[w], np.eye(cfg.N)) < 1e-13
        assert relerr(q[w], q_o) < 1e-9, (w, relerr(q[w], q_o))     # cond(R0) ~ 1e2-1e3 enters both methods
        assert abs(ldr[w] - ldr_o) < RTOL * max(1.0, abs(ldr_o))
    # already orthonormal: unchanged, log det R = 0
    phi_d = _dev(pb.phi)
    _, ldr_d, _ = ctx.orthogonalize(phi_d)
    assert relerr(phi_d.cpu().numpy(), pb.phi) < 1e-13
    assert float(ldr_d.abs().max()) < 1e-12
    # rank-deficient walker -> info > 0 for that walker only
    bad = pb.phi.copy()
    bad[0][:, -1] = bad[0][:, 0]
    bad_d = _dev(bad)
    _, _, info_d = ctx.orthogonalize(bad_d)
    info = info_d.cpu().numpy()
    assert info[0] > 0 and np.all(info[1:] == 0)


def test_mixed_estimator(case):
    ctx = case["ctx"]
    rng = np.random.default_rng(5)
    nw = 7
    e = rng.standard_normal((nw, 3)) + 1j * rng.standard_normal((nw, 3))
    w = rng.random(nw)
    out = ctx.mixed_estimator(_dev(e), _dev(w)).cpu().numpy()
    num, den = orc.mixed_estimator(w, e)
    assert relerr(out[:3], num) < 1e-14 and abs(out[3] - den) < 1e-14 * den


def _compare_block(cfg, pb, ctx, Lh, ht, nsteps, dtau, sample, tol_phi=1e-8):
    nw = pb.phi.shape[0]
    xs = synth.make_block_fields(cfg, nsteps, nw)
    b1 = orc.onebody_half_propagator(pb.h1, dtau)
    ctx.set_onebody(_dev(pb.h1), dtau)
    phi_d, w_d = _dev(pb.phi), _dev(np.ones(nw))
    energy_d, emixed_d, ldr_d, info_d = ctx.block(phi_d, w_d, _dev(xs), dtau, cfg.order)
    phi_g, w_g, e_g = phi_d.cpu().numpy(), w_d.cpu().numpy(), energy_d.cpu().numpy()
    em_g, ldr_g = emixed_d.cpu().numpy(), ldr_d.cpu().numpy()
    assert np.all(info_d.cpu().numpy() == 0)
    idx = list(sample)
    phi_o, w_o, e_o, (num, den), ldr_o = orc.block(cfg.mesh, pb.L, Lh, ht, pb.psi_t, b1, pb.phi[idx], np.ones(len(idx)),
                                                   xs[:, idx], dtau, cfg.order)
    for i, w in enumerate(idx):
        assert relerr(phi_g[w], phi_o[i]) < tol_phi, ("phi", w, relerr(phi_g[w], phi_o[i]))
        assert abs(w_g[w] - w_o[i]) <= 1e-8 * max(w_o[i], 1e-3), ("weight", w, w_g[w], w_o[i])
        assert relerr(e_g[w], e_o[i]) < 1e-8, ("energy", w, relerr(e_g[w], e_o[i]))
        assert abs(ldr_g[w] - ldr_o[i]) < 1e-8 * max(1.0, abs(ldr_o[i])), ("logdetR", w)
        assert relerr(np.conj(phi_g[w].T) @ phi_g[w], np.eye(cfg.N)) < 1e-12
    # the mixed estimator is over ALL walkers: check it against the GPU's own weights and energies (exact sum order)
    assert relerr(em_g[:3], np.einsum('w,wc->c', w_g, e_g)) < 1e-13
    assert abs(em_g[3] - w_g.sum()) <= 1e-13 * max(w_g.sum(), 1e-300)
    if len(idx) == nw:
        assert relerr(em_g[:3], num) <= 1e-8 and abs(em_g[3].real - den) <= 1e-8 * den
    return w_g


def test_block_small_shapes(case):
    cfg, pb = case["cfg"], case["pb"]
    w = _compare_block(cfg, pb, case["ctx"], case["Lh"], case["ht"], 3, cfg.dtau, range(pb.phi.shape[0]))
    assert np.all(w > 0)                                          # physically scaled steps: nobody is killed
    # zero steps: energy of the input walkers, weights unchanged, walkers orthonormalised (already are)
    _compare_block(cfg, pb, case["ctx"], case["Lh"], case["ht"], 0, cfg.dtau, range(pb.phi.shape[0]))


def test_block_unscaled_inputs_kill_walkers_consistently():
    """BASELINE.json's unscaled L: large steps, the phaseless projection zeroes weights; GPU and oracle agree on who dies."""
    from paper_2003_09468_b200 import binding
    cfg = SHAPES["C1"]
    pb = synth.make_problem(cfg)
    ctx = binding.from_problem(pb)
    Lh, ht = orc.half_rotate(pb.L, pb.psi_t, pb.h1)
    _compare_block(cfg, pb, ctx, Lh, ht, 2, cfg.dtau, range(cfg.nw), tol_phi=1e-7)
    ctx.close()


def test_block_c3_full_size_sampled_walkers():
    from paper_2003_09468_b200 import binding
    cfg = synth.CONFIGS["C3"]
    pb = synth.make_problem(cfg, l_scale=0.01)
    ctx = binding.from_problem(pb)
    Lh, ht = orc.half_rotate(pb.L, pb.psi_t, pb.h1)
    w = _compare_block(cfg, pb, ctx, Lh, ht, 2, cfg.dtau, [0, 17])
    assert w[0] > 0 and w[17] > 0                                 # the compared walkers survive both steps
    ctx.close()


def test_block_argument_errors(case):
    from paper_2003_09468_b200 import binding
    cfg, pb, ctx = case["cfg"], case["pb"], case["ctx"]
    ctx.set_onebody(_dev(pb.h1), cfg.dtau)
    nw = pb.phi.shape[0]
    xs = _dev(synth.make_block_fields(cfg, 1, nw))
    with pytest.raises(binding.AfqmcError):
        ctx.block(_dev(pb.phi), _dev(np.ones(nw)), xs, -1.0, cfg.order)
    with pytest.raises(binding.AfqmcError):
        ctx.block(_dev(pb.phi), _dev(np.ones(nw)), xs, cfg.dtau, 99)
