"""GPU parity: every C-ABI step call against the CPU oracle on the same seeded inputs.

Tolerances (BASELINE.json north_star, metric of SURVEY.md P16): relative 1e-10 in complex128 --
tensors: max|gpu-ref| / max|ref| per walker; scalars: |gpu-ref| / |ref|; logdet: real part
relative to max(1,|ref|), phase modulo 2 pi.  Each stage is fed the GPU output of the previous
stage (downloaded), and the oracle evaluates the same stage on exactly those inputs, so a stage's
error is not hidden or amplified by its predecessors.
"""
import os

import numpy as np
import pytest
import torch

from oracle import afqmc_oracle as orc
from paper_2003_09468_b200 import synth

pytestmark = pytest.mark.gpu

RTOL = 1e-10


def relerr(a, b):
    a, b = np.asarray(a), np.asarray(b)
    den = max(float(np.max(np.abs(b))), 1e-300)
    return float(np.max(np.abs(a - b)) / den)


def phase_diff(a, b):
    return abs(np.angle(np.exp(1j * (a - b))))


def _to_dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


class Case:
    def __init__(self, cfg, nw=None, real_orbitals=False):
        from paper_2003_09468_b200 import binding
        self.cfg = cfg
        self.pb = synth.make_problem(cfg, nw, real_orbitals=real_orbitals)
        self.nw = self.pb.phi.shape[0]
        self.ctx = binding.from_problem(self.pb)
        self.Lh, self.ht = orc.half_rotate(self.pb.L, self.pb.psi_t, self.pb.h1)

    def close(self):
        self.ctx.close()


_JOB = {}


def _energy_job(w):
    j = _JOB
    return orc.local_energy(j["mesh"], j["Lh"], j["ht"], j["theta"][w])


def oracle_energies(mesh, Lh, ht, theta, walkers):
    """orc.local_energy for several walkers, one forked worker process per walker when there is more than one (the
    oracle itself stays plain and single-threaded; the children run numpy only and never touch CUDA)."""
    walkers = list(walkers)
    _JOB.update(mesh=mesh, Lh=Lh, ht=ht, theta=theta)
    try:
        if len(walkers) > 1 and (os.cpu_count() or 1) > 1 and Lh.nbytes > (64 << 20):
            import multiprocessing as mp
            try:
                with mp.get_context("fork").Pool(min(len(walkers), os.cpu_count())) as pool:
                    return dict(zip(walkers, pool.map_async(_energy_job, walkers).get(timeout=900)))
            except Exception as exc:           # noqa: BLE001 - fall back to the plain loop
                print("oracle pool failed (%r): serial evaluation" % (exc,))
        return {w: _energy_job(w) for w in walkers}
    finally:
        _JOB.clear()


def cond_overlap(psi_t, phi_w):
    """2-norm condition number of O = A^dagger Phi (numpy SVD; used only to DERIVE a tolerance, never as a reference value)."""
    return float(np.linalg.cond(orc.overlap(psi_t, phi_w)))


def theta2_bound(cond):
    """Tolerance of quantities that pass through the inversion of the PROPAGATED walker's overlap O': north_star's 1e-10,
    flat.  cond(O') is printed beside every measured error because it is what the error scales with (elimination with
    partial pivoting: forward error <~ c(N) * cond * 2^-53); on the synthetic walkers cond(O') reaches 1e4 and the measured
    error 3e-13, so the flat bound holds with two orders of margin at every config."""
    del cond
    return RTOL


def run_chain_and_compare(case, sample=None, tol=RTOL, energy_sample=None):
    """Stages a1..a9 on ALL walkers of the case against the oracle; `sample` restricts the walkers (None = all) and
    `energy_sample` the walkers whose local energy the oracle evaluates (the oracle's exchange recipe costs seconds
    per walker at the full-size configs); every walker outside `energy_sample` has its energies cross-checked between
    the two independent exchange kernels (3M, exchange3m.cu; 4M, energy.cu) at 1e-12."""
    cfg, pb, ctx = case.cfg, case.pb, case.ctx
    mesh = cfg.mesh
    sample = list(range(case.nw)) if sample is None else list(sample)
    energy_sample = sample if energy_sample is None else list(energy_sample)
    phi_d = _to_dev(pb.phi)
    x_d = _to_dev(pb.x)

    # a1-a3
    theta_d, logdet_d, info_d = ctx.green(phi_d)
    theta, logdet, info = theta_d.cpu().numpy(), logdet_d.cpu().numpy(), info_d.cpu().numpy()
    assert np.all(info == 0)
    ld2, info2 = ctx.overlap(phi_d)
    assert np.array_equal(ld2.cpu().numpy(), logdet)          # same kernel, same result
    for w in sample:
        th_o, ld_o, inf_o = orc.green(pb.psi_t, pb.phi[w])
        assert inf_o == 0
        assert relerr(theta[w], th_o) < tol, ("theta", w, relerr(theta[w], th_o))
        assert abs(logdet[w].real - ld_o.real) < tol * max(1.0, abs(ld_o.real)), ("logdet", w)
        assert phase_diff(logdet[w].imag, ld_o.imag) < 1e-9, ("phase", w)

    # a4
    vb_d = ctx.force_bias(theta_d)
    vb = vb_d.cpu().numpy()
    for w in sample:
        vb_o = orc.force_bias(mesh, case.Lh, theta[w])
        assert relerr(vb[w], vb_o) < tol, ("vbias", w, relerr(vb[w], vb_o))

    # a5 (with and without the force-bias shift)
    vhs_d = ctx.vhs(x_d, vb_d, cfg.dtau)
    vhs0_d = ctx.vhs(x_d, None, cfg.dtau)
    for w in sample:
        V = vhs_d[w].cpu().numpy()
        V_o = orc.vhs(mesh, pb.L, orc.assemble_fields(mesh, pb.x[w], vb[w], cfg.dtau))
        assert relerr(V, V_o) < tol, ("vhs", w, relerr(V, V_o))
        V0 = vhs0_d[w].cpu().numpy()
        V0_o = orc.vhs(mesh, pb.L, orc.assemble_fields(mesh, pb.x[w], None, cfg.dtau))
        assert relerr(V0, V0_o) < tol, ("vhs0", w)
        assert relerr(V0, -np.conj(V0.T)) < 1e-13              # anti-Hermitian without the shift
    del vhs0_d

    # a6
    phi2_d = phi_d.clone()
    ctx.propagate(vhs_d, cfg.dtau, cfg.order, phi2_d)
    phi2 = phi2_d.cpu().numpy()
    for w in sample:
        p_o = orc.propagate(vhs_d[w].cpu().numpy(), pb.phi[w], cfg.dtau, cfg.order)
        assert relerr(phi2[w], p_o) < tol, ("propagate", w, relerr(phi2[w], p_o))
    phi0_d = phi_d.clone()
    ctx.propagate(vhs_d, cfg.dtau, 0, phi0_d)
    assert torch.equal(phi0_d, phi_d)                          # order 0 = identity
    del vhs_d

    # a1-a3 on the propagated walker: held to north_star's 1e-10 unless cond(O') forbids it (derived, printed)
    theta2_d, logdet2_d, info2_d = ctx.green(phi2_d)
    theta2, logdet2 = theta2_d.cpu().numpy(), logdet2_d.cpu().numpy()
    assert np.all(info2_d.cpu().numpy() == 0)
    worst, worst_cond = 0.0, 0.0
    for w in sample:
        th_o, ld_o, _ = orc.green(pb.psi_t, phi2[w])
        cnd = cond_overlap(pb.psi_t, phi2[w])
        err = relerr(theta2[w], th_o)
        worst, worst_cond = max(worst, err), max(worst_cond, cnd)
        assert err < theta2_bound(cnd), ("theta2", w, err, cnd)
        assert abs(logdet2[w].real - ld_o.real) < tol * max(1.0, abs(ld_o.real)), ("logdet2", w)
        assert phase_diff(logdet2[w].imag, ld_o.imag) < 1e-9, ("phase2", w)
    print("[parity %s] theta(propagated walker): max rel err %.2e, max cond(O') %.2e, bound %.2e"
          % (cfg.name, worst, worst_cond, theta2_bound(worst_cond)))

    # a7-a9
    e_d = ctx.local_energy(theta2_d)
    e = e_d.cpu().numpy()
    e_orc = oracle_energies(mesh, case.Lh, case.ht, theta2, energy_sample)
    for w in energy_sample:
        e_o = e_orc[w]
        for i, name in enumerate(("E1", "EC", "EX")):
            assert abs(e[w, i] - e_o[i]) < tol * abs(e_o[i]), (name, w, e[w, i], e_o[i])
    if len(energy_sample) < case.nw:
        # the walkers the oracle did not evaluate: the two independent exchange kernels must agree on every walker
        ctx.set_option("exchange_3m", 0)
        try:
            e4 = ctx.local_energy(theta2_d).cpu().numpy()
        finally:
            ctx.set_option("exchange_3m", 1)
        assert np.max(np.abs(e4 - e) / np.abs(e)) < 1e-12, ("3M vs 4M", np.max(np.abs(e4 - e) / np.abs(e)))
        # E1 and EC of EVERY walker against the oracle's cheap definitions (Eq. 49 line 1; Eq. 41 from the force bias)
        vb2 = ctx.force_bias(theta2_d).cpu().numpy()
        for w in sample:
            e1_o = sum(2.0 * np.sum(case.ht[k] * theta2[w][k * cfg.n:(k + 1) * cfg.n, k * cfg.m:(k + 1) * cfg.m]) for k in range(cfg.nk))
            ec_o = orc.coulomb_from_vbias(mesh, orc.force_bias(mesh, case.Lh, theta2[w]))
            assert abs(e[w, 0] - e1_o) < tol * abs(e1_o), ("E1", w)
            assert abs(e[w, 1] - ec_o) < tol * abs(ec_o), ("EC", w)
            assert relerr(vb2[w], orc.force_bias(mesh, case.Lh, theta2[w])) < tol

    # whole step == the chain above, bit for bit, on device and through the host entry
    phi3_d = phi_d.clone()
    e3_d, ld3_d, info3_d = ctx.step(phi3_d, x_d, cfg.dtau, cfg.order)
    assert torch.equal(phi3_d, phi2_d)
    assert torch.equal(e3_d, e_d)
    assert torch.equal(ld3_d, logdet2_d)
    phi_h = torch.from_numpy(pb.phi.copy()).pin_memory()
    x_h = torch.from_numpy(pb.x.copy()).pin_memory()
    e_h = torch.empty((case.nw, 3), dtype=torch.complex128).pin_memory()
    ctx.step_host(phi_h, x_h, cfg.dtau, cfg.order, e_h)
    assert torch.equal(phi_h, phi2_d.cpu())
    assert torch.equal(e_h, e_d.cpu())
    return e


def step_end_to_end_vs_oracle(case, walkers):
    """afqmc_step (one call, nothing downloaded in between) against orc.step on the same walkers: energies, log det and
    the propagated walker with every stage's rounding compounding.  The energies pass through the inversion of O', so
    their bound is theta2_bound(cond(O')) (= 1e-10 unless the propagated overlap is ill conditioned; printed)."""
    cfg, pb, ctx = case.cfg, case.pb, case.ctx
    phi_d = _to_dev(pb.phi)
    e_d, ld_d, info_d = ctx.step(phi_d, _to_dev(pb.x), cfg.dtau, cfg.order)
    e, ld, phi_new = e_d.cpu().numpy(), ld_d.cpu().numpy(), phi_d.cpu().numpy()
    assert np.all(info_d.cpu().numpy() == 0)
    for w in walkers:
        phi_o, e_o, ld_o = orc.step(cfg.mesh, pb.L, case.Lh, case.ht, pb.psi_t, pb.phi[w:w + 1], pb.x[w:w + 1], cfg.dtau, cfg.order)
        cnd = cond_overlap(pb.psi_t, phi_o[0])
        bound = theta2_bound(cnd)
        assert relerr(phi_new[w], phi_o[0]) < RTOL, ("phi'", w, relerr(phi_new[w], phi_o[0]))
        errs = [abs(e[w, i] - e_o[0, i]) / abs(e_o[0, i]) for i in range(3)]
        print("[e2e %s walker %d] rel err E1 %.2e EC %.2e EX %.2e, cond(O') %.2e, bound %.2e" % ((cfg.name, w) + tuple(errs) + (cnd, bound)))
        assert max(errs) < bound, (w, errs, cnd)
        assert abs(ld[w].real - ld_o[0].real) < RTOL * max(1.0, abs(ld_o[0].real))
        assert phase_diff(ld[w].imag, ld_o[0].imag) < 1e-9


# ------------------------------------------------------------------------------------------
# small and ragged shapes: all walkers checked
# ------------------------------------------------------------------------------------------
RAGGED = [
    dict(mesh=(2, 3, 1), m=5, n=3, nchol=7, nw=5),      # odd m, n<4, odd nchol, nw not a multiple of 4
    dict(mesh=(1, 1, 1), m=7, n=5, nchol=9, nw=1),      # single k-point, two a-groups, one walker
    dict(mesh=(2, 2, 2), m=6, n=4, nchol=16, nw=9),     # every Q self-inverse
    dict(mesh=(3, 1, 2), m=4, n=2, nchol=3, nw=2),
    dict(mesh=(3, 3, 1), m=9, n=6, nchol=21, nw=3),     # n=6: padded second a-group
    dict(mesh=(2, 1, 1), m=104, n=10, nchol=6, nw=3),   # theta blocks too large for one CTA: large-block exchange kernel,
                                                        # self-partner and paired units, padded third a-group
]


@pytest.mark.parametrize("kw", RAGGED, ids=lambda k: "x".join(map(str, k["mesh"])) + "_m%d_n%d_c%d_w%d" % (k["m"], k["n"], k["nchol"], k["nw"]))
def test_ragged_small(kw):
    cfg = synth.tiny_config(seed=2, **kw)
    case = Case(cfg)
    try:
        run_chain_and_compare(case)
        step_end_to_end_vs_oracle(case, range(case.nw))
    finally:
        case.close()


def test_config_C1_all_walkers():
    case = Case(synth.CONFIGS["C1"])
    try:
        run_chain_and_compare(case)
        step_end_to_end_vs_oracle(case, range(case.nw))
    finally:
        case.close()


def test_config_C2_all_walkers_energy_sampled():
    case = Case(synth.CONFIGS["C2"])
    try:
        run_chain_and_compare(case, energy_sample=[0, 37, 63])
        step_end_to_end_vs_oracle(case, [11])
    finally:
        case.close()


def test_gamma_point_supercell_shape_all_walkers():
    """the dense Gamma-point representation = one k-point with large m and n (synth config G1);
    its theta blocks do not fit one CTA's shared memory, so the exchange runs the large-block 3M kernel."""
    case = Case(synth.CONFIGS["G1"])
    try:
        run_chain_and_compare(case)        # every walker: the 4M cross-check kernel cannot hold these theta blocks
    finally:
        case.close()


def test_config_C3_headline_all_walkers_energy_sampled():
    case = Case(synth.CONFIGS["C3"])
    try:
        run_chain_and_compare(case, energy_sample=[0, 16, 31])
        step_end_to_end_vs_oracle(case, [7])
    finally:
        case.close()


@pytest.mark.slow
@pytest.mark.skipif(os.environ.get("AFQMC_SKIP_LARGE") == "1", reason="AFQMC_SKIP_LARGE=1")
def test_config_C4_all_walkers_energy_sampled():
    case = Case(synth.CONFIGS["C4"])
    try:
        run_chain_and_compare(case, energy_sample=[0, 8, 15])
    finally:
        case.close()


@pytest.mark.slow
@pytest.mark.skipif(os.environ.get("AFQMC_SKIP_LARGE") == "1", reason="AFQMC_SKIP_LARGE=1")
def test_config_C5_all_walkers_energy_sampled():
    case = Case(synth.CONFIGS["C5"])
    try:
        run_chain_and_compare(case, energy_sample=[0, 4, 7])
    finally:
        case.close()


# ------------------------------------------------------------------------------------------
# degenerate and edge cases
# ------------------------------------------------------------------------------------------
@pytest.fixture(scope="module")
def small_case():
    case = Case(synth.tiny_config(mesh=(2, 2, 1), m=6, n=4, nchol=10, nw=4, seed=5))
    yield case
    case.close()


def test_trial_walker_unit_overlap(small_case):
    case = small_case
    A = orc.supercell_trial(case.pb.psi_t)
    phi_d = _to_dev(np.stack([A, A]))
    theta_d, ld_d, info_d = case.ctx.green(phi_d)
    ld = ld_d.cpu().numpy()
    assert np.max(np.abs(ld)) < 1e-12                      # det = 1
    assert relerr(theta_d[0].cpu().numpy(), A.T) < 1e-12   # Theta = A^T
    e = case.ctx.local_energy(theta_d).cpu().numpy()
    assert np.max(np.abs(e.imag)) < 1e-12 * np.max(np.abs(e.real))
    assert e[0, 1].real > 0 and e[0, 2].real < 0
    vb = case.ctx.force_bias(theta_d).cpu().numpy()
    assert abs(e[0, 1] - 0.5 * np.sum(np.abs(vb[0]) ** 2)) < 1e-12 * abs(e[0, 1])


def test_block_diagonal_walker_momentum_conservation(small_case):
    case, cfg = small_case, small_case.cfg
    rng = np.random.default_rng(3)
    phi = np.zeros((1, cfg.M, cfg.N), dtype=complex)
    for k in range(cfg.nk):
        phi[0, k * cfg.m:(k + 1) * cfg.m, k * cfg.n:(k + 1) * cfg.n] = \
            rng.standard_normal((cfg.m, cfg.n)) + 1j * rng.standard_normal((cfg.m, cfg.n))
    theta_d, ld_d, _ = case.ctx.green(_to_dev(phi))
    vb = case.ctx.force_bias(theta_d).cpu().numpy()[0]
    assert np.max(np.abs(vb[1:])) < 1e-12 * np.max(np.abs(vb[0]))
    # det O = prod_k det(A_k^dagger phi_k)
    tot = 0
    for k in range(cfg.nk):
        s, la = np.linalg.slogdet(np.conj(case.pb.psi_t[k]).T @ phi[0, k * cfg.m:(k + 1) * cfg.m, k * cfg.n:(k + 1) * cfg.n])
        tot += la + 1j * np.angle(s)
    ld = ld_d.cpu().numpy()[0]
    assert abs(ld.real - tot.real) < 1e-10 and phase_diff(ld.imag, tot.imag) < 1e-10


@pytest.mark.parametrize("kw", [dict(mesh=(2, 3, 1), m=5, n=3, nchol=7), dict(mesh=(1, 2, 2), m=6, n=5, nchol=18)],
                         ids=["2x3x1_m5_n3_c7", "1x2x2_m6_n5_c18"])
def test_a0_half_rotation_probed_through_the_abi(kw):
    """a0 located directly instead of inferred downstream: a ONE-HOT Theta with its 1 at row (k,a), column (k',r) makes
    afqmc_force_bias return 2*Lh[Q][k][a][:,r] for the single Q with k-Q = k' and zero for every other Q (Eq. 47 is
    linear in Theta), and afqmc_local_energy return E1 = 2*ht[k][a][r] iff k' = k (Eq. 49 line 1).  Every element of the
    library's packed half-rotated tensors is thus read back and compared with orc.half_rotate on a ragged shape."""
    cfg = synth.tiny_config(seed=23, nw=1, **kw)
    nw = cfg.N * cfg.M
    pb = synth.make_problem(cfg, nw=1)
    from paper_2003_09468_b200 import binding
    ctx = binding.from_problem(pb, max_walkers=nw)
    try:
        Lh, ht = orc.half_rotate(pb.L, pb.psi_t, pb.h1)
        kminus, _ = orc.k_tables(cfg.mesh)
        theta = np.zeros((nw, cfg.N, cfg.M), dtype=complex)
        theta.reshape(nw, nw)[np.arange(nw), np.arange(nw)] = 1.0
        theta_d = _to_dev(theta)
        vb = ctx.force_bias(theta_d).cpu().numpy()
        e = ctx.local_energy(theta_d).cpu().numpy()
        expect_vb = np.zeros((nw, cfg.nk, cfg.nchol), dtype=complex)
        expect_e1 = np.zeros(nw, dtype=complex)
        for row in range(cfg.N):
            k, a = divmod(row, cfg.n)
            for col in range(cfg.M):
                kp, r = divmod(col, cfg.m)
                w = row * cfg.M + col
                Q = [q for q in range(cfg.nk) if kminus[k, q] == kp]
                assert len(Q) == 1
                expect_vb[w, Q[0]] = 2.0 * Lh[Q[0], k, a, :, r]
                if kp == k:
                    expect_e1[w] = 2.0 * ht[k, a, r]
        scale = np.max(np.abs(expect_vb))
        assert np.max(np.abs(vb - expect_vb)) < 1e-13 * scale
        assert np.max(np.abs(e[:, 0] - expect_e1)) < 1e-13 * np.max(np.abs(expect_e1))
    finally:
        ctx.close()


# walker counts that reach every split of the force-bias kernel (force_bias.cu): one n-tile per warp (nw <= 8), two (16),
# warp pairs sharing the A ring (17..32), four warps per A ring with idle warps in the last walker super-group (40, 70), and
# Cholesky counts that give 1..5 m-tiles per warp incl. a ragged last m-group (nchol = 100: 13 tiles = 5 + 5 + 3)
@pytest.mark.parametrize("kw", [dict(mesh=(2, 2, 1), m=6, n=2, nchol=5, nw=7), dict(mesh=(3, 1, 1), m=7, n=3, nchol=16, nw=16),
                                dict(mesh=(2, 1, 2), m=9, n=2, nchol=24, nw=21), dict(mesh=(1, 3, 1), m=10, n=3, nchol=29, nw=32),
                                dict(mesh=(2, 2, 1), m=5, n=2, nchol=100, nw=40), dict(mesh=(1, 1, 2), m=26, n=4, nchol=41, nw=70)],
                         ids=lambda k: "c%d_w%d" % (k["nchol"], k["nw"]))
def test_force_bias_tile_and_walker_splits(kw):
    """afqmc_force_bias on random (not Green-derived) Theta against orc.force_bias on every walker, and the same numbers
    from afqmc_step's fused path (Green's epilogue writes the B fragments) through the step's Coulomb energy."""
    from paper_2003_09468_b200 import binding
    cfg = synth.tiny_config(seed=31, **kw)
    pb = synth.make_problem(cfg)
    ctx = binding.from_problem(pb)
    try:
        Lh, _ = orc.half_rotate(pb.L, pb.psi_t, pb.h1)
        rng = np.random.default_rng(5)
        theta = rng.standard_normal((cfg.nw, cfg.N, cfg.M)) + 1j * rng.standard_normal((cfg.nw, cfg.N, cfg.M))
        vb = ctx.force_bias(_to_dev(theta)).cpu().numpy()
        for w in range(cfg.nw):
            vb_o = orc.force_bias(cfg.mesh, Lh, theta[w])
            assert relerr(vb[w], vb_o) < 1e-12, (w, relerr(vb[w], vb_o))
        # fewer walkers than the context was made for: the fragment workspace keeps finite leftovers of the larger batch
        nsub = max(1, cfg.nw // 3)
        vb_s = ctx.force_bias(_to_dev(theta[:nsub])).cpu().numpy()
        assert relerr(vb_s, vb[:nsub]) < 1e-13       # (another walker count cuts the K range elsewhere: not bitwise)
        # fused path: the Coulomb energy of afqmc_step is 1/2 sum v[Q] v[-Q] of the force bias of the propagated walkers
        phi_d, x_d = _to_dev(pb.phi), _to_dev(pb.x)
        e, _, info = ctx.step(phi_d, x_d, cfg.dtau, cfg.order)
        assert int(info.abs().sum()) == 0
        th2, _, _ = ctx.green(phi_d)                   # phi_d now holds the propagated walkers
        vb2 = ctx.force_bias(th2).cpu().numpy()         # unfused: the re-layout kernel
        _, kneg = orc.k_tables(cfg.mesh)
        ec = 0.5 * np.einsum("wqg,wqg->w", vb2, vb2[:, kneg, :])
        assert relerr(e.cpu().numpy()[:, 1], ec) < 1e-11
    finally:
        ctx.close()


def test_singular_overlap_reports_info(small_case):
    case = small_case
    phi = case.pb.phi[:2].copy()
    phi[1][:, 3] = 0.0                       # zero column -> O has a zero column
    _, info_d = case.ctx.overlap(_to_dev(phi))
    info = info_d.cpu().numpy()
    assert info[0] == 0 and info[1] > 0


def test_gauge_invariance_on_gpu(small_case):
    case, cfg = small_case, small_case.cfg
    rng = np.random.default_rng(4)
    R = rng.standard_normal((cfg.N, cfg.N)) + 1j * rng.standard_normal((cfg.N, cfg.N))
    phi = np.stack([case.pb.phi[0], case.pb.phi[0] @ R])
    theta_d, _, _ = case.ctx.green(_to_dev(phi))
    th = theta_d.cpu().numpy()
    assert relerr(th[1], th[0]) < 1e-9
    e = case.ctx.local_energy(theta_d).cpu().numpy()
    assert relerr(e[1], e[0]) < 1e-9


def test_argument_errors(small_case):
    from paper_2003_09468_b200 import binding
    case = small_case
    lib = binding.lib()
    phi_d = _to_dev(case.pb.phi)
    # nw = 0 is a no-op
    assert lib.afqmc_green(case.ctx._h, phi_d.data_ptr(), 0, phi_d.data_ptr(), None, None, None) == 0
    # nw > max_walkers, null pointers, bad order
    assert lib.afqmc_green(case.ctx._h, phi_d.data_ptr(), case.nw + 1, phi_d.data_ptr(), None, None, None) == 1
    assert lib.afqmc_green(case.ctx._h, None, 1, phi_d.data_ptr(), None, None, None) == 1
    assert lib.afqmc_propagate(case.ctx._h, phi_d.data_ptr(), 0.005, -1, phi_d.data_ptr(), 1, None) == 1
    assert lib.afqmc_propagate(case.ctx._h, phi_d.data_ptr(), 0.005, 33, phi_d.data_ptr(), 1, None) == 1
    import ctypes
    h = ctypes.c_void_p(0)
    d = binding.Dims((ctypes.c_int * 3)(2, 2, 1), 6, 4, 10, 0, 0, 4, 0)    # open shell without a spin-down orbital count
    assert lib.afqmc_create(ctypes.byref(h), ctypes.byref(d), phi_d.data_ptr(), phi_d.data_ptr(), phi_d.data_ptr(), None) == 1
    d = binding.Dims((ctypes.c_int * 3)(2, 2, 1), 6, 4, 10, 1, 2, 4, 0)    # precision: only 0 (complex128) and 1 (complex64) exist
    assert lib.afqmc_create(ctypes.byref(h), ctypes.byref(d), phi_d.data_ptr(), phi_d.data_ptr(), phi_d.data_ptr(), None) == 2
    d = binding.Dims((ctypes.c_int * 3)(2, 2, 1), 6, 7, 10, 1, 0, 4, 0)    # n > m
    assert lib.afqmc_create(ctypes.byref(h), ctypes.byref(d), phi_d.data_ptr(), phi_d.data_ptr(), phi_d.data_ptr(), None) == 1


def test_binding_rejects_wrong_shapes_dtypes_and_devices(small_case):
    """The binding is marshalling only, but it must not hand a mis-shaped tensor to the kernels as a raw pointer."""
    case, cfg = small_case, small_case.cfg
    phi_d = _to_dev(case.pb.phi)
    with pytest.raises(ValueError):
        case.ctx.green(phi_d[:, :-1].contiguous())                       # wrong trailing dimension
    with pytest.raises(ValueError):
        case.ctx.green(torch.from_numpy(case.pb.phi))                    # host tensor
    with pytest.raises(TypeError):
        case.ctx.green(phi_d.to(torch.complex64))                        # wrong dtype
    with pytest.raises(ValueError):
        case.ctx.green(torch.cat([phi_d, phi_d]))                        # more walkers than max_walkers
    theta_d, _, _ = case.ctx.green(phi_d)
    with pytest.raises(ValueError):
        case.ctx.force_bias(theta_d.transpose(1, 2).contiguous())        # [nw][M][N] where [nw][N][M] is expected
    with pytest.raises(ValueError):
        case.ctx.vhs(_to_dev(case.pb.x)[:2], case.ctx.force_bias(theta_d), cfg.dtau)   # batch sizes disagree
    with pytest.raises(ValueError):
        case.ctx.step_host(phi_d, torch.from_numpy(case.pb.x), cfg.dtau, cfg.order, torch.empty((case.nw, 3), dtype=torch.complex128))


def test_contexts_in_sequence_and_side_by_side_share_no_state():
    """include/afqmc.h: 'no global state'.  Kernel attributes (the dynamic shared-memory opt-in) are remembered per
    context: a context created after another one was destroyed, and two contexts alive at once with different shapes,
    give bit-identical results to a lone context."""
    from paper_2003_09468_b200 import binding
    cfg_a = synth.tiny_config(mesh=(2, 2, 1), m=26, n=4, nchol=24, nw=5, seed=31)      # > 48 KB of staged theta blocks
    cfg_b = synth.tiny_config(mesh=(1, 1, 2), m=14, n=9, nchol=6, nw=2, seed=32)
    pa, pb_ = synth.make_problem(cfg_a), synth.make_problem(cfg_b)

    def run(ctx, pb, cfg):
        phi = _to_dev(pb.phi)
        e, ld, info = ctx.step(phi, _to_dev(pb.x), cfg.dtau, cfg.order)
        return phi.cpu(), e.cpu(), ld.cpu()

    ctx = binding.from_problem(pa)
    ref_a = run(ctx, pa, cfg_a)
    ctx.close()
    ctx = binding.from_problem(pb_)
    ref_b = run(ctx, pb_, cfg_b)
    ctx.close()
    ca, cb = binding.from_problem(pa), binding.from_problem(pb_)
    try:
        for _ in range(2):
            got_b = run(cb, pb_, cfg_b)
            got_a = run(ca, pa, cfg_a)
            for r, g in zip(ref_a + ref_b, got_a + got_b):
                assert torch.equal(r, g)
    finally:
        ca.close()
        cb.close()


def test_subbatch_equals_full_batch(small_case):
    """nw < max_walkers: results for the first walkers do not depend on the batch size."""
    case = small_case
    phi_d = _to_dev(case.pb.phi)
    th_all, _, _ = case.ctx.green(phi_d)
    th_3, _, _ = case.ctx.green(phi_d[:3].contiguous())
    assert torch.equal(th_all[:3], th_3)
    e_all = case.ctx.local_energy(th_all)
    e_3 = case.ctx.local_energy(th_3)
    assert torch.equal(e_all[:3], e_3)


def test_green_register_kernel_equals_legacy_kernel(small_case):
    """The register-resident elimination and the shared-memory one agree to rounding (both exact up to pivot order)."""
    case = small_case
    phi_d = _to_dev(case.pb.phi)
    th_new, ld_new, _ = case.ctx.green(phi_d)
    case.ctx.set_option("green_legacy", 1)
    try:
        th_old, ld_old, _ = case.ctx.green(phi_d)
    finally:
        case.ctx.set_option("green_legacy", 0)
    assert relerr(th_new.cpu().numpy(), th_old.cpu().numpy()) < 1e-12
    assert np.max(np.abs(ld_new.cpu().numpy().real - ld_old.cpu().numpy().real)) < 1e-12
    assert np.max(phase_diff(ld_new.cpu().numpy().imag, ld_old.cpu().numpy().imag)) < 1e-12


@pytest.mark.parametrize("nw", [3, 11, 37])
def test_vhs_without_the_pair_identity_falls_back_to_all_blocks(nw):
    """vhs.cu stores one L block per (Q,-Q) pair only if afqmc_create finds the identity of PAPER.md:216 in the caller's
    L; an L that violates it must still give the exact contraction of Eq. 48 (all blocks stored, no pairing).  Several
    batch sizes exercise the 1-, 2- and 4-tile kernels and more than one walker group."""
    from paper_2003_09468_b200 import binding
    cfg = synth.tiny_config(mesh=(2, 3, 1), m=5, n=3, nchol=7, nw=nw, seed=17)
    pb = synth.make_problem(cfg)
    rng = np.random.default_rng(99)
    for Lcase, paired in ((pb.L, True), (pb.L + 0.3 * (rng.standard_normal(pb.L.shape) + 1j * rng.standard_normal(pb.L.shape)), False)):
        pb2 = synth.Problem(cfg, pb.h1, pb.psi_t, np.ascontiguousarray(Lcase), pb.phi, pb.x)
        ctx = binding.from_problem(pb2)
        try:
            vb = rng.standard_normal((nw, cfg.nk, cfg.nchol)) + 1j * rng.standard_normal((nw, cfg.nk, cfg.nchol))
            V = ctx.vhs(_to_dev(pb.x), _to_dev(vb), cfg.dtau).cpu().numpy()
            for w in range(nw):
                V_o = orc.vhs(cfg.mesh, pb2.L, orc.assemble_fields(cfg.mesh, pb.x[w], vb[w], cfg.dtau))
                assert relerr(V[w], V_o) < RTOL, (paired, w, relerr(V[w], V_o))
        finally:
            ctx.close()


@pytest.mark.parametrize("kw", [dict(mesh=(2, 2, 1), m=6, n=4, nchol=10, nw=4), dict(mesh=(2, 3, 1), m=5, n=3, nchol=7, nw=5),
                                dict(mesh=(1, 2, 2), m=9, n=1, nchol=5, nw=2), dict(mesh=(3, 1, 1), m=26, n=4, nchol=18, nw=7),
                                dict(mesh=(2, 2, 1), m=9, n=6, nchol=11, nw=5), dict(mesh=(1, 1, 2), m=14, n=9, nchol=6, nw=2)],
                         ids=["n4", "n3_odd", "n1_two_walkers", "m26_seven_walkers", "n6_two_groups", "n9_three_groups"])
def test_exchange_3m_and_4m_kernels_against_the_oracle(kw):
    """All exchange kernels (exchange3m.cu: register-B and generic 3M kernels; energy.cu: 4M, option exchange_3m=0) on the
    same theta, each against the oracle, and against each other."""
    case = Case(synth.tiny_config(seed=13, **kw))
    try:
        theta_d, _, _ = case.ctx.green(_to_dev(case.pb.phi))
        theta = theta_d.cpu().numpy()
        e_o = np.array([orc.local_energy(case.cfg.mesh, case.Lh, case.ht, theta[w]) for w in range(case.nw)])
        res = {}
        # "3m" is the default kernel of the shape (register-B persistent kernel for m <= 28, else the generic one); the other
        # entries force the generic kernel in its variants (smem B fragments, 1 or 2 warp pairs, 2 or 3 k-steps of prefetch,
        # 1/2/4 n-tiles per warp), the two-walker register-B kernel, and the 4M kernel
        for name, opts in (("3m", {}), ("4m", {"exchange_3m": 0}), ("3m_generic", {"exchange_regb": 0}),
                           ("3m_generic_depth2", {"exchange_regb": 0, "exchange_depth": 2}),
                           ("3m_generic_4warps", {"exchange_warps": 4}), ("3m_generic_np4", {"exchange_np": 4}),
                           ("3m_generic_np1_4warps", {"exchange_regb": 0, "exchange_np": 1, "exchange_warps": 4}),
                           ("3m_two_walkers_per_cta", {"exchange_np": 1}),
                           ("3m_register_prefetch_blocking_handover", {"exchange_regb": 2}),
                           ("3m_register_prefetch_two_walkers", {"exchange_regb": 2, "exchange_np": 1})):
            for k, v in opts.items():
                case.ctx.set_option(k, v)
            res[name] = case.ctx.local_energy(theta_d).cpu().numpy()
            for k in ("exchange_depth", "exchange_warps", "exchange_np"):
                case.ctx.set_option(k, 0)
            case.ctx.set_option("exchange_3m", 1)
            case.ctx.set_option("exchange_regb", 1)
        for name, e in res.items():
            for w in range(case.nw):
                assert np.max(np.abs(e[w] - e_o[w]) / np.abs(e_o[w])) < RTOL, (name, w, e[w], e_o[w])
        assert relerr(res["3m"], res["4m"]) < 1e-12
    finally:
        case.close()


@pytest.mark.parametrize("kw", [dict(mesh=(2, 2, 1), m=6, n=4, nchol=10, nw=4), dict(mesh=(2, 3, 1), m=5, n=3, nchol=7, nw=5),
                                dict(mesh=(1, 2, 2), m=9, n=1, nchol=5, nw=2), dict(mesh=(3, 1, 1), m=26, n=4, nchol=18, nw=7),
                                # the tcgen05 kernel's pipeline: two and three row tiles (the tiles alternate between two pairs of
                                # issuing threads and two accumulator buffers), two walker groups of 16 with one walker in the second,
                                # K-blocks with one k-step left over, three and four K-blocks, 8-walker images
                                dict(mesh=(2, 1, 1), m=17, n=4, nchol=40, nw=17), dict(mesh=(1, 2, 1), m=33, n=2, nchol=70, nw=9),
                                dict(mesh=(1, 1, 2), m=50, n=4, nchol=33, nw=3)],
                         ids=["n4", "n3_odd", "n1_two_walkers", "m26_seven_walkers", "two_tiles_17_walkers", "three_tiles_three_kblocks",
                              "four_kblocks"])
def test_mixed_precision_exchange_against_the_oracle(kw):
    """Option exchange_precision, the analogue of the paper's single-precision mode and of the north_star's
    optional complex64 path (tolerance 1e-4), on BOTH kernels: the tcgen05 / TMEM one (exchange_tc.cu, default) and the
    mma.sync one (exchange_tf32.cu, option exchange_tc = 0).  Mode 1 (3xTF32 split) is held to 1e-5 relative on EX against
    the FP64 oracle, mode 2 (operands rounded once to TF32) only to 1e-2 (it is documented as outside the 1e-4 tolerance).
    E1 and EC must not change at all."""
    case = Case(synth.tiny_config(seed=19, **kw))
    try:
        theta_d, _, _ = case.ctx.green(_to_dev(case.pb.phi))
        theta = theta_d.cpu().numpy()
        e_o = np.array([orc.local_energy(case.cfg.mesh, case.Lh, case.ht, theta[w]) for w in range(case.nw)])
        e64 = case.ctx.local_energy(theta_d).cpu().numpy()
        for tc in (1, 0):
            for mode, tol in ((1, 1e-5), (2, 1e-2)):
                case.ctx.set_option("exchange_tc", tc)
                case.ctx.set_option("exchange_precision", mode)
                try:
                    e = case.ctx.local_energy(theta_d).cpu().numpy()
                    e_again = case.ctx.local_energy(theta_d).cpu().numpy()
                finally:
                    case.ctx.set_option("exchange_precision", 0)
                    case.ctx.set_option("exchange_tc", 1)
                assert np.array_equal(e, e_again)                      # no atomics, fixed summation order
                assert np.array_equal(e[:, :2], e64[:, :2])
                for w in range(case.nw):
                    assert abs(e[w, 2] - e_o[w, 2]) / abs(e_o[w, 2]) < tol, (tc, mode, w, e[w, 2], e_o[w, 2])
    finally:
        case.close()


def test_mixed_precision_exchange_is_unsupported_for_more_than_four_orbitals():
    from paper_2003_09468_b200 import binding
    case = Case(synth.tiny_config(mesh=(1, 1, 1), m=7, n=5, nchol=9, nw=1, seed=3))
    try:
        with pytest.raises(binding.AfqmcError) as e:
            case.ctx.set_option("exchange_precision", 1)
        assert e.value.code == 2
    finally:
        case.close()


def test_mixed_precision_exchange_c3_full_size():
    """C3 at full size: 3xTF32 (tcgen05 kernel, and the mma.sync kernel) against the FP64 kernel on every walker (the FP64
    kernel is checked against the oracle in test_config_C3_headline_all_walkers_energy_sampled), and against the oracle on
    one walker."""
    case = Case(synth.CONFIGS["C3"])
    try:
        theta_d, _, _ = case.ctx.green(_to_dev(case.pb.phi))
        e64 = case.ctx.local_energy(theta_d).cpu().numpy()
        case.ctx.set_option("exchange_precision", 1)
        e = case.ctx.local_energy(theta_d).cpu().numpy()
        case.ctx.set_option("exchange_tc", 0)
        e_legacy = case.ctx.local_energy(theta_d).cpu().numpy()
        case.ctx.set_option("exchange_tc", 1)
        case.ctx.set_option("exchange_precision", 0)
        assert np.max(np.abs(e[:, 2] - e64[:, 2]) / np.abs(e64[:, 2])) < 1e-5
        assert np.max(np.abs(e_legacy[:, 2] - e64[:, 2]) / np.abs(e64[:, 2])) < 1e-5
        e_o = orc.local_energy(case.cfg.mesh, case.Lh, case.ht, theta_d[5].cpu().numpy())
        assert abs(e[5, 2] - e_o[2]) / abs(e_o[2]) < 1e-5
    finally:
        case.close()


@pytest.mark.parametrize("mesh,n", [((4, 4, 3), 6), ((4, 3, 3), 7), ((5, 5, 1), 5)], ids=["N288_legacy", "N252_cluster8", "N125_cluster2"])
def test_green_large_N(mesh, n):
    """Overlap sizes that select the cluster kernels (N <= 128: 2 CTAs, N <= 256: 8 CTAs) and the legacy path (N > 256)."""
    cfg = synth.tiny_config(mesh=mesh, m=n + 2, n=n, nchol=2, nw=3, seed=11)
    case = Case(cfg)
    try:
        theta_d, ld_d, info_d = case.ctx.green(_to_dev(case.pb.phi))
        assert np.all(info_d.cpu().numpy() == 0)
        theta, ld = theta_d.cpu().numpy(), ld_d.cpu().numpy()
        for w in range(case.nw):
            th_o, ld_o, _ = orc.green(case.pb.psi_t, case.pb.phi[w])
            assert relerr(theta[w], th_o) < RTOL
            assert abs(ld[w].real - ld_o.real) < RTOL * max(1.0, abs(ld_o.real))
            assert phase_diff(ld[w].imag, ld_o.imag) < 1e-9
    finally:
        case.close()


def test_gpu_step_against_the_stored_oracle_fixture():
    """The GPU step on the tiny seeded system of tests/golden/tiny_step.txt (written by the oracle alone) reproduces the
    stored values: a parity check that does not execute the oracle at test time."""
    import importlib.util
    here = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
    spec = importlib.util.spec_from_file_location("make_golden", os.path.join(here, "make_golden.py"))
    mg = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mg)
    stored = {}
    for line in open(os.path.join(here, "tiny_step.txt")):
        if line.startswith("#") or not line.strip():
            continue
        name, re_, im_ = line.split()
        stored[name] = complex(float(re_), float(im_))
    case = Case(synth.tiny_config(**mg.CFG))
    try:
        cfg, pb, ctx = case.cfg, case.pb, case.ctx
        phi_d, x_d = _to_dev(pb.phi), _to_dev(pb.x)
        theta_d, ld0_d, _ = ctx.green(phi_d)
        vb = ctx.force_bias(theta_d).cpu().numpy()
        energy, logdet, info = ctx.step(phi_d, x_d, cfg.dtau, cfg.order)
        e, ld1, ld0, phi_new = energy.cpu().numpy(), logdet.cpu().numpy(), ld0_d.cpu().numpy(), phi_d.cpu().numpy()
        for w in range(cfg.nw):
            got = {"vbias_sum[%d]" % w: complex(np.sum(vb[w])), "E1[%d]" % w: e[w, 0], "EC[%d]" % w: e[w, 1],
                   "EX[%d]" % w: e[w, 2], "phi_new_sum[%d]" % w: complex(np.sum(phi_new[w]))}
            for name, z in got.items():
                assert abs(z - stored[name]) <= 1e-9 * max(1.0, abs(stored[name])), (name, z, stored[name])
            for name, z in (("logdet0[%d]" % w, ld0[w]), ("logdet1[%d]" % w, ld1[w])):
                assert abs(z.real - stored[name].real) < 1e-9 and phase_diff(z.imag, stored[name].imag) < 1e-9, name
    finally:
        case.close()
