"""Pins of the oracle's AFQMC-block functions against things other than
themselves: the real-field (Hermitian) restatement of the Hubbard-Stratonovich transformation, a Gauss-Hermite
quadrature of Eq. 12/15-16, Wick's theorem, scipy's expm, numpy's QR, brute-force loops.  CPU only."""
import numpy as np
import pytest
import scipy.linalg

from oracle import afqmc_oracle as orc
from paper_2003_09468_b200 import synth


def relerr(a, b):
    a = np.asarray(a)
    b = np.asarray(b)
    return float(np.max(np.abs(a - b)) / max(np.max(np.abs(b)), 1e-300))


@pytest.fixture(scope="module", params=[(2, 3, 1), (2, 2, 1), (3, 1, 1)])
def tiny(request):
    cfg = synth.tiny_config(mesh=request.param, m=3, n=2, nchol=3, nw=2, seed=5)
    pb = synth.make_problem(cfg)
    Lh, ht = orc.half_rotate(pb.L, pb.psi_t, pb.h1)
    A = orc.supercell_trial(pb.psi_t)
    Lsc = orc.supercell_L(cfg.mesh, pb.L)
    vops = orc.hermitian_hs_operators(cfg.mesh, Lsc, cfg.nchol)
    B1 = orc.onebody_half_propagator(pb.h1, cfg.dtau)
    return dict(cfg=cfg, pb=pb, Lh=Lh, ht=ht, A=A, Lsc=Lsc, vops=vops, B1=B1)


# ---------------------------------------------------------------- real-field basis (Eq. 8-11)
def test_hs_operators_are_hermitian_and_square_to_h2prime(tiny):
    vops, Lsc = tiny["vops"], tiny["Lsc"]
    for v in vops:
        assert relerr(v, np.conj(v.T)) < 1e-14
    # (1/2) sum_j v_j^2 == (1/2) sum_Gamma L_Gamma L_Gamma^dagger  (one-body part of H2', Eq. 8 with v_hat = i v)
    lhs = 0.5 * np.einsum('jpr,jrs->ps', vops, vops)
    rhs = 0.5 * np.einsum('prg,srg->ps', Lsc, np.conj(Lsc))
    assert relerr(lhs, rhs) < 1e-13
    # and the two-body part: sum_j v_j (x) v_j == sum_Gamma L_Gamma (x) L_Gamma^dagger  (Eq. 20)
    lhs4 = np.einsum('jpr,jqs->pqrs', vops, vops)
    rhs4 = orc.eri_from_L(Lsc)
    assert relerr(lhs4, rhs4) < 1e-13


def test_real_fields_times_hermitian_ops_equal_complex_fields_times_L(tiny):
    cfg, pb, vops, Lsc = tiny["cfg"], tiny["pb"], tiny["vops"], tiny["Lsc"]
    x = pb.x[0]
    xi = orc.assemble_fields(cfg.mesh, x, None, cfg.dtau)            # = -i z
    V = orc.dense_vhs(Lsc, xi.reshape(-1))                           # = -i sum z L
    assert relerr(np.einsum('j,jpr->pr', x.reshape(-1), vops), 1j * V) < 1e-13


# ---------------------------------------------------------------- one-body half steps (Eq. 7, 13)
def test_onebody_half_propagator_vs_scipy_expm(tiny):
    pb, cfg, B1 = tiny["pb"], tiny["cfg"], tiny["B1"]
    for k in range(cfg.nk):
        assert relerr(B1[k], scipy.linalg.expm(-0.5 * cfg.dtau * pb.h1[k])) < 1e-13
        assert relerr(B1[k] @ B1[k], scipy.linalg.expm(-cfg.dtau * pb.h1[k])) < 1e-13
        assert relerr(B1[k], np.conj(B1[k].T)) < 1e-14


def test_apply_onebody_is_the_block_diagonal_product(tiny):
    pb, B1 = tiny["pb"], tiny["B1"]
    dense = scipy.linalg.block_diag(*B1)
    assert relerr(orc.apply_onebody(B1, pb.phi[0]), dense @ pb.phi[0]) < 1e-14


# ---------------------------------------------------------------- hybrid weight (Eq. 15-19)
def test_hybrid_step_matches_real_basis_definition(tiny):
    cfg, pb = tiny["cfg"], tiny["pb"]
    nonzero = 0
    for w in range(cfg.nw):
        for dtau in (1e-4, 1e-3, cfg.dtau, 0.05):
            B1 = orc.onebody_half_propagator(pb.h1, dtau)
            phi_p, logI, dth_p, fac_p, info = orc.hybrid_step(cfg.mesh, pb.L, tiny["Lh"], pb.psi_t, B1, pb.phi[w],
                                                              pb.x[w], dtau, cfg.order)
            phi_d, I_d, dth_d, fac_d = orc.dense_hybrid_step(tiny["A"], tiny["vops"], orc.supercell_h1(B1), pb.phi[w],
                                                             pb.x[w].reshape(-1), dtau, cfg.order)
            assert info == 0
            assert relerr(phi_p, phi_d) < 1e-12
            assert abs(np.exp(logI) - I_d) / abs(I_d) < 1e-11
            assert abs(dth_p - dth_d) < 1e-11
            assert abs(fac_p - fac_d) <= 1e-11 * max(fac_d, 1.0)
            nonzero += fac_d > 0
    assert nonzero >= 3           # the comparison is not vacuous (large steps on these inputs flip the phase)


def test_phaseless_projection_kills_and_wraps():
    mesh = (1, 1, 1)
    x = np.zeros((1, 2))
    vb = np.zeros((1, 2), dtype=complex)
    # phase change of the overlap ratio: 2 * 0.9 = 1.8 rad > pi/2 -> killed
    _, dth, fac = orc.hybrid_weight(mesh, x, vb, 0.01, 0.0 + 0.0j, 0.3 + 0.9j)
    assert abs(dth - 1.8) < 1e-15 and fac == 0.0
    # 2 * 3.0 = 6.0 rad wraps to 6 - 2 pi = -0.283...: survives with |I| cos
    logI, dth, fac = orc.hybrid_weight(mesh, x, vb, 0.01, 0.0 + 0.0j, 0.3 + 3.0j)
    assert abs(dth - (6.0 - 2 * np.pi)) < 1e-14
    assert abs(fac - np.exp(0.6) * np.cos(6.0 - 2 * np.pi)) < 1e-13
    # no fields, no force bias, same determinant: factor 1
    _, dth, fac = orc.hybrid_weight(mesh, x, vb, 0.01, 1.0 + 0.5j, 1.0 + 0.5j)
    assert dth == 0.0 and fac == 1.0


def test_importance_function_by_quadrature():
    """Eq. 12 vs Eq. 15-16: int p(x) I(x, xbar) dx = <Psi_T| int p(x) B(x) dx |phi> / <Psi_T|phi> for EVERY shift
    xbar (contour shift of an entire integrand), and int p(x) B(x) dx = exp(-dtau/2 sum_j v_j^2 ... ) so that
    (1 - <I>)/dtau -> <H2'>_mixed (Wick) as dtau -> 0.  Gauss-Hermite quadrature over 2 real fields."""
    cfg = synth.tiny_config(mesh=(2, 1, 1), m=3, n=1, nchol=1, nw=1, seed=11)
    pb = synth.make_problem(cfg)
    A = orc.supercell_trial(pb.psi_t)
    Lsc = orc.supercell_L(cfg.mesh, pb.L)
    vops = orc.hermitian_hs_operators(cfg.mesh, Lsc, cfg.nchol)
    assert vops.shape[0] == 2
    B1 = np.eye(cfg.M, dtype=complex)                            # isolate the two-body propagator
    phi = pb.phi[0]
    G = orc.dense_green(A, phi)
    h2p = orc.dense_h2prime_mixed(vops, G)
    nodes, wts = np.polynomial.hermite_e.hermegauss(24)           # weight exp(-x^2/2)
    wts = wts / np.sqrt(2 * np.pi)
    slopes = []
    for dtau in (1e-2, 1e-3):
        avg = {}
        for name, xbar in (("force_bias", None), ("zero", np.zeros(2)), ("other", np.array([0.3 - 0.2j, -0.1 + 0.4j]))):
            tot = 0.0 + 0.0j
            for i, x0 in enumerate(nodes):
                for j, x1 in enumerate(nodes):
                    _, I, _, _ = orc.dense_hybrid_step(A, vops, B1, phi, np.array([x0, x1]), dtau, 40, xbar_override=xbar)
                    tot += wts[i] * wts[j] * I
            avg[name] = tot
        assert abs(avg["force_bias"] - avg["zero"]) < 1e-11
        assert abs(avg["other"] - avg["zero"]) < 1e-11
        slopes.append((1.0 - avg["zero"]) / dtau)
    # first-order agreement with the Wick value, improving linearly with dtau
    e1, e2 = abs(slopes[0] - h2p), abs(slopes[1] - h2p)
    assert e2 < 2e-2 * abs(h2p) + 1e-6
    assert e2 < 0.2 * e1


def test_h2prime_wick_equals_two_body_energy_plus_one_body_part(tiny):
    vops, A, pb, Lsc = tiny["vops"], tiny["A"], tiny["pb"], tiny["Lsc"]
    G = orc.dense_green(A, pb.phi[1])
    V = orc.eri_from_L(Lsc)
    e = orc.dense_energy(np.zeros_like(G), V, G)                  # (0, EC, EX), pinned by brute force elsewhere
    onebody = 2.0 * 0.5 * np.einsum('jpr,jrs,ps->', vops, vops, G)
    assert abs(orc.dense_h2prime_mixed(vops, G) - (e[1] + e[2] + onebody)) < 1e-11 * abs(e[1])


# ---------------------------------------------------------------- orthogonalisation
def test_orthogonalize_vs_numpy_qr_and_invariants(tiny):
    cfg, pb = tiny["cfg"], tiny["pb"]
    rng = np.random.default_rng(2)
    R0 = rng.standard_normal((cfg.N, cfg.N)) + 1j * rng.standard_normal((cfg.N, cfg.N))
    phi = pb.phi[0] @ R0                                           # a non-orthonormal walker
    q, ldr = orc.orthogonalize(phi)
    assert relerr(np.conj(q.T) @ q, np.eye(cfg.N)) < 1e-13
    qn, rn = np.linalg.qr(phi)                                     # library routine; fix the phase convention
    ph = np.diag(rn) / np.abs(np.diag(rn))
    assert relerr(q, qn * ph) < 1e-12
    r = np.conj(q.T) @ phi
    assert relerr(np.tril(r, -1), np.zeros_like(r)) < 1e-12 or np.max(np.abs(np.tril(r, -1))) < 1e-12
    assert np.all(np.diag(r).real > 0) and np.max(np.abs(np.diag(r).imag)) < 1e-12
    assert abs(ldr - np.log(abs(np.linalg.det(R0)))) < 1e-11 * max(1.0, abs(ldr))   # phi[0] is orthonormal: det R = |det R0|
    # idempotent
    q2, ldr2 = orc.orthogonalize(q)
    assert relerr(q2, q) < 1e-13 and abs(ldr2) < 1e-13
    # the determinant changes by det R only; Theta and the energy do not change (gauge invariance)
    th0, ld0, _ = orc.green(pb.psi_t, phi)
    th1, ld1, _ = orc.green(pb.psi_t, q)
    assert relerr(th1, th0) < 1e-11
    assert abs((ld0 - ld1).real - ldr) < 1e-11 * max(1.0, abs(ldr))
    e0 = orc.local_energy(cfg.mesh, tiny["Lh"], tiny["ht"], th0)
    e1 = orc.local_energy(cfg.mesh, tiny["Lh"], tiny["ht"], th1)
    assert relerr(e1, e0) < 1e-10


# ---------------------------------------------------------------- mixed estimator (Eq. 34-35)
def test_mixed_estimator_bruteforce():
    rng = np.random.default_rng(4)
    w = rng.random(5)
    e = rng.standard_normal((5, 3)) + 1j * rng.standard_normal((5, 3))
    num, den = orc.mixed_estimator(w, e)
    for c in range(3):
        assert abs(num[c] - sum(w[i] * e[i, c] for i in range(5))) < 1e-14
    assert abs(den - sum(w)) < 1e-15
    # equal weights: the plain average of the total local energy
    num, den = orc.mixed_estimator(np.ones(5), e)
    assert abs(np.sum(num) / den - np.mean(np.sum(e, axis=1))) < 1e-14


# ---------------------------------------------------------------- block composition
def test_block_is_the_composition_of_its_parts(tiny):
    cfg, pb, Lh, ht, B1 = tiny["cfg"], tiny["pb"], tiny["Lh"], tiny["ht"], tiny["B1"]
    dtau = 1e-3
    B1 = orc.onebody_half_propagator(pb.h1, dtau)
    xs = synth.make_block_fields(cfg, 3)
    w0 = np.array([1.0, 0.7])
    phi_o, w_o, e_o, (num, den), ldr = orc.block(cfg.mesh, pb.L, Lh, ht, pb.psi_t, B1, pb.phi, w0, xs, dtau, cfg.order)
    for w in range(cfg.nw):
        p = pb.phi[w]
        wt = w0[w]
        for s in range(3):
            p, _, _, f, _ = orc.hybrid_step(cfg.mesh, pb.L, Lh, pb.psi_t, B1, p, xs[s, w], dtau, cfg.order)
            wt *= f
        assert abs(wt - w_o[w]) <= 1e-13 * wt
        th, _, _ = orc.green(pb.psi_t, p)
        assert relerr(e_o[w], orc.local_energy(cfg.mesh, Lh, ht, th)) < 1e-12
        q, l = orc.orthogonalize(p)
        assert relerr(phi_o[w], q) < 1e-12 and abs(l - ldr[w]) < 1e-12
        assert relerr(np.conj(phi_o[w].T) @ phi_o[w], np.eye(cfg.N)) < 1e-13
    assert np.all(w_o >= 0) and np.any(w_o > 0)
    assert relerr(num, np.einsum('w,wc->c', w_o, e_o)) < 1e-13 and abs(den - w_o.sum()) < 1e-14


def test_free_projection_limit_is_unitary_and_weight_is_overlap_ratio(tiny):
    """vbias -> 0 limit of Eq. 16: I = overlap ratio; and with B1 = 1 the two-body propagator of real fields
    is unitary as dtau -> 0 (anti-Hermitian exponent)."""
    cfg, pb = tiny["cfg"], tiny["pb"]
    x = pb.x[0]
    vb0 = np.zeros((cfg.nk, cfg.nchol), dtype=complex)
    logI, dth, fac = orc.hybrid_weight(cfg.mesh, x, vb0, 1e-3, 0.2 + 0.1j, 0.25 + 0.3j)
    assert abs(logI - 2 * (0.05 + 0.2j)) < 1e-15
    assert abs(dth - 0.4) < 1e-15 and abs(fac - np.exp(0.1) * np.cos(0.4)) < 1e-14
