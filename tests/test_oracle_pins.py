"""Pins for the CPU oracle (oracle/afqmc_oracle.py) -- CPU only, no CUDA.

Each test pins a part of the oracle to something other than itself: a closed form, an
invariant the mathematics fixes, brute force in explicit Python loops on tiny inputs, a
textbook special case, or a library routine (numpy.linalg) -- chosen so that a dropped term,
wrong sign/index or transposed operand fails at least one of them.  The paper prints no
worked numerical example for this path, so there are no printed values.
"""
import itertools

import numpy as np
import pytest

from oracle import afqmc_oracle as orc
from paper_2003_09468_b200 import synth

TOL = 1e-11


def relerr(a, b):
    a = np.asarray(a)
    b = np.asarray(b)
    den = max(np.max(np.abs(b)), 1e-300)
    return float(np.max(np.abs(a - b)) / den)


@pytest.fixture(scope="module", params=[(2, 3, 1), (2, 2, 2), (3, 1, 2)])
def tiny(request):
    cfg = synth.tiny_config(mesh=request.param, m=3, n=2, nchol=4, nw=2, seed=3)
    pb = synth.make_problem(cfg)
    Lh, ht = orc.half_rotate(pb.L, pb.psi_t, pb.h1)
    A = orc.supercell_trial(pb.psi_t)
    Lsc = orc.supercell_L(cfg.mesh, pb.L)
    H = orc.supercell_h1(pb.h1)
    return dict(cfg=cfg, pb=pb, Lh=Lh, ht=ht, A=A, Lsc=Lsc, H=H)


# ---------------------------------------------------------------- k-point arithmetic
@pytest.mark.parametrize("mesh", [(2, 2, 2), (3, 3, 3), (4, 4, 4), (2, 3, 1), (1, 1, 1)])
def test_kpoint_tables_agree_and_group_laws(mesh):
    kminus_o, neg_o = orc.k_tables(mesh)
    kminus_s, neg_s = synth.kpoint_tables(mesh)      # independent implementation
    assert np.array_equal(kminus_o, kminus_s)
    assert np.array_equal(neg_o, neg_s)
    nk = len(neg_o)
    assert np.array_equal(neg_o[neg_o], np.arange(nk))          # -(-Q) = Q
    assert np.array_equal(kminus_o[:, 0], np.arange(nk))        # k - 0 = k
    for k in range(nk):
        assert sorted(kminus_o[k]) == list(range(nk))           # Q -> k-Q is a bijection
        for Q in range(nk):
            # (k-Q) - (-Q) = k
            assert kminus_o[kminus_o[k, Q], neg_o[Q]] == k
    # explicit coordinates on the 3x3x3 mesh: index (i1*3+i2)*3+i3
    if mesh == (3, 3, 3):
        assert orc.k_index(mesh, (1, 2, 0)) == 15
        assert orc.k_sub(mesh, 0, 15) == orc.k_index(mesh, (2, 1, 0)) == 21
        assert orc.k_neg(mesh, 15) == 21


# ---------------------------------------------------------------- L structure, Eq. 20
def test_supercell_L_momentum_conservation_and_pair_symmetry(tiny):
    cfg, Lsc = tiny["cfg"], tiny["Lsc"]
    nk, m, nchol = cfg.nk, cfg.m, cfg.nchol
    coords = orc.k_coords(cfg.mesh)
    g = np.array(cfg.mesh)
    for Q in range(nk):
        blkQ = Lsc[:, :, Q * nchol:(Q + 1) * nchol]
        for kp in range(nk):
            for kr in range(nk):
                sub = blkQ[kp * m:(kp + 1) * m, kr * m:(kr + 1) * m]
                ok = np.all((np.array(coords[kp]) - np.array(coords[kr]) - np.array(coords[Q])) % g == 0)
                if not ok:
                    assert np.all(sub == 0)          # zero outside k_r = k_p - Q
                else:
                    assert np.any(sub != 0)
        mQ = orc.k_neg(cfg.mesh, Q)
        blkm = Lsc[:, :, mQ * nchol:(mQ + 1) * nchol]
        # L^{-Q}_{rp} = conj(L^{Q}_{pr})
        assert relerr(blkm, np.conj(np.transpose(blkQ, (1, 0, 2)))) < 1e-15


def test_eri_symmetries(tiny):
    V = orc.eri_from_L(tiny["Lsc"])
    # brute-force one element of Eq. 20
    Lsc = tiny["Lsc"]
    p, q, r, s = 1, 4, 2, 3
    ref = sum(Lsc[p, r, g] * np.conj(Lsc[s, q, g]) for g in range(Lsc.shape[2]))
    assert abs(V[p, q, r, s] - ref) < 1e-14
    # v_pqrs = conj(v_rspq)  (Hermiticity) holds for any L
    assert relerr(V, np.conj(np.transpose(V, (2, 3, 0, 1)))) < 1e-14
    # v_pqrs = v_qpsr (electron exchange) needs the (Q,-Q) structure of the generator
    assert relerr(V, np.transpose(V, (1, 0, 3, 2))) < 1e-13


# ---------------------------------------------------------------- LU / determinant / inverse
def _cofactor_det(a):
    n = a.shape[0]
    if n == 1:
        return a[0, 0]
    tot = 0
    for j in range(n):
        minor = np.delete(np.delete(a, 0, axis=0), j, axis=1)
        tot += (-1) ** j * a[0, j] * _cofactor_det(minor)
    return tot


@pytest.mark.parametrize("nn", [1, 2, 3, 5, 6])
def test_lu_det_vs_cofactor_expansion(nn):
    rng = np.random.default_rng(10 + nn)
    a = rng.standard_normal((nn, nn)) + 1j * rng.standard_normal((nn, nn))
    lu, perm, sign, info = orc.lu_factor(a)
    assert info == 0
    ld = orc.lu_logdet(lu, sign)
    det = _cofactor_det(a)
    assert abs(np.exp(ld) - det) < 1e-12 * abs(det)


@pytest.mark.parametrize("nn", [4, 32, 108])
def test_lu_vs_numpy_and_inverse(nn):
    rng = np.random.default_rng(nn)
    a = rng.standard_normal((nn, nn)) + 1j * rng.standard_normal((nn, nn))
    lu, perm, sign, info = orc.lu_factor(a)
    ld = orc.lu_logdet(lu, sign)
    s, la = np.linalg.slogdet(a)
    assert abs(ld.real - la) < 1e-11 * max(1, abs(la))
    assert abs(np.exp(1j * ld.imag) - s) < 1e-11
    # P A = L U
    Lm = np.tril(lu, -1) + np.eye(nn)
    Um = np.triu(lu)
    assert relerr(Lm @ Um, a[perm]) < 1e-12
    inv = orc.lu_inverse(lu, perm)
    assert relerr(a @ inv, np.eye(nn)) < 1e-10
    assert relerr(inv @ a, np.eye(nn)) < 1e-10


def test_lu_singular_reports_info():
    a = np.array([[1, 2, 3], [2, 4, 6], [1, 0, 1]], dtype=complex)
    a[:, 1] = 0
    _, _, _, info = orc.lu_factor(a)
    assert info == 2


def test_det_multiplicative_under_gauge(tiny):
    pb, cfg = tiny["pb"], tiny["cfg"]
    rng = np.random.default_rng(5)
    R = rng.standard_normal((cfg.N, cfg.N)) + 1j * rng.standard_normal((cfg.N, cfg.N))
    _, ld0, _ = orc.green(pb.psi_t, pb.phi[0])
    _, ld1, _ = orc.green(pb.psi_t, pb.phi[0] @ R)
    s, la = np.linalg.slogdet(R)
    assert abs((ld1.real - ld0.real) - la) < 1e-10
    assert abs(np.exp(1j * (ld1.imag - ld0.imag)) - s) < 1e-10


# ---------------------------------------------------------------- overlap / Green
def test_trial_walker_gives_unit_overlap_and_trial_density(tiny):
    pb, A, cfg = tiny["pb"], tiny["A"], tiny["cfg"]
    O = orc.overlap(pb.psi_t, A)
    assert relerr(O, np.eye(cfg.N)) < 1e-14
    th, ld, info = orc.green(pb.psi_t, A)
    assert info == 0 and abs(ld) < 1e-13               # det = 1
    assert relerr(th, A.T) < 1e-13                      # Theta = A^T
    G = np.conj(A) @ th
    assert relerr(G, np.conj(A @ np.conj(A.T))) < 1e-13  # trial density (transposed)


def test_overlap_blocks_equal_dense_product(tiny):
    pb, A = tiny["pb"], tiny["A"]
    assert relerr(orc.overlap(pb.psi_t, pb.phi[1]), orc.dense_overlap(A, pb.phi[1])) < 1e-14
    # brute force for a few entries: O_ij = sum_P conj(A_Pi) Phi_Pj
    phi = pb.phi[1]
    for i, j in [(0, 0), (3, 7), (5, 2)]:
        ref = sum(np.conj(A[P, i]) * phi[P, j] for P in range(A.shape[0]))
        assert abs(orc.overlap(pb.psi_t, phi)[i, j] - ref) < 1e-14


def test_green_invariants(tiny):
    pb, A, cfg = tiny["pb"], tiny["A"], tiny["cfg"]
    for w in range(cfg.nw):
        th, ld, info = orc.green(pb.psi_t, pb.phi[w])
        assert info == 0
        assert relerr(th, orc.dense_theta(A, pb.phi[w])) < 1e-11     # Eq. 30 via numpy inverse
        assert relerr(th @ np.conj(A), np.eye(cfg.N)) < 1e-11         # Theta A^* = 1
        G = np.conj(A) @ th
        assert relerr(G @ G, G) < 1e-11                               # projector
        assert abs(np.trace(G) - cfg.N) < 1e-11
        # Eq. 27 == Eq. 28 transposed
        O = np.conj(A.T) @ pb.phi[w]
        G27 = pb.phi[w] @ np.linalg.inv(O) @ np.conj(A.T)             # indexed [r][p]
        assert relerr(G, G27.T) < 1e-11


def test_block_diagonal_walker_factorises_determinant(tiny):
    pb, cfg = tiny["pb"], tiny["cfg"]
    rng = np.random.default_rng(7)
    nk, m, n = cfg.nk, cfg.m, cfg.n
    phi = np.zeros((cfg.M, cfg.N), dtype=complex)
    prod = 0.0
    for k in range(nk):
        blk = rng.standard_normal((m, n)) + 1j * rng.standard_normal((m, n))
        phi[k * m:(k + 1) * m, k * n:(k + 1) * n] = blk
        s, la = np.linalg.slogdet(np.conj(pb.psi_t[k]).T @ blk)
        prod += la + 1j * np.angle(s)
    _, ld, _ = orc.green(pb.psi_t, phi)
    assert abs(ld.real - prod.real) < 1e-11
    assert abs(np.exp(1j * ld.imag) - np.exp(1j * prod.imag)) < 1e-11


def test_gauge_invariance_of_theta_and_energy(tiny):
    pb, cfg, Lh, ht = tiny["pb"], tiny["cfg"], tiny["Lh"], tiny["ht"]
    rng = np.random.default_rng(9)
    R = rng.standard_normal((cfg.N, cfg.N)) + 1j * rng.standard_normal((cfg.N, cfg.N))
    th0, _, _ = orc.green(pb.psi_t, pb.phi[0])
    th1, _, _ = orc.green(pb.psi_t, pb.phi[0] @ R)
    assert relerr(th1, th0) < 1e-9
    e0 = orc.local_energy(cfg.mesh, Lh, ht, th0)
    e1 = orc.local_energy(cfg.mesh, Lh, ht, th1)
    assert relerr(e1, e0) < 1e-9


# ---------------------------------------------------------------- half rotation
def test_half_rotation_bruteforce(tiny):
    pb, Lh, ht, cfg = tiny["pb"], tiny["Lh"], tiny["ht"], tiny["cfg"]
    rng = np.random.default_rng(0)
    for _ in range(20):
        Q, k = rng.integers(cfg.nk, size=2)
        a, g, r = rng.integers(cfg.n), rng.integers(cfg.nchol), rng.integers(cfg.m)
        ref = sum(np.conj(pb.psi_t[k][p, a]) * pb.L[Q, k, g, p, r] for p in range(cfg.m))
        assert abs(Lh[Q, k, a, g, r] - ref) < 1e-14
    k, a, q = 1, 1, 2
    ref = sum(np.conj(pb.psi_t[k][p, a]) * pb.h1[k][p, q] for p in range(cfg.m))
    assert abs(ht[k, a, q] - ref) < 1e-14
    # dense statement: Lh_sc[(k,a),(k-Q,r),Gamma] = (A^dagger L_sc)
    A, Lsc = tiny["A"], tiny["Lsc"]
    Lh_sc = np.einsum('pa,prg->arg', np.conj(A), Lsc)
    Q, k = 1, 0
    kq = orc.k_sub(cfg.mesh, k, Q)
    n, m, nc = cfg.n, cfg.m, cfg.nchol
    blk = Lh_sc[k * n:(k + 1) * n, kq * m:(kq + 1) * m, Q * nc:(Q + 1) * nc]      # [a][r][g]
    assert relerr(np.transpose(blk, (0, 2, 1)), Lh[Q, k]) < 1e-14


# ---------------------------------------------------------------- force bias
def test_force_bias_matches_definition(tiny):
    pb, cfg, Lh, A, Lsc = tiny["pb"], tiny["cfg"], tiny["Lh"], tiny["A"], tiny["Lsc"]
    for w in range(cfg.nw):
        th, _, _ = orc.green(pb.psi_t, pb.phi[w])
        vb = orc.force_bias(cfg.mesh, Lh, th)
        G = orc.dense_green(A, pb.phi[w])
        ref = orc.dense_vbias(Lsc, G).reshape(cfg.nk, cfg.nchol)
        assert relerr(vb, ref) < TOL
        # brute force one entry of 2 sum_pr L_pr G_pr
        Gam = 1 * cfg.nchol + 2
        bf = 2 * sum(Lsc[p, r, Gam] * G[p, r] for p in range(cfg.M) for r in range(cfg.M))
        assert abs(vb[1, 2] - bf) < 1e-11 * max(1.0, abs(bf))


def test_force_bias_momentum_conservation_and_reality(tiny):
    pb, cfg, Lh, A = tiny["pb"], tiny["cfg"], tiny["Lh"], tiny["A"]
    rng = np.random.default_rng(11)
    nk, m, n = cfg.nk, cfg.m, cfg.n
    phi = np.zeros((cfg.M, cfg.N), dtype=complex)
    for k in range(nk):
        phi[k * m:(k + 1) * m, k * n:(k + 1) * n] = rng.standard_normal((m, n)) + 1j * rng.standard_normal((m, n))
    th, _, _ = orc.green(pb.psi_t, phi)
    vb = orc.force_bias(cfg.mesh, Lh, th)
    assert np.max(np.abs(vb[1:])) < 1e-12 * np.max(np.abs(vb[0]))    # only Q = 0 survives
    thT, _, _ = orc.green(pb.psi_t, A)
    vbT = orc.force_bias(cfg.mesh, Lh, thT)
    assert np.max(np.abs(vbT[0].imag)) < 1e-12 * np.max(np.abs(vbT[0].real))  # Hermitian G, Hermitian L^0


# ---------------------------------------------------------------- vHS and field assembly
def test_vhs_matches_dense_and_is_linear(tiny):
    pb, cfg, Lsc = tiny["pb"], tiny["cfg"], tiny["Lsc"]
    rng = np.random.default_rng(13)
    xi = rng.standard_normal((cfg.nk, cfg.nchol)) + 1j * rng.standard_normal((cfg.nk, cfg.nchol))
    xi2 = rng.standard_normal((cfg.nk, cfg.nchol)) + 1j * rng.standard_normal((cfg.nk, cfg.nchol))
    V = orc.vhs(cfg.mesh, pb.L, xi)
    assert relerr(V, orc.dense_vhs(Lsc, xi.reshape(-1))) < 1e-13
    V2 = orc.vhs(cfg.mesh, pb.L, xi2)
    assert relerr(orc.vhs(cfg.mesh, pb.L, 2 * xi - 1j * xi2), 2 * V - 1j * V2) < 1e-13
    # brute force one entry
    P, R = 4, 7
    bf = sum(Lsc[P, R, g] * xi.reshape(-1)[g] for g in range(Lsc.shape[2]))
    assert abs(V[P, R] - bf) < 1e-13


def test_fields_without_force_bias_give_antihermitian_vhs(tiny):
    pb, cfg = tiny["pb"], tiny["cfg"]
    xi = orc.assemble_fields(cfg.mesh, pb.x[0], None, cfg.dtau)
    V = orc.vhs(cfg.mesh, pb.L, xi)
    assert relerr(V, -np.conj(V.T)) < 1e-13            # vHS = -i * Hermitian
    # z has unit variance per real degree of freedom: sum |z|^2 == sum x^2 exactly
    z = 1j * xi
    assert abs(np.sum(np.abs(z) ** 2) - np.sum(pb.x[0] ** 2)) < 1e-10


def test_field_shift_is_eq17_in_this_basis(tiny):
    """exponent = -sqrt(dtau) vHS must equal  i sqrt(dtau) sum z rho  -  dtau sum_Q vbias[-Q] rho_Q
    (R7): check the shift part against the dense definition."""
    pb, cfg, Lsc, A = tiny["pb"], tiny["cfg"], tiny["Lsc"], tiny["A"]
    G = orc.dense_green(A, pb.phi[0])
    vb = orc.dense_vbias(Lsc, G).reshape(cfg.nk, cfg.nchol)
    xi_full = orc.assemble_fields(cfg.mesh, pb.x[0], vb, cfg.dtau)
    xi_free = orc.assemble_fields(cfg.mesh, pb.x[0], None, cfg.dtau)
    lhs = -np.sqrt(cfg.dtau) * (orc.dense_vhs(Lsc, (xi_full - xi_free).reshape(-1)))
    _, neg = orc.k_tables(cfg.mesh)
    rhs = -cfg.dtau * orc.dense_vhs(Lsc, vb[neg].reshape(-1))
    assert relerr(lhs, rhs) < 1e-12


# ---------------------------------------------------------------- Taylor propagator
def test_taylor_order_zero_and_one(tiny):
    pb, cfg = tiny["pb"], tiny["cfg"]
    rng = np.random.default_rng(17)
    V = rng.standard_normal((cfg.M, cfg.M)) + 1j * rng.standard_normal((cfg.M, cfg.M))
    assert np.array_equal(orc.propagate(V, pb.phi[0], cfg.dtau, 0), pb.phi[0])
    p1 = orc.propagate(V, pb.phi[0], cfg.dtau, 1)
    assert relerr(p1, pb.phi[0] - np.sqrt(cfg.dtau) * V @ pb.phi[0]) < 1e-14


def test_taylor_matches_explicit_power_series(tiny):
    pb, cfg = tiny["pb"], tiny["cfg"]
    xi = orc.assemble_fields(cfg.mesh, pb.x[0], None, cfg.dtau)
    V = orc.vhs(cfg.mesh, pb.L, xi)
    s = -np.sqrt(cfg.dtau)
    acc = np.zeros_like(pb.phi[0])
    P = np.eye(cfg.M, dtype=complex)
    fact = 1.0
    for j in range(7):
        if j > 0:
            P = P @ (s * V)
            fact *= j
        acc = acc + (P / fact) @ pb.phi[0]
    assert relerr(orc.propagate(V, pb.phi[0], cfg.dtau, 6), acc) < 1e-13


def test_taylor_converges_to_exact_exponential_with_slope_7_2(tiny):
    pb, cfg = tiny["pb"], tiny["cfg"]
    xi = orc.assemble_fields(cfg.mesh, pb.x[0], None, 1.0)   # dtau only enters via the shift (none here)
    V = orc.vhs(cfg.mesh, pb.L, xi)
    Hh = 1j * V                                              # Hermitian
    assert relerr(Hh, np.conj(Hh.T)) < 1e-13
    errs = []
    dts = [1e-2, 1e-3, 1e-4]
    for dt in dts:
        approx = orc.propagate(V, pb.phi[0], dt, 6)
        exact = orc.exact_exp_apply(Hh, pb.phi[0], 1j * np.sqrt(dt))   # exp(-sqrt(dt) V) = exp(i sqrt(dt) Hh)
        errs.append(relerr(approx, exact))
    slopes = [np.log10(errs[i] / errs[i + 1]) for i in range(len(errs) - 1)]
    assert errs[0] < 1e-3 and errs[2] < 1e-10
    assert abs(slopes[0] - 3.5) < 0.3 and abs(slopes[1] - 3.5) < 0.3                        # remainder ~ (sqrt dt)^7
    # unitary limit: Phi'^dagger Phi' -> Phi^dagger Phi
    p = orc.propagate(V, pb.phi[0], 1e-4, 6)
    assert relerr(np.conj(p.T) @ p, np.conj(pb.phi[0].T) @ pb.phi[0]) < 1e-10


# ---------------------------------------------------------------- energies
def test_dense_energy_bruteforce_loops():
    """Explicit p,q,r,s loops of Eq. 36 on a tiny system pin the einsum index strings."""
    cfg = synth.tiny_config(mesh=(2, 1, 1), m=2, n=1, nchol=3, nw=1, seed=4)
    pb = synth.make_problem(cfg)
    A = orc.supercell_trial(pb.psi_t)
    Lsc = orc.supercell_L(cfg.mesh, pb.L)
    H = orc.supercell_h1(pb.h1)
    V = orc.eri_from_L(Lsc)
    G = orc.dense_green(A, pb.phi[0])
    M = cfg.M
    e1 = sum(2 * H[p, q] * G[p, q] for p in range(M) for q in range(M))
    ec = ex = 0
    for p, q, r, s in itertools.product(range(M), repeat=4):
        ec += 0.5 * 4 * V[p, q, r, s] * G[p, r] * G[q, s]
        ex += -0.5 * 2 * V[p, q, r, s] * G[p, s] * G[q, r]
    e = orc.dense_energy(H, V, G)
    assert abs(e[0] - e1) < 1e-12 and abs(e[1] - ec) < 1e-12 and abs(e[2] - ex) < 1e-12


def test_two_electron_textbook_case():
    """Nk = 1, n = 1 (two electrons, opposite spin, one spatial orbital phi = trial):
    E = 2 h_aa + J_aa with J = (aa|aa): EC + EX = 2J - J = J."""
    cfg = synth.tiny_config(mesh=(1, 1, 1), m=4, n=1, nchol=5, nw=1, seed=8)
    pb = synth.make_problem(cfg)
    Lh, ht = orc.half_rotate(pb.L, pb.psi_t, pb.h1)
    a = pb.psi_t[0][:, 0]
    th, _, _ = orc.green(pb.psi_t, orc.supercell_trial(pb.psi_t))
    e = orc.local_energy(cfg.mesh, Lh, ht, th)
    haa = np.conj(a) @ pb.h1[0] @ a
    # J = sum_g |a^dag L_g a|^2   (L^0 Hermitian per gamma at Q=0)
    J = sum(abs(np.conj(a) @ pb.L[0, 0, g] @ a) ** 2 for g in range(cfg.nchol))
    assert abs(e[0] - 2 * haa) < 1e-12
    assert abs(e[1] - 2 * J) < 1e-12 and abs(e[2] + J) < 1e-12


def test_local_energy_matches_four_index_definition(tiny):
    pb, cfg, Lh, ht, A, Lsc, H = (tiny[k] for k in ("pb", "cfg", "Lh", "ht", "A", "Lsc", "H"))
    V = orc.eri_from_L(Lsc)
    for w in range(cfg.nw):
        th, _, _ = orc.green(pb.psi_t, pb.phi[w])
        e = orc.local_energy(cfg.mesh, Lh, ht, th)
        G = orc.dense_green(A, pb.phi[w])
        ref = orc.dense_energy(H, V, G)
        for i in range(3):
            assert abs(e[i] - ref[i]) < 1e-11 * abs(ref[i]), (i, e[i], ref[i])
        # Coulomb from the force bias (bilinear), and NOT (1/2) sum |v|^2 in general
        vb = orc.force_bias(cfg.mesh, Lh, th)
        assert abs(orc.coulomb_from_vbias(cfg.mesh, vb) - ref[1]) < 1e-11 * abs(ref[1])
        assert abs(0.5 * np.sum(np.abs(vb) ** 2) - ref[1]) > 1e-3 * abs(ref[1])


def test_energy_at_trial_is_real_with_signs(tiny):
    pb, cfg, Lh, ht, A = (tiny[k] for k in ("pb", "cfg", "Lh", "ht", "A"))
    th, _, _ = orc.green(pb.psi_t, A)
    e = orc.local_energy(cfg.mesh, Lh, ht, th)
    assert np.max(np.abs(e.imag)) < 1e-12 * np.max(np.abs(e.real))
    vb = orc.force_bias(cfg.mesh, Lh, th)
    assert abs(e[1] - 0.5 * np.sum(np.abs(vb) ** 2)) < 1e-12 * abs(e[1])   # EC = 1/2 sum |v|^2 >= 0
    assert e[1].real > 0 and e[2].real < 0


def test_exchange_involution_T2_is_T1_of_partner(tiny):
    """T2(Q,k,k')[a,b,g] == T1(-Q,k'-Q,k-Q)[a,b,g] -- lets the GPU halve the GEMMs."""
    pb, cfg, Lh = tiny["pb"], tiny["cfg"], tiny["Lh"]
    th, _, _ = orc.green(pb.psi_t, pb.phi[0])
    G = orc.reshape_theta(th, cfg.nk, cfg.n, cfg.m)
    mesh = cfg.mesh

    def T1(Q, k, kp):
        return np.einsum('agr,br->bag', Lh[Q, k], G[orc.k_sub(mesh, kp, Q), orc.k_sub(mesh, k, Q)])

    def T2(Q, k, kp):
        return np.einsum('bgs,as->abg', Lh[orc.k_neg(mesh, Q), orc.k_sub(mesh, kp, Q)], G[k, kp])

    for Q, k, kp in [(1, 0, 2), (3, 4, 1), (0, 2, 2), (5 % cfg.nk, 1, 0)]:
        Qm, k2, kp2 = orc.k_neg(mesh, Q), orc.k_sub(mesh, kp, Q), orc.k_sub(mesh, k, Q)
        assert relerr(T2(Q, k, kp), T1(Qm, k2, kp2)) < 1e-13


def test_full_step_runs_and_is_consistent(tiny):
    pb, cfg, Lh, ht = tiny["pb"], tiny["cfg"], tiny["Lh"], tiny["ht"]
    phi2, e, ld = orc.step(cfg.mesh, pb.L, Lh, ht, pb.psi_t, pb.phi, pb.x, cfg.dtau, cfg.order)
    assert phi2.shape == pb.phi.shape and e.shape == (cfg.nw, 3) and np.all(np.isfinite(e))
    th2, ld2, _ = orc.green(pb.psi_t, phi2[1])
    assert abs(ld2 - ld[1]) < 1e-12


# ---------------------------------------------------------------- stored fixture (regression guard of the oracle)
def test_oracle_reproduces_the_stored_tiny_step():
    """tests/golden/tiny_step.txt was written by tests/golden/make_golden.py from the oracle alone; the oracle must keep
    reproducing it (a deliberate change of the oracle's arithmetic regenerates the file and cites its reason)."""
    import importlib.util
    import os
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
    rows = dict(mg.compute())
    assert set(rows) == set(stored)
    for name, z in rows.items():
        assert abs(z - stored[name]) <= 1e-12 * max(1.0, abs(stored[name])), name
