"""Pins for the OPEN-SHELL oracle functions (oracle/afqmc_oracle.py, `*_uhf`) -- CPU only.

Eq. 36 with its explicit spin sums is the definition; each function is pinned to something other than
itself: explicit Python loops over p,q,r,s,sigma,sigma' of Eq. 36, the exact one-electron cancellation E_C + E_X = 0, the
closed-shell limit (two equal channels reproduce the closed-shell functions, which are pinned in test_oracle_pins.py), and
level P == level D on tiny meshes with N_up != N_dn.
"""
import numpy as np
import pytest

from oracle import afqmc_oracle as orc
from paper_2003_09468_b200 import synth

TOL = 1e-11


def relerr(a, b):
    a, b = np.asarray(a), np.asarray(b)
    return float(np.max(np.abs(a - b)) / max(np.max(np.abs(b)), 1e-300))


@pytest.fixture(scope="module", params=[((2, 3, 1), 3, 2, 1), ((2, 2, 1), 4, 3, 2), ((1, 1, 2), 3, 1, 2)],
                ids=["2x3x1_up2_dn1", "2x2x1_up3_dn2", "1x1x2_up1_dn2"])
def uhf(request):
    mesh, m, n_up, n_dn = request.param
    cfg = synth.tiny_config(mesh=mesh, m=m, n=n_up, nchol=4, nw=2, seed=7)
    pb, psi_dn, phi_dn = synth.make_open_shell(cfg, n_dn)
    Lh_up, ht_up = orc.half_rotate(pb.L, pb.psi_t, pb.h1)
    Lh_dn, ht_dn = orc.half_rotate(pb.L, psi_dn, pb.h1)
    Lsc = orc.supercell_L(cfg.mesh, pb.L)
    return dict(cfg=cfg, pb=pb, psi=(pb.psi_t, psi_dn), phi=(pb.phi, phi_dn), Lh=(Lh_up, Lh_dn), ht=(ht_up, ht_dn),
                A=(orc.supercell_trial(pb.psi_t), orc.supercell_trial(psi_dn)), Lsc=Lsc, H=orc.supercell_h1(pb.h1),
                V=orc.eri_from_L(Lsc))


def test_dense_energy_uhf_against_explicit_spin_orbital_loops():
    """Eq. 36 written as plain loops over spin ORBITALS on a very small system: E = sum h G + 1/2 sum v [G G - G G] with
    the spin-orbital Green's function G_{(p s),(r s')} = delta_{s s'} G^s_pr and v_{(ps)(qt)(rs')(st')} = v_pqrs delta_{s s'} delta_{t t'}."""
    rng = np.random.default_rng(0)
    M = 3
    Lsc = rng.standard_normal((M, M, 4)) + 1j * rng.standard_normal((M, M, 4))
    V = orc.eri_from_L(Lsc)
    H = rng.standard_normal((M, M)) + 1j * rng.standard_normal((M, M))
    G = [rng.standard_normal((M, M)) + 1j * rng.standard_normal((M, M)) for _ in range(2)]
    e1 = ec = ex = 0.0
    for s in range(2):
        for p in range(M):
            for q in range(M):
                e1 += H[p, q] * G[s][p, q]
    for s in range(2):
        for t in range(2):
            for p in range(M):
                for q in range(M):
                    for r in range(M):
                        for u in range(M):
                            ec += 0.5 * V[p, q, r, u] * G[s][p, r] * G[t][q, u]
                            if s == t:
                                ex += -0.5 * V[p, q, r, u] * G[s][p, u] * G[s][q, r]
    got = orc.dense_energy_uhf(H, V, G[0], G[1])
    assert relerr(got, [e1, ec, ex]) < 1e-13


def test_one_electron_has_no_two_body_energy(uhf):
    """A single electron (one occupied spin-up orbital, no spin-down electron) does not interact with itself: the Coulomb
    and exchange terms of Eq. 36 cancel EXACTLY, whatever the walker.  Fixes the relative sign and the 1/2 of both terms
    and the delta_{sigma sigma'} on the exchange."""
    cfg, A_up = uhf["cfg"], uhf["A"][0]
    rng = np.random.default_rng(5)
    a = A_up[:, :1]
    phi = a + 0.3 * (rng.standard_normal(a.shape) + 1j * rng.standard_normal(a.shape))
    G = orc.dense_green(a, phi)
    e = orc.dense_energy_uhf(uhf["H"], uhf["V"], G, np.zeros_like(G))
    assert abs(e[1] + e[2]) < 1e-12 * abs(e[1])
    assert abs(e[1]) > 1e-3                      # (the two terms are not trivially zero)


def test_two_like_spin_electrons_exchange_differs_from_opposite_spins(uhf):
    """Same two orbitals occupied with parallel spins (both in the up channel) or antiparallel (one per channel): E1 and E_C
    agree (the total density is the same when the walker is the trial and the orbitals are orthonormal columns of one
    matrix), E_X differs by exactly the cross term -sum v G^a_ps G^b_qr - (a<->b)... checked through its definition."""
    A_up = uhf["A"][0]
    if A_up.shape[1] < 2:
        pytest.skip("needs two occupied orbitals")
    a, b = A_up[:, :1], A_up[:, 1:2]
    Ga, Gb = orc.dense_green(a, a), orc.dense_green(b, b)
    Gab = orc.dense_green(A_up[:, :2], A_up[:, :2])
    assert relerr(Gab, Ga + Gb) < 1e-12                                    # orthonormal orbitals: densities add
    par = orc.dense_energy_uhf(uhf["H"], uhf["V"], Gab, np.zeros_like(Gab))
    anti = orc.dense_energy_uhf(uhf["H"], uhf["V"], Ga, Gb)
    assert abs(par[0] - anti[0]) < 1e-12 * abs(par[0]) and abs(par[1] - anti[1]) < 1e-12 * abs(par[1])
    cross = -0.5 * (np.einsum('pqrs,ps,qr->', uhf["V"], Ga, Gb) + np.einsum('pqrs,ps,qr->', uhf["V"], Gb, Ga))
    assert abs((par[2] - anti[2]) - cross) < 1e-12 * abs(cross)


def test_closed_shell_limit_of_every_uhf_function(uhf):
    """Two EQUAL channels reproduce the closed-shell functions (factors 2, 4, 2 by hand there, spin sums here)."""
    cfg, pb = uhf["cfg"], uhf["pb"]
    A, Lsc, H, V = uhf["A"][0], uhf["Lsc"], uhf["H"], uhf["V"]
    Lh, ht = uhf["Lh"][0], uhf["ht"][0]
    for w in range(cfg.nw):
        G = orc.dense_green(A, pb.phi[w])
        assert relerr(orc.dense_energy_uhf(H, V, G, G), orc.dense_energy(H, V, G)) < TOL
        assert relerr(orc.dense_vbias_uhf(Lsc, G, G), orc.dense_vbias(Lsc, G)) < TOL
        th, _, _ = orc.green(pb.psi_t, pb.phi[w])
        assert relerr(orc.force_bias_uhf(cfg.mesh, Lh, Lh, th, th), orc.force_bias(cfg.mesh, Lh, th)) < TOL
        assert relerr(orc.local_energy_uhf(cfg.mesh, (Lh, Lh), (ht, ht), (th, th)), orc.local_energy(cfg.mesh, Lh, ht, th)) < TOL
    (pu, pd), e, ld = orc.step_uhf(cfg.mesh, pb.L, (Lh, Lh), (ht, ht), (pb.psi_t, pb.psi_t), (pb.phi, pb.phi), pb.x, cfg.dtau, cfg.order)
    p0, e0, ld0 = orc.step(cfg.mesh, pb.L, Lh, ht, pb.psi_t, pb.phi, pb.x, cfg.dtau, cfg.order)
    assert relerr(pu, p0) < TOL and relerr(pd, p0) < TOL and relerr(e, e0) < 1e-10
    assert np.max(np.abs(ld.real - 2 * ld0.real)) < 1e-10
    assert np.max(np.abs(np.angle(np.exp(1j * (ld.imag - 2 * ld0.imag))))) < 1e-10


def test_level_p_equals_level_d_open_shell(uhf):
    cfg = uhf["cfg"]
    for w in range(cfg.nw):
        G = [orc.dense_green(uhf["A"][s], uhf["phi"][s][w]) for s in range(2)]
        th = [orc.green(uhf["psi"][s], uhf["phi"][s][w])[0] for s in range(2)]
        # half-rotated Green's function and the full one: G = A^* Theta (Eq. 29)
        for s in range(2):
            assert relerr(np.conj(uhf["A"][s]) @ th[s], G[s]) < TOL
        vb_d = orc.dense_vbias_uhf(uhf["Lsc"], G[0], G[1]).reshape(cfg.nk, cfg.nchol)
        assert relerr(orc.force_bias_uhf(cfg.mesh, uhf["Lh"][0], uhf["Lh"][1], th[0], th[1]), vb_d) < TOL
        e_d = orc.dense_energy_uhf(uhf["H"], uhf["V"], G[0], G[1])
        e_p = orc.local_energy_uhf(cfg.mesh, uhf["Lh"], uhf["ht"], th)
        assert relerr(e_p, e_d) < TOL
        # the Coulomb term is the bilinear form of the spin-summed force bias (Eq. 41 / step 3)
        assert abs(e_p[1] - orc.coulomb_from_vbias(cfg.mesh, vb_d)) < TOL * abs(e_p[1])


def test_open_shell_step_composition(uhf):
    """step_uhf = per-spin Green, spin-summed force bias, ONE vHS, the same propagator on both channels, energy of the new
    walker: re-assembled here from the single-channel pieces (level D energy at the end)."""
    cfg, pb = uhf["cfg"], uhf["pb"]
    (pu, pd), e, ld = orc.step_uhf(cfg.mesh, pb.L, uhf["Lh"], uhf["ht"], uhf["psi"], uhf["phi"], pb.x, cfg.dtau, cfg.order)
    for w in range(cfg.nw):
        G = [orc.dense_green(uhf["A"][s], uhf["phi"][s][w]) for s in range(2)]
        vb = orc.dense_vbias_uhf(uhf["Lsc"], G[0], G[1]).reshape(cfg.nk, cfg.nchol)
        V = orc.dense_vhs(uhf["Lsc"], orc.assemble_fields(cfg.mesh, pb.x[w], vb, cfg.dtau).reshape(-1))
        new = [orc.taylor_apply(V, uhf["phi"][s][w], cfg.dtau, cfg.order) for s in range(2)]
        assert relerr(pu[w], new[0]) < TOL and relerr(pd[w], new[1]) < TOL
        G2 = [orc.dense_green(uhf["A"][s], new[s]) for s in range(2)]
        assert relerr(e[w], orc.dense_energy_uhf(uhf["H"], uhf["V"], G2[0], G2[1])) < 1e-9
        det = np.prod([np.linalg.det(orc.dense_overlap(uhf["A"][s], new[s])) for s in range(2)])
        assert abs(ld[w].real - np.log(abs(det))) < 1e-10
        assert abs(np.angle(np.exp(1j * (ld[w].imag - np.angle(det))))) < 1e-10
