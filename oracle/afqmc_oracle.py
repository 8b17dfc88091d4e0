"""CPU ORACLE for the k-point ph-AFQMC per-walker step  --  TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` leg may import this file.  It shares no code with the CUDA library
(`paper_2003_09468_b200/csrc`): no kernels, headers, helpers, tables or pre/post-processing.
It imports nothing from the product package.

Everything is complex128 (numpy), written for readability against the paper
(`/root/reference/PAPER.md`, arxiv 2003.09468), not for speed.  Library primitives used as
steps: ``numpy.matmul`` / ``einsum`` (a matrix product) and ``numpy.linalg.eigh`` (only in the
exact-exponential reference of level D).  There is no blocking, fusion or reordering beyond
what the cited definition or algorithm states.

Two levels:

* **Level D (definition)** -- dense supercell objects and explicit 4-index sums:
  Eq. 20, Eq. 26-30 (:135-146), Eq. 25/37 (:131,:178), Eq. 36 (:171),
  Eq. 33 (:158) and the Taylor series of :160.  Tiny sizes only.
* **Level P (production)** -- the k-blocked algorithm the GPU implements and is compared
  with: Eq. 47 (:220), Eq. 48 (:224), Eq. 49 (:230-236) evaluated by the paper's
  steps 1-3 (:306-319) literally (both T^1 and T^2 for every (Q,k,k')).

Pins (tests/test_oracle_pins.py): level P == level D on tiny meshes; level D against
closed forms and invariants (O = 1 and Theta = A^T at Phi = Psi_T; G^2 = G, Tr G = N;
brute-force cofactor determinant; numpy.linalg.slogdet; exact exponential as dtau -> 0 with
slope 7/2; anti-Hermitian vHS without force bias; momentum conservation; gauge invariance
Phi -> Phi R).  No function here is "parity unpinned"; the field-assembly rule
(`assemble_fields`, reading R7) and the Taylor order (R8) are conventions pinned
only by level D of this file, as DESIGN.md states.

The AFQMC-block functions at the end of the file (one-body half steps, hybrid weight,
orthogonalisation, mixed estimator, block) are pinned by tests/test_oracle_block_pins.py (real-field Hermitian
restatement, Gauss-Hermite quadrature of Eq. 12/16, Wick's theorem, scipy expm, numpy QR); none is "parity
unpinned".  `numpy.linalg.det` / `inv` appear only in level D.

The OPEN-SHELL functions (two spin channels with N_up != N_dn; Eq. 36 and Eq. 49 with their
explicit sigma, sigma' sums) follow the closed-shell ones section by section (`*_uhf`); they are
pinned by tests/test_oracle_open_shell_pins.py (explicit p,q,r,s,sigma,sigma' loops, the one-electron self-interaction
cancellation E_C + E_X = 0, the closed-shell limit, level P == level D); none is "parity unpinned".

Layouts (row-major, last index fastest):
  L[Q][k][gamma][p][r]   p at k-point k, r at k-Q
  psi_t[k][p][a]         trial, block diagonal in k
  h1[k][p][q]            one-body Hamiltonian, block diagonal     (Eq. 45)
  phi[w][M][N]           dense walker, row (k,p), column (k,a)
  theta[w][N][M]         half-rotated Green's function, Eq. 30
  vbias[w][Q][gamma], x[w][Q][gamma] (real), vhs[w][M][M], energy[w][3] = (E1, EC, EX)
"""
from __future__ import annotations

import numpy as np

C128 = np.complex128


# --------------------------------------------------------------------------------------
# k-point index arithmetic (Gamma-centred regular mesh; index (i1*g2+i2)*g3+i3)
# --------------------------------------------------------------------------------------
def k_coords(mesh):
    g1, g2, g3 = mesh
    return [(i1, i2, i3) for i1 in range(g1) for i2 in range(g2) for i3 in range(g3)]


def k_index(mesh, c):
    g1, g2, g3 = mesh
    return ((c[0] % g1) * g2 + (c[1] % g2)) * g3 + (c[2] % g3)


def k_sub(mesh, k, Q):
    """Index of k - Q (k_r = k_p - Q)."""
    ck, cq = k_coords(mesh)[k], k_coords(mesh)[Q]
    return k_index(mesh, (ck[0] - cq[0], ck[1] - cq[1], ck[2] - cq[2]))


def k_neg(mesh, Q):
    cq = k_coords(mesh)[Q]
    return k_index(mesh, (-cq[0], -cq[1], -cq[2]))


def k_tables(mesh):
    nk = mesh[0] * mesh[1] * mesh[2]
    kminus = np.array([[k_sub(mesh, k, Q) for Q in range(nk)] for k in range(nk)])
    neg = np.array([k_neg(mesh, Q) for Q in range(nk)])
    return kminus, neg


# --------------------------------------------------------------------------------------
# LEVEL D : dense supercell definitions
# --------------------------------------------------------------------------------------
def supercell_trial(psi_t):
    """A (M x N), block diagonal in k."""
    nk, m, n = psi_t.shape
    A = np.zeros((nk * m, nk * n), dtype=C128)
    for k in range(nk):
        A[k * m:(k + 1) * m, k * n:(k + 1) * n] = psi_t[k]
    return A


def supercell_h1(h1):
    """h (M x M), block diagonal in k (Eq. 45)."""
    nk, m, _ = h1.shape
    H = np.zeros((nk * m, nk * m), dtype=C128)
    for k in range(nk):
        H[k * m:(k + 1) * m, k * m:(k + 1) * m] = h1[k]
    return H


def supercell_L(mesh, L):
    """L_sc[P][R][Gamma], Gamma = (Q,gamma); zero unless k_R = k_P - Q."""
    nk, _, nchol, m, _ = L.shape
    Lsc = np.zeros((nk * m, nk * m, nk * nchol), dtype=C128)
    for Q in range(nk):
        for k in range(nk):
            kq = k_sub(mesh, k, Q)
            # L[Q,k] is [gamma][p][r] -> [p][r][gamma]
            Lsc[k * m:(k + 1) * m, kq * m:(kq + 1) * m, Q * nchol:(Q + 1) * nchol] = \
                np.transpose(L[Q, k], (1, 2, 0))
    return Lsc


def eri_from_L(Lsc):
    """v_pqrs = sum_Gamma L_{pr,Gamma} conj(L_{sq,Gamma})   (Eq. 20)."""
    return np.einsum('prg,sqg->pqrs', Lsc, np.conj(Lsc))


def dense_overlap(A, phi):
    """O = A^dagger Phi  (the matrix inverted in Eq. 27)."""
    return np.conj(A.T) @ phi


def dense_theta(A, phi):
    """Eq. 30: Theta = (Phi^T A^*)^{-1} Phi^T, via numpy's inverse (level D only)."""
    return np.linalg.inv(phi.T @ np.conj(A)) @ phi.T


def dense_green(A, phi):
    """Eq. 28-29: G_pr = [A^* Theta]_pr = <c_p^dag c_r>."""
    return np.conj(A) @ dense_theta(A, phi)


def dense_vbias(Lsc, G):
    """v_Gamma = 2 sum_pr L_{pr,Gamma} G_pr (Eq. 25/37 without the -sqrt(dtau) c_pm prefactor;
    the 2 is the closed-shell spin sum)."""
    return 2.0 * np.einsum('prg,pr->g', Lsc, G)


def dense_energy(H, V, G):
    """Eq. 36 for a closed shell (both spins share G):
    E1 = 2 sum h_pq G_pq;  EC = (1/2) 4 sum v_pqrs G_pr G_qs;  EX = -(1/2) 2 sum v_pqrs G_ps G_qr."""
    e1 = 2.0 * np.einsum('pq,pq->', H, G)
    ec = 0.5 * 4.0 * np.einsum('pqrs,pr,qs->', V, G, G)
    ex = -0.5 * 2.0 * np.einsum('pqrs,ps,qr->', V, G, G)
    return np.array([e1, ec, ex], dtype=C128)


def dense_vhs(Lsc, xi):
    """vHS_pr = sum_Gamma xi_Gamma L_{pr,Gamma} (the contraction of Eq. 33/48)."""
    return np.einsum('prg,g->pr', Lsc, xi)


def taylor_apply(vhs, phi, dtau, order):
    """Phi' = sum_{j=0..order} (s V)^j / j!  Phi with s = -sqrt(dtau), by repeated
    multiplication T_j = (s/j) V T_{j-1} (R7(v), R8)."""
    s = -np.sqrt(dtau)
    term = phi.astype(C128).copy()
    out = term.copy()
    for j in range(1, order + 1):
        term = (s / j) * (vhs @ term)
        out = out + term
    return out


def exact_exp_apply(herm, phi, scale):
    """exp(scale * herm) Phi for a HERMITIAN matrix `herm` by eigendecomposition."""
    w, U = np.linalg.eigh(herm)
    return (U * np.exp(scale * w)) @ (np.conj(U.T) @ phi)


# --------------------------------------------------------------------------------------
# LEVEL P : the k-blocked production algorithm
# --------------------------------------------------------------------------------------
def half_rotate(L, psi_t, h1):
    """a0.  Lh[Q][k][a][gamma][r] = sum_p conj(A_k[p,a]) L[Q][k][gamma][p][r],
    stored 'transposed' as (a gamma, r) like steps 2(a)/(b) use it;
    ht[k][a][q] = sum_p conj(A_k[p,a]) h_k[p,q]  (first line of Eq. 49)."""
    nk, _, nchol, m, _ = L.shape
    n = psi_t.shape[2]
    Lh = np.empty((nk, nk, n, nchol, m), dtype=C128)
    for Q in range(nk):
        for k in range(nk):
            Ak = np.conj(psi_t[k])          # [p][a]
            for g in range(nchol):
                Lh[Q, k, :, g, :] = Ak.T @ L[Q, k, g]     # [a][r]
    ht = np.empty((nk, n, m), dtype=C128)
    for k in range(nk):
        ht[k] = np.conj(psi_t[k]).T @ h1[k]
    return Lh, ht


def overlap(psi_t, phi_w):
    """a1.  O = A^dagger Phi assembled as Nk row blocks A_k^dagger Phi[k rows, :]."""
    nk, m, n = psi_t.shape
    N = nk * n
    O = np.empty((N, N), dtype=C128)
    for k in range(nk):
        O[k * n:(k + 1) * n, :] = np.conj(psi_t[k]).T @ phi_w[k * m:(k + 1) * m, :]
    return O


def lu_factor(O):
    """a2.  LU with partial (row) pivoting, column by column (Doolittle, unblocked).
    Returns (LU packed, perm, sign, info); info = j+1 of the first exactly-zero pivot, else 0."""
    a = O.astype(C128).copy()
    nn = a.shape[0]
    perm = np.arange(nn)
    sign = 1.0
    info = 0
    for j in range(nn):
        p = j + int(np.argmax(np.abs(a[j:, j])))
        if a[p, j] == 0:
            if info == 0:
                info = j + 1
            continue
        if p != j:
            a[[j, p], :] = a[[p, j], :]
            perm[[j, p]] = perm[[p, j]]
            sign = -sign
        a[j + 1:, j] /= a[j, j]
        a[j + 1:, j + 1:] -= np.outer(a[j + 1:, j], a[j, j + 1:])
    return a, perm, sign, info


def lu_logdet(lu, sign):
    """log det O = sum_j log(u_jj) (+ i pi if the permutation is odd): log|det| + i arg det."""
    d = np.diag(lu)
    logabs = np.sum(np.log(np.abs(d)))
    phase = np.sum(np.angle(d)) + (np.pi if sign < 0 else 0.0)
    phase = (phase + np.pi) % (2 * np.pi) - np.pi
    return complex(logabs, phase)


def lu_inverse(lu, perm):
    """O^{-1} from the factors: solve L U X = P I by forward then back substitution."""
    nn = lu.shape[0]
    X = np.eye(nn, dtype=C128)[perm, :]
    for j in range(nn):                     # L y = P I   (unit lower)
        X[j + 1:, :] -= np.outer(lu[j + 1:, j], X[j, :])
    for j in range(nn - 1, -1, -1):         # U x = y
        X[j, :] /= lu[j, j]
        X[:j, :] -= np.outer(lu[:j, j], X[j, :])
    return X


def green(psi_t, phi_w):
    """a1-a3 for one walker: returns (Theta [N][M], logdet, info).
    Theta = (Phi^T A^*)^{-1} Phi^T = (Phi O^{-1})^T, Eq. 30."""
    O = overlap(psi_t, phi_w)
    lu, perm, sign, info = lu_factor(O)
    if info != 0:
        return np.full((O.shape[0], phi_w.shape[0]), np.nan, dtype=C128), complex(np.nan, np.nan), info
    Oinv = lu_inverse(lu, perm)
    theta = (phi_w @ Oinv).T
    return np.ascontiguousarray(theta), lu_logdet(lu, sign), 0


def force_bias(mesh, Lh, theta_w):
    """a4.  vbias[Q][gamma] = 2 sum_k sum_{a,r} Lh[Q][k][a][gamma][r] Theta[(k,a),(k-Q,r)]
    (the half-rotated contraction at the core of Eq. 47, = 2 X_gamma of Eq. 37)."""
    nk, _, n, nchol, m = Lh.shape
    vb = np.zeros((nk, nchol), dtype=C128)
    for Q in range(nk):
        for k in range(nk):
            kq = k_sub(mesh, k, Q)
            blk = theta_w[k * n:(k + 1) * n, kq * m:(kq + 1) * m]     # [a][r]
            vb[Q] += 2.0 * np.einsum('agr,ar->g', Lh[Q, k], blk)
    return vb


def assemble_fields(mesh, x_w, vbias_w, dtau):
    """Field assembly, reading R7 (the paper's Eq. 8/17/24/47/48 are mutually
    inconsistent in signs and factors of i):
      (i)   one real field x[Q][gamma] per (Q,gamma);
      (ii)  z_Q = x_Q if -Q == Q; for idx(Q) < idx(-Q): z_Q = (x_Q + i x_{-Q})/sqrt2,
            z_{-Q} = conj(z_Q);
      (iii) zbar_{Q,gamma} = -i sqrt(dtau) vbias_{-Q,gamma}   (Eq. 17 in this basis; 0 if no vbias);
      (iv)  xi = -i (z - zbar).
    """
    nk = x_w.shape[0]
    z = np.zeros(x_w.shape, dtype=C128)
    for Q in range(nk):
        mq = k_neg(mesh, Q)
        if mq == Q:
            z[Q] = x_w[Q]
        elif Q < mq:
            z[Q] = (x_w[Q] + 1j * x_w[mq]) / np.sqrt(2.0)
            z[mq] = np.conj(z[Q])
    zbar = np.zeros_like(z)
    if vbias_w is not None:
        for Q in range(nk):
            zbar[Q] = -1j * np.sqrt(dtau) * vbias_w[k_neg(mesh, Q)]
    return -1j * (z - zbar)


def vhs(mesh, L, xi_w):
    """a5.  V[(k,p),(k-Q,r)] = sum_gamma L[Q][k][gamma][p][r] xi[Q][gamma]   (Eq. 48);
    each (k,k') block of the M x M matrix receives exactly one Q = k - k'."""
    nk, _, nchol, m, _ = L.shape
    V = np.zeros((nk * m, nk * m), dtype=C128)
    for Q in range(nk):
        for k in range(nk):
            kq = k_sub(mesh, k, Q)
            V[k * m:(k + 1) * m, kq * m:(kq + 1) * m] += np.einsum('gpr,g->pr', L[Q, k], xi_w[Q])
    return V


def propagate(vhs_w, phi_w, dtau, order):
    """a6.  Same recurrence as level D."""
    return taylor_apply(vhs_w, phi_w, dtau, order)


def reshape_theta(theta_w, nk, n, m):
    """Step 1: G[(k1 a),(k2 q)] -> G[k1][k2][a][q]."""
    return np.ascontiguousarray(theta_w.reshape(nk, n, nk, m).transpose(0, 2, 1, 3))


def local_energy(mesh, Lh, ht, theta_w):
    """a7-a9 for one walker, by the paper's steps 1-3, closed shell.

    Returns (E1, EC, EX).  Spin factors: E1 x2; the traces v_j carry x2 each so EC = (1/2) v1 v2
    has x4 (sigma, sigma' independent); EX x2 (delta_{sigma sigma'} in Eq. 49)."""
    nk, _, n, nchol, m = Lh.shape
    G = reshape_theta(theta_w, nk, n, m)                    # step 1
    e1 = 0.0 + 0.0j
    for k in range(nk):                                     # Eq. 49 line 1
        e1 += 2.0 * np.sum(ht[k] * G[k, k])
    ex = 0.0 + 0.0j
    ec = 0.0 + 0.0j
    for Q in range(nk):
        mQ = k_neg(mesh, Q)
        v1 = np.zeros(nchol, dtype=C128)
        v2 = np.zeros(nchol, dtype=C128)
        for k in range(nk):
            kq = k_sub(mesh, k, Q)
            for kp in range(nk):
                kpq = k_sub(mesh, kp, Q)
                # 2(a): T1[b,a,g] = sum_r Lh[Q,k][a,g,r] G[k'-Q, k-Q][b,r]
                T1 = np.einsum('agr,br->bag', Lh[Q, k], G[kpq, kq])
                # 2(b): T2[a,b,g] = sum_s Lh[-Q,k'-Q][b,g,s] G[k, k'][a,s]
                T2 = np.einsum('bgs,as->abg', Lh[mQ, kpq], G[k, kp])
                # 2(c)
                ex += -0.5 * 2.0 * np.einsum('bag,abg->', T1, T2)
                # 2(d): the trace is a density only when k'-Q == k
                if kpq == k:
                    v1 += 2.0 * np.einsum('aag->g', T1)
                    v2 += 2.0 * np.einsum('aag->g', T2)
        ec += 0.5 * np.sum(v1 * v2)                         # step 3, summed over Q
    return np.array([e1, ec, ex], dtype=C128)


def coulomb_from_vbias(mesh, vbias_w):
    """EC = (1/2) sum_Q sum_gamma vbias[Q] vbias[-Q]  (bilinear; Eq. 41)."""
    nk = vbias_w.shape[0]
    ec = 0.0 + 0.0j
    for Q in range(nk):
        ec += 0.5 * np.sum(vbias_w[Q] * vbias_w[k_neg(mesh, Q)])
    return ec


# --------------------------------------------------------------------------------------
# One full step for a batch (the composition bench.py times)
# --------------------------------------------------------------------------------------
def step(mesh, L, Lh, ht, psi_t, phi, x, dtau, order):
    """overlap+green, force bias, vHS, propagate on Phi; then overlap+green+local energy on Phi'.
    Returns (phi_new [nw][M][N], energy [nw][3], logdet_new [nw])."""
    nw = phi.shape[0]
    phi_new = np.empty_like(phi)
    energy = np.empty((nw, 3), dtype=C128)
    logdet = np.empty(nw, dtype=C128)
    for w in range(nw):
        th, _, _ = green(psi_t, phi[w])
        vb = force_bias(mesh, Lh, th)
        xi = assemble_fields(mesh, x[w], vb, dtau)
        V = vhs(mesh, L, xi)
        phi_new[w] = propagate(V, phi[w], dtau, order)
        th2, ld, _ = green(psi_t, phi_new[w])
        energy[w] = local_energy(mesh, Lh, ht, th2)
        logdet[w] = ld
    return phi_new, energy, logdet


# ======================================================================================
# The AFQMC block around the step:  one-body half steps (Eq. 7, 13,
# PAPER.md:54, :85), hybrid importance function and phaseless weight update (Eq. 15-19,
# PAPER.md:93-105), walker orthogonalisation and the mixed estimator (Eq. 34-35);
# "a block is 20 iterations of the propagation step followed by an energy evaluation and walker
# orthogonalization ... the 'hybrid' method is used for propagation".
# ======================================================================================

# ---- level D: the real-field (Hermitian) basis of the Hubbard-Stratonovich operators ----
def hermitian_hs_operators(mesh, Lsc, nchol):
    """One HERMITIAN M x M matrix v_j per real field x[Q][gamma] (j = Q*nchol + gamma), so that
    H2' = (1/2) sum_Gamma rho_Gamma rho_Gamma^dagger = (1/2) sum_j v_j^2 (Eq. 8-9, with
    the paper's v_hat = i v) and sum_j x_j v_j = sum_Gamma z_Gamma L_Gamma with the z of
    `assemble_fields`:
        -Q == Q          : v = L_Q                             (Hermitian by the (Q,-Q) identity)
        idx(Q) < idx(-Q) : v_Q = (L_Q + L_{-Q})/sqrt2,  v_{-Q} = i (L_Q - L_{-Q})/sqrt2.
    rho_Gamma = sum_pr L_{pr,Gamma} c_p^dag c_r and rho_{(-Q,gamma)} = rho_{(Q,gamma)}^dagger."""
    nk = mesh[0] * mesh[1] * mesh[2]
    Mdim = Lsc.shape[0]
    v = np.zeros((nk * nchol, Mdim, Mdim), dtype=C128)
    for Q in range(nk):
        mq = k_neg(mesh, Q)
        for g in range(nchol):
            LQ = Lsc[:, :, Q * nchol + g]
            LmQ = Lsc[:, :, mq * nchol + g]
            if mq == Q:
                v[Q * nchol + g] = LQ
            elif Q < mq:
                v[Q * nchol + g] = (LQ + LmQ) / np.sqrt(2.0)
                v[mq * nchol + g] = 1j * (LQ - LmQ) / np.sqrt(2.0)
    return v


def dense_expm_hermitian(Hm, scale):
    """exp(scale * Hm) for a Hermitian matrix by eigendecomposition."""
    w, U = np.linalg.eigh(Hm)
    return (U * np.exp(scale * w)) @ np.conj(U.T)


def dense_hybrid_step(A, vops, B1, phi_w, x_flat, dtau, order, xbar_override=None):
    """Level D of one hybrid propagation step for one walker, entirely in the real-field basis; `B1` is the
    DENSE M x M one-body half-step propagator (`supercell_h1` of the per-k blocks)
    (Eq. 13, 15-19; closed shell, both spins share phi):
        G      = Green's function of phi (Eq. 29);   <v_j> = 2 sum_pr (v_j)_pr G_pr
        xbar_j = -i sqrt(dtau) <v_j>                  (Eq. 17 with v_hat_j = i v_j)
        B(x - xbar) = B1 * Taylor_order( i sqrt(dtau) sum_j (x_j - xbar_j) v_j ) * B1   (Eq. 13)
        ratio  = [det(A^dag phi') / det(A^dag phi)]^2                          (two spin channels)
        I      = ratio * exp(x.xbar - xbar.xbar/2)                             (Eq. 16)
        dtheta = arg(ratio)                                                     (Eq. 19)
        factor = |I| max(0, cos dtheta)                                         (Eq. 18)
    `xbar_override` replaces the force-bias shift by any (complex) shift: Eq. 12 and 15-16 describe the same
    integral for every shift, which is what the quadrature pin checks.
    Returns (phi', I, dtheta, factor)."""
    G = dense_green(A, phi_w)
    vavg = 2.0 * np.einsum('jpr,pr->j', vops, G)
    xbar = -1j * np.sqrt(dtau) * vavg
    if xbar_override is not None:
        xbar = np.asarray(xbar_override, dtype=C128)
    xs = x_flat - xbar
    V = np.einsum('j,jpr->pr', xs, vops)
    t = B1 @ phi_w
    # Taylor series of exp(i sqrt(dtau) V) applied to t
    term = t.copy()
    out = t.copy()
    for j in range(1, order + 1):
        term = (1j * np.sqrt(dtau) / j) * (V @ term)
        out = out + term
    phi_new = B1 @ out
    d_old = np.linalg.det(dense_overlap(A, phi_w))
    d_new = np.linalg.det(dense_overlap(A, phi_new))
    ratio = (d_new / d_old) ** 2
    I = ratio * np.exp(np.sum(x_flat * xbar) - 0.5 * np.sum(xbar * xbar))
    dtheta = float(np.angle(ratio))
    factor = float(np.abs(I) * max(0.0, np.cos(dtheta)))
    return phi_new, I, dtheta, factor


def dense_h2prime_mixed(vops, G):
    """<Psi_T| (1/2) sum_j v_j^2 |phi> / <Psi_T|phi> for a closed shell by Wick's theorem with
    G_pr = <c_p^dag c_r> (per spin):  <c_p^dag c_r c_q^dag c_s> = G_pr G_qs + G_ps (delta_rq - G_qr), so
    <v^2> = (2 tr_pr v G)^2 + 2 sum v_pr v_rs G_ps - 2 sum v_pr v_qs G_ps G_qr."""
    tot = 0.0 + 0.0j
    for v in vops:
        t1 = 2.0 * np.einsum('pr,pr->', v, G)
        t2 = 2.0 * np.einsum('pr,rs,ps->', v, v, G)
        t3 = 2.0 * np.einsum('pr,qs,ps,qr->', v, v, G, G)
        tot += 0.5 * (t1 * t1 + t2 - t3)
    return tot


# ---- level P: what the GPU library computes ----
def onebody_half_propagator(h1p, dtau):
    """B1[k] = exp(-dtau/2 * h1p[k]) per k-point (H1' is block diagonal in k, Eq. 45, PAPER.md:210;
    the half steps of Eq. 7/13).  `h1p` is whatever one-body operator the caller propagates with
    (the paper's H1' = H1 + v0, Eq. 10; v0 is outside this build's scope)."""
    return np.stack([dense_expm_hermitian(h1p[k], -0.5 * dtau) for k in range(h1p.shape[0])])


def apply_onebody(B1, phi_w):
    """Phi[(k,:), :] <- B1[k] Phi[(k,:), :]  (block-diagonal one-body propagator, Eq. 13)."""
    nk, m, _ = B1.shape
    out = np.empty_like(phi_w)
    for k in range(nk):
        out[k * m:(k + 1) * m, :] = B1[k] @ phi_w[k * m:(k + 1) * m, :]
    return out


def hybrid_weight(mesh, x_w, vbias_w, dtau, logdet_old, logdet_new):
    """Eq. 16, 18, 19 in the (Q,gamma) field basis of `assemble_fields`:
    with z, zbar as there (zbar_{Q} = -i sqrt(dtau) vbias_{-Q}),
        x.xbar = sum_{Q,gamma} z_Q zbar_{-Q},   xbar.xbar = sum_{Q,gamma} zbar_Q zbar_{-Q}
    (the real-field bilinear forms written in the complex basis; pinned against level D),
        log ratio = 2 (logdet_new - logdet_old)          (closed shell: both spin channels)
        log I = log ratio + x.xbar - xbar.xbar/2;  dtheta = Im log ratio wrapped to (-pi, pi];
        factor = |I| max(0, cos dtheta).
    Returns (log I (complex), dtheta, factor)."""
    nk = x_w.shape[0]
    z = np.zeros(x_w.shape, dtype=C128)
    for Q in range(nk):
        mq = k_neg(mesh, Q)
        if mq == Q:
            z[Q] = x_w[Q]
        elif Q < mq:
            z[Q] = (x_w[Q] + 1j * x_w[mq]) / np.sqrt(2.0)
            z[mq] = np.conj(z[Q])
    zbar = np.zeros_like(z)
    for Q in range(nk):
        zbar[Q] = -1j * np.sqrt(dtau) * vbias_w[k_neg(mesh, Q)]
    xxb = 0.0 + 0.0j
    xbxb = 0.0 + 0.0j
    for Q in range(nk):
        mq = k_neg(mesh, Q)
        xxb += np.sum(z[Q] * zbar[mq])
        xbxb += np.sum(zbar[Q] * zbar[mq])
    logratio = 2.0 * (logdet_new - logdet_old)
    logI = logratio + xxb - 0.5 * xbxb
    dtheta = float((logratio.imag + np.pi) % (2 * np.pi) - np.pi)
    if dtheta == -np.pi:
        dtheta = np.pi
    factor = float(np.exp(logI.real) * max(0.0, np.cos(dtheta)))
    return logI, dtheta, factor


def orthogonalize(phi_w):
    """Walker orthogonalisation: thin QR  Phi = Q R  with R upper triangular and a
    REAL POSITIVE diagonal (which makes Q unique), by modified Gram-Schmidt column by column.
    Returns (Q [M][N], log det R = sum_j log r_jj, real).  The Slater determinant changes only by the
    factor det R: Theta, vbias and the local energy are invariant (gauge invariance, R14)."""
    q = phi_w.astype(C128).copy()
    nn = q.shape[1]
    logdet_r = 0.0
    for j in range(nn):
        for i in range(j):
            rij = np.vdot(q[:, i], q[:, j])           # q_i^dagger a_j
            q[:, j] = q[:, j] - rij * q[:, i]
        rjj = np.sqrt(np.vdot(q[:, j], q[:, j]).real)
        q[:, j] = q[:, j] / rjj
        logdet_r += np.log(rjj)
    return q, logdet_r


def mixed_estimator(weight, energy):
    """Eq. 35: E_mixed = sum_w weight_w E_L[phi_w] / sum_w weight_w, E_L = E1 + EC + EX.
    Returns (numerator [3] complex = sum_w weight_w (E1, EC, EX)_w, denominator = sum_w weight_w)."""
    num = np.einsum('w,wc->c', weight.astype(np.float64), energy)
    return num, float(np.sum(weight))


def hybrid_step(mesh, L, Lh, psi_t, B1, phi_w, x_w, dtau, order):
    """One hybrid propagation step for one walker (Eq. 13, 15-19): force bias, vHS, B1 * Taylor * B1,
    overlap ratio and weight factor.  Returns (phi', log I, dtheta, factor, info)."""
    th, ld_old, info = green(psi_t, phi_w)
    vb = force_bias(mesh, Lh, th)
    xi = assemble_fields(mesh, x_w, vb, dtau)
    V = vhs(mesh, L, xi)
    t = apply_onebody(B1, phi_w)
    t = propagate(V, t, dtau, order)
    phi_new = apply_onebody(B1, t)
    lu, perm, sign, info2 = lu_factor(overlap(psi_t, phi_new))
    ld_new = lu_logdet(lu, sign)
    logI, dtheta, factor = hybrid_weight(mesh, x_w, vb, dtau, ld_old, ld_new)
    return phi_new, logI, dtheta, factor, max(info, info2)


def block(mesh, L, Lh, ht, psi_t, B1, phi, weight, x, dtau, order):
    """One AFQMC block: x.shape[0] hybrid propagation steps, then the local energy of
    every walker and the mixed estimator, then walker orthogonalisation.
      phi [nw][M][N], weight [nw] real, x [nsteps][nw][Nk][nchol] real.
    Returns (phi_out, weight_out, energy [nw][3], (num, den) of Eq. 35, logdetR [nw])."""
    nsteps, nw = x.shape[0], phi.shape[0]
    phi = phi.astype(C128).copy()
    weight = weight.astype(np.float64).copy()
    for s in range(nsteps):
        for w in range(nw):
            phi[w], _, _, factor, _ = hybrid_step(mesh, L, Lh, psi_t, B1, phi[w], x[s, w], dtau, order)
            weight[w] *= factor
    energy = np.empty((nw, 3), dtype=C128)
    logdet_r = np.empty(nw)
    for w in range(nw):
        th, _, _ = green(psi_t, phi[w])
        energy[w] = local_energy(mesh, Lh, ht, th)
    num, den = mixed_estimator(weight, energy)
    for w in range(nw):
        phi[w], logdet_r[w] = orthogonalize(phi[w])
    return phi, weight, energy, (num, den), logdet_r


# ======================================================================================
# OPEN SHELL: two spin channels, N_up != N_dn allowed.
# Eq. 36:  E = sum_{pq,s} h_pq G^s_pq + 1/2 sum_{pqrs} v_pqrs sum_{s,s'} [ G^s_pr G^s'_qs - delta_{ss'} G^s_ps G^s_qr ]
# Eq. 49 is the same in k-blocked, half-rotated form with its explicit sigma sums.
# A channel is (trial A^s [Nk][m][n_s], walker Phi^s [M][N_s]); the closed shell is the case A^up = A^dn, Phi^up = Phi^dn,
# where these functions reduce to the closed-shell ones above (factors 2, 4, 2).
# ======================================================================================

# ---- level D ----
def dense_vbias_uhf(Lsc, G_up, G_dn):
    """v_Gamma = sum_sigma sum_pr L_{pr,Gamma} G^sigma_pr  (Eq. 25/37 summed over spin, no prefactor)."""
    return np.einsum('prg,pr->g', Lsc, G_up) + np.einsum('prg,pr->g', Lsc, G_dn)


def dense_energy_uhf(H, V, G_up, G_dn):
    """Eq. 36 with both spin sums explicit:
    E1 = sum_s sum_pq h_pq G^s_pq;  EC = 1/2 sum_{s,s'} sum v_pqrs G^s_pr G^s'_qs;
    EX = -1/2 sum_s sum v_pqrs G^s_ps G^s_qr   (delta_{ss'}: exchange only between like spins)."""
    e1 = 0.0 + 0.0j
    ec = 0.0 + 0.0j
    ex = 0.0 + 0.0j
    for Gs in (G_up, G_dn):
        e1 += np.einsum('pq,pq->', H, Gs)
        ex += -0.5 * np.einsum('pqrs,ps,qr->', V, Gs, Gs)
        for Gt in (G_up, G_dn):
            ec += 0.5 * np.einsum('pqrs,pr,qs->', V, Gs, Gt)
    return np.array([e1, ec, ex], dtype=C128)


# ---- level P ----
def force_bias_uhf(mesh, Lh_up, Lh_dn, theta_up, theta_dn):
    """a4, open shell: vbias[Q][gamma] = sum_sigma sum_k sum_{a,r} Lh^sigma[Q][k][a][gamma][r] Theta^sigma[(k,a),(k-Q,r)]
    (Eq. 47 with its spin sum).  `force_bias` above carries the closed-shell factor 2 = two equal channels."""
    return 0.5 * (force_bias(mesh, Lh_up, theta_up) + force_bias(mesh, Lh_dn, theta_dn))


def local_energy_uhf(mesh, Lh_s, ht_s, theta_s):
    """a7-a9, open shell, by the paper's steps 1-3 with the loop over sigma of step 2 written out.
    `Lh_s`, `ht_s`, `theta_s` are 2-tuples (up, dn).  The traces v_1, v_2 of step 2(d) are summed over BOTH spins before
    step 3 multiplies them (the Coulomb term couples the channels: sigma, sigma' independent in Eq. 49), while the exchange
    contribution of step 2(c) is accumulated per spin (delta_{sigma sigma'})."""
    nk = Lh_s[0].shape[0]
    nchol = Lh_s[0].shape[3]
    e1 = 0.0 + 0.0j
    ex = 0.0 + 0.0j
    ec = 0.0 + 0.0j
    G_s = []
    for Lh, ht, theta_w in zip(Lh_s, ht_s, theta_s):
        n, m = Lh.shape[2], Lh.shape[4]
        G = reshape_theta(theta_w, nk, n, m)                # step 1, per spin
        G_s.append(G)
        for k in range(nk):                                 # Eq. 49 line 1
            e1 += np.sum(ht[k] * G[k, k])
    for Q in range(nk):
        mQ = k_neg(mesh, Q)
        v1 = np.zeros(nchol, dtype=C128)
        v2 = np.zeros(nchol, dtype=C128)
        for Lh, G in zip(Lh_s, G_s):                        # step 2: "for each (sigma, Q, k, k')"
            for k in range(nk):
                kq = k_sub(mesh, k, Q)
                for kp in range(nk):
                    kpq = k_sub(mesh, kp, Q)
                    T1 = np.einsum('agr,br->bag', Lh[Q, k], G[kpq, kq])        # 2(a)
                    T2 = np.einsum('bgs,as->abg', Lh[mQ, kpq], G[k, kp])       # 2(b)
                    ex += -0.5 * np.einsum('bag,abg->', T1, T2)                # 2(c)
                    if kpq == k:                                                # 2(d)
                        v1 += np.einsum('aag->g', T1)
                        v2 += np.einsum('aag->g', T2)
        ec += 0.5 * np.sum(v1 * v2)                                            # step 3, summed over Q
    return np.array([e1, ec, ex], dtype=C128)


def step_uhf(mesh, L, Lh_s, ht_s, psi_t_s, phi_s, x, dtau, order):
    """The timed composition for open-shell walkers: per walker, Green's function of both channels, the spin-summed force
    bias, ONE vHS (spin independent), the same Taylor propagator on both channels, then overlap + Green + local energy of
    the new walker.  phi_s = (phi_up [nw][M][N_up], phi_dn [nw][M][N_dn]).
    Returns ((phi_up', phi_dn'), energy [nw][3], logdet [nw] = log det O_up + log det O_dn)."""
    nw = phi_s[0].shape[0]
    out = (np.empty_like(phi_s[0]), np.empty_like(phi_s[1]))
    energy = np.empty((nw, 3), dtype=C128)
    logdet = np.empty(nw, dtype=C128)
    for w in range(nw):
        th = [green(psi_t_s[s], phi_s[s][w])[0] for s in range(2)]
        vb = force_bias_uhf(mesh, Lh_s[0], Lh_s[1], th[0], th[1])
        xi = assemble_fields(mesh, x[w], vb, dtau)
        V = vhs(mesh, L, xi)
        th2, ld = [], 0.0 + 0.0j
        for s in range(2):
            out[s][w] = propagate(V, phi_s[s][w], dtau, order)
            t2, l2, _ = green(psi_t_s[s], out[s][w])
            th2.append(t2)
            ld += l2
        energy[w] = local_energy_uhf(mesh, Lh_s, ht_s, th2)
        logdet[w] = complex(ld.real, (ld.imag + np.pi) % (2 * np.pi) - np.pi)
    return out, energy, logdet
