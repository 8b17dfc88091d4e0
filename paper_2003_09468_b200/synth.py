"""Seeded synthetic inputs for the k-point AFQMC step (shared by tests, oracle runs and bench).

This module holds NONE of the method's arithmetic: it only draws random tensors with the
shapes, value distributions and symmetry structure of the paper's workloads and hands the
same host arrays to both the CUDA library and the CPU oracle.  The recipe is the one in
BASELINE.json `configs` / SURVEY.md 8(d) and is restated in DESIGN.md ("Input recipe"):

* mesh g1 x g2 x g3, k-point linear index (i1*g2 + i2)*g3 + i3 (Gamma-centred regular
  grid);
* ``L[Q][k][gamma][p][r]`` (p at k, r at k-Q) ~ CN(0, 1/m), built so that the
  block at (-Q, k-Q) is the conjugate transpose (per gamma) of the block at (Q, k)
  (the (Q,-Q) identity of PAPER.md:216); the self-partner blocks (Q = 0) are (G + G^H)/sqrt 2;
* ``h1[k]`` Hermitian (G + G^H)/2 with G ~ CN(0,1);
* ``psi_t[k]``: Q factor of the thin QR of an m x n CN(0,1) matrix (trial block-diagonal in
  k);
* walkers: QR-orthonormalised (trial + 0.1 CN(0,1)) as dense M x N matrices;
* fields x ~ N(0,1) real, one per (walker, Q, gamma).

CN(0, s2) means E|z|^2 = s2 (real and imaginary parts N(0, s2/2) each).
The draw order is fixed: h1, psi_t, L (canonical blocks in (Q,k) index order), walkers, x.
"""
from __future__ import annotations

from dataclasses import dataclass, field
import numpy as np


@dataclass(frozen=True)
class Config:
    name: str
    mesh: tuple
    m: int
    n: int
    nchol: int
    nw: int
    dtau: float = 0.005
    order: int = 6
    seed: int = 0

    @property
    def nk(self) -> int:
        return self.mesh[0] * self.mesh[1] * self.mesh[2]

    @property
    def M(self) -> int:
        return self.nk * self.m

    @property
    def N(self) -> int:
        return self.nk * self.n


# The five BASELINE.json configs (C1..C5).  C3 is the headline benchmark.
CONFIGS = {
    "C1": Config("C1", (2, 2, 2), 8, 4, 32, 4),
    "C2": Config("C2", (2, 2, 2), 26, 4, 160, 64),
    "C3": Config("C3", (3, 3, 3), 26, 4, 200, 32),
    "C4": Config("C4", (3, 3, 3), 52, 4, 400, 16),
    "C5": Config("C5", (4, 4, 4), 26, 4, 200, 8),
    # NOT a BASELINE.json config: the dense Gamma-point supercell shape of SURVEY.md 8(f) NEXT-4 (one k-point, large m and n:
    # the 2x2x2 cell of C2 written as a single cell), which runs the same kernels at a very different
    # tile shape (n = 32 occupied orbitals: eight a-groups in the exchange kernel, N = 32, M = 208).
    "G1": Config("G1", (1, 1, 1), 208, 32, 1040, 16),
}


def kpoint_tables(mesh):
    """Index tables of the regular mesh: ``kminus[k, Q]`` = index of k-Q, ``neg[Q]`` = index of -Q.

    Pure index bookkeeping, needed only to place the conjugate-transpose partner blocks.
    """
    g1, g2, g3 = mesh
    nk = g1 * g2 * g3
    coords = np.array([(a, b, c) for a in range(g1) for b in range(g2) for c in range(g3)])
    g = np.array(mesh)

    def lin(c):
        return (c[..., 0] * g2 + c[..., 1]) * g3 + c[..., 2]

    kminus = lin((coords[:, None, :] - coords[None, :, :]) % g)  # [k, Q]
    neg = lin((-coords) % g)
    assert kminus.shape == (nk, nk)
    return kminus.astype(np.int64), neg.astype(np.int64)


def _cn(rng, shape, var):
    z = rng.standard_normal(shape + (2,))
    z *= np.sqrt(var / 2.0)
    return z.view(np.complex128)[..., 0]


def _rn(rng, shape, var):
    """Real draws of the same variance, stored as complex128 with zero imaginary parts (real orbitals)."""
    return (rng.standard_normal(shape) * np.sqrt(var)).astype(np.complex128)


@dataclass
class Problem:
    cfg: Config
    h1: np.ndarray      # [Nk][m][m]
    psi_t: np.ndarray   # [Nk][m][n]
    L: np.ndarray       # [Nk(Q)][Nk(k)][nchol][m][m]
    phi: np.ndarray     # [nw][M][N]
    x: np.ndarray       # [nw][Nk][nchol] float64
    extra: dict = field(default_factory=dict)


def make_hamiltonian(cfg: Config, rng, real_orbitals=False):
    """`real_orbitals`: h1, psi_t and L are drawn REAL (same shapes, variances and symmetry structure): the dense Gamma-point
    supercell representation with real orbitals of PAPER.md:260, :276-284.  Walkers stay complex."""
    nk, m, n, nchol = cfg.nk, cfg.m, cfg.n, cfg.nchol
    kminus, neg = kpoint_tables(cfg.mesh)
    _cn = globals()["_rn"] if real_orbitals else globals()["_cn"]
    g = _cn(rng, (nk, m, m), 1.0)
    h1 = 0.5 * (g + np.conj(np.swapaxes(g, -1, -2)))
    psi_t = np.empty((nk, m, n), dtype=np.complex128)
    for k in range(nk):
        q, _ = np.linalg.qr(_cn(rng, (m, n), 1.0))
        psi_t[k] = q
    L = np.empty((nk, nk, nchol, m, m), dtype=np.complex128)
    for Q in range(nk):
        for k in range(nk):
            Qp, kp = int(neg[Q]), int(kminus[k, Q])
            if (Qp, kp) < (Q, k):
                continue  # filled as the partner of an earlier canonical block
            blk = _cn(rng, (nchol, m, m), 1.0 / m)
            if (Qp, kp) == (Q, k):
                blk = (blk + np.conj(np.swapaxes(blk, -1, -2))) / np.sqrt(2.0)
                L[Q, k] = blk
            else:
                L[Q, k] = blk
                L[Qp, kp] = np.conj(np.swapaxes(blk, -1, -2))
    return np.ascontiguousarray(h1), np.ascontiguousarray(psi_t), L


def make_walkers(cfg: Config, psi_t, rng, nw=None, noise=0.1):
    nk, m, n = cfg.nk, cfg.m, cfg.n
    nw = cfg.nw if nw is None else nw
    A = np.zeros((cfg.M, cfg.N), dtype=np.complex128)
    for k in range(nk):
        A[k * m:(k + 1) * m, k * n:(k + 1) * n] = psi_t[k]
    phi = np.empty((nw, cfg.M, cfg.N), dtype=np.complex128)
    for w in range(nw):
        q, _ = np.linalg.qr(A + noise * _cn(rng, (cfg.M, cfg.N), 1.0))
        phi[w] = q
    return phi


def make_problem(cfg: Config, nw=None, l_scale=1.0, real_orbitals=False) -> Problem:
    """`l_scale` multiplies L after the draw (same random stream).  1.0 is BASELINE.json's recipe, whose
    sqrt(dtau)*vHS has norm 2-16 (R9): every kernel is tested there, but in a hybrid AFQMC block such
    steps rotate the overlap phase by more than pi/2 and the phaseless projection sets most weights to 0.  The
    block tests and the block bench therefore also use a 'physically scaled' L (l_scale ~ 0.05-0.1, steps of
    norm < 1), as SURVEY.md P9 suggests; shapes and structure are unchanged."""
    rng = np.random.default_rng(cfg.seed)
    h1, psi_t, L = make_hamiltonian(cfg, rng, real_orbitals)
    if l_scale != 1.0:
        L *= l_scale
    phi = make_walkers(cfg, psi_t, rng, nw)
    x = rng.standard_normal((phi.shape[0], cfg.nk, cfg.nchol))
    return Problem(cfg, h1, psi_t, L, phi, x)


def tiny_config(mesh=(2, 3, 1), m=3, n=2, nchol=4, nw=2, seed=1, dtau=0.005, order=6):
    """Small configs for the definition-level (dense 4-index) oracle checks."""
    return Config("tiny%dx%dx%d" % tuple(mesh), tuple(mesh), m, n, nchol, nw, dtau, order, seed)


def make_block_fields(cfg: Config, nsteps: int, nw=None, seed_offset=7):
    """Auxiliary fields for one AFQMC block (a block = `nsteps` propagation steps, 20 in the
    paper): x[nsteps][nw][Nk][nchol] ~ N(0,1), from their own stream `seed + seed_offset` so the single-step
    inputs of `make_problem` are unchanged.  Initial weights are 1 (the caller's array)."""
    nw = cfg.nw if nw is None else nw
    rng = np.random.default_rng(cfg.seed + seed_offset)
    return rng.standard_normal((nsteps, nw, cfg.nk, cfg.nchol))


# ---- open-shell inputs: a second spin channel with its own occupied count ----
def make_open_shell(cfg: Config, n_dn: int, nw=None, seed_offset=101):
    """Adds a spin-DOWN channel with `n_dn` occupied orbitals per k-point to `make_problem(cfg)` (whose trial and walkers
    become the spin-UP channel, n_up = cfg.n): an independent random orthonormal trial block per k and walkers drawn the same
    way (trial + 0.1 CN(0,1), thin QR), from their own stream `seed + seed_offset`.  Returns (problem, psi_t_dn [Nk][m][n_dn],
    phi_dn [nw][M][Nk*n_dn]); the Hamiltonian and the fields are shared by both channels."""
    pb = make_problem(cfg, nw)
    rng = np.random.default_rng(cfg.seed + seed_offset)
    nk, m = cfg.nk, cfg.m
    psi_dn = np.empty((nk, m, n_dn), dtype=np.complex128)
    for k in range(nk):
        q, _ = np.linalg.qr(_cn(rng, (m, n_dn), 1.0))
        psi_dn[k] = q
    cfg_dn = Config(cfg.name + "_dn", cfg.mesh, m, n_dn, cfg.nchol, pb.phi.shape[0], cfg.dtau, cfg.order, cfg.seed)
    phi_dn = make_walkers(cfg_dn, psi_dn, rng, pb.phi.shape[0])
    return pb, psi_dn, phi_dn
