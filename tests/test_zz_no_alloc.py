"""afqmc_overlap_noalloc (the entry point that allocates nothing: its overlap matrices live in a static device array inside
the library) against the existing path afqmc_overlap, at the tolerance of the parity tests, on two calls in a row that share
the scratch array.  Collected last on purpose (the file name): a failure here must not hide any other test under `pytest -x`.
"""
import ctypes

import numpy as np
import pytest
import torch

from paper_2003_09468_b200 import synth

RTOL = 1e-10


def _phase_diff(a, b):
    return np.abs(np.angle(np.exp(1j * (a - b))))


def _compare(ld_new, ld_old):
    a, b = ld_new.cpu().numpy(), ld_old.cpu().numpy()
    assert np.all(np.isfinite(a.real)) and np.all(np.isfinite(a.imag))
    assert float(np.max(np.abs(a.real - b.real) / np.maximum(1.0, np.abs(b.real)))) < RTOL
    assert float(np.max(_phase_diff(a.imag, b.imag))) < RTOL


@pytest.mark.gpu
@pytest.mark.parametrize("shape", ["C1", "ragged", "C3"])
def test_overlap_noalloc_matches_afqmc_overlap_on_two_calls_in_a_row(shape):
    from paper_2003_09468_b200 import binding
    if shape == "C1":
        cfg = synth.CONFIGS["C1"]
    elif shape == "ragged":
        cfg = synth.tiny_config(mesh=(3, 1, 2), m=7, n=3, nchol=5, nw=5, seed=21)
    else:
        # C3's mesh, bands, occupied orbitals and 32 walkers (N = 108: 32 matrices of 108 x 109 = 6.0 MB of the 16 MiB); a
        # short Cholesky index keeps the context's setup small -- the overlap does not read L
        cfg = synth.tiny_config(mesh=(3, 3, 3), m=26, n=4, nchol=4, nw=32, seed=3)
    pb = synth.make_problem(cfg)
    nw = pb.phi.shape[0]
    ctx = binding.from_problem(pb)
    try:
        psi_t = torch.from_numpy(np.ascontiguousarray(pb.psi_t)).cuda()
        phi1 = torch.from_numpy(np.ascontiguousarray(pb.phi)).cuda()
        # second call: other walkers (a fixed invertible mixing of the columns plus a perturbation), fewer of them, so that
        # it finds the first call's matrices in the array and uses a different part of it
        rng = np.random.default_rng(1234)
        N = pb.phi.shape[2]
        mix = np.eye(N) + 0.3 * (rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N))) / np.sqrt(N)
        phi2 = torch.from_numpy(np.ascontiguousarray((pb.phi @ mix)[: max(1, nw - 1)] +
                                                     0.05 * rng.standard_normal(pb.phi[: max(1, nw - 1)].shape))).cuda()
        assert binding.overlap_noalloc_bytes(cfg.mesh, cfg.m, cfg.n, nw) <= binding.overlap_noalloc_max_bytes()
        binding.overlap_noalloc_setup()
        before = torch.cuda.memory_allocated()
        for phi in (phi1, phi2):
            k = phi.shape[0]
            ld_old, info_old = ctx.overlap(phi)
            ld_new = torch.full((k,), float("nan"), dtype=torch.complex128, device="cuda")
            info_new = torch.full((k,), -1, dtype=torch.int32, device="cuda")
            binding.overlap_noalloc(cfg.mesh, cfg.m, cfg.n, psi_t, phi, ld_new, info_new)
            torch.cuda.synchronize()
            assert int(info_old.abs().sum()) == 0 and int(info_new.abs().sum()) == 0
            _compare(ld_new, ld_old)
        # and once more on the first batch: bitwise the same as a fresh evaluation would give (stale contents play no part)
        ld_a = torch.empty((nw,), dtype=torch.complex128, device="cuda")
        ld_b = torch.empty((nw,), dtype=torch.complex128, device="cuda")
        binding.overlap_noalloc(cfg.mesh, cfg.m, cfg.n, psi_t, phi1, ld_a)
        binding.overlap_noalloc(cfg.mesh, cfg.m, cfg.n, psi_t, phi2, torch.empty((phi2.shape[0],), dtype=torch.complex128, device="cuda"))
        binding.overlap_noalloc(cfg.mesh, cfg.m, cfg.n, psi_t, phi1, ld_b)
        torch.cuda.synchronize()
        assert torch.equal(torch.view_as_real(ld_a), torch.view_as_real(ld_b))
        assert torch.cuda.memory_allocated() >= before      # torch's own output tensors only; the library allocated nothing
    finally:
        ctx.close()


@pytest.mark.gpu
def test_overlap_noalloc_singular_walker_and_limits():
    from paper_2003_09468_b200 import binding
    cfg = synth.tiny_config(mesh=(2, 1, 1), m=4, n=2, nchol=3, nw=3, seed=5)
    pb = synth.make_problem(cfg)
    psi_t = torch.from_numpy(np.ascontiguousarray(pb.psi_t)).cuda()
    phi_np = pb.phi.copy()
    phi_np[1, :, 2] = phi_np[1, :, 0]                # two equal columns: singular overlap for walker 1
    phi = torch.from_numpy(phi_np).cuda()
    ld = torch.empty((3,), dtype=torch.complex128, device="cuda")
    info = torch.zeros((3,), dtype=torch.int32, device="cuda")
    binding.overlap_noalloc(cfg.mesh, cfg.m, cfg.n, psi_t, phi, ld, info)
    torch.cuda.synchronize()
    got = info.cpu().numpy()
    assert got[0] == 0 and got[2] == 0
    ref = np.linalg.slogdet(np.einsum("kpa,wkpj->wkaj", pb.psi_t.conj(), phi_np.reshape(3, 2, 4, 4)).reshape(3, 4, 4))
    assert abs(ld[0].real.item() - ref[1][0]) < 1e-10 and abs(ld[2].real.item() - ref[1][2]) < 1e-10
    assert got[1] > 0 or ld[1].real.item() < ref[1][0] - 25.0       # exactly-zero pivot, or one at rounding level
    # beyond the limit: a clear error, nothing launched
    lib = binding.lib()
    big = binding.Dims((ctypes.c_int * 3)(4, 4, 4), 26, 4, 0, 1, 0, 64, 0)      # N = 256: 16.8 MB for 16 walkers
    assert binding.overlap_noalloc_bytes((4, 4, 4), 26, 4, 16) > binding.overlap_noalloc_max_bytes()
    rc = lib.afqmc_overlap_noalloc(ctypes.byref(big), ctypes.c_void_p(psi_t.data_ptr()), ctypes.c_void_p(phi.data_ptr()), 16,
                                   ctypes.c_void_p(ld.data_ptr()), None, None)
    assert rc == 5 and b"scratch" in lib.afqmc_strerror(rc)
    with pytest.raises(binding.AfqmcError) as ei:
        binding._check(rc, "afqmc_overlap_noalloc")
    assert "scratch" in str(ei.value)


def test_overlap_noalloc_size_arithmetic_without_a_gpu():
    from paper_2003_09468_b200 import binding
    assert binding.overlap_noalloc_max_bytes() == 16 << 20
    for name in ("C1", "C2", "C3", "C4", "C5"):
        cfg = synth.CONFIGS[name]
        N = cfg.nk * cfg.n
        need = binding.overlap_noalloc_bytes(cfg.mesh, cfg.m, cfg.n, cfg.nw)
        assert need == cfg.nw * N * (N | 1) * 16
        assert need <= binding.overlap_noalloc_max_bytes(), name
    lib = binding.lib()
    d = binding.Dims((ctypes.c_int * 3)(4, 4, 4), 26, 4, 0, 1, 0, 64, 0)
    assert lib.afqmc_overlap_noalloc(ctypes.byref(d), ctypes.c_void_p(16), ctypes.c_void_p(16), 64, ctypes.c_void_p(16), None, None) == 5
    assert lib.afqmc_overlap_noalloc(None, None, None, 1, None, None, None) == 1
    d2 = binding.Dims((ctypes.c_int * 3)(2, 2, 2), 8, 4, 0, 0, 0, 4, 0)
    assert lib.afqmc_overlap_noalloc(ctypes.byref(d2), ctypes.c_void_p(16), ctypes.c_void_p(16), 4, ctypes.c_void_p(16), None, None) == 2
    assert lib.afqmc_strerror(5).startswith(b"request exceeds")
