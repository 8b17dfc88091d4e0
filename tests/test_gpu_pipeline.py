"""afqmc_step_host_begin / afqmc_step_host_end (two host-buffer steps in flight): every step of a pipelined sequence of
different walker batches returns bit for bit what the synchronous afqmc_step_host returns for that batch -- the host-link
traffic of neighbouring steps overlaps, their arithmetic does not change.  The synchronous call itself is compared with the
oracle in test_gpu_parity.py."""
import numpy as np
import pytest
import torch

from paper_2003_09468_b200 import synth

pytestmark = pytest.mark.gpu


def _batches(pb, nbatch, nw):
    """nbatch different walker batches from the problem's walkers: column mixings with fixed seeds (any invertible mixing is
    a valid walker), and their own fields."""
    rng = np.random.default_rng(77)
    N = pb.phi.shape[2]
    out = []
    for b in range(nbatch):
        mix = np.eye(N) + 0.2 * (rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N))) / np.sqrt(N)
        phi = np.ascontiguousarray((pb.phi[:nw] @ mix))
        x = rng.standard_normal(pb.x[:nw].shape)
        out.append((phi, x))
    return out


@pytest.mark.parametrize("shape", ["C1", "ragged", "C2"])
def test_pipelined_host_steps_equal_the_synchronous_call(shape):
    from paper_2003_09468_b200 import binding
    if shape == "C1":
        cfg, nw = synth.CONFIGS["C1"], 4
    elif shape == "ragged":
        cfg, nw = synth.tiny_config(mesh=(3, 1, 2), m=7, n=3, nchol=5, nw=5, seed=11), 5
    else:
        cfg, nw = synth.CONFIGS["C2"], 24          # fewer walkers than the context's maximum
    pb = synth.make_problem(cfg)
    ctx = binding.from_problem(pb)
    try:
        nb = 5
        batches = _batches(pb, nb, nw)
        pin = lambda a: torch.from_numpy(a).pin_memory()
        phi_in = [pin(p) for p, _ in batches]
        x_in = [pin(x) for _, x in batches]
        # reference: the synchronous call, one batch at a time (phi in place)
        ref = []
        for b in range(nb):
            ph = pin(batches[b][0].copy())
            e = torch.empty((nw, 3), dtype=torch.complex128).pin_memory()
            ld = torch.empty((nw,), dtype=torch.complex128).pin_memory()
            info = torch.empty((nw,), dtype=torch.int32).pin_memory()
            ctx.step_host(ph, x_in[b], cfg.dtau, cfg.order, e, ld, info)
            ref.append((ph.clone(), e.clone(), ld.clone(), info.clone()))
        # pipelined: two in flight, outputs into per-batch buffers; inputs are left untouched (phi_out != phi_in)
        out = [(torch.empty_like(phi_in[b]).pin_memory(), torch.empty((nw, 3), dtype=torch.complex128).pin_memory(),
                torch.empty((nw,), dtype=torch.complex128).pin_memory(), torch.empty((nw,), dtype=torch.int32).pin_memory())
               for b in range(nb)]
        for rep in range(2):               # the second pass reuses both slots' staging buffers
            for o in out:
                o[0].zero_(); o[1].zero_()
            for b in range(nb):
                ctx.step_host_begin(b & 1, phi_in[b], x_in[b], cfg.dtau, cfg.order, out[b][0], out[b][1], out[b][2], out[b][3])
            ctx.step_host_end(0)
            ctx.step_host_end(1)
            for b in range(nb):
                assert torch.equal(phi_in[b], torch.from_numpy(batches[b][0])), "input buffer was modified"
                for got, want, name in zip(out[b], ref[b], ("phi", "energy", "logdet", "info")):
                    assert torch.equal(torch.view_as_real(got) if got.is_complex() else got,
                                       torch.view_as_real(want) if want.is_complex() else want), (rep, b, name)
        # in place (phi_out = phi_in), a synchronous call while a slot is busy, and end on an idle slot
        ph0, ph1 = pin(batches[0][0].copy()), pin(batches[1][0].copy())
        e0 = torch.empty((nw, 3), dtype=torch.complex128).pin_memory()
        e1 = torch.empty((nw, 3), dtype=torch.complex128).pin_memory()
        ctx.step_host_begin(1, ph1, x_in[1], cfg.dtau, cfg.order, ph1, e1)
        ctx.step_host(ph0, x_in[0], cfg.dtau, cfg.order, e0)        # completes slot 1 first, then runs
        ctx.step_host_end(1)
        ctx.step_host_end(0)
        assert torch.equal(torch.view_as_real(ph0), torch.view_as_real(ref[0][0]))
        assert torch.equal(torch.view_as_real(ph1), torch.view_as_real(ref[1][0]))
        assert torch.equal(torch.view_as_real(e0), torch.view_as_real(ref[0][1]))
        assert torch.equal(torch.view_as_real(e1), torch.view_as_real(ref[1][1]))
        with pytest.raises(binding.AfqmcError):
            ctx.step_host_begin(2, ph0, x_in[0], cfg.dtau, cfg.order, ph0, e0)
    finally:
        ctx.close()
