"""Runs ONE C-ABI call of the step a few times on a synthetic config: the command line that the ncu captures under
`profiles/` name (a whole `bench.py` run replays every kernel ~40 times under `ncu --set full`; this runs just the call).

  python -m paper_2003_09468_b200.run_call --config C3 --call local_energy --reps 2 [--walkers 8] [--option exchange_regb=2 ...]

calls: green, force_bias, vhs, propagate, local_energy, step.  Inputs: `synth.make_problem` of the config (seeded); Theta
is the Green's function of the config's walkers; nothing here is timed or checked (tests/ and bench.py do that).
"""
from __future__ import annotations

import argparse

import torch

from . import binding, synth


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", default="C3", choices=sorted(synth.CONFIGS))
    ap.add_argument("--call", default="local_energy", choices=["green", "force_bias", "vhs", "propagate", "local_energy", "step"])
    ap.add_argument("--reps", type=int, default=2)
    ap.add_argument("--precision", type=int, default=0)
    ap.add_argument("--walkers", type=int, default=0, help="use only the first N walkers of the config (0 = all)")
    ap.add_argument("--option", action="append", default=[], help="name=value, passed to afqmc_set_option")
    a = ap.parse_args()
    cfg = synth.CONFIGS[a.config]
    pb = synth.make_problem(cfg)
    ctx = binding.from_problem(pb, precision=a.precision)
    for o in a.option:
        k, v = o.split("=")
        ctx.set_option(k, int(v))
    cd = torch.complex64 if a.precision == 1 else torch.complex128
    rd = torch.float32 if a.precision == 1 else torch.float64
    nw = a.walkers if a.walkers > 0 else pb.phi.shape[0]
    phi = torch.from_numpy(pb.phi[:nw].copy()).cuda().to(cd)
    x = torch.from_numpy(pb.x[:nw].copy()).cuda().to(rd)
    theta, _, _ = ctx.green(phi)
    vb = ctx.force_bias(theta)
    vhs = ctx.vhs(x, vb, cfg.dtau) if a.call in ("vhs", "propagate") else None
    out = None
    for _ in range(a.reps):
        if a.call == "green":
            out = ctx.green(phi)[0]
        elif a.call == "force_bias":
            out = ctx.force_bias(theta)
        elif a.call == "vhs":
            out = ctx.vhs(x, vb, cfg.dtau)
        elif a.call == "propagate":
            out = ctx.propagate(vhs, cfg.dtau, cfg.order, phi.clone())
        elif a.call == "local_energy":
            out = ctx.local_energy(theta)
        else:
            out = ctx.step(phi.clone(), x, cfg.dtau, cfg.order)[0]
    torch.cuda.synchronize()
    print("%s x %d on %s: ok (|out| sum %.6e)" % (a.call, a.reps, a.config, float(out.abs().sum())))
    ctx.close()


if __name__ == "__main__":
    main()
