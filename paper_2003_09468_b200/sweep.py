"""Walker-batch sweep: time per walker of each stage of the step as a function of the
number of walkers processed together, in the spirit of Fig. 3-5 of the paper (speedup of the
energy evaluation, the propagation and the Green's function with the batch size Nw, at 8 and 27 k-points).

    python -m paper_2003_09468_b200.sweep [--configs C2 C3] [--walkers 1 2 4 8 16 32 64] [--reps 5] [--md out.md]

Every stage is the library's own kernel path through the C-ABI (afqmc_step with stage timers); inputs are the
seeded synthetic tensors of `synth` with the shapes of the named config and `nw` walkers.  "Speedup" of a stage
at batch size nw is  t(1 walker) * nw / t(nw walkers), the paper's definition ("with respect to sequential
execution ... but processing all walkers simultaneously").  No arithmetic of the method lives here.
"""
from __future__ import annotations

import argparse
import json
import sys

STAGE_GROUPS = {
    "green (a1-a3)": ("green",),
    "force bias (a4)": ("force_bias",),
    "vHS (a5)": ("vhs",),
    "propagate (a6)": ("propagate",),
    "energy (a7-a9)": ("force_bias2", "exchange", "finalize"),
}


def run_config(name, walkers, reps):
    import torch
    from . import binding, synth
    cfg = synth.CONFIGS[name]
    nmax = max(walkers)
    pb = synth.make_problem(cfg, nw=nmax)
    ctx = binding.from_problem(pb, max_walkers=nmax)
    ctx.set_option("timers", 1)
    phi_all = torch.from_numpy(pb.phi).cuda()
    x_all = torch.from_numpy(pb.x).cuda()
    rows = []
    for nw in walkers:
        x = x_all[:nw].contiguous()
        acc = {}
        for it in range(reps + 2):
            phi = phi_all[:nw].clone()
            ctx.step(phi, x, cfg.dtau, cfg.order)
            torch.cuda.synchronize()
            if it >= 2:
                for k, v in ctx.stage_times().items():
                    acc[k] = acc.get(k, 0.0) + v / reps
        row = {"config": name, "nw": nw, "step_ms": sum(acc.values())}
        for g, keys in STAGE_GROUPS.items():
            row[g] = sum(acc[k] for k in keys)
        rows.append(row)
    ctx.close()
    base = rows[0]
    for r in rows:
        r["speedup"] = {g: base[g] * r["nw"] / base["nw"] / r[g] for g in STAGE_GROUPS}
        r["speedup"]["step"] = base["step_ms"] * r["nw"] / base["nw"] / r["step_ms"]
    return rows


def to_markdown(rows):
    out = []
    for name in sorted({r["config"] for r in rows}):
        sel = [r for r in rows if r["config"] == name]
        out.append("### %s\n" % name)
        out.append("| walkers | step ms | ms per walker | " + " | ".join("%s ms (speedup)" % g for g in STAGE_GROUPS) + " | step speedup |")
        out.append("|---|---|---|" + "---|" * (len(STAGE_GROUPS) + 1))
        for r in sel:
            cells = ["%.3f (x%.1f)" % (r[g], r["speedup"][g]) for g in STAGE_GROUPS]
            out.append("| %d | %.3f | %.3f | %s | x%.1f |" % (r["nw"], r["step_ms"], r["step_ms"] / r["nw"], " | ".join(cells),
                                                             r["speedup"]["step"]))
        out.append("")
    return "\n".join(out)


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__.split("\n\n")[0])
    ap.add_argument("--configs", nargs="+", default=["C2", "C3"])
    ap.add_argument("--walkers", nargs="+", type=int, default=[1, 2, 4, 8, 16, 32, 64])
    ap.add_argument("--reps", type=int, default=5)
    ap.add_argument("--md", default=None, help="also write the tables as markdown to this file")
    args = ap.parse_args(argv)
    rows = []
    for name in args.configs:
        rows += run_config(name, sorted(args.walkers), args.reps)
    for r in rows:
        print(json.dumps(r))
    md = to_markdown(rows)
    if args.md:
        with open(args.md, "w") as f:
            f.write(md + "\n")
    print(md, file=sys.stderr)


if __name__ == "__main__":
    main()
