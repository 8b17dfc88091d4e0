#!/usr/bin/env python
"""bench.py -- walker-steps/s (incl. local energy) of the k-point ph-AFQMC step on B200.

One "step" = one pass of the whole hot path over the walker batch (afqmc_step: green, force bias,
vHS, 6th-order Taylor propagation, green on the new walkers, local energy with the exchange
contraction).  Workload at N=1: BASELINE.json config C3 (3x3x3 k-mesh,
m=26, n=4, nchol=200, 32 walkers, complex128), the config the metric is quoted on; seeded synthetic
inputs (paper_2003_09468_b200/synth.py).  N>1: independent replicas, one per GPU/rank, walkers
sharded by rank with no data-path collective (weak scaling).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C3] [--impl ours|reference]

Prints ONE JSON line on rank 0.  `--impl reference` times the CPU oracle (oracle/afqmc_oracle.py, as
it stands) on the host cores on a bounded sample (one walker per "step").
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "walker-steps/s incl. local energy"
UNIT = "walker-steps/s"

# dram__bytes_read.sum + dram__bytes_write.sum of ONE exchange-kernel launch: bench.py cannot measure DRAM traffic itself, so
# it reads the committed ncu capture of the default exchange kernel (a text file; profiles/r02l_summary.md names the command;
# the `--set full` capture of the same kernel one commit earlier is profiles/r02c_ncu_exchange.md).  Only the configuration
# that was captured has a value.
EXCHANGE_DRAM_CAPTURES = {"C3": "profiles/r02l_exchange_dram.csv"}


def exchange_dram_traffic(config_name):
    """(bytes per launch, source) from the committed ncu CSV, or (None, None)."""
    rel = EXCHANGE_DRAM_CAPTURES.get(config_name)
    if not rel:
        return None, None
    try:
        import csv
        total, seen = 0.0, set()
        with open(os.path.join(ROOT, rel), newline="") as f:
            for row in csv.reader(f):
                if len(row) >= 15 and row[12] in ("dram__bytes_read.sum", "dram__bytes_write.sum") and row[12] not in seen:
                    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}[row[13]]
                    total += float(row[14].replace(",", "")) * scale
                    seen.add(row[12])
        if len(seen) != 2:
            return None, None
        return total, rel + " (command: profiles/r02l_summary.md)"
    except (OSError, KeyError, ValueError):
        return None, None


def load_measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return json.load(open(p))
        except Exception:
            pass
    return None


class ClockSampler(threading.Thread):
    """Samples nvidia-smi clocks / throttle reasons every 200 ms while the timed region runs."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index = index
        self.samples = []
        self._halt = threading.Event()

    def run(self):
        while not self._halt.is_set():
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                      "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5).stdout
                f = [v.strip() for v in out.strip().split(",")]
                if len(f) >= 7:
                    self.samples.append(f)
            except Exception:
                pass
            self._halt.wait(0.2)

    def stop(self):
        self._halt.set()
        self.join(timeout=3)

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unsampled"]}
        sm = sorted(float(s[0]) for s in self.samples)
        reasons = []
        for i, name in enumerate(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")):
            if any(s[3 + i].lower().startswith("active") for s in self.samples):
                reasons.append(name)
        pw = max(float(s[2]) for s in self.samples)
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(self.samples[0][1]), "power_w_max": pw,
                "samples": len(sm), "reasons": reasons}


# ---- the CPU oracle on the host cores: one worker PROCESS per core, one walker per worker call.  The oracle itself is
# untouched (plain single-threaded numpy); the pool only runs several walkers side by side, which is how the step shards
# (walkers are independent).  Workers are forked BEFORE this process touches CUDA, inherit the problem copy-on-write and
# run numpy only.
_ORC = {}


def _oracle_job(w):
    from threadpoolctl import threadpool_limits
    o = _ORC
    with threadpool_limits(limits=1):
        t0 = time.perf_counter()
        o["orc"].step(o["cfg"].mesh, o["pb"].L, o["Lh"], o["ht"], o["pb"].psi_t, o["pb"].phi[w:w + 1], o["pb"].x[w:w + 1],
                      o["cfg"].dtau, o["cfg"].order)
        return time.perf_counter() - t0


def host_cores():
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


class OraclePool:
    """`cores` forked workers that each run orc.step for one walker at a time."""

    def __init__(self, cfg, pb, cores):
        import multiprocessing as mp
        from threadpoolctl import threadpool_limits
        from oracle import afqmc_oracle as orc
        with threadpool_limits(limits=1):
            Lh, ht = orc.half_rotate(pb.L, pb.psi_t, pb.h1)
        _ORC.update(orc=orc, cfg=cfg, pb=pb, Lh=Lh, ht=ht)
        self.cores = max(1, int(cores))
        self.pool = mp.get_context("fork").Pool(self.cores) if self.cores > 1 else None

    def run(self, walkers):
        """Wall seconds to do one full oracle step for each walker of `walkers`, `cores` at a time."""
        t0 = time.perf_counter()
        if self.pool is None:
            for w in walkers:
                _oracle_job(w)
        else:
            self.pool.map(_oracle_job, list(walkers), chunksize=1)
        return time.perf_counter() - t0

    def close(self):
        if self.pool is not None:
            self.pool.close()
            self.pool.join()
        _ORC.clear()


def run_reference(args):
    """The CPU oracle as the reference arm: each 'step' is the full step (overlap .. local energy) for one walker per
    host core in use, all cores side by side (bounded sample of the config's walker batch; work is linear in walkers)."""
    from paper_2003_09468_b200 import replicas, synth
    rank, _, world = replicas.rank_env()
    if rank != 0:
        return
    cfg = synth.CONFIGS[args.config]
    cores = min(host_cores() if args.cores <= 0 else args.cores, cfg.nw)
    pb = synth.make_problem(cfg, nw=cores)
    pool = OraclePool(cfg, pb, cores)
    try:
        for _ in range(args.warmup):
            pool.run(range(cores))
        tot = sum(pool.run(range(cores)) for _ in range(args.steps))
    finally:
        pool.close()
    value = cores * args.steps / tot
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "c128", "data": "synthetic",
        "config": {"workload": "%s: %dx%dx%d k-mesh, m=%d, n=%d, nchol=%d, complex128; %d walkers per step (one per host core)"
                               % ((cfg.name,) + tuple(cfg.mesh) + (cfg.m, cfg.n, cfg.nchol, cores))},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": "%d timed passes, each the full step (overlap..local energy) of %d walkers of %s side by side, "
                                   "one single-threaded numpy oracle process per core" % (args.steps, cores, cfg.name)},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def run_ours(args):
    import numpy as np
    from paper_2003_09468_b200 import replicas, synth

    rank, local_rank, world = replicas.rank_env()
    cfg = synth.CONFIGS[args.config]
    # replicas: every rank has the same Hamiltonian and its own seeded walkers/fields (weak scaling); rank r owns the
    # global walkers [r*nw, (r+1)*nw) of the nw*world walkers of the job
    pb = synth.make_problem(cfg)
    nw = cfg.nw
    w_lo, w_hi = replicas.shard_walkers(nw * world, rank, world)
    assert w_hi - w_lo == nw
    if rank > 0:
        rng = np.random.default_rng(cfg.seed + 1000 + rank)
        pb.phi = synth.make_walkers(cfg, pb.psi_t, rng)
        pb.x = rng.standard_normal(pb.x.shape)

    # ---- CPU baseline: the oracle on a bounded sample, on all host cores (rank 0, N=1 only); runs BEFORE CUDA is touched
    # so that the worker processes can be forked safely ----
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        cores = min(host_cores() if args.cores <= 0 else args.cores, nw)
        pool = OraclePool(cfg, pb, cores)
        try:
            t1 = pool.run(range(cores))                       # one walker per core
            passes = 1
            while t1 < 8.0 and passes < 64:                   # small configs: repeat until ~10 s of wall time
                t1 += pool.run(range(cores))
                passes += 1
        finally:
            pool.close()
        cpu = {"value": cores * passes / t1, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": "%d pass(es) of %d of the %d walkers of %s, full step each (work is linear in walkers), one "
                         "single-threaded numpy oracle process per host core, %.1f s wall" % (passes, cores, nw, cfg.name, t1)}

    import torch
    import torch.distributed as dist
    from paper_2003_09468_b200 import binding
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    ctx = binding.from_problem(pb)
    ctx.set_option("timers", 1)
    phi0 = torch.from_numpy(pb.phi).cuda()
    phi = phi0.clone()
    x = torch.from_numpy(pb.x).cuda()
    energy = torch.empty((nw, 3), dtype=torch.complex128, device="cuda")
    logdet = torch.empty((nw,), dtype=torch.complex128, device="cuda")
    info = torch.empty((nw,), dtype=torch.int32, device="cuda")

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---------------- device-resident timing ----------------
    for _ in range(args.warmup):
        phi.copy_(phi0)
        ctx.step(phi, x, cfg.dtau, cfg.order, energy, logdet, info)
    torch.cuda.synchronize()
    sampler = ClockSampler(local_rank)
    sampler.start()
    stage_acc = {k: 0.0 for k in ctx.STAGES}
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    l0 = ctx.launch_count()
    barrier()
    t_wall0 = time.perf_counter()
    for i in range(args.steps):
        phi.copy_(phi0)                       # restore the walkers (outside the event pair)
        ev[i][0].record()
        ctx.step(phi, x, cfg.dtau, cfg.order, energy, logdet, info)
        ev[i][1].record()
        ev[i][1].synchronize()
        for k, v in ctx.stage_times().items():
            stage_acc[k] += v
    barrier()
    t_wall = time.perf_counter() - t_wall0
    launches = ctx.launch_count() - l0
    dev_ms = sum(a.elapsed_time(b) for a, b in ev)
    assert int(info.abs().sum().item()) == 0
    e_dev = energy.cpu().numpy().copy()

    # ---------------- the 4M exchange kernel (energy.cu) for comparison: a few untimed-for-the-metric steps -------------
    ex_flops_default = ctx.exchange_flops(nw)
    ctx.set_option("exchange_3m", 0)
    ex_flops_4m = ctx.exchange_flops(nw)
    ex4_ms = 0.0
    for i in range(4):
        phi.copy_(phi0)
        ctx.step(phi, x, cfg.dtau, cfg.order, energy, logdet, info)
        torch.cuda.synchronize()
        if i > 0:
            ex4_ms += ctx.stage_times()["exchange"] / 3
    e_4m = energy.cpu().numpy().copy()
    ctx.set_option("exchange_3m", 1)
    assert np.max(np.abs(e_4m - e_dev) / np.abs(e_dev)) < 1e-10, "3M and 4M exchange kernels disagree"

    # ---------------- optional mixed-precision exchange (exchange_tf32.cu): extra information, NOT the headline ----------
    mixed = {}
    for mode, label in ((1, "3xTF32"), (2, "1xTF32")):
        try:
            ctx.set_option("exchange_precision", mode)
        except binding.AfqmcError:            # more than 4 occupied orbitals per k-point: FP64 kernels only
            mixed[label] = None
            continue
        tot = exm = 0.0
        for i in range(4):
            phi.copy_(phi0)
            ctx.step(phi, x, cfg.dtau, cfg.order, energy, logdet, info)
            torch.cuda.synchronize()
            if i > 0:
                stt = ctx.stage_times()
                tot += sum(stt.values()) / 3
                exm += stt["exchange"] / 3
        e_m = energy.cpu().numpy()
        mixed[label] = {"ms_per_step": tot, "exchange_ms": exm, "walker_steps_per_s": nw / (tot * 1e-3),
                        "max_rel_err_EX_vs_fp64": float(np.max(np.abs(e_m[:, 2] - e_dev[:, 2]) / np.abs(e_dev[:, 2])))}
    ctx.set_option("exchange_precision", 0)

    # ---------------- end to end through the host-buffer C-ABI call ----------------
    # (stage timers off: the per-stage events are only needed for the device-timed steps above; nine event records per step
    # cost the pipelined host entry 0.15 ms per step)
    ctx.set_option("timers", 0)
    phi_h0 = torch.from_numpy(pb.phi).pin_memory()
    phi_h = torch.empty_like(phi_h0).pin_memory()
    x_h = torch.from_numpy(pb.x).pin_memory()
    e_h = torch.empty((nw, 3), dtype=torch.complex128).pin_memory()
    ld_h = torch.empty((nw,), dtype=torch.complex128).pin_memory()
    info_h = torch.empty((nw,), dtype=torch.int32).pin_memory()
    e2e_t = 0.0
    for i in range(max(1, args.warmup // 2) + args.steps):
        phi_h.copy_(phi_h0)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        ctx.step_host(phi_h, x_h, cfg.dtau, cfg.order, e_h, ld_h, info_h)   # synchronises before returning
        dt = time.perf_counter() - t0
        if i >= max(1, args.warmup // 2):
            e2e_t += dt
    assert np.array_equal(e_h.numpy(), e_dev), "host-entry step disagrees with the device step"
    # the same through the pipelined host entry (afqmc_step_host_begin / _end, two steps in flight): every step uploads its
    # walkers and fields from pinned memory and downloads the propagated walkers, energies, log det and info; the upload of a
    # step overlaps the kernels of the step before it.  K steps, one timed region from the first begin to the last end.
    outs = [(torch.empty_like(phi_h0).pin_memory(), torch.empty_like(e_h).pin_memory(), torch.empty_like(ld_h).pin_memory(),
             torch.empty_like(info_h).pin_memory()) for _ in range(2)]

    def run_pipelined(nsteps):
        for i in range(nsteps):
            o = outs[i & 1]
            ctx.step_host_begin(i & 1, phi_h0, x_h, cfg.dtau, cfg.order, o[0], o[1], o[2], o[3])
        ctx.step_host_end(0)
        ctx.step_host_end(1)

    run_pipelined(max(2, args.warmup))
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    run_pipelined(args.steps)
    e2e_pipe_t = time.perf_counter() - t0
    sampler.stop()
    for o in outs[:min(2, args.steps)]:
        assert np.array_equal(o[1].numpy(), e_dev), "pipelined host-entry step disagrees with the device step"
        assert torch.equal(o[0], phi_h), "pipelined host-entry walkers disagree with the synchronous host-entry walkers"
    h2d = phi_h.numel() * 16 + x_h.numel() * 8
    d2h = phi_h.numel() * 16 + e_h.numel() * 16 + ld_h.numel() * 16 + info_h.numel() * 4

    # max over ranks (the only torch.distributed traffic of the run besides the barriers)
    dev_ms_max = replicas.max_over_ranks(dev_ms, device="cuda")
    e2e_ms_max = replicas.max_over_ranks(e2e_t * 1e3, device="cuda")
    e2e_pipe_ms_max = replicas.max_over_ranks(e2e_pipe_t * 1e3, device="cuda")

    if rank == 0:
        value = replicas.aggregate_throughput(nw, args.steps, world, dev_ms_max)
        e2e_sync_value = replicas.aggregate_throughput(nw, args.steps, world, e2e_ms_max)
        e2e_value = replicas.aggregate_throughput(nw, args.steps, world, e2e_pipe_ms_max)
        # ---- roofline of the dominant kernel (exchange contraction, a9) ----
        ex_ms = stage_acc["exchange"] / args.steps
        ex_flops = ex_flops_default
        achieved = ex_flops / (ex_ms * 1e-3) / 1e12
        peak_probe = binding.probe_fp64(1, 20000)          # DMMA issue-rate probe, this GPU, now
        # algorithmic bytes of one exchange launch = the METHOD's bytes: the half-rotated tensor once + Theta once, 16 bytes
        # per complex number; beside it what the kernel's own packed operand occupies (Lx3t: the three A
        # variants Re+Im, Re, Im stored = 24 bytes per element, K padded to k-steps)
        ctx_alg_bytes = cfg.nk ** 2 * cfg.n * cfg.nchol * cfg.m * 16 + nw * cfg.N * cfg.M * 16
        ksf, tail = ((cfg.m // 4, 1) if cfg.m % 4 in (1, 2) else ((cfg.m + 3) // 4, 0))
        packed_bytes = cfg.nk ** 2 * ((cfg.n + 3) // 4) * ((cfg.nchol + 3) // 4) * (3 * ksf + tail) * 64 * 8 + nw * cfg.N * cfg.M * 16
        peaks = load_measured_peaks()
        roofline = {
            "kernel": "exchange (a9), afqmc_local_energy", "bound": "tensor", "achieved": achieved,
            "peak": peak_probe, "unit": "TFLOP/s", "frac": achieved / peak_probe,
            "traffic": exchange_dram_traffic(cfg.name)[0],
            "traffic_unit": "bytes per launch (DRAM read+write)",
            "traffic_source": exchange_dram_traffic(cfg.name)[1],
            "algorithmic_bytes": float(ctx_alg_bytes),
            "packed_operand_bytes": float(packed_bytes),
            "peak_source": "live FP64 DMMA.8x8x4 probe (afqmc_probe_fp64); MEASURED_PEAKS.json has no FP64 entry",
            "flops_per_launch": ex_flops, "ms_per_launch": ex_ms,
            "flops_note": "EXECUTED real flops of the default kernel (3M complex product when n <= 4: 6 per complex "
                          "multiply-add, unpadded; the K = m padding to 4 is not counted)",
            "variant_4m": {"ms_per_launch": ex4_ms, "flops_per_launch": ex_flops_4m,
                           "achieved": ex_flops_4m / (ex4_ms * 1e-3) / 1e12, "frac": ex_flops_4m / (ex4_ms * 1e-3) / 1e12 / peak_probe,
                           "note": "one real GEMM with 8 flops per complex multiply-add (energy.cu), option exchange_3m=0"},
            "share_of_step": ex_ms / (dev_ms_max / args.steps),
        }
        if peaks and "bf16_tflops" in peaks:
            roofline["peak_alt_bf16_ratio"] = peaks["bf16_tflops"] * 45.0 / 2250.0
        # sanity check of the probe from the record itself: 148 SMs x 128 FP64 flops per clock (one DMMA.8x8x4 = 512 flops per
        # 16 cycles and SM sub-partition) x the SM clock sampled during the timed region
        clk = sampler.summary()
        if clk and clk.get("sm_mhz"):
            roofline["peak_check"] = {"formula": "num_sms * 128 flop/clk * sm_mhz", "num_sms": 148, "sm_mhz": clk["sm_mhz"],
                                      "tflops": 148 * 128 * clk["sm_mhz"] * 1e6 / 1e12}
        stages = {k: v / args.steps for k, v in stage_acc.items()}
        # the other kernel the north_star names: force bias (a4).  EXECUTED flops: 3M complex product, 6 Nk^2 n m nchol real
        # flops per walker (the plain definition / a real embedding costs 8); the stage time includes the reduction kernel
        # that sums the stream-K partial tiles
        fb_flops = ctx.force_bias_flops(nw)
        fb_flops_def = 8.0 * nw * cfg.nk ** 2 * cfg.n * cfg.m * cfg.nchol
        fb_ms = stages["force_bias"]
        fb_bytes = 16.0 * cfg.nk ** 2 * cfg.n * cfg.m * cfg.nchol + 16.0 * nw * cfg.nk ** 2 * cfg.n * cfg.m
        force_bias_roofline = {"kernel": "force bias (a4), afqmc_force_bias", "bound": "tensor", "flops_per_launch": fb_flops,
                               "ms_per_launch": fb_ms, "achieved": fb_flops / (fb_ms * 1e-3) / 1e12, "peak": peak_probe,
                               "unit": "TFLOP/s", "frac": fb_flops / (fb_ms * 1e-3) / 1e12 / peak_probe,
                               "flops_note": "EXECUTED real flops (3M complex product, 6 per complex multiply-add)",
                               "definition_flops": fb_flops_def,
                               "definition_rate_tflops": fb_flops_def / (fb_ms * 1e-3) / 1e12,
                               "algorithmic_bytes": fb_bytes,
                               "hbm_gbs": fb_bytes / (fb_ms * 1e-3) / 1e9,
                               "hbm_frac": (fb_bytes / (fb_ms * 1e-3) / 1e9 / peaks["hbm_gbs"]) if peaks and "hbm_gbs" in peaks else None}
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dev_ms_max / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "c128", "data": "synthetic",
            "config": {"workload": "%s: %dx%dx%d k-mesh, m=%d, n=%d, nchol=%d, %d walkers/GPU, complex128, "
                                   "dtau=%g, Taylor order %d; step = green+force_bias+vhs+propagate+green+local_energy"
                                   % ((cfg.name,) + tuple(cfg.mesh) + (cfg.m, cfg.n, cfg.nchol, nw, cfg.dtau, cfg.order)),
                       "l2": "inputs larger than L2 (L %.2f GB, packed Lh %.2f GB, vhs %.2f GB per step)"
                             % (pb.L.nbytes / 1e9, 2 * cfg.nk ** 2 * cfg.n * cfg.nchol * cfg.m * 16 / 1e9,
                                nw * cfg.M ** 2 * 16 / 1e9),
                       "parallelism": "replicas x%d (walkers sharded by rank, no collective)" % world},
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "call": "afqmc_step_host_begin / afqmc_step_host_end, two steps in flight: every step uploads phi and x from "
                            "pinned host memory and downloads phi', energy, logdet, info; the upload of step i+1 runs during the "
                            "kernels of step i; host wall clock over the K steps",
                    "ms_per_step": e2e_pipe_ms_max / args.steps,
                    "one_step_at_a_time": {"value": e2e_sync_value, "ms_per_step": e2e_ms_max / args.steps,
                                           "call": "afqmc_step_host (returns when the step's results are in the host buffers)"}},
            "gpu_launches": int(launches),
            "clocks": sampler.summary(),
            "roofline": roofline,
            "force_bias_roofline": force_bias_roofline,
            "mixed_precision_exchange": dict(mixed, note="option exchange_precision: exchange energy on the TF32 tensor cores "
                                             "(boundary complex128, everything else FP64); extra information, the headline "
                                             "value above is the all-FP64 path"),
            "stage_ms": stages,
            "exchange_tflops": achieved,
            "wall_s_timed_region": t_wall,
        }
        if cpu is not None:
            line["cpu_baseline"] = cpu
    ctx.close()
    # ---- the paper's measured unit (Fig. 2): a BLOCK = 20 hybrid propagation steps + one energy
    # evaluation + walker orthogonalisation (afqmc_block), on the same shapes with the 'physically scaled' L of
    # synth.make_problem (l_scale: the unscaled synthetic L makes the phaseless projection kill every walker).
    # Extra information beside the headline metric; N=1 only.
    if world == 1 and rank == 0 and not args.no_block:
        del phi, phi0
        torch.cuda.empty_cache()
        l_scale, nsteps_blk = 0.01, 20
        pb.L *= l_scale
        bctx = binding.from_problem(pb)
        bctx.set_onebody(torch.from_numpy(pb.h1).cuda(), cfg.dtau)
        xs = torch.from_numpy(synth.make_block_fields(cfg, nsteps_blk, nw)).cuda()
        phi_b0 = torch.from_numpy(pb.phi).cuda()
        blk_ms = []
        for it in range(4):
            phi_b = phi_b0.clone()
            wt = torch.ones(nw, dtype=torch.float64, device="cuda")
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            l0b = bctx.launch_count()
            e0.record()
            _, emixed, _, binfo = bctx.block(phi_b, wt, xs, cfg.dtau, cfg.order)
            e1.record()
            torch.cuda.synchronize()
            if it > 0:
                blk_ms.append(e0.elapsed_time(e1))
            blk_launches = bctx.launch_count() - l0b
        em = emixed.cpu().numpy()
        line["block"] = {
            "definition": "%d hybrid steps (green, force bias, vHS, B1*Taylor%d*B1, overlap, phaseless weight) + local energy "
                          "+ mixed estimator + Cholesky-QR2 orthogonalisation (afqmc_block; PAPER.md:274)" % (nsteps_blk, cfg.order),
            "ms_per_block": sum(blk_ms) / len(blk_ms), "blocks_timed": len(blk_ms), "walkers": nw,
            "walker_blocks_per_s": nw / (sum(blk_ms) / len(blk_ms) * 1e-3), "l_scale": l_scale,
            "gpu_launches_per_block": int(blk_launches), "surviving_walkers": int((wt > 0).sum().item()),
            "info_nonzero": int((binfo != 0).sum().item()),
            "e_mixed": [float((em[0] + em[1] + em[2]).real / em[3].real) if em[3].real > 0 else None][0],
        }
        bctx.close()
    # ---- the optional complex64 boundary (afqmc_dims.precision = 1): extra information, N=1 only ----
    if world == 1 and rank == 0 and not args.no_block:
        torch.cuda.empty_cache()
        pb64 = synth.make_problem(cfg)
        c64 = binding.from_problem(pb64, precision=1)
        c64.set_option("timers", 1)
        phi64_0 = torch.from_numpy(pb64.phi).to(torch.complex64).cuda()
        x32 = torch.from_numpy(pb64.x).to(torch.float32).cuda()
        ms64 = []
        for it in range(4):
            p64 = phi64_0.clone()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            e0.record()
            e64, _, _ = c64.step(p64, x32, cfg.dtau, cfg.order)
            e1.record()
            torch.cuda.synchronize()
            if it > 0:
                ms64.append(e0.elapsed_time(e1))
        st64 = c64.stage_times()
        err = np.abs(e64.cpu().numpy().astype(np.complex128) - e_dev) / np.abs(e_dev)
        line["complex64_path"] = {"ms_per_step": sum(ms64) / len(ms64), "walker_steps_per_s": nw / (sum(ms64) / len(ms64) * 1e-3),
                                  "max_rel_diff_vs_complex128": [float(err[:, i].max()) for i in range(3)],
                                  "stage_ms": st64,
                                  "stage_ms_complex128": {k: stages[k] for k in ("force_bias", "vhs", "exchange")},
                                  "note": "afqmc_dims.precision = 1: complex64 arrays at the boundary, the vHS and force-bias operands "
                                          "STORED in single precision (half the HBM bytes, FP64 accumulation), FP64 small algebra, 3xTF32 "
                                          "exchange; extra information (the energies are those of the polynomial-propagated walkers, "
                                          "whose FP32 storage error is amplified by the synthetic step size, DESIGN.md R9)"}
        c64.close()
    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="C3")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cores", type=int, default=0, help="host cores for the CPU oracle (0 = all available to the process)")
    ap.add_argument("--no-block", action="store_true", help="skip the extra 20-step block measurement")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3
    from paper_2003_09468_b200 import replicas
    if replicas.needs_launch(args.gpus):
        # `python bench.py --gpus N` without torchrun: start the N ranks (one per GPU) and let rank 0 print the line
        sys.exit(replicas.launch_ranks(os.path.abspath(__file__), sys.argv[1:], args.gpus))
    _, _, world = replicas.rank_env()
    if world != args.gpus:
        raise SystemExit("bench.py: --gpus %d but WORLD_SIZE=%d" % (args.gpus, world))
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
