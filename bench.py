#!/usr/bin/env python
"""bench.py -- electron moves/s of the particle-by-particle sweep (SPO-VGL + ratio + inverse update).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config large] [--delay 0] [--impl ours|reference]

One STEP is one full sweep of the configuration: every electron of every walker is proposed once
(qmc_sweep with nsweeps = 1): S0 proposal, S1 stencil, S2 SPO-VGL gather, S3 ratio, S4 Metropolis
test, S5 inverse update.  Default workload: BASELINE.json's "large supercell"
(128^3 grid, N = 1024, 512 walkers, 8.6 GB fp32 table, 4.3 GB of fp64 inverses).  Inputs are
seeded and synthetic (paper_1802_06922_b200/inputs.py).  Prints ONE JSON line on rank 0.

Multi-GPU (torchrun, one rank per GPU): walkers are independent Markov chains, so
each rank runs its own 512 walkers against its own replica of the table; there is no data-path
collective ("scaling": "weak").  Time = max over ranks.

--impl reference times the fp64 CPU oracle (oracle/qmc_oracle.c), as it stands, on the host cores,
on a bounded sample of the same workload.
"""
import argparse
import json
import os
import statistics
import sys
import threading
import time

import numpy as np
import torch

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1802_06922_b200 import inputs, sharding  # noqa: E402

METRIC = "electron moves/s at N=1024 (spline VGL+ratio+SM update); HBM GB/s vs peak"
UNIT = "moves/s"
# delayed ranks measured by default per config, the first one is the headline (BASELINE.json: large =
# rank-16 vs rank-1; very large names rank-32, which is measured beside rank-16: at N = 2048 the
# rank-16 window is the faster one on this kernel)
DEFAULT_DELAY = {"tiny": [0], "small": [16, 0], "mid": [16, 0], "large": [16, 0], "xlarge": [16, 32, 0]}
# further arms reported as variants (fewer timed steps each): (delay rank, fp32-stored inverse)
EXTRA_ARMS = {"large": [(16, True), (0, True), (20, False), (24, False), (32, False), (0, False, "drift"), (16, False, "updn"),
                        (16, False, "jastrow"), (16, True, "aw")],
              "mid": [(16, True), (16, False, "updn")], "xlarge": [(16, True), (24, False)],
              # L2-resident configs: the sweep is launch-bound; the same sweep replayed from a CUDA graph
              "tiny": [(0, False, "graph")], "small": [(16, False, "graph"), (0, False, "graph")]}
# dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed `ncu --set full` captures
# (profiles/r01_rank1_summary.md: kernel unchanged since; profiles/r02_delayed_summary.md), config `large`
# keyed by (kernel, delay rank); value = (bytes per launch, the file the figure comes from)
NCU_TRAFFIC = {("sm_update", 0): (6.725e9, "profiles/r01_rank1_summary.md"),
               ("delayed_flush", 16): (8.612e9, "profiles/r02_delayed_summary.md")}


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


class ClockSampler:
    """Samples SM clock and throttle reasons with NVML every 100 ms while the timed region runs."""

    def __init__(self, index):
        self.samples, self.power, self.reasons, self.max_mhz = [], [], set(), None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def _run(self):
        nv = self.nv
        names = {
            getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksThrottleReasonSwPowerCap", 0x4): "sw_power_cap",
            getattr(nv, "nvmlClocksThrottleReasonHwPowerBrakeSlowdown", 0x80): "hw_power_brake",
        }
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            try:
                self.power.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0)      # W
            except Exception:
                pass
            self._stop.wait(0.1)

    def start(self):
        if self.nv is not None:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()

    def stop(self):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()
        med = statistics.median(self.samples) if self.samples else None
        pw = statistics.median(self.power) if self.power else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "power_w": pw}


def cpu_sample(x, coefs_np, target_s=15.0):
    """The oracle, as it stands, on a bounded sample of the workload: W walkers (a whole number per
    thread) x the first M electron moves of a sweep, sized for about `target_s` seconds.
    Returns (moves/s, cores, sample text, seconds)."""
    import oracle
    cores = len(os.sched_getaffinity(0))
    nthreads = max(1, min(cores, oracle.max_threads(), 32, x.pos.shape[0]))
    nel = x.cfg.norb
    probe = min(8, nel)

    def setup(nwc):
        pos = np.ascontiguousarray(x.pos[:nwc])
        B, ld, sg = oracle.init_walkers(coefs_np, x.lattice, pos, nthreads=nthreads)       # untimed set-up
        return pos, B, ld, sg, np.ascontiguousarray(x.delta[:1, :, :nwc]), np.ascontiguousarray(x.unif[:1, :, :nwc])

    pos, B, ld, sg, delta, unif = setup(nthreads)
    oracle.sweep(coefs_np, x.lattice, pos, B, ld, sg, delta, unif, iel_count=probe, nthreads=nthreads)   # page the table in
    t0 = time.perf_counter()
    oracle.sweep(coefs_np, x.lattice, pos, B, ld, sg, delta, unif, iel_count=probe, nthreads=nthreads)
    t_move = (time.perf_counter() - t0) / probe            # one electron step of `nthreads` walkers
    m = int(min(nel, max(probe, target_s / max(t_move, 1e-6))))
    per_thread = int(max(1, min(x.pos.shape[0] // nthreads, round(target_s / max(t_move * m, 1e-6)))))
    nwc = nthreads * per_thread
    if per_thread > 1:
        pos, B, ld, sg, delta, unif = setup(nwc)
    for attempt in range(2):
        t0 = time.perf_counter()
        out = oracle.sweep(coefs_np, x.lattice, pos, B, ld, sg, delta, unif, iel_count=m, nthreads=nthreads)
        dt = time.perf_counter() - t0
        grow = int(min(x.pos.shape[0] // nthreads, per_thread * target_s / max(dt, 1e-3)))
        if attempt or dt >= 0.6 * target_s or grow <= per_thread:
            break
        per_thread, nwc = grow, nthreads * grow          # the probe over-estimated the cost: enlarge the sample once
        pos, B, ld, sg, delta, unif = setup(nwc)
    acc = float(out["accept"][0, :m].mean())
    text = (f"{nwc} walkers x first {m} electron moves of one sweep of config '{x.cfg.name}' "
            f"(accept {acc:.2f}), {nthreads} OpenMP threads, {dt:.1f} s")
    return nwc * m / dt, nthreads, text, dt


def run_reference(args, rank, world):
    """--impl reference: the CPU oracle arm (rank 0 only)."""
    if rank != 0:
        return
    cfg = inputs.CONFIGS[args.config]
    dev = "cuda" if torch.cuda.is_available() else "cpu"
    x = inputs.make_inputs(cfg, device=dev, nw=min(cfg.nw, 64), nsweeps=1)
    coefs_np = x.coefs_numpy()
    x.coefs = None
    if dev == "cuda":
        torch.cuda.empty_cache()
    vals, secs = [], []
    per_step = max(5.0, min(30.0, 120.0 / max(1, args.steps + args.warmup)))
    info = None
    for i in range(args.warmup + args.steps):
        v, cores, text, dt = cpu_sample(x, coefs_np, target_s=per_step)
        if i >= args.warmup:
            vals.append(v)
            secs.append(dt)
            info = (cores, text)
    value = float(np.mean(vals))
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "impl": "reference", "n_gpus": 0,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * float(np.mean(secs)),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic (seeded; paper_1802_06922_b200/inputs.py)",
        "config": {"workload": args.config, "grid": list(cfg.grid), "N": cfg.norb,
                   "sample": info[1]},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": info[0], "kind": "oracle", "sample": info[1]},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def flush_micro(args, api, spline, cfg, pos_np, nw, nel, dev, peak, fp64_peak):
    """Kernel-level timing of the delayed flush on real window data: per repetition, K standalone steps
    (qmc_spo_vgl -> qmc_det_ratio -> qmc_det_accept_update with ~81 % of the walkers accepting each step),
    then qmc_det_flush bracketed by the library's per-kernel CUDA events (kind `delayed_flush`)."""
    ranks = [args.delay] if args.delay >= 2 else [16, 24, 32]
    g = torch.Generator(device=dev).manual_seed(1234)
    for K in ranks:
        for fp32 in ([True] if args.fp32_inverse else [False, True]):
            pos = torch.from_numpy(pos_np).to(dev)
            det = api.Det.init(spline, pos, delay_rank=K, fp32_inverse=fp32)
            times, paccs = [], []
            for rep in range(args.warmup + args.steps):
                k0 = (rep * K) % max(1, nel - K)
                pacc = torch.zeros(nw, device=dev)
                for l in range(K):
                    k = k0 + l
                    newpos = pos[:, k] + cfg.sigma * torch.randn((nw, 3), dtype=torch.float64, device=dev, generator=g)
                    phi = api.spo_vgl(spline, newpos, want_gl=False)
                    R = det.ratio(k, phi)
                    acc = ((torch.rand(nw, device=dev, generator=g) < 0.81) & torch.isfinite(R) & (R.abs() > 0.05)).to(torch.uint8)
                    det.accept_update(k, phi, R, acc)
                    pos[:, k] = torch.where(acc.bool()[:, None], newpos, pos[:, k])
                    pacc += acc
                det.profile(True)
                det.flush()
                torch.cuda.synchronize()
                prof = det.profile_read()
                det.profile(False)
                if rep >= args.warmup:
                    times.append(prof["delayed_flush"][0])
                    paccs.append(float(pacc.mean().item()))
            ms = float(np.median(times))
            pbar = float(np.mean(paccs))
            eb = det.storage_bytes
            byt = nw * 2 * eb * nel * det.ld + nw * pbar * (8 * det.ld + 4 * spline.row_pitch)
            fl = 4.0 * pbar * nw * nel * nel
            print(json.dumps({"flush_micro": True, "workload": args.config, "N": nel, "walkers": nw, "rank": K,
                              "storage": "f32" if fp32 else "f64", "accepted_per_window": pbar, "flush_ms": ms,
                              "GB/s": byt / ms / 1e6, "frac_of_hbm_peak": byt / ms / 1e6 / peak,
                              "fp64_TFLOP/s": fl / ms / 1e9, "frac_of_fp64_dmma_peak": fl / ms / 1e9 / fp64_peak,
                              "ring": os.environ.get("QMC_FLUSH_RING", "1")}), flush=True)
            det.destroy()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="large", choices=list(inputs.CONFIGS))
    ap.add_argument("--delay", type=int, default=-1,
                    help="inverse update: 0 = Sherman-Morrison rank-1; k >= 2 = delayed rank-k; default: the "
                         "config's delayed rank as the headline AND rank-1 as a variant in the same line")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--fp32-inverse", action="store_true", help="store the inverse in fp32 (QMC_DET_FP32_INVERSE)")
    ap.add_argument("--accept-windows", action="store_true",
                    help="with --delay <= 16: delayed windows close on an accept count (QMC_DET_ACCEPT_WINDOWS); the "
                         "default run (no --delay) uses it for the headline arm of mid / large / xlarge and reports the "
                         "step-count windows as a variant")
    ap.add_argument("--no-variants", action="store_true", help="skip the extra variant arms of the default run")
    ap.add_argument("--flush-micro", action="store_true",
                    help="time qmc_det_flush alone: windows filled through qmc_det_ratio / qmc_det_accept_update "
                         "(81 %% of --delay steps accepted), one JSON line per (rank, storage) with the flush kernel's "
                         "CUDA-event time; a kernel-level A/B tool (QMC_FLUSH_RING=0 selects flush.cu), not the metric")
    ap.add_argument("--walkers", type=int, default=0, help="override walkers per GPU (debug)")
    ap.add_argument("--probe-fp64", action="store_true",
                    help="print the fp64-pipe microbenchmark table (qmc_probe_fp64_pipe: DMMA / DFMA / mixed by warps "
                         "per SM and accumulator chains) and exit; not the metric")
    args = ap.parse_args()

    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # `python bench.py --gpus N`: launch N ranks (one per GPU) of this script, as the driver's
        # torchrun command does, and let rank 0 print the line
        import subprocess
        port = 29500 + os.getpid() % 2000
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        sys.exit(subprocess.call(cmd))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.gpus != world and rank == 0:
        print(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}; running {world} rank(s)", file=sys.stderr)
    if args.impl == "reference":
        run_reference(args, rank, world)
        return
    args.warmup = max(args.warmup, 3)

    from paper_1802_06922_b200 import api
    api.load_library()                       # no fallback: raises if the CUDA library is missing
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (use --impl reference for the CPU oracle)"
    torch.cuda.set_device(local_rank)
    if args.probe_fp64:
        if rank == 0:
            for mode, name in ((0, "dmma"), (1, "dfma"), (2, "dmma+2dfma")):
                for warps in (4, 8, 16, 32):
                    for chains in (1, 2, 4, 8):
                        a_, b_ = api.probe_fp64_pipe(mode, warps, chains)
                        print(json.dumps({"probe": "fp64_pipe", "mix": name, "warps_per_sm": warps, "chains_per_warp": chains,
                                          "dmma_TFLOP/s": round(a_, 2), "dfma_TFLOP/s": round(b_, 2)}), flush=True)
        return
    dev = torch.device("cuda", local_rank)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    cfg = inputs.CONFIGS[args.config]
    nw = args.walkers or cfg.nw
    nel = cfg.norb
    nsteps_total = args.warmup + args.steps
    # every rank draws the inputs of all ranks and keeps its own walkers (weak scaling)
    x = inputs.make_inputs(cfg, device=dev, nw=nw * world, nsweeps=nsteps_total)
    pos_np, delta_np, unif_np = sharding.shard_inputs(x.pos, x.delta, x.unif, rank, world)
    assert pos_np.shape[0] == nw

    spline = api.Spline.create(x.coefs, x.lattice)
    torch.cuda.synchronize()
    coefs_np = None
    want_cpu = rank == 0 and world == 1 and not args.no_cpu_baseline
    if want_cpu:
        coefs_np = x.coefs_numpy()
    x.coefs = None
    torch.cuda.empty_cache()

    delta = torch.from_numpy(delta_np).to(dev)
    unif = torch.from_numpy(unif_np).to(dev)
    delta_h = torch.from_numpy(delta_np).pin_memory()
    unif_h = torch.from_numpy(unif_np).pin_memory()
    peak, peak_src = measured_peaks()
    fp64_peak = api.probe_fp64_dmma()        # TFLOP/s, measured live (MEASURED_PEAKS.json has no fp64 figure)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    def max_over_ranks(ms):
        return sharding.max_over_ranks(ms, device=dev)

    def run_arm(delay, fp32=False, mode=None, steps=None):
        """W warm-up sweeps + K timed sweeps with the inverse update `delay` (0 = rank-1), device
        resident; then the same K sweeps end to end from pinned host buffers.  fp32: the inverse is
        stored in single precision (QMC_DET_FP32_INVERSE)."""
        nsteps = args.steps if steps is None else min(args.steps, steps)
        nsteps_total = args.warmup + nsteps
        pos = torch.from_numpy(pos_np).to(dev)
        accept = torch.zeros(unif.shape, dtype=torch.uint8, device=dev)
        ratios = torch.zeros(unif.shape, dtype=torch.float64, device=dev)
        t0 = time.perf_counter()
        det = api.Det.init(spline, pos, delay_rank=delay, fp32_inverse=fp32, accept_windows=(mode == "aw"))
        torch.cuda.synchronize()
        t_init = time.perf_counter() - t0

        drift_tau = float(cfg.sigma) ** 2 if mode == "drift" else 0.0     # chi = the config's Gaussian displacements
        wf = det2 = pos2 = jas = graph = None
        if mode == "jastrow":     # one- and two-body B-spline Jastrow factor (eq. 28-33), seeded parameters
            jx = inputs.make_jastrow(cfg, x.lattice, nother=0, nw=1)
            jas = api.Jastrow(jx.funcs, f_same=jx.f_same, f_opp=jx.f_opp, lattice=x.lattice, ions=jx.ions, ion_func=jx.ion_func)
        if mode == "updn":        # closed shell: a second determinant of the same orbitals at other positions
            g = torch.Generator(device=dev).manual_seed(inputs.BASE_SEED + 77 + rank)
            lat_t = torch.tensor(x.lattice, dtype=torch.float64, device=dev)
            pos2 = torch.rand((nw, nel, 3), dtype=torch.float64, device=dev, generator=g) @ lat_t
            det2 = api.Det.init(spline, pos2, delay_rank=delay, fp32_inverse=fp32)
            wf = api.Wavefunction(det, det2)
            delta2 = torch.cat([delta, cfg.sigma * torch.randn(delta.shape, dtype=torch.float64, device=dev, generator=g)], dim=1)
            unif2 = torch.cat([unif, torch.rand(unif.shape, dtype=torch.float64, device=dev, generator=g)], dim=1)
            accept = torch.zeros(unif2.shape, dtype=torch.uint8, device=dev)
            ratios = torch.zeros(unif2.shape, dtype=torch.float64, device=dev)

        d_buf = u_buf = r_buf = a_buf = None

        def step(i):
            if wf is not None:
                wf.sweep(pos, pos2, delta2[i:i + 1], unif2[i:i + 1], ratios_out=ratios[i:i + 1], accept_out=accept[i:i + 1])
            elif graph is not None:     # fresh random numbers into the graph's static buffers, replay, keep the outputs
                d_buf.copy_(delta[i:i + 1]); u_buf.copy_(unif[i:i + 1])
                graph.replay()
                ratios[i:i + 1].copy_(r_buf); accept[i:i + 1].copy_(a_buf)
            else:
                api.sweep(det, pos, delta[i:i + 1], unif[i:i + 1], ratios_out=ratios[i:i + 1], accept_out=accept[i:i + 1],
                          drift_tau=drift_tau, jastrow=jas)

        # ---- device-resident timing: inputs in HBM, CUDA events on the launching stream, no
        #      per-kernel instrumentation inside the timed region
        for i in range(args.warmup):
            step(i)
        if mode == "graph":       # capture one sweep (after the eager warm-up sweeps), then replay it
            d_buf, u_buf = delta[0:1].clone(), unif[0:1].clone()
            r_buf, a_buf = torch.zeros_like(u_buf), torch.zeros(u_buf.shape, dtype=torch.uint8, device=dev)
            torch.cuda.synchronize()
            c0 = api.launch_count()
            graph = api.SweepGraph(det, pos, d_buf, u_buf, ratios_out=r_buf, accept_out=a_buf)
            graph_launches = api.launch_count() - c0      # kernels of one sweep, recorded in the graph
            step(0)
        barrier()
        launches0 = api.launch_count()
        sampler = ClockSampler(local_rank)
        sampler.start()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for i in range(args.warmup, nsteps_total):
            step(i)
        e1.record()
        barrier()
        clocks = sampler.stop()
        launches = api.launch_count() - launches0
        if mode == "graph":
            launches = graph_launches * nsteps             # replayed by the graph: counted at capture
        ms = max_over_ranks(e0.elapsed_time(e1))
        nmoved = (2 if wf is not None else 1) * nel          # electrons moved per walker and sweep
        moves = nsteps * nmoved * nw * world
        value = moves / (ms * 1e-3)
        acc_rate = float(accept[args.warmup:nsteps_total].to(torch.float64).mean().item())

        # ---- per-kernel split: a SECOND pass of `nprof` sweeps with every launch bracketed by CUDA
        #      events (qmc_det_profile); the walk goes on with the random numbers of the first timed sweeps
        nprof = min(nsteps, 5)
        if graph is not None:     # the per-kernel split needs eager launches (events are recorded by the library)
            graph = None
        det.profile(True)
        if det2 is not None:
            det2.profile(True)
        e0.record()
        for i in range(args.warmup, args.warmup + nprof):
            step(i)
        e1.record()
        barrier()
        prof = det.profile_read()
        det.profile(False)
        if det2 is not None:
            p2 = det2.profile_read()
            det2.profile(False)
            prof = {k: (prof[k][0] + p2[k][0], prof[k][1] + p2[k][1]) for k in prof}
        ms_prof = e0.elapsed_time(e1)
        n_acc = float(accept[args.warmup:args.warmup + nprof].to(torch.float64).sum().item())

        # ---- roofline of the dominant kernel (rank-local, from the per-launch CUDA events)
        ld, npitch, K, eb = det.ld, spline.row_pitch, det.delay_rank, det.storage_bytes
        per_launch = {   # algorithmic bytes per launch; eb = bytes per stored element of B
            # (accept windows too: the scratch is a ring indexed by electron, every proposal is evaluated once)
            "spo_vgl": (nprof * nmoved * nw * (2 if drift_tau else 1) / max(prof["spo_vgl"][1], 1)) * (64 + 5) * npitch * 4,
            "ratio_rowcopy": nw * ((eb + 8) * ld + 4 * nel) * (0.75 if drift_tau else 1.0),   # drift: averaged with the propose kernel
            "sm_update": (n_acc / max(prof["sm_update"][1], 1)) * (2 * eb * nel * ld + 12 * nel),
            # (accept windows: a launch serves the walkers that still have moves to apply -- about n_acc / K
            #  full windows plus one partial window per walker and sweep in all)
            "delayed_flush": ((n_acc / max(K, 1) + 0.5 * nw * nprof) / max(prof["delayed_flush"][1], 1) if mode == "aw" else nw)
                             * 2 * eb * nel * ld + (n_acc / max(prof["delayed_flush"][1], 1)) * (8 * ld + 4 * npitch),
            # window: K rows of B0 and K vectors in, R' rows out
            "delayed_window": nw * max(K, 1) * (eb * ld + 4 * npitch) + (n_acc / max(prof["delayed_window"][1], 1)) * 8 * ld,
        }
        kernels = {}
        for k, (kms, kn) in prof.items():
            if not kn:
                continue
            kernels[k] = {"ms": kms, "launches": kn, "avg_us": 1e3 * kms / kn, "share_of_step": kms / ms_prof}
            if k in per_launch:
                gbs = per_launch[k] / (kms / kn * 1e-3) / 1e9
                kernels[k].update({"bytes_per_launch": per_launch[k], "GB/s": gbs, "frac_of_hbm_peak": gbs / peak})
        if "delayed_flush" in kernels:   # two fp64 contractions on the tensor cores: 4 p N^2 flop per walker
            kf = kernels["delayed_flush"]
            fl = 4.0 * (n_acc / kf["launches"]) * nel * nel
            tf = fl / (kf["avg_us"] * 1e-6) / 1e12
            kf.update({"flops_per_launch": fl, "fp64_TFLOP/s": tf, "fp64_dmma_peak_TFLOP/s": fp64_peak,
                       "frac_of_fp64_dmma_peak": tf / fp64_peak,
                       "min_ms_hbm": kf["bytes_per_launch"] / (peak * 1e9) * 1e3,
                       "min_ms_fp64": fl / (fp64_peak * 1e12) * 1e3})
        dom = max(kernels, key=lambda k: kernels[k]["ms"])
        kd = kernels[dom]
        # DRAM bytes per launch are an ncu measurement (no profiler runs inside bench.py): quoted from the
        # committed capture of the same kernel and launch shape, with its source; null for other shapes
        traffic, traffic_src = None, None
        if args.config == "large" and nw == cfg.nw and not fp32 and (dom, K) in NCU_TRAFFIC:
            traffic, traffic_src = NCU_TRAFFIC[(dom, K)]
        if dom == "delayed_flush" and kd["min_ms_fp64"] > kd["min_ms_hbm"]:
            # the contraction, not the pass over B, bounds this rank: report against the fp64 tensor peak
            roofline = {"bound": "tensor", "kernel": dom, "achieved": kd["fp64_TFLOP/s"], "peak": fp64_peak,
                        "unit": "TFLOP/s", "frac": kd["frac_of_fp64_dmma_peak"], "traffic": traffic, "traffic_source": traffic_src,
                        "peak_source": "measured live: qmc_probe_fp64_dmma (DMMA.8x8x4 issue loop)",
                        "launches": kd["launches"], "avg_us": kd["avg_us"], "flops_per_launch": kd["flops_per_launch"],
                        "share_of_step": kd["share_of_step"]}
        else:
            roofline = {"bound": "hbm", "kernel": dom, "achieved": kd.get("GB/s"), "peak": peak, "unit": "GB/s",
                        "frac": kd.get("frac_of_hbm_peak"), "traffic": traffic, "traffic_source": traffic_src, "peak_source": peak_src,
                        "launches": kd["launches"], "avg_us": kd["avg_us"], "bytes_per_launch": kd.get("bytes_per_launch"),
                        "share_of_step": kd["share_of_step"]}

        # ---- end to end through the C ABI with HOST buffers (pinned): H2D of pos/delta/unif and D2H
        #      of pos/ratios/decisions inside the timed region, every step
        e2e = None
        if mode in (None, "aw"):
            pos_h = pos.cpu().pin_memory()
            ratios_h = torch.zeros(unif_h.shape, dtype=torch.float64).pin_memory()
            accept_h = torch.zeros(unif_h.shape, dtype=torch.uint8).pin_memory()

            def step_host(i):
                api.sweep_host(det, pos_h, delta_h[i:i + 1], unif_h[i:i + 1], ratios_out=ratios_h[i:i + 1],
                               accept_out=accept_h[i:i + 1])

            step_host(0)
            barrier()
            e0.record()
            for i in range(args.warmup, nsteps_total):
                step_host(i)
            e1.record()
            barrier()
            ms_e2e = max_over_ranks(e0.elapsed_time(e1))
            h2d = pos_h.numel() * 8 + delta_h[0].numel() * 8 + unif_h[0].numel() * 8
            d2h = pos_h.numel() * 8 + ratios_h[0].numel() * 8 + accept_h[0].numel()
            e2e = {"value": moves / (ms_e2e * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d * world,
                   "d2h_bytes_per_step": d2h * world}
        update = "sherman-morrison rank-1" if K == 0 else f"delayed rank-{K} (same result as rank-1)"
        if fp32:
            update += ", fp32-stored inverse (fp64 arithmetic; R:A19)"
        if mode == "drift":
            update += f", drift moves tau = {drift_tau:.4g} (eq. 11-13)"
        if mode == "jastrow":
            update += ", one- and two-body B-spline Jastrow factor (eq. 28-33)"
            jas.destroy()
        if mode == "graph":
            update += ", sweep replayed from a CUDA graph (api.SweepGraph)"
        if mode == "aw":
            update += f", windows closed on {K} accepted moves (QMC_DET_ACCEPT_WINDOWS)"
        if mode == "updn":
            update += f", D_up D_dn: 2 x {nel} electrons per walker (eq. 26)"
            wf.destroy()
            det2.destroy()
        det.destroy()
        return {"value": value, "ms_per_step": ms / nsteps, "steps": nsteps, "update": update, "accept_rate": acc_rate,
                "kernel_split": f"second pass of {nprof} sweeps with per-launch CUDA events ({ms_prof / nprof:.2f} ms per sweep)",
                "init_s": t_init, "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roofline,
                "kernels": kernels, "spline_evals_per_s": value * nel * (2 if drift_tau else 1)}

    if args.flush_micro:
        flush_micro(args, api, spline, cfg, pos_np, nw, nel, dev, peak, fp64_peak)
        spline.destroy()
        return

    ws_table, ws_binv = cfg.table_bytes() / 1e9, nw * nel * nel * 8 / 1e9
    l2_note = (f"working set ({ws_table:.2f} GB table + {ws_binv:.2f} GB inverses) "
               + ("exceeds the 126 MB L2; no flush needed" if ws_table + ws_binv > 0.5 else
                  "fits L2: numbers are L2-resident, not HBM rooflines"))
    delays = [args.delay] if args.delay >= 0 else DEFAULT_DELAY.get(args.config, [0])
    # the headline arm of the HBM-resident configs closes its windows on 16 ACCEPTED moves (same result; every
    # flush then applies a full window); the step-count windows of round 1 are reported beside it
    aw_default = args.delay < 0 and not args.fp32_inverse and args.config in ("mid", "large", "xlarge")
    def arm_mode(i, dl):
        if 2 <= dl <= 16 and (args.accept_windows or (aw_default and i == 0)):
            return "aw"
        return None
    arms = [run_arm(dl, fp32=args.fp32_inverse, mode=arm_mode(i, dl)) for i, dl in enumerate(dict.fromkeys(delays))]
    if aw_default and not args.no_variants:
        arms.append(run_arm(16, steps=10))
    if args.delay < 0 and not args.fp32_inverse and not args.no_variants:
        arms += [run_arm(a[0], fp32=a[1], mode=a[2] if len(a) > 2 else None, steps=5) for a in EXTRA_ARMS.get(args.config, [])]
    main_arm = arms[0]
    line = {
        "metric": METRIC, "value": main_arm["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": main_arm["ms_per_step"], "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic (seeded; paper_1802_06922_b200/inputs.py)",
        "config": {"workload": args.config, "grid": list(cfg.grid), "N": nel, "walkers_per_gpu": nw,
                   "update": main_arm["update"],
                   "step": "one full sweep (N electron moves x walkers)",
                   "l2": l2_note,
                   "spo_dtype": "f32", "accept_rate": main_arm["accept_rate"], "init_s": main_arm["init_s"]},
        "clocks": main_arm["clocks"], "e2e": main_arm["e2e"], "gpu_launches": main_arm["gpu_launches"],
        "roofline": main_arm["roofline"], "kernels": main_arm["kernels"], "kernel_split": main_arm["kernel_split"],
        "spline_evals_per_s": main_arm["spline_evals_per_s"],
    }
    if len(arms) > 1:
        line["variants"] = {a["update"]: {k: a[k] for k in ("value", "ms_per_step", "steps", "accept_rate", "clocks", "e2e",
                                                            "gpu_launches", "roofline", "kernels")} for a in arms[1:]}

    if want_cpu:
        xs = inputs.QmcInputs(cfg, x.lattice, None, pos_np, delta_np, unif_np)
        v, cores, text, _ = cpu_sample(xs, coefs_np)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": text}
    if rank == 0:
        print(json.dumps(line), flush=True)
    spline.destroy()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
