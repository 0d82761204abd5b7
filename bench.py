#!/usr/bin/env python
"""bench.py -- split-step cell-updates/s of the B200 Schroedinger-Newton stepper (libsn.so).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C5_512] [--impl reference]

A bench "step" is one full Strang step K(dtau/2) N(dtau) K(dtau/2) of PAPER.md:42-44 eq. (1),(2)
(method: PAPER.md:113) over the whole grid, i.e. one pass of every row S1-S11 of SURVEY.md 8(a).
The timed region is ONE sn_step(K) call (adjacent half kinetics merged inside the call, as a user
would run it) bracketed by barrier + synchronize, CUDA events on the stream the kernels run on.
Default workload: BASELINE.json configs[4] at 512^3 (the size north_star's 60 % HBM target names);
the state (1 GiB) is far larger than L2 (126 MB), so no L2 flush is needed between steps.

One JSON line on stdout (rank 0).  Extra objects: roofline (dominant kernel, per-launch CUDA
events measured in a second K-step run right after the timed one), cpu_baseline (the float64
oracle as it stands, on the host cores, on a bounded sample), e2e (sn_set_state from pinned
host memory + sn_step(K) + sn_get_state to pinned host memory + sn_diagnostics, all inside the
timed region), clocks (NVML samples during the timed region).

Multi-GPU: the path does not shard (every transform is global; "replicas only");
--gpus N runs N independent replicas, one per rank, with no data-path collective.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "split-step cell-updates/sec (complex64)"
UNIT = "cell-updates/s"

# Algorithmic bytes per cell of each pass kind (complex64 = 8 B, half spectrum
# = 4 B per cell of the full grid).  hs = the half-spectrum array, (N0/2+1)/N0 of a full complex array.
PASS_BYTES_PER_CELL = {
    "H_NLKIN": 20.0,   # read phi^ (4) + read psi (8) + write psi (8)
    "S_KIN": 16.0,     # read + write psi
    "X_KIN": 16.0,
    "H_R2C": 12.0,     # read psi (8) + write rho^ (4)
    "S_FFT": 8.0,      # read + write half spectrum
    "X_POISSON": 8.0,
    "H_SRC": 24.0,     # eq. (12): read F[lap rho] (4) + psi (8) + beta, gamma (8), write F[s] (4)
    "H_BOHM": 20.0,    # eq. (15) Bohm phase: read F[lap sqrt(rho)] (4) + psi (8), write psi (8)
    "R_STEPS": 16.0,   # cluster-resident kernel (64^2 / 128^2): ONE launch = all K steps, psi read once and written once
}
B_MIN = {2: 64.0, 3: 112.0}  # SURVEY.md 8(d) minimal-pass byte count per cell-update
B_OWN = {2: 56.0, 3: 88.0}   # bytes this design's pass list has to move per cell-update
# ncu dram__bytes_read.sum + dram__bytes_write.sum per launch, C5_512, from profiles/r02z_final_C5_512.md
# (end-of-round capture, build of commit 3eb3bad; the same values as in profiles/r02g of commit 163e14c: the commits in
# between changed twiddle loads, register use and shared-memory stores, not DRAM traffic)
NCU_TRAFFIC_C5_512 = {"H_NLKIN": 2.634e9, "S_KIN": 2.089e9, "X_KIN": 2.089e9, "H_R2C": 1.577e9, "S_FFT": 1.019e9,
                      "X_POISSON": 1.020e9}


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy read+write)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """NVML samples of SM clock and throttle reasons while the timed region runs."""

    REASONS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap"}

    def __init__(self, index: int):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nv = pynvml
            self._h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self._nv = None

    def _run(self):
        nv = self._nv
        while not self._stop.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM)))
                r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self._h))
                for bit, name in self.REASONS.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            self._stop.wait(0.01)

    def __enter__(self):
        if self._nv is not None:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()

    def summary(self):
        return {"sm_mhz": int(statistics.median(self.samples)) if self.samples else None,
                "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


def oracle_rate(cfg_name: str, budget_s: float, inputs):
    """Time the float64 oracle as it stands on a bounded sample of the workload (host cores)."""
    from oracle import snref  # test infrastructure: only this leg and --impl reference touch it
    from oracle.snref import Oracle
    base = inputs.CONFIGS[cfg_name]
    # bounded sample: the same recipe (seed, constants, box) resampled so that one step is ~1 s of CPU
    if base.cells > 128 ** 3 and len(base.dims) == 3:
        cfg = inputs.scaled(base, (128, 128, 128))
    elif base.cells > 1024 ** 2 and len(base.dims) == 2:
        cfg = inputs.scaled(base, (1024, 1024), L=base.L * 1024 / base.dims[0])
    else:
        cfg = base
    psi0 = cfg.initial_state().astype(np.complex128)
    orc = Oracle.from_config(cfg)
    orc.set_state(psi0)
    t0 = time.perf_counter()
    orc.step(1)
    t1 = time.perf_counter() - t0
    k = int(max(2, min(cfg.steps, budget_s / max(t1, 1e-6))))
    t0 = time.perf_counter()
    orc.step(k)
    dt = time.perf_counter() - t0
    cores = snref.num_threads()
    # the same program on ONE host thread too (the paper's single-thread comparison, Fig. 1):
    # a third of the budget, at least two steps
    snref.set_num_threads(1)
    k1 = int(max(2, min(k, budget_s / 3.0 / max(t1 * cores, 1e-6))))
    t0 = time.perf_counter()
    orc.step(k1)
    dt1 = time.perf_counter() - t0
    snref.set_num_threads(cores)
    orc.close()
    return {"value": cfg.cells * k / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{base.name} recipe on a {'x'.join(map(str, cfg.dims))} grid, {k} Strang steps, float64, "
                      f"{dt:.1f} s wall",
            "single_thread": {"value": cfg.cells * k1 / dt1, "steps": k1, "wall_s": dt1}}, cfg, k, dt


def run_reference(args, inputs):
    """--impl reference: the oracle (oracle/snref.c) timed on the host cores; rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    base = inputs.CONFIGS[args.workload]
    from oracle.snref import Oracle
    from oracle import snref
    cfg = inputs.scaled(base, (128, 128, 128)) if (len(base.dims) == 3 and base.cells > 128 ** 3) else (
        inputs.scaled(base, (1024, 1024), L=base.L * 1024 / base.dims[0]) if base.cells > 1024 ** 2 else base)
    orc = Oracle.from_config(cfg)
    orc.set_state(cfg.initial_state().astype(np.complex128))
    orc.step(args.warmup)
    t0 = time.perf_counter()
    orc.step(args.steps)
    dt = time.perf_counter() - t0
    orc.close()
    value = cfg.cells * args.steps / dt
    sample = (f"each step = one float64 Strang step of the {base.name} recipe resampled on a "
              f"{'x'.join(map(str, cfg.dims))} grid (bounded sample of {'x'.join(map(str, base.dims))})")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": base.name, "dims": list(base.dims), "sample_dims": list(cfg.dims)},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": snref.num_threads(), "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def run_slab(args, cfg, psi0, dev, barrier):
    """--slab R: the decomposed step on one GPU (R contexts, one stream); one JSON line, no per-pass roofline."""
    import torch
    from paper_1909_08354_b200 import slab
    R, K = args.slab, args.steps
    grp = slab.LocalSlabGroup(cfg.dims, cfg.L, cfg.A, cfg.B, cfg.C, cfg.D, cfg.g, cfg.dtau, R, device=dev)
    grp.set_state(psi0)
    n0 = grp.norm()
    grp.step(args.warmup)
    stream = torch.cuda.current_stream()
    reps = []
    for r in range(args.repeats):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        l0, x0 = grp.launch_count(), grp.exchanged_elems
        barrier()
        e0.record(stream)
        grp.step(K)
        e1.record(stream)
        barrier()
        launches, moved = grp.launch_count() - l0, (grp.exchanged_elems - x0) * 8
        reps.append(e0.elapsed_time(e1))
    n1 = grp.norm()
    grp.close()
    ms = statistics.median(reps)
    print(json.dumps({
        "metric": METRIC, "value": cfg.cells * K / (ms * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": K, "warmup": args.warmup,
        "ms_per_step": ms / K, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
        "dtype": "complex64 (f32 arithmetic)", "data": "synthetic",
        "config": {"workload": f"{cfg.name}: {'x'.join(map(str, cfg.dims))}", "dims": list(cfg.dims),
                   "parallelism": f"slab decomposition, {R} virtual ranks on ONE GPU (sn_slab_exchange_local: device-to-device "
                                  f"block copies stand in for the all-to-all; not a multi-GPU measurement)"},
        "gpu_launches": launches, "exchange_bytes_per_step": moved / K,
        "exchange_bytes_per_cell_update": moved / K / cfg.cells,
        "repeats": {"n": len(reps), "ms_per_step_min": min(reps) / K, "ms_per_step_max": max(reps) / K},
        "checks": {"norm_before": n0, "norm_after": n1}}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--workload", default="C5_512")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--cpu-budget", type=float, default=15.0, help="seconds of oracle work for cpu_baseline")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--batch", type=int, default=0,
                    help="an ensemble of this many independent systems in one context (sn_create_batch; every "
                         "member a shifted, rescaled copy of the workload's state)")
    ap.add_argument("--bohm", type=float, default=0.0,
                    help="with --extras: also the Bohm term c_B V_B of eq. (15) with this coefficient")
    ap.add_argument("--order4", action="store_true",
                    help="time sn_step_order4 (Yoshida composition of three Strang steps per step) instead of sn_step")
    ap.add_argument("--extras", action="store_true",
                    help="NEXT-1 row: also run with the pressure potential 0.02 ln(rho) (eq. (16)) and the "
                         "phi_C table of eq. (11) as external potential and the beta, gamma tables of eq. (12) "
                         "(DESIGN.md section 8)")
    ap.add_argument("--dtype", default="c64", choices=["c64", "c128"],
                    help="c64: complex64 (BASELINE.json's metric); c128: the complex128 path (SURVEY.md 8(f) item 3, the "
                         "precision the paper benchmarked): same step, 16 B per cell of state, float64 arithmetic")
    ap.add_argument("--dispatch", type=int, default=0, choices=[0, 1, 2],
                    help="sn_set_option(SN_OPT_DISPATCH): 0 default, 1 first-path kernels only, 2 pipelined wherever instantiated")
    ap.add_argument("--graph-steps", type=int, default=0,
                    help="sn_set_option(SN_OPT_GRAPH_STEPS): interior steps per replayed CUDA graph (launch-bound grids)")
    ap.add_argument("--slab", type=int, default=0,
                    help="time the slab-decomposed step (NEXT-2, DESIGN.md section 7) as this many virtual ranks on ONE GPU: "
                         "the local passes of every rank plus the all-to-all exchanges done as device-to-device copies")
    ap.add_argument("--repeats", type=int, default=5,
                    help="timed repetitions of the K-step call (SURVEY.md 8(d): median of >= 5); value = median")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "b200" else args.warmup
    args.repeats = max(args.repeats, 1)

    # --gpus N without a launcher: become N replica processes (torchrun sets WORLD_SIZE; plain `python bench.py
    # --gpus 8` must not silently run one replica and print n_gpus 1)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        import socket
        with socket.socket() as so:
            so.bind(("127.0.0.1", 0))
            port = so.getsockname()[1]
        os.execv(sys.executable, [sys.executable, "-m", "torch.distributed.run", "--nnodes=1",
                                  f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1", "--master-port",
                                  str(port), os.path.abspath(__file__), *sys.argv[1:]])

    from paper_1909_08354_b200 import inputs
    if args.impl == "reference":
        run_reference(args, inputs)
        return

    import torch
    import torch.distributed as dist
    from paper_1909_08354_b200 import build as _build
    _build.build()                                      # no-op when libsn.so is up to date (it travels with the snapshot)
    from paper_1909_08354_b200 import replicas, sn

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    if world != args.gpus:
        raise SystemExit(f"bench.py --gpus {args.gpus} launched with WORLD_SIZE={world}: one rank per GPU")
    # SN_BENCH_BACKEND=gloo: dry run of the multi-rank plumbing on a box with fewer GPUs than ranks (ranks share
    # devices; replicas do not wait on one another).  Default nccl, one rank per GPU, as the driver launches it.
    backend = os.environ.get("SN_BENCH_BACKEND", "nccl")
    if backend != "nccl":
        local = local % torch.cuda.device_count()
    torch.cuda.set_device(local)
    dev = f"cuda:{local}"
    if world > 1:
        if backend == "nccl":
            dist.init_process_group("nccl", device_id=torch.device(dev))
        else:
            dist.init_process_group(backend)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    cfg = inputs.CONFIGS[args.workload]
    nd = len(cfg.dims)
    K, W = args.steps, args.warmup
    psi0 = cfg.initial_state()                          # seeded synthetic state, complex64
    f64 = args.dtype == "c128"
    esz = 16 if f64 else 8                              # bytes per complex value
    if f64:
        psi0 = psi0.astype(np.complex128)               # same rounded recipe state, carried in double
    if args.batch:
        rng = np.random.default_rng(1)
        mem = [np.roll(psi0, tuple(int(rng.integers(n)) for n in cfg.dims), axis=tuple(range(nd))) *
               np.complex64(0.8 + 0.4 * b / args.batch) for b in range(args.batch)]
        psi0 = np.ascontiguousarray(np.stack(mem, axis=1).astype(psi0.dtype))   # storage layout [n0][batch][...]
        del mem
    host_in = torch.from_numpy(psi0).pin_memory()
    host_out = torch.empty_like(host_in).pin_memory()
    dev_in = host_in.to(dev, non_blocking=True)

    if args.slab:
        run_slab(args, cfg, psi0, dev, barrier)
        return

    stream = torch.cuda.current_stream()
    sim = sn.Simulation.from_config(cfg, device=dev, stream=stream, batch=args.batch or None,
                                    features=(sn.FEAT_VEXT | sn.FEAT_SOURCE) if args.extras else 0,
                                    dtype="complex128" if f64 else "complex64")
    if args.extras:
        # eq. (16) n = 1: V_pressure = w ln(rho), w = 0.02; eq. (11): phi_C = ln[1 - (r0/(r + r0))^lambda], lambda = 1,
        # r0 = 2, radius softened to sqrt(r^2 + 1) (the grid has a point at r = 0)
        ax = [inputs.coords(n, cfg.L) for n in cfg.dims]
        r2 = sum(np.square(a).reshape([-1 if i == k else 1 for i in range(nd)]) for k, a in enumerate(ax))
        rs = np.sqrt(r2 + 1.0)
        f = 2.0 / (rs + 2.0)
        sim.set_local_terms(0.02, 1e-12, 0.0, 1.0)
        sim.set_external_potential(np.log(1.0 - f).astype(np.float32))
        # eq. (12) with eq. (9),(10): gamma = (1 - f)/2, beta = lambda f/(r + r0)
        sim.set_source_tables((f / (rs + 2.0)).astype(np.float32), (0.5 * (1.0 - f)).astype(np.float32))
        if args.bohm:
            sim.set_bohm(args.bohm, 1e-4)               # eq. (15): + nu^2 V_B
        del rs, f, r2
    if args.dispatch:
        sim.set_option(sn.OPT_DISPATCH, args.dispatch)
    if args.graph_steps:
        sim.set_option(sn.OPT_GRAPH_STEPS, args.graph_steps)
    step = sim.step_order4 if args.order4 else sim.step
    sim.set_state(dev_in)
    step(W)                                             # untimed warm-up steps
    barrier()

    # ---- timed region: exactly K Strang steps, state resident in HBM; repeated, each repetition bracketed by
    # barrier + synchronize with its own event pair; the reported time is the MEDIAN repetition ----
    reps = []
    with ClockSampler(local) as clk:
        for r in range(args.repeats):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            n0 = sim.launch_count()
            barrier()
            e0.record(stream)
            step(K)
            e1.record(stream)
            barrier()
            launches = sim.launch_count() - n0
            reps.append(e0.elapsed_time(e1))

    # ---- per-launch CUDA events over the same K steps (roofline of the dominant kernel) ----
    sim.profile(True)
    step(K)
    prof = sim.profile_read(reset=True)
    sim.profile(False)
    norm_after = sim.diagnostics()["norm"]

    # ---- e2e: host buffers through the public API, copies inside the timed region ----
    barrier()
    t0 = time.perf_counter()
    sim.set_state(host_in)
    step(K)
    sim.get_state(host_out)
    d = sim.diagnostics()
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    sim.close()

    # max over ranks (per repetition), then the median repetition
    red = replicas.max_over_ranks(reps + [e2e_s * 1e3], device=dev if backend == "nccl" else "cpu")
    reps, e2e_ms = red[:-1], red[-1]
    ms = statistics.median(reps)

    if rank == 0:
        cells = cfg.cells * max(1, args.batch)
        value = replicas.whole_job_rate(cells, K, world, ms)
        peak, peak_src = load_peaks()
        tot = sum(v[0] for v in prof.values()) or 1.0
        dom = max(prof, key=lambda k: prof[k][0])
        dom_ms = prof[dom][0] / prof[dom][1]
        hs_frac = (cfg.dims[0] // 2 + 1) / (cfg.dims[0] / 2)   # exact half-spectrum factor on the 4-byte terms
        def bytes_per_cell(kind):
            """algorithmic bytes per cell of the full grid for one launch of this pass kind"""
            return bytes_per_cell_c64(kind) * (esz / 8.0)   # complex128: every array is twice as wide

        def bytes_per_cell_c64(kind):
            if kind == "H_NLKIN":
                return 16.0 + 4.0 * hs_frac
            if kind == "H_R2C":
                return 8.0 + 4.0 * hs_frac
            if kind in ("S_FFT", "X_POISSON"):
                return 8.0 * hs_frac
            if kind == "X_KIN":
                return 16.0 + (4.0 if args.extras else 0.0)              # + the external potential table
            if kind == "H_SRC":
                return 16.0 + 8.0 * hs_frac
            if kind == "H_BOHM":
                return 16.0 + 4.0 * hs_frac
            return PASS_BYTES_PER_CELL.get(kind, 0.0)
        bpc = bytes_per_cell(dom)
        achieved = bpc * cells / (dom_ms * 1e-3) / 1e9
        out = {
            "metric": METRIC if not f64 else "split-step cell-updates/sec (complex128)", "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "complex128 (f64 arithmetic)" if f64 else "complex64 (f32 arithmetic)", "data": "synthetic",
            "config": {"workload": f"{cfg.name}{' x%d ensemble' % args.batch if args.batch else ''}{'+next1(0.02 ln rho, phi_C, beta/gamma tables of eq. (12))' if args.extras else ''}: {'x'.join(map(str, cfg.dims))} periodic, L={cfg.L}, A={cfg.A}, "
                                   f"B={cfg.B}, C={cfg.C}, D={cfg.D:.6g}, g={list(cfg.g)}, dtau={cfg.dtau}",
                       "dims": list(cfg.dims), "parallelism": "replicas only" if world > 1 else "single GPU",
                       "l2": "state %d B/cell x %d cells = %.0f MiB > 126 MB L2, no flush needed" % (
                           esz, cells, cells * esz / 2 ** 20) if cells * esz > 126e6 else
                       "state fits L2: launch/L2-bound regime, HBM fraction is an effective figure only",
                       "timed_call": f"one {'sn_step_order4' if args.order4 else 'sn_step'}({K}) (merged half kinetics) per "
                                     f"repetition; value = median of {len(reps)} repetitions"},
            "repeats": {"n": len(reps), "ms_per_step_median": ms / K, "ms_per_step_min": min(reps) / K,
                        "ms_per_step_max": max(reps) / K},
            "gpu_launches": launches,
            "clocks": clk.summary(),
            "roofline": {
                "bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak,
                "traffic": NCU_TRAFFIC_C5_512.get(dom) if cfg.name == "C5_512" and not args.extras and not f64 and not args.batch else None,
                "traffic_source": "ncu --set full dram__bytes_read.sum + dram__bytes_write.sum per launch, profiles/r02z_final_C5_512.md",
                "note": ("R_STEPS = the cluster-resident kernel: one launch advances all K steps with the state in distributed "
                         "shared memory, HBM sees 16 B/cell per CALL; it is latency-bound inside the cluster, so every HBM "
                         "fraction of this line is an effective figure only") if dom == "R_STEPS" else None,
                "algorithmic_bytes_per_launch": bpc * cells, "peak_source": peak_src,
                "bytes_per_cell": bpc, "avg_launch_ms": dom_ms, "share_of_step": prof[dom][0] / tot,
                "per_pass": {k: {"ms_per_launch": v[0] / v[1], "launches": v[1], "share": v[0] / tot,
                                 "bytes_per_cell": bytes_per_cell(k),
                                 "achieved_GBps": bytes_per_cell(k) * cells / (v[0] / v[1] * 1e-3) / 1e9,
                                 "frac_of_measured_peak": bytes_per_cell(k) * cells / (v[0] / v[1] * 1e-3) / 1e9 / peak}
                             for k, v in sorted(prof.items())},
                "step": {"b_min_bytes_per_cell_update": B_MIN[nd] * (esz / 8.0),
                         "achieved_GBps_over_b_min": B_MIN[nd] * (esz / 8.0) * cells * K / (ms * 1e-3) / 1e9,
                         "frac_of_measured_peak": B_MIN[nd] * (esz / 8.0) * cells * K / (ms * 1e-3) / 1e9 / peak,
                         "frac_of_8TBps_nominal": B_MIN[nd] * (esz / 8.0) * cells * K / (ms * 1e-3) / 8e12,
                         "own_bytes_per_cell_update": B_OWN[nd] * (esz / 8.0),
                         "achieved_GBps_over_own_bytes": B_OWN[nd] * (esz / 8.0) * cells * K / (ms * 1e-3) / 1e9,
                         "own_frac_of_measured_peak": B_OWN[nd] * (esz / 8.0) * cells * K / (ms * 1e-3) / 1e9 / peak},
            },
            "e2e": {"value": replicas.whole_job_rate(cells, K, world, e2e_ms), "unit": UNIT,
                    "h2d_bytes_per_step": cells * esz / K, "d2h_bytes_per_step": (cells * esz + 40) / K,
                    "call": f"sn_set_state(pinned host) + sn_step({K}) + sn_get_state(pinned host) + sn_diagnostics",
                    "h2d_bytes_per_call": cells * esz, "d2h_bytes_per_call": cells * esz + 40, "ms_per_call": e2e_ms},
            "checks": {"norm_after_timed_steps": norm_after, "norm_after_e2e": d["norm"]},
        }
        if world == 1 and not args.no_cpu_baseline:
            out["cpu_baseline"] = oracle_rate(args.workload, args.cpu_budget, inputs)[0]
        print(json.dumps(out))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
