#!/usr/bin/env python
"""bench.py -- throughput of the QSS-chemistry hot path (wdot + analytical QSS Jacobian, fp64) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 2]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

A "step" is one pass of the whole hot path (rate constants -> QSS closure -> wdot ->
analytical Jacobian with the chain rule, Eq. 2-4, 6, 7, 9) over one batch of synthetic cells: one
`qss_eval_jac` call with the wdot output enabled.  Workload at N=1: BASELINE.json configs[1] (the mid-size
35+18-species, 270-reaction synthetic mechanism, 2^20 cells), the config the metric's target is quoted on.
At N>1 every rank evaluates its own 2^20 cells (cells are independent: no data-path collective; "weak").

Prints ONE JSON line (rank 0).  Keys: DESIGN.md "Measurement".
`--impl reference` times the CPU oracle (oracle/, as it stands) on the host cores on a bounded sample of the
same workload; the oracle is never used on the product path.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "cells/sec for wdot+analytical QSS Jacobian (fp64) per B200; % of roofline"
UNIT = "cells/s"
ORACLE_SAMPLE = {1: 4096, 2: 1 << 15, 3: 1 << 12, 4: 1 << 15, 5: 1 << 9}   # cells of the CPU-oracle sample
FP64_LANES_PER_SM = 64          # 148 SMs x 64 fp64 FMA lanes x 1.965 GHz
EXPECTED_JAC_VARIANT = {1: 3, 2: 3, 4: 3, 3: 0, 5: 0}   # the kernel each BASELINE config is expected to run on
CALLS = {"jac+wdot": "qss_eval_jac with the wdot output (the metric)", "jac": "qss_eval_jac alone", "wdot": "qss_eval_wdot alone",
         "jac+wdot+energy": "qss_eval_jac with wdot, then qss_eval_energy: the full (N+1)x(N+1) Jacobian and the temperature right-hand side",
         "jac_full": "qss_eval_jac_full: the full (N+1)x(N+1) Jacobian, wdot and Tdot in one call (two launches)",
         "energy": "qss_eval_energy alone (on a Jacobian computed before the timed region)",
         "jac_const": "qss_eval_jac_approx, constant-QSS AJ", "jac_zero": "qss_eval_jac_approx, zero-QSS AJ",
         "aos": "qss_jac_to_aos alone: the (N+1) x (N+1) Jacobian (computed before the timed region) as one contiguous row-major matrix per cell",
         "newton": "qss_newton_solve alone: x = (I - gamma J)^-1 (wdot, Tdot) on a full Jacobian computed before the timed region",
         "jac+wdot+energy+newton": "qss_eval_jac with wdot, qss_eval_energy, qss_newton_solve: one Newton direction of an implicit step",
         "sums_thread": "qss_bench_species_sums mode 0: mapping micro-benchmark, species sums with lane = cell (not on the path)",
         "sums_warp": "qss_bench_species_sums mode 1: mapping micro-benchmark, species sums with a warp per cell and SHFL reductions (not on the path)",
         "ignition": "qss_ignition_advance: one adaptive attempt with two full Newton iterations (accept / reject, step control and ignition time on the device), state restored before every step",
         "bdf1": "qss_bdf1_advance: one backward-Euler substep with two full Newton iterations (two kernels each: Jacobian, fused Newton step), state restored before every step"}


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "MEASURED_PEAKS.json", float(d.get("sm_max_mhz", 1965.0))
    return 6650.0, "fallback (B200_PROFILING.md)", 1965.0


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 100 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--id={index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                       "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.p = None

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.p.terminate()
        try:
            out, _ = self.p.communicate(timeout=5)
        except Exception:
            self.p.kill(); out = ""
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.strip().splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def run_reference(args, cfg: int, rank: int):
    """The oracle, as it stands, on the host cores (rank 0 only)."""
    if rank != 0:
        return
    import numpy as np
    import oracle
    import qss_synth
    mech = qss_synth.config_mechanism(cfg)
    n = ORACLE_SAMPLE[cfg]
    C, T = qss_synth.config_states(cfg, n)
    n = min(n, C.shape[1])
    om = oracle.OracleMech(mech)
    # every host core this process may use, also under torchrun (which exports OMP_NUM_THREADS=1 to its ranks)
    cores = max(oracle.max_threads(), len(os.sched_getaffinity(0)))
    for _ in range(args.warmup):
        oracle.evaluate(om, C, T, min(n, 256), want_jac=True, nthreads=cores)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.evaluate(om, C, T, n, want_jac=True, nthreads=cores)
    dt = (time.perf_counter() - t0) / args.steps
    v = n / dt
    sample = f"first {n} cells of cfg{cfg} per step (explicit-formula fp64 oracle, OpenMP over cells)"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic", "config": _config(cfg, mech, n, args.gpus),
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def _cpu_model():
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return None


def _config(cfg, mech, n_cells, n_gpus):
    return {"workload": f"BASELINE.json configs[{cfg - 1}] (cfg{cfg}): synthetic QSS mechanism {mech.n_nqss} transported + "
                        f"{mech.n_qss} QSS species, {mech.n_reac} reactions; {n_cells} cells per GPU; Jacobian "
                        f"{mech.n_nqss}x{mech.n_nqss + 1} per cell + wdot",
            "cfg": cfg, "n_nqss": mech.n_nqss, "n_qss": mech.n_qss, "n_reac": mech.n_reac, "cells_per_gpu": n_cells,
            "parallelism": f"cells sharded over {n_gpus} GPU(s), no collective",
            "l2_policy": "inputs (C,T) and outputs (J,wdot) per step exceed the 126 MB L2; no flush needed"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config index (1-based); default 2 = configs[1]")
    ap.add_argument("--cells", type=int, default=0, help="override the cell count (0 = the config's)")
    ap.add_argument("--call", default="jac+wdot", choices=sorted(CALLS), help="which C-ABI call(s) a step is: " + "; ".join(f"{k}: {v}" for k, v in CALLS.items()))
    ap.add_argument("--allow-fallback", action="store_true", help="do not fail when the library selected another kernel variant than the expected one")
    ap.add_argument("--ld-pad", type=int, default=64, help="cells of padding behind the workload in every row (leading dimension = cells + pad; default 64: row strides that are "
                    "powers of two are avoided, DESIGN.md section 5); -1: the leading dimension of the input generator")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    cfg = args.config
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # plain `python bench.py --gpus N`: launch the N ranks ourselves, the way the driver does (one process per GPU)
        port = 29500 + os.getpid() % 2000
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
               "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        raise SystemExit(subprocess.run(cmd).returncode)
    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, cfg, rank)
        return

    import numpy as np
    import torch
    import qss_synth
    import paper_2405_05974_b200 as qss
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libqss has no CPU fallback")
    ndev = torch.cuda.device_count()
    local = local % ndev                     # more ranks than devices (a 1-GPU box): the ranks share a device, timing is then not a scaling number
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        if world <= ndev:
            dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        else:
            dist.init_process_group("gloo")  # NCCL refuses two ranks on one device; the group only carries the barrier and the max of the times
    dev = torch.device("cuda", local)

    mech = qss_synth.config_mechanism(cfg)
    n_full = qss_synth.CONFIGS[cfg]["n_cells"]
    n = args.cells or n_full
    C, T = qss_synth.config_states(cfg, n)
    n = min(n, C.shape[1]) if cfg == 4 else n
    if args.ld_pad >= 0:        # the same states with another leading dimension (padding cells repeat cell 0)
        ld2 = n + args.ld_pad
        C2 = np.empty((C.shape[0], ld2)); T2 = np.empty(ld2)
        C2[:, :n] = C[:, :n]; T2[:n] = T[:n]; C2[:, n:] = C[:, :1]; T2[n:] = T[0]
        C, T = C2, T2
    ld = C.shape[1]
    t_create = time.perf_counter()
    qm = qss.QssMech(mech, local)            # includes the run-time specialisation of the Jacobian kernel (NVRTC), untimed below
    t_create = time.perf_counter() - t_create
    N = qm.N
    Cd = torch.from_numpy(C).to(dev); Td = torch.from_numpy(T).to(dev)
    J = torch.empty((N, N + 1, ld), dtype=torch.float64, device=dev)
    W = torch.empty((N, ld), dtype=torch.float64, device=dev)
    qm.workspace(True)
    stream = torch.cuda.current_stream()
    if os.environ.get("QSS_BENCH_ADDR"):        # (diagnostic: device addresses of the buffers, for layout experiments)
        print("addr", {k: hex(v.data_ptr()) for k, v in dict(C=Cd, T=Td, J=J, W=W, ws=qm.workspace(True)).items()}, "ld", ld, file=sys.stderr)

    qm.workspace(False)
    expect = EXPECTED_JAC_VARIANT.get(cfg)
    forced = "QSS_VARIANT" in os.environ or "QSS_JIT" in os.environ
    if expect is not None and qm.info.kernel_variant_jac != expect and not args.allow_fallback and not forced:
        raise SystemExit(f"bench.py: cfg{cfg} ran on kernel variant {qm.info.kernel_variant_jac}, expected {expect} (run-time compilation unavailable?); "
                         "--allow-fallback times it anyway")
    tdot = torch.empty((ld,), dtype=torch.float64, device=dev); erow = torch.empty((N + 1, ld), dtype=torch.float64, device=dev)
    B = X = gam = None
    if "newton" in args.call:        # wdot and Tdot are written straight into the right-hand side (no copies in a step)
        B = torch.empty((N + 1, ld), dtype=torch.float64, device=dev)
        W = B[:N]; tdot = B[N]
    if args.call in ("energy", "newton", "jac+wdot+energy+newton", "aos"):
        qm.eval_jac(Cd, Td, n, jac=J, wdot=W, want_wdot=True)
    AOS = None
    if args.call == "aos":
        qm.eval_energy(Cd, Td, W, J, n, tdot=tdot, erow=erow)
        AOS = torch.empty((n, N + 1, N + 1), dtype=torch.float64, device=dev)
    if "newton" in args.call:
        # right-hand side (wdot, Tdot); gamma_c = theta_c / max|J_c|, theta log-uniform in [1e-2, 1e3] (seeded): from "explicit would do" to stiff
        qm.eval_energy(Cd, Td, W, J, n, tdot=tdot, erow=erow)
        X = torch.empty_like(B)
        jmax = torch.maximum(J.abs().amax((0, 1)), erow.abs().amax(0))
        g = torch.Generator(device=dev); g.manual_seed(7)
        gam = torch.exp(np.log(10.0) * (torch.rand(ld, dtype=torch.float64, device=dev, generator=g) * 5.0 - 2.0)) / torch.where(jmax > 0, jmax, torch.ones_like(jmax))
        del jmax
        qm.newton_solve(J, erow, gam, B, n, x=X)        # (first call: run-time compilation, outside the timed region)
        torch.cuda.synchronize()
        assert bool(torch.isfinite(X[:, :n]).all())
    Qm = None
    if args.call.startswith("sums_"):        # rates of progress: seeded normal values (the arithmetic does not depend on them)
        g = torch.Generator(device=dev); g.manual_seed(11)
        Qm = torch.randn((qm.info.n_reac, ld), dtype=torch.float64, device=dev, generator=g)
    launches_per_step = {"jac+wdot+energy": 2, "jac+wdot+energy+newton": 3, "bdf1": 4, "ignition": 4, "jac_full": 2}.get(args.call, 1)
    if args.call in ("bdf1", "ignition"):
        # h_c = 3 / max|J_c| at the initial state (a few of the fastest time scales per substep); the state is restored before every step
        del J
        torch.cuda.empty_cache()
        Jt, Wt = qm.eval_jac(Cd, Td, n, want_wdot=True)
        td0, er0 = qm.eval_energy(Cd, Td, Wt, Jt, n)
        jmax = torch.maximum(Jt.abs().amax((0, 1)), er0.abs().amax(0))
        dtd = 3.0 / torch.where(jmax > 0, jmax, torch.ones_like(jmax))
        del Jt, Wt, td0, er0, jmax
        torch.cuda.empty_cache()
        C0, T0 = Cd.clone(), Td.clone()
        bdf_ws = qm.bdf1_advance(Cd, Td, dtd, 1, 2, n)
        torch.cuda.synchronize()
        J = None
        if args.call == "ignition":
            dt0 = dtd.clone(); tcur = torch.zeros(ld, dtype=torch.float64, device=dev); tign = torch.full((ld,), float("nan"), dtype=torch.float64, device=dev)

    def step():
        if args.call in ("jac+wdot", "jac+wdot+energy", "jac+wdot+energy+newton"):
            qm.eval_jac(Cd, Td, n, jac=J, wdot=W, want_wdot=True)
            if args.call != "jac+wdot":
                qm.eval_energy(Cd, Td, W, J, n, tdot=tdot, erow=erow)
            if args.call == "jac+wdot+energy+newton":
                qm.newton_solve(J, erow, gam, B, n, x=X)
        elif args.call == "newton":
            qm.newton_solve(J, erow, gam, B, n, x=X)
        elif args.call.startswith("sums_"):
            qm.bench_species_sums(0 if args.call == "sums_thread" else 1, Qm, n, wdot=W)
        elif args.call == "bdf1":
            Cd.copy_(C0); Td.copy_(T0)
            qm.bdf1_advance(Cd, Td, dtd, 1, 2, n, workspace=bdf_ws)
        elif args.call == "ignition":
            Cd.copy_(C0); Td.copy_(T0); dtd.copy_(dt0); tcur.zero_()
            qm.ignition_advance(Cd, Td, dtd, tcur, 1.0e30, 1, 2, n, t_ign=tign, T0=T0, workspace=bdf_ws)
        elif args.call == "jac_full":
            qm.eval_jac_full(Cd, Td, n, jac=J, wdot=W, tdot=tdot, erow=erow)
        elif args.call == "jac":
            qm.eval_jac(Cd, Td, n, jac=J)
        elif args.call == "energy":
            qm.eval_energy(Cd, Td, W, J, n, tdot=tdot, erow=erow)
        elif args.call == "aos":
            qm.jac_to_aos(J, erow, n, out=AOS)
        elif args.call in ("jac_const", "jac_zero"):
            qm.eval_jac_approx(Cd, Td, 1 if args.call == "jac_const" else 2, n, jac=J)
        else:
            qm.eval_wdot(Cd, Td, n, wdot=W)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- fp64 FMA-pipe peak, measured in the same run (roofline denominator cross-check)
    sink = torch.zeros(8, dtype=torch.float64, device=dev)
    sms = torch.cuda.get_device_properties(dev).multi_processor_count
    qss.bench_dfma(sms * 8, 200, sink); torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream); nf = qss.bench_dfma(sms * 8, 4000, sink); e1.record(stream); torch.cuda.synchronize()
    dfma_slots_s = nf / (e0.elapsed_time(e1) * 1e-3)

    for _ in range(args.warmup):
        step()
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    evs = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    evs[0].record(stream)
    for i in range(args.steps):
        step()
        evs[i + 1].record(stream)
    barrier()
    clocks = sampler.stop() if sampler else None
    total_ms = evs[0].elapsed_time(evs[-1])
    launch_ms = [evs[i].elapsed_time(evs[i + 1]) for i in range(args.steps)]
    from paper_2405_05974_b200.shard import max_over_ranks
    total_ms_max = max_over_ranks(total_ms, dist, dev if (dist is None or dist.get_backend() == "nccl") else None)
    value = world * n * args.steps / (total_ms_max * 1e-3)

    # ---- end to end through the C-ABI host-buffer call: pinned host buffers, H2D + D2H inside the timed region
    e2e = None
    if not args.no_e2e and args.call == "jac+wdot":
        del J, W
        torch.cuda.empty_cache()
        Ch = torch.from_numpy(C).pin_memory(); Th = torch.from_numpy(T).pin_memory()
        Jh = torch.empty((N, N + 1, ld), dtype=torch.float64).pin_memory()
        Wh = torch.empty((N, ld), dtype=torch.float64).pin_memory()
        scratch = torch.empty(qm.host_scratch_bytes(n, ld) + 256, dtype=torch.uint8, device=dev)
        ke = max(1, min(args.steps, 3))
        qm.eval_jac_host(Ch, Th, Jh, Wh, scratch, n)
        barrier()
        t0 = time.perf_counter()
        for _ in range(ke):
            qm.eval_jac_host(Ch, Th, Jh, Wh, scratch, n)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        e2e = {"value": world * n * ke / max_over_ranks(dt, dist, dev if (dist is None or dist.get_backend() == "nccl") else None), "unit": UNIT,
               "h2d_bytes_per_step": int((N + 1) * ld * 8), "d2h_bytes_per_step": int((N * (N + 1) + N) * ld * 8),
               "steps": ke, "api": "qss_eval_jac_host (C-ABI, pinned host buffers, copies + kernel + sync timed by wall clock)"}
        assert bool(torch.isfinite(Wh[:, :n]).all())

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant (only) kernel: qss Jacobian kernel
    hbm_gbs, peak_src, sm_max_mhz = _peaks()
    info = qm.info
    avg_s = statistics.mean(launch_ms) * 1e-3
    if args.call == "wdot":
        bytes_cell, slots_cell = info.bytes_wdot, info.slots_wdot
    elif args.call == "energy":        # reads C, T, wdot and J once, writes the row and tdot; 2 N (N+1) + ~30 N fp64 slots
        bytes_cell, slots_cell = 8.0 * (N * (N + 1) + 2 * N + 1) + 8.0 * (N + 2), 2.0 * N * (N + 1) + 30.0 * N
    elif args.call == "aos":           # reads and writes the (N+1)^2 matrix once; no arithmetic
        bytes_cell, slots_cell = 16.0 * (N + 1) * (N + 1), 0.0
    elif args.call == "newton":        # reads the (N+1)^2 matrix, b and gamma once, writes x; n^3/3 + n^2 fp64 FMA slots (elimination + substitutions)
        nn = N + 1
        bytes_cell, slots_cell = 8.0 * (nn * nn + 2 * nn + 1), nn ** 3 / 3.0 + nn * nn
    elif args.call.startswith("sums_"):   # reads Q once, writes wdot; one multiply-add per non-zero of the net stoichiometric matrix (~4 per reaction)
        bytes_cell, slots_cell = 8.0 * (info.n_reac + N), 4.0 * info.n_reac
    elif args.call in ("bdf1", "ignition"):          # two Newton iterations: the three heavy calls twice (the residual / update kernels move 5 (N+1) doubles each)
        nn = N + 1
        bytes_cell = 2.0 * ((info.bytes_jac + 8.0 * N) + (8.0 * (N * nn + 2 * N + 1) + 8.0 * (N + 2)) + 8.0 * (nn * nn + 2 * nn + 1) + 8.0 * 9 * nn)
        slots_cell = 2.0 * (info.slots_jac + 2.0 * N * nn + 30.0 * N + nn ** 3 / 3.0 + nn * nn)
    else:
        bytes_cell, slots_cell = info.bytes_jac + (8.0 * N if args.call.startswith("jac+wdot") else 0.0), info.slots_jac
        if args.call == "jac_full":      # + wdot, Tdot, the energy row; + 2 N (N+1) + ~30 N slots for the row
            bytes_cell += 8.0 * (2 * N + 2); slots_cell += 2.0 * N * (N + 1) + 30.0 * N
    bytes_launch = bytes_cell * n
    slots_launch = slots_cell * n
    fp64_peak_slots = sms * FP64_LANES_PER_SM * sm_max_mhz * 1e6
    t_hbm = bytes_launch / (hbm_gbs * 1e9); t_alu = slots_launch / fp64_peak_slots
    if t_alu >= t_hbm:
        roof = {"bound": "alu", "achieved": 2 * slots_launch / avg_s / 1e12, "peak": 2 * fp64_peak_slots / 1e12, "unit": "TFLOP/s"}
    else:
        roof = {"bound": "hbm", "achieved": bytes_launch / avg_s / 1e9, "peak": hbm_gbs, "unit": "GB/s"}
    roof["frac"] = roof["achieved"] / roof["peak"]
    traffic = None
    try:        # bytes of one launch from the committed ncu capture of the same workload and kernel variant, else null
        with open(os.path.join(ROOT, "profiles", "r02_traffic.txt")) as f:
            tj = json.load(f)
        if args.call == "jac+wdot" and tj["cfg"] == cfg and tj["cells"] == n and tj["kernel_variant"] == info.kernel_variant_jac:
            traffic = tj["dram_bytes_per_launch"]
    except Exception:
        traffic = None
    roof.update({"traffic": traffic, "traffic_unit": "bytes per launch (dram read + write) from the committed ncu capture of this workload and kernel variant (profiles/r02_traffic.txt); not measurable inside this run",
                 "kernel": "qss_mapbench_kernel" if args.call.startswith("sums_") else "qss_energy_kernel" if args.call == "energy" else "qss_jac_aos_kernel" if args.call == "aos" else "qss_newton_kernel" if args.call == "newton" else "the 4 launches of one substep (Jacobian kernel, fused Newton step; twice)" if args.call in ("bdf1", "ignition") else ("qss wdot kernel (qss_eval_wdot)" if args.call == "wdot" else f"qss jacobian kernel, variant {info.kernel_variant_jac} ({CALLS[args.call]})"),
                 "launch_ms_avg": avg_s * 1e3, "launch_ms_min": min(launch_ms),
                 "alg_fp64_slots_per_cell": slots_cell, "alg_bytes_per_cell": bytes_cell,
                 "t_alu_ms": t_alu * 1e3, "t_hbm_ms": t_hbm * 1e3,
                 "hbm_achieved_gbs": bytes_launch / avg_s / 1e9, "hbm_frac": bytes_launch / avg_s / 1e9 / hbm_gbs,
                 "peak_source": f"alu: {sms} SMs x {FP64_LANES_PER_SM} fp64 FMA lanes x {sm_max_mhz:.0f} MHz (nominal; DESIGN.md); "
                                f"hbm: {peak_src}",
                 "dfma_measured_tflops": 2 * dfma_slots_s / 1e12})

    cpu = None
    if not args.no_cpu:
        import oracle
        ns = min(ORACLE_SAMPLE[cfg], n)
        Cs = np.ascontiguousarray(C[:, :ns]); Ts = np.ascontiguousarray(T[:ns])
        om = oracle.OracleMech(mech)
        oracle.evaluate(om, Cs, Ts, min(ns, 256), want_jac=True)
        t0 = time.perf_counter()
        oracle.evaluate(om, Cs, Ts, ns, want_jac=True)
        dt = time.perf_counter() - t0
        n1 = max(32, ns // 16)      # single-thread figure on a 16x smaller sample
        t0 = time.perf_counter()
        oracle.evaluate(om, Cs, Ts, n1, want_jac=True, nthreads=1)
        dt1 = time.perf_counter() - t0
        cpu = {"value": ns / dt, "unit": UNIT, "cores": oracle.max_threads(), "kind": "oracle",
               "sample": f"first {ns} cells of the same cfg{cfg} input, explicit-formula fp64 oracle, OpenMP over cells, {dt:.2f} s",
               "value_1thread": n1 / dt1, "sample_1thread": f"first {n1} cells, one thread, {dt1:.2f} s",
               "cpu_model": _cpu_model()}

    print(json.dumps({
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": total_ms_max / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic", "config": dict(_config(cfg, mech, n, world), call=args.call, ld=int(ld)),
        "clocks": clocks, "e2e": e2e, "gpu_launches": args.steps * launches_per_step, "roofline": roof, "cpu_baseline": cpu,
        "kernel_variant": {"wdot": info.kernel_variant_wdot, "jac": info.kernel_variant_jac}, "mech_create_s": t_create,
        "call": args.call}))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
