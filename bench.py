#!/usr/bin/env python
"""bench.py -- throughput of the batched-LM hot path on B200 (contract: see DESIGN.md section 6).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--workload C4|C2|C3|C5]

One "step" = one pass of the whole hot path (S0..S10: load seeds + targets, the on-device LM loop,
store) over one batch of synthetic input: ``lm_reset`` + ``lm_run(max_iters)``.  The headline
workload is BASELINE.json configs[3] (4096 trajectories x 300 waypoints, 7-DoF Panda, 50 LM
iterations) -- the configuration the north_star's roofline target is quoted on.  Metric:
waypoint-LM-iterations/s (executed iterations only), whole job.

N > 1 (torchrun): every rank refines its own batch of the same shape (trajectories are
independent units, no data-path collective) -> weak scaling; time = max over ranks.

`--impl reference` times the fp64 CPU oracle (oracle/) on the host cores on a bounded sample of
the same workload (rank 0 only).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "waypoint_lm_iterations_per_sec"
UNIT = "waypoint-iterations/s"

# Algorithmic FLOPs per waypoint-iteration (DESIGN.md section 6 / SURVEY.md section 8d; FMA = 2).
ALG_FLOP = {7: 1459.0, 8: 1762.0}
# the dual 6 x 6 variant (LM_SOLVER_DUAL): Jacobian 84, J J^T + lambda 42 d + 6, Cholesky 70,
# solves 72, J^T y 12 d, update 3 d, FK 48 d + 6, residual 77, accept 5
ALG_FLOP_DUAL = {7: 1055.0, 8: 1160.0}
# FP32 FMA-pipe peak derived from the guide's unit counts and clocks: 148 SMs x 128 lanes x 2 x f_max
SM_COUNT, FP32_LANES = 148, 128
# Numbers that only an ncu capture can give (DRAM bytes per launch, executed FP32 flop per waypoint-iteration) live in
# profiles/ncu_constants.json, each entry naming the capture it was read from and the SHA-256 of the kernel sources it
# was taken with; an entry whose hash does not match the sources of this checkout is reported as null (stale).
HOT_SOURCES = ("lm_device.cuh", "lm_kernels.cuh", "lm_specs.cuh")
TRAJ_SOURCES = ("lm_traj.cuh", "lm_coll.cuh", "lm_device.cuh", "lm_traj_launch.h")


def source_hash(files) -> str:
    import hashlib
    h = hashlib.sha256()
    for f in files:
        h.update(open(os.path.join(ROOT, "paper_2309_09102_b200", "csrc", f), "rb").read())
    return h.hexdigest()[:16]


def ncu_constant(key: str, field: str, files):
    """profiles/ncu_constants.json[key][field] if the entry was captured with the current kernel sources, else None."""
    try:
        e = json.load(open(os.path.join(ROOT, "profiles", "ncu_constants.json")))[key]
    except (OSError, KeyError, ValueError):
        return None
    return e.get(field) if e.get("source_sha256_16") == source_hash(files) else None


def load_peaks() -> dict:
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    d = {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "_source": "fallback"}
    if os.path.exists(p):
        d = json.load(open(p))
        d["_source"] = "measured"
    # FP32 pipe peak, derived: SMs x FP32 lanes x 2 x the maximum SM clock
    d["alu_tflops"] = SM_COUNT * FP32_LANES * 2 * d["sm_max_mhz"] * 1e6 / 1e12
    return d


def alg_bytes_per_waypoint(d: int) -> float:
    """S0 + S10 traffic per waypoint per run: seeds 4d + target 28 in;
    q 4d + lambda, |r|, pos, rot 16 + iters/status 4 + mask 8 out."""
    return 4 * d + 28 + 4 * d + 16 + 4 + 8


# ------------------------------------------------------------------ clocks sampler

class ClockSampler:
    """SM clock and throttle reasons sampled through NVML every 10 ms while the timed region runs
    (the same counters `nvidia-smi --query-gpu=clocks.sm,clocks_event_reasons.*` prints)."""
    REASONS = {"hw_slowdown": 0x8, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20, "sw_power_cap": 0x4}

    def __init__(self, index: int):
        self.index, self.sm, self.bits, self.power = index, [], [], []
        self.stop_flag, self.thread, self.err, self.sm_max = threading.Event(), None, None, None

    def _loop(self, h, nv):
        while not self.stop_flag.is_set():
            try:
                self.sm.append(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM))
                self.bits.append(nv.nvmlDeviceGetCurrentClocksEventReasons(h)
                                 if hasattr(nv, "nvmlDeviceGetCurrentClocksEventReasons")
                                 else nv.nvmlDeviceGetCurrentClocksThrottleReasons(h))
                self.power.append(nv.nvmlDeviceGetPowerUsage(h) / 1000.0)
            except Exception as e:  # noqa: BLE001
                self.err = repr(e)
                return
            time.sleep(0.01)

    def start(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            idx = self.index
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            if vis and all(x.strip().isdigit() for x in vis.split(",")):
                idx = int(vis.split(",")[self.index])
            h = nv.nvmlDeviceGetHandleByIndex(idx)
            self.sm_max = nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM)
            self.thread = threading.Thread(target=self._loop, args=(h, nv), daemon=True)
            self.thread.start()
        except Exception as e:  # noqa: BLE001
            self.err = repr(e)
        return self

    def stop(self) -> dict:
        self.stop_flag.set()
        if self.thread is not None:
            self.thread.join(timeout=2)
        if not self.sm:
            return {"sm_mhz": None, "sm_max_mhz": self.sm_max, "samples": 0, "reasons": [], "error": self.err}
        reasons = sorted(n for n, b in self.REASONS.items() if any(x & b for x in self.bits))
        return {"sm_mhz": float(np.median(self.sm)), "sm_min_mhz": float(min(self.sm)), "sm_max_mhz": float(self.sm_max),
                "power_w_max": float(max(self.power)), "samples": len(self.sm), "reasons": reasons}


# ------------------------------------------------------------------ distributed plumbing

def dist_env():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def dist_init(backend: str):
    import torch.distributed as dist
    rank, _, world = dist_env()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29511")
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, world


def dist_barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def dist_max_sum(ms: float, units: float, device) -> tuple:
    """(max over ranks of ms, sum over ranks of units) -- the only cross-rank quantities of the
    path (trajectories are independent units; there is no data-path collective)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return ms, units
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    u = torch.tensor([units], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def spawn_ranks(n: int, argv: list) -> int:
    """Re-run this script as n ranks of one node under torch.distributed.run (one process per GPU, LOCAL_RANK = device
    index), exactly as the driver launches the N > 1 bench; returns its exit code.  Rank 0's JSON line passes through."""
    import socket
    import subprocess
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__)] + list(argv)
    return subprocess.call(cmd)


def run_dist_selftest(args) -> None:
    """The N > 1 plumbing without a GPU (tests/test_dist_cpu.py): process group over gloo, the barrier, the MAX of the
    per-rank times and the SUM of the per-rank units -- everything that crosses ranks in run_gpu -- and rank 0's line."""
    import torch
    rank, world = dist_init("gloo")
    dist_barrier()
    ms, units = dist_max_sum(1.0 + rank, 1.0, torch.device("cpu"))
    dist_barrier()
    if rank == 0:
        print(json.dumps({"selftest": "dist", "n_gpus": world, "requested": args.gpus, "ms_max": ms, "units_sum": units}), flush=True)


def rank_seed_offset(rank: int) -> int:
    """Each rank draws its own batch (weak scaling): the workload seed is offset by 1000 * rank."""
    return 1000 * rank


# ------------------------------------------------------------------ workloads

def make_workload(name: str, fk, B: int | None, n: int | None, rank: int = 0):
    from paper_2309_09102_b200 import workloads as wl
    kw = {"seed_offset": rank_seed_offset(rank)}
    if B:
        kw["B"] = B
    if n:
        kw["n"] = n
    if name == "C4":
        return wl.config4(fk, **kw)
    if name == "C2":
        return wl.config2(fk, **kw)
    if name == "C3":
        return wl.config3(fk, **kw)
    if name == "C5":
        kw.setdefault("B", 4096)
        kw.setdefault("n", 300)
        return wl.config5(fk, **kw)
    raise SystemExit(f"unknown workload {name}")


def workload_desc(w) -> dict:
    return {"workload": f"{w.name}: {w.B} trajectories x {w.n} waypoints, {w.chain.dof}-DoF {w.chain.name}, "
                        f"tol={w.tol:g}, max_iters={w.max_iters}, lambda0={w.lambda0:g}",
            "B": w.B, "n": w.n, "dof": int(w.chain.dof), "max_iters": w.max_iters, "tol": w.tol}


# ------------------------------------------------------------------ CPU oracle legs

def time_oracle(w, n_traj: int, steps: int = 1, warmup: int = 0, nthreads: int = 0) -> dict:
    """The oracle as it stands, on the host cores, on the first n_traj trajectories of w."""
    from oracle import lm_oracle as orc
    sub = w.subset(slice(0, min(n_traj, w.B)))
    prm = orc.Params(lambda0=sub.lambda0, tol=sub.tol)
    tp, tq, s = sub.target_pos.astype(np.float64), sub.target_quat.astype(np.float64), sub.seeds.astype(np.float64)
    times, executed = [], 0
    for i in range(warmup + steps):
        t0 = time.perf_counter()
        st = orc.lm_run(sub.chain, prm, tp, tq, s, sub.max_iters, nthreads=nthreads)
        dt = time.perf_counter() - t0
        if i >= warmup:
            times.append(dt)
            executed += st.executed
    total = float(sum(times))
    return {"value": executed / total, "unit": UNIT, "cores": nthreads if nthreads > 0 else orc.num_threads(), "kind": "oracle",
            "sample": f"first {sub.B} of {w.B} trajectories ({sub.W} waypoints, {executed // max(steps, 1)} "
                      f"waypoint-iterations per step), fp64, OpenMP over waypoints",
            "seconds": total, "ms_per_step": 1e3 * total / max(steps, 1), "traj_per_s": sub.B * steps / total}


def run_reference(args) -> None:
    rank, _, world = dist_env()
    if rank != 0:
        return
    from oracle import lm_oracle as orc
    from paper_2309_09102_b200 import workloads as wl
    chain = wl.random_chain_8dof(3) if args.workload == "C3" else wl.panda_chain()
    n_traj = args.ref_traj or 16
    # only the sampled trajectories are generated (the generators are per-trajectory independent
    # in distribution, the sample is a prefix of a smaller batch of the same recipe)
    w = make_workload(args.workload, lambda q: orc.fk(chain, q), n_traj, args.n)
    r = time_oracle(w, n_traj, steps=args.steps, warmup=min(args.warmup, 1))
    full = workload_desc(w)
    full["workload"] += f" [oracle timed on a {n_traj}-trajectory sample of the {args.B or 4096}-trajectory workload]"
    line = {"impl": "reference", "metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": int(args.gpus), "gpus_used": 0,
            "steps": args.steps, "warmup": min(args.warmup, 1), "ms_per_step": r["ms_per_step"],
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": full,
            "cpu_baseline": {k: r[k] for k in ("value", "unit", "cores", "kind", "sample")},
            "e2e": {"value": r["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


# ------------------------------------------------------------------ GPU legs

def run_gpu(args) -> None:
    import torch
    from paper_2309_09102_b200 import build as lm_build, lm

    rank, local_rank, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the batched-LM path has no CPU fallback)")
    if not os.path.exists(lm_build.LIB_PATH):
        lm_build.build()
    torch.cuda.set_device(local_rank)
    device = torch.device("cuda", local_rank)
    if world > 1:
        dist_init("nccl")

    from paper_2309_09102_b200 import workloads as wl
    chain = wl.random_chain_8dof(3) if args.workload == "C3" else wl.panda_chain()
    fk = lm.device_fk(chain, device=str(device))
    w = make_workload(args.workload, fk, args.B, args.n, rank)
    d = int(chain.dof)
    prm = lm.lm_default_params(lambda0=w.lambda0, tol=w.tol)
    stream = torch.cuda.Stream(device=device)
    solver = lm.Solver(chain, w.B, w.n, w.target_pos, w.target_quat, w.seeds, params=prm, device=str(device), stream=stream)
    if args.block:
        solver.set_launch(args.block)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=device)  # > 126 MB L2

    def one_step():
        solver.reset()
        solver.run(w.max_iters)

    with torch.cuda.stream(stream):
        for _ in range(max(args.warmup, 3)):
            flush.zero_()
            one_step()
        stream.synchronize()
        iters_per_step, conv_traj = solver.fetch_totals()

        # ---- device-timed steps: CUDA events on the launching stream, L2 flushed between steps
        sampler = ClockSampler(local_rank).start()
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
        dist_barrier()
        torch.cuda.synchronize(device)
        launches0 = lm.lm_launch_count()
        wall0 = time.perf_counter()
        for a, b in evs:
            flush.zero_()
            a.record(stream)
            one_step()
            b.record(stream)
        torch.cuda.synchronize(device)
        wall = time.perf_counter() - wall0
        launches = lm.lm_launch_count() - launches0
        dist_barrier()
        clocks = sampler.stop()
    step_ms = [a.elapsed_time(b) for a, b in evs]
    total_ms = float(sum(step_ms))
    units = float(iters_per_step) * args.steps
    total_ms_all, units_all = dist_max_sum(total_ms, units, device)
    value = units_all / (total_ms_all * 1e-3)

    # ---- end to end through the C ABI with HOST buffers: lm_init (H2D) + lm_run + lm_fetch (D2H)
    e2e_chunks = max(1, min(16, w.B))
    e2e = measure_e2e(lm, torch, chain, w, prm, device, max(1, min(args.steps, 5)), chunks=e2e_chunks)
    e2e_plain = measure_e2e(lm, torch, chain, w, prm, device, max(1, min(args.steps, 5)), chunks=0)
    e2e_ms_all, e2e_units_all = dist_max_sum(e2e["ms_total"], e2e["units"], device)
    e2e_value = e2e_units_all / (e2e_ms_all * 1e-3)

    if rank != 0:
        return
    peaks = load_peaks()
    ms_kernel = total_ms / args.steps  # the step IS one launch of lm_iterate_kernel
    flop = ALG_FLOP.get(d, 1459.0 * d / 7.0) * iters_per_step
    peak_tf = SM_COUNT * FP32_LANES * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12
    achieved_tf = flop / (ms_kernel * 1e-3) / 1e12
    hbm_bytes = alg_bytes_per_waypoint(d) * w.W
    fma_tf = lm.lm_fp32_peak(int(stream.cuda_stream))
    full_size = (args.B is None and args.n is None)
    roofline = {"bound": "alu", "achieved": achieved_tf, "peak": peak_tf, "unit": "TFLOP/s",
                "frac": achieved_tf / peak_tf,
                "traffic": ncu_constant(f"lm_iterate_{solver.kernel_name}_{args.workload}", "dram_bytes_per_launch", HOT_SOURCES) if full_size else None,
                "kernel": f"lm_iterate_kernel<{d}, {solver.kernel_name}>", "kernel_ms": ms_kernel,
                "peak_measured_fma": fma_tf, "frac_of_measured_fma": achieved_tf / fma_tf if fma_tf > 0 else None,
                "alg_flop_per_waypoint_iteration": ALG_FLOP.get(d),
                "ncu_executed_flop_per_waypoint_iteration": ncu_constant(f"lm_iterate_{solver.kernel_name}_{args.workload}", "executed_flop_per_waypoint_iteration", HOT_SOURCES) if full_size else None,
                "peak_how": f"derived: {SM_COUNT} SMs x {FP32_LANES} FP32 lanes x 2 x {peaks['sm_max_mhz']:.0f} MHz "
                            f"(sm_max_mhz {peaks['_source']})",
                "hbm": {"alg_bytes": hbm_bytes, "achieved_gbs": hbm_bytes / (ms_kernel * 1e-3) / 1e9,
                        "peak_gbs": peaks["hbm_gbs"], "frac": hbm_bytes / (ms_kernel * 1e-3) / 1e9 / peaks["hbm_gbs"],
                        "peak_source": peaks["_source"]}}
    if roofline["ncu_executed_flop_per_waypoint_iteration"]:
        roofline["executed_tflops"] = roofline["ncu_executed_flop_per_waypoint_iteration"] * iters_per_step / (ms_kernel * 1e-3) / 1e12
    ref_traj = min(args.ref_traj or 256, w.B)
    cpu = time_oracle(make_workload(args.workload, fk, ref_traj, w.n), ref_traj)
    cpu1 = time_oracle(make_workload(args.workload, fk, min(16, w.B), w.n), min(16, w.B), nthreads=1)
    cfg = workload_desc(w)
    cfg.update({"parallelism": f"dp{world} (independent batches, no collective)", "l2": "flushed between steps (256 MiB write)",
                "block_threads": args.block or 128, "kernel": solver.kernel_name,
                "targets": "poses of the seeded joint paths / anchors through the library's fp32 lm_fk (the parity tests "
                           "build theirs with the oracle's fp64 FK; bench.py may run the oracle only in its cpu_baseline leg)"})
    extra = {}
    if args.workload == "C4" and full_size:
        # what an unregistered robot gets: the generic (run-time chain structure) kernel on the same workload
        extra["generic_kernel_C4"] = time_kernel_option(lm, torch, w, device, stream, peak_tf, lm.LM_OPT_GENERIC_KERNEL, 1)
        # ... and after lm_specialize: the same kernel template compiled at run time (NVRTC) for the structure of a chain that
        # has no ahead-of-time kernel -- here the Panda with a rotated flange tool on the same inputs
        extra["jit_specialized_C4"] = time_jit(lm, torch, w, device, stream, peak_tf)
        # the lane-group alternative the north star names (2 / 4 lanes per waypoint), measured beside the product kernel
        extra["lane_group_variants"] = {f"{g}_lanes": time_kernel_option(lm, torch, w, device, stream, peak_tf, lm.LM_OPT_LANES_PER_WAYPOINT, g)
                                        for g in (2, 4)}
        extra["lane_group_variants"]["1_lane"] = {"ms_per_step": ms_kernel, "frac_of_derived_peak": achieved_tf / peak_tf}
        # BASELINE.json configs[2]: 2048 x 300, 8-DoF chain with a prismatic joint, to |r| < tol or 50 iterations
        extra["c3_8dof"] = time_c3(lm, torch, wl, device, stream, peak_tf)
        # BASELINE.json configs[4], compact: B x n grid, exactly 20 iterations
        extra["sweep_C5"] = time_sweep_c5(lm, torch, wl, fk, device, stream)
        # the paper's own batch shape: K = 175 plans of one path
        extra["paper_shape_K175_n300"] = time_paper_shape(lm, torch, wl, fk, device, stream)
        # the "to convergence" statistic of the metric, on BASELINE.json configs[1] (512 x 300, tol 1e-5)
        extra["to_convergence_C2"] = time_to_convergence(lm, torch, wl, fk, device, stream)
        extra["variant_dual"] = time_dual_variant(lm, torch, w, device, stream, peak_tf)
        # lm_step: one iteration per launch, the state round-trips through HBM (report both bounds)
        extra["single_step_C4"] = time_single_step(lm, torch, w, solver, stream, peak_tf, peaks)
        # the trajectory-level step on the same workload
        extra["trajectory_step"] = time_traj_step(lm, torch, w, solver, stream, peaks)
        # the paper's alternating schedule with anytime bookkeeping (NEXT-2), valid trajectories per second
        extra["schedule_C2"] = time_plan(lm, torch, wl, fk, device, stream)
        # the global discrete search over K candidates of one path (NEXT-4 iii)
        extra["search_K175_n300"] = time_search(lm, torch, wl, fk, device, stream)
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": total_ms_all / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic", "config": cfg,
            "trajectories_per_sec": w.B * world * args.steps / (total_ms_all * 1e-3),
            "converged_trajectories_per_step": conv_traj,
            "waypoint_iterations_per_step": iters_per_step, "wall_s_timed_region": wall,
            "clocks": clocks, "gpu_launches": int(launches),
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": e2e["h2d"], "d2h_bytes_per_step": e2e["d2h"],
                    "ms_per_step": e2e_ms_all / e2e["steps"],
                    "how": f"lm_pipe_solve(pinned host inputs -> host q, |r|, iters, status; {e2e_chunks} chunks pipelined over the handle's copy-in / kernel / copy-out streams)",
                    "unpipelined_ms_per_step": e2e_plain["ms_total"] / e2e_plain["steps"],
                    "unpipelined_how": "lm_init(LM_MEM_HOST, pinned) + lm_run + lm_fetch"},
            "roofline": roofline,
            "cpu_baseline": {**{k: cpu[k] for k in ("value", "unit", "cores", "kind", "sample")},
                             "single_thread": {k: cpu1[k] for k in ("value", "unit", "cores", "sample")}}}
    line.update(extra)
    print(json.dumps(line))


def traj_step_alg_bytes(d: int, refine: int = 1, fused: bool = True) -> float:
    """HBM bytes one trajectory-level LM iteration must move per waypoint, fp32 words.
    Fused path (the solve kernels' producers assemble in shared memory; J^T J, g, rho never exist in HBM):
      factor + solve   q d + target 7 in, -S^-1 NA + z d + delta d out, -S^-1 NA + z d back in     = 2 NA + 4 d + 7
      each refinement  q d + delta d + target 7 + -S^-1 NA in, z d out, NA + 2 d back in, delta d out = 2 NA + 6 d + 7
      trial cost       q d + delta d + target 7 in, candidate q d + 3 cost terms out               = 3 d + 10
      decision         3 cost terms in.
    Unfused path (small batches, collision rows): + the round trip of w_p^2 J^T J, g (2 (NA + d)) and of rho (2 d); the
    inputs q, delta, target are then read by the per-waypoint kernels instead of the solve kernels."""
    na = d * (d + 1) // 2
    words = (2 * na + 4 * d + 7) + refine * (2 * na + 6 * d + 7) + (3 * d + 10) + 3
    if not fused:
        words += 2 * (na + d) + refine * (2 * d)
    return 4.0 * words


def traj_step_alg_flop(d: int, refine: int = 1) -> dict:
    """Counted FP32 work of ONE trajectory-level LM iteration per waypoint (FMA = 2; DESIGN.md section 10 has the table).
    The per-waypoint pieces are those of the pose step (FK 48 d + 6, residual 77, Jacobian 12 d,
    J^T J + lambda 7 d^2, J^T r 12 d at d = 7: 342 / 77 / 84 / 343 / 84); the block-tridiagonal pieces follow from the
    elimination S_i = D_i - w^4 S_{i-1}^-1 with the off-diagonal block -w_diff^2 I."""
    fk, res, jac, jtj, jtr = 48.0 * d + 6.0, 77.0, 12.0 * d, 7.0 * d * d, 12.0 * d
    matvec = 2.0 * d * d                                     # symmetric d x d block times a vector
    assemble = fk + res + jac + jtj + jtr + 4.0 * d          # + the differencing part of g_i and of the diagonal
    eliminate = d ** 3 + matvec + d * (d + 1)                # Cholesky + inverse of S_i (d^3), z_i update, S update
    substitute = matvec + 2.0 * d                            # x_i = -S_i^-1 (z_i - w^2 x_{i+1})
    rho = fk + res + jac + 12.0 * d + jtr + 6.0 * d          # r + J delta, J^T(...), lambda delta and differencing terms
    resolve = 2.0 * (matvec + 2.0 * d)                       # forward and backward pass on the stored -S^-1
    cost = fk + res + 5.0 * d                                # trial point, its pose and differencing cost
    parts = {"assemble": assemble, "eliminate": eliminate, "substitute": substitute, "refine_rho": refine * rho,
             "refine_resolve": refine * resolve, "trial_cost": cost}
    parts["total"] = float(sum(parts.values()))
    return parts


def traj_step_method_bytes(d: int) -> float:
    """What the METHOD must move per waypoint-iteration whatever the data flow: q (4 d) + target (28) in, q (4 d) out."""
    return 8.0 * d + 28.0


def traj_step_alg_bytes_round1(d: int, refine: int = 1) -> float:
    """The round-1 data flow (every kernel through HBM, candidate normal equations written by the trial kernel): the
    figure VERDICT r1 recomputed the 0.546 from; kept so that the two rounds can be compared on one scale."""
    na = d * (d + 1) // 2
    return 4.0 * ((3 * na + 4 * d) + refine * ((3 * d + 7) + (2 * na + 5 * d)) + (na + 4 * d + 10) + 3)


def time_traj_step(lm, torch, w, solver, stream, peaks, iters: int = 10, reps: int = 5) -> dict:
    """The trajectory-level LM step (lm_traj_run: stacked pose + differencing residual, block-tridiagonal
    solve per trajectory) on the SAME workload, after 4 pose-only iterations; CUDA events around
    lm_traj_run(iters) on the launching stream, best of `reps` after one warm-up.  The CPU leg times the
    oracle of that step (oracle/lm_traj_oracle.c) on a few trajectories."""
    d = int(w.chain.dof)
    tp = lm.lm_traj_default_params(w_pose=1.0, w_diff=0.3)
    solver.traj_attach(tp)
    ts = []
    with torch.cuda.stream(stream):
        for i in range(reps + 1):
            solver.reset()
            solver.run(4)
            solver.traj_reset()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            l0 = lm.lm_launch_count()
            a.record(stream)
            solver.traj_run(iters)
            b.record(stream)
            stream.synchronize()
            launches = lm.lm_launch_count() - l0
            if i >= 1:
                ts.append(a.elapsed_time(b))
        g = solver.traj_fetch()
        # the same iterations with the robot-robot collision rows (NEXT-3; synthetic Panda capsules, 9 pairs)
        coll = None
        if w.chain.name == "panda":
            from paper_2309_09102_b200 import workloads as wl_
            solver.traj_set_capsules(wl_.panda_capsules(), 1.0, 0.05)
            tc = []
            for i in range(reps + 1):
                solver.reset()
                solver.run(4)
                solver.traj_reset()
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(stream)
                solver.traj_run(iters)
                b.record(stream)
                stream.synchronize()
                if i >= 1:
                    tc.append(a.elapsed_time(b))
            gc_ = solver.traj_fetch()
            # ... and with the robot-environment rows as well (synthetic scene: 3 cuboids, 10 capsule-cuboid pairs)
            solver.traj_set_obstacles(wl_.panda_scene(), 1.0, 0.05)
            te = []
            for i in range(reps + 1):
                solver.reset()
                solver.run(4)
                solver.traj_reset()
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(stream)
                solver.traj_run(iters)
                b.record(stream)
                stream.synchronize()
                if i >= 1:
                    te.append(a.elapsed_time(b))
            ge_ = solver.traj_fetch()
            solver.traj_set_capsules(None)
            # the same rows when the 32 trajectories of every tile are candidates for ONE path (the paper's use: K plans
            # of one problem): the lanes of a warp are then near the same obstacles and walk similar pair lists
            corr_ms, corr_active = time_correlated_tiles(lm, torch, w, wl_, stream, iters, reps)
            coll = {"ms_per_iteration": float(min(tc)) / iters, "capsules": 7, "pairs": 9, "w_coll": 1.0, "d_safe_m": 0.05,
                    "trajectories_with_active_pairs": int((gc_["cost_coll"] > 0).sum()),
                    "with_environment_rows": {"ms_per_iteration": float(min(te)) / iters, "cuboids": 3, "pairs": 10,
                                              "trajectories_with_active_pairs": int((ge_["cost_coll"] > 0).sum()),
                                              "tiles_of_32_candidates_per_path": {"ms_per_iteration": corr_ms, "trajectories_with_active_pairs": corr_active}}}
    # the same step without the refinement re-solve (refine_steps = 0: 3 launches per iteration instead of 5).  At this
    # workload's weights the fp32 block elimination alone is within 1e-5 rad of the fp64 oracle (bar 1e-4; the refinement
    # matters when w_diff^2 + lambda is small), so it is an option, not the default.
    solver.traj_attach(lm.lm_traj_default_params(w_pose=1.0, w_diff=0.3, refine_steps=0))
    t0_ = []
    with torch.cuda.stream(stream):
        for i in range(reps + 1):
            solver.reset()
            solver.run(4)
            solver.traj_reset()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            solver.traj_run(iters)
            b.record(stream)
            stream.synchronize()
            if i >= 1:
                t0_.append(a.elapsed_time(b))
    ms0 = float(min(t0_)) / iters
    fused = (w.B + 31) // 32 >= 96  # LM_TL_FUSED_MIN_TILES (csrc/lm_traj.cuh); no collision rows in this leg
    alg0 = traj_step_alg_bytes(d, 0, fused) * w.W
    norefine = {"ms_per_iteration": ms0, "design_bytes_per_waypoint_iteration": traj_step_alg_bytes(d, 0, fused),
                "hbm_design_traffic_frac": alg0 / (ms0 * 1e-3) / 1e9 / peaks["hbm_gbs"],
                "alu_frac": traj_step_alg_flop(d, 0)["total"] * w.W / (ms0 * 1e-3) / 1e12 / peaks["alu_tflops"]}
    ms_iter = float(min(ts)) / iters
    alg = traj_step_alg_bytes(d, int(tp.refine_steps), fused) * w.W
    alg_r1 = traj_step_alg_bytes_round1(d, int(tp.refine_steps)) * w.W
    flop = traj_step_alg_flop(d, int(tp.refine_steps))
    out = {"workload": f"{w.name}: {w.B} x {w.n}, after 4 pose-only iterations; w_pose=1, w_diff=0.3, refine=1, {iters} iterations",
           "ms_per_iteration": ms_iter, "waypoint_iterations_per_sec": w.W / (ms_iter * 1e-3),
           "trajectory_iterations_per_sec": w.B / (ms_iter * 1e-3), "gpu_launches_per_run": int(launches),
           "accepted_fraction": float(np.mean([bin(int(m)).count("1") for m in g["mask"]])) / iters,
           "cost_diff_mean": float(g["cost_diff"].mean()), "with_self_collision_rows": coll,
           "without_refinement": norefine,
           # Three fractions, none of them near 1: the step is bound by issue slots and by the latency of the sequential
           # block elimination (one block of 32 trajectories per SM), DESIGN.md section 10.
           "roofline": {"bound": "alu", "binding_limit": "issue slots / latency of the sequential block elimination, one tile of 32 trajectories per SM",
                        "achieved": flop["total"] * w.W / (ms_iter * 1e-3) / 1e12, "peak": peaks["alu_tflops"], "unit": "TFLOP/s",
                        "frac": flop["total"] * w.W / (ms_iter * 1e-3) / 1e12 / peaks["alu_tflops"],
                        "traffic": ncu_constant("traj_iteration_C4", "dram_bytes_per_iteration", TRAJ_SOURCES) if (w.B, w.n) == (4096, 300) else None,
                        "alg_flop_per_waypoint_iteration": flop,
                        "hbm_method": {"bytes_per_waypoint_iteration": traj_step_method_bytes(d),
                                       "what": "q and target in, q out: the method's own input + output, whatever the data flow",
                                       "achieved_gbs": traj_step_method_bytes(d) * w.W / (ms_iter * 1e-3) / 1e9,
                                       "frac": traj_step_method_bytes(d) * w.W / (ms_iter * 1e-3) / 1e9 / peaks["hbm_gbs"]},
                        "hbm_design_traffic": {"bytes_per_waypoint_iteration": traj_step_alg_bytes(d, int(tp.refine_steps), fused),
                                               "what": "the bytes of THIS design's data flow (the factor -S^-1 and z spilled to HBM and read back); "
                                                       "measured DRAM traffic matches it by construction",
                                               "achieved_gbs": alg / (ms_iter * 1e-3) / 1e9, "peak_gbs": peaks["hbm_gbs"],
                                               "frac": alg / (ms_iter * 1e-3) / 1e9 / peaks["hbm_gbs"],
                                               "frac_on_round1_bytes": alg_r1 / (ms_iter * 1e-3) / 1e9 / peaks["hbm_gbs"],
                                               "round1_bytes_per_waypoint_iteration": traj_step_alg_bytes_round1(d, int(tp.refine_steps))},
                        "path": "fused (producer warps assemble in shared memory)" if fused else "unfused (per-waypoint kernels through HBM)",
                        "peak_source": peaks["_source"]}}
    try:
        from oracle import lm_oracle as orc, lm_traj_oracle as torc
        nb = min(8, w.B)
        sub = w.subset(slice(0, nb))
        q0 = orc.lm_run(sub.chain, orc.Params(lambda0=sub.lambda0, tol=0.0), sub.target_pos.astype(np.float64),
                        sub.target_quat.astype(np.float64), sub.seeds.astype(np.float64), 4).q.reshape(nb, sub.n, d)
        t0 = time.perf_counter()
        st = torc.lm_run(sub.chain, orc.Params(), torc.TrajParams(w_pose=1.0, w_diff=0.3),
                         sub.target_pos.astype(np.float64).reshape(nb, sub.n, 3),
                         sub.target_quat.astype(np.float64).reshape(nb, sub.n, 4), q0, 2)
        dt = time.perf_counter() - t0
        out["cpu_baseline"] = {"value": st.executed * sub.n / dt, "unit": UNIT, "cores": orc.num_threads(), "kind": "oracle",
                               "sample": f"{nb} trajectories x {sub.n} waypoints x 2 iterations, fp64 banded Cholesky, OpenMP over trajectories"}
    except Exception as e:  # noqa: BLE001
        out["cpu_baseline"] = {"error": repr(e)}
    return out


def time_correlated_tiles(lm, torch, w, wl_, stream, iters: int, reps: int):
    """The headline workload with every tile of 32 trajectories replaced by 32 noisy copies (seed noise N(0, 0.02)) of
    its first trajectory, all collision rows on: (ms per trajectory-level iteration, trajectories with active rows)."""
    B, n, d = w.B, w.n, int(w.chain.dof)
    tp = w.target_pos.reshape(B, n, 3).copy()
    tq = w.target_quat.reshape(B, n, 4).copy()
    sd = w.seeds.reshape(B, n, d).copy()
    rng = np.random.default_rng(0)
    for t0 in range(0, B, 32):
        t1 = min(B, t0 + 32)
        tp[t0:t1], tq[t0:t1] = tp[t0], tq[t0]
        sd[t0:t1] = sd[t0] + rng.normal(size=(t1 - t0, n, d)).astype(np.float32) * np.float32(0.02)
    sd = np.clip(sd, w.chain.q_lo.astype(np.float32) + np.float32(1e-4), w.chain.q_hi.astype(np.float32) - np.float32(1e-4))
    s = lm.Solver(w.chain, B, n, tp.reshape(-1, 3), tq.reshape(-1, 4), sd.reshape(-1, d), params=lm.lm_default_params(tol=0.0),
                  device=str(stream.device), stream=stream)
    s.traj_attach(lm.lm_traj_default_params(w_pose=1.0, w_diff=0.3))
    s.traj_set_capsules(wl_.panda_capsules(), 1.0, 0.05)
    s.traj_set_obstacles(wl_.panda_scene(), 1.0, 0.05)
    s.traj_set_cost_lanes(1)  # the caller knows its tiles are candidates of one path: a warp takes one waypoint of 32 trajectories
    ts = []
    with torch.cuda.stream(stream):
        for i in range(reps + 1):
            s.reset()
            s.run(4)
            s.traj_reset()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            s.traj_run(iters)
            b.record(stream)
            stream.synchronize()
            if i >= 1:
                ts.append(a.elapsed_time(b))
        g = s.traj_fetch()
    s.close()
    return float(min(ts)) / iters, int((g["cost_coll"] > 0).sum())


def time_plan(lm, torch, wl, fk, device, stream, cycles: int = 3, reps: int = 5) -> dict:
    """The paper's schedule (lm_plan_run) on configs[1] (512 x 300, Panda): `cycles` x
    [pose-only phase, record, one trajectory-level step] + a final pose phase and record.  Reports valid
    trajectories (0.1 mm / 0.1 deg at every waypoint, no joint step above 7 deg) per second."""
    w = wl.config2(fk)
    prm = lm.lm_default_params(lambda0=w.lambda0, tol=w.tol)
    s = lm.Solver(w.chain, w.B, w.n, w.target_pos, w.target_quat, w.seeds, params=prm, device=str(device), stream=stream)
    s.traj_attach(lm.lm_traj_default_params(w_pose=1.0, w_diff=1.0))
    s.plan_attach(lm.lm_plan_default_params(pose_iters=10))
    out = {}
    with torch.cuda.stream(stream):
        for cyc in (0, cycles):
            ts = []
            for i in range(reps + 1):
                s.set_state(w.seeds)
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                l0 = lm.lm_launch_count()
                a.record(stream)
                s.plan_run(cyc)
                b.record(stream)
                stream.synchronize()
                launches = lm.lm_launch_count() - l0
                if i >= 1:
                    ts.append(a.elapsed_time(b))
            g = s.plan_fetch()
            ms = float(min(ts))
            out[f"cycles_{cyc}"] = {"ms": ms, "gpu_launches": int(launches), "valid_trajectories": g["valid_trajectories"],
                                    "valid_trajectories_per_sec": g["valid_trajectories"] / (ms * 1e-3),
                                    "mean_length_of_valid_rad": float(np.nanmean(g["length"])) if g["valid_trajectories"] else None}
    s.close()
    out["workload"] = f"C2: {w.B} x {w.n}, tol={w.tol:g}, pose_iters=10, w_pose=1, w_diff=1"
    return out


def time_single_step(lm, torch, w, solver, stream, peak_tf: float, peaks: dict, nsteps: int = 20, reps: int = 5) -> dict:
    """lm_step on the headline workload: `nsteps` launches of one LM iteration each (state in / out of HBM every
    launch, FK recomputed at entry), CUDA events around the launches on the launching stream, best of `reps`.
    Per waypoint-iteration: 1459 + one more FK (342) + residual (77) = 1878 FLOP (d = 7; SURVEY 8d counts 1.87 k) and
    4 (2d + 18) bytes (q, lambda, iters|status, 64-bit mask both ways, targets in, |r| / pos / rot error out)."""
    d = int(w.chain.dof)
    flop = ALG_FLOP.get(d, 1459.0 * d / 7.0) + 48.0 * d + 6.0 + 77.0
    nbytes = 4.0 * (2 * d + 18)
    ts = []
    with torch.cuda.stream(stream):
        for i in range(reps + 1):
            solver.reset()
            solver.step()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            for _ in range(nsteps):
                solver.step()
            b.record(stream)
            stream.synchronize()
            if i >= 1:
                ts.append(a.elapsed_time(b) / nsteps)
    ms = float(min(ts))
    W = w.B * w.n
    tf = flop * W / (ms * 1e-3) / 1e12
    gbs = nbytes * W / (ms * 1e-3) / 1e9
    return {"ms_per_lm_step": ms, "waypoint_iterations_per_sec": W / (ms * 1e-3), "alg_flop_per_waypoint_iteration": flop,
            "alg_bytes_per_waypoint_iteration": nbytes, "alu": {"achieved_tflops": tf, "frac_of_derived_peak": tf / peak_tf},
            "hbm": {"achieved_gbs": gbs, "peak_gbs": peaks["hbm_gbs"], "frac": gbs / peaks["hbm_gbs"]},
            "note": "tol = 0 workload: every waypoint executes every step"}


def time_search(lm, torch, wl, fk, device, stream, K: int = 175, n: int = 300, reps: int = 10) -> dict:
    """lm_search on K synthetic candidate trajectories of one n-waypoint path (Panda): median
    CUDA-event time of one call (edge costs + penalties, the layered dynamic program, backtracking, xi gather) after
    3 warm-ups.  The CPU leg runs the oracle (oracle/lm_search_oracle.py, fp32 decisions) once on the same input."""
    import time as _time
    from oracle import lm_search_oracle as sorc
    ch = wl.panda_chain()
    q = wl.search_candidates(ch, K, n, 2, limit_frac=0.02)
    tp = np.zeros((K * n, 3), np.float32)                      # the search reads joint values only
    tq = np.tile(np.array([[1, 0, 0, 0]], np.float32), (K * n, 1))
    s = lm.Solver(ch, K, n, tp, tq, q.reshape(K * n, ch.dof), device=str(device), stream=stream)
    ts = []
    with torch.cuda.stream(stream):
        for i in range(reps + 3):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            l0 = lm.lm_launch_count()
            a.record(stream)
            s.search(to_host=False)
            b.record(stream)
            stream.synchronize()
            launches = lm.lm_launch_count() - l0
            if i >= 3:
                ts.append(a.elapsed_time(b))
        g = s.search()
    s.close()
    pen = sorc.penalties(q, ch.q_lo.astype(np.float32), ch.q_hi.astype(np.float32), ch.joint_type,
                         margin_rev=np.float32(np.deg2rad(1.5)), margin_pris=np.float32(0.03))
    t0 = _time.perf_counter()
    choice, xi, cost, mj = sorc.search(q, pen, dtype=np.float32)
    cpu_s = _time.perf_counter() - t0
    ms = float(np.median(ts))
    return {"workload": f"{K} candidates x {n} waypoints, Panda, synthetic (workloads.search_candidates)", "ms": ms,
            "gpu_launches": int(launches), "edges_per_sec": (n - 1) * K * K / (ms * 1e-3), "mjac_rad": g["mjac"],
            "candidates_used": int(len(set(g["choice"].tolist()))), "same_choice_as_oracle": bool(np.array_equal(g["choice"], choice)),
            "cpu_baseline": {"ms": cpu_s * 1e3, "kind": "oracle", "cores": 1, "sample": "the same input, once"}}


def _time_runs(torch, s, stream, max_iters: int, reps: int, flush=None):
    ts = []
    with torch.cuda.stream(stream):
        for i in range(reps + 3):
            if flush is not None:
                flush.zero_()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            s.reset()
            a.record(stream)
            s.run(max_iters)
            b.record(stream)
            stream.synchronize()
            if i >= 3:
                ts.append(a.elapsed_time(b))
        iters, conv = s.fetch_totals()
    return float(np.median(ts)), iters, conv


def time_kernel_option(lm, torch, w, device, stream, peak_tf: float, option: int, value: int, reps: int = 10) -> dict:
    """lm_reset + lm_run on the headline workload with one lm_set_option knob changed (median CUDA-event time)."""
    d = int(w.chain.dof)
    prm = lm.lm_default_params(lambda0=w.lambda0, tol=w.tol)
    s = lm.Solver(w.chain, w.B, w.n, w.target_pos, w.target_quat, w.seeds, params=prm, device=str(device), stream=stream)
    lm.lm_set_option(s._ctx, option, value)
    ms, iters, _ = _time_runs(torch, s, stream, w.max_iters, reps)
    name = s.kernel_name
    s.close()
    tf = ALG_FLOP.get(d, 1459.0 * d / 7.0) * iters / (ms * 1e-3) / 1e12
    return {"kernel": name, "ms_per_step": ms, "waypoint_iterations_per_sec": iters / (ms * 1e-3), "achieved_tflops": tf,
            "frac_of_derived_peak": tf / peak_tf}


def time_jit(lm, torch, w, device, stream, peak_tf: float, reps: int = 10) -> dict:
    """lm_specialize on a chain whose structure is not registered (Panda + rotated tool; the headline's targets and seeds):
    generic kernel, then the run-time specialised one; compile time of the first call."""
    import copy
    ch = copy.deepcopy(w.chain)
    ch.name = "panda_rotated_tool"
    ch.tool = np.array([0.01, -0.02, 0.107, 0.9238795325112867, 0.2, -0.1, 0.3104])
    ch.tool[3:] /= np.linalg.norm(ch.tool[3:])
    d = int(ch.dof)
    prm = lm.lm_default_params(lambda0=w.lambda0, tol=w.tol)
    s = lm.Solver(ch, w.B, w.n, w.target_pos, w.target_quat, w.seeds, params=prm, device=str(device), stream=stream)
    out = {"chain": "Panda with a rotated flange tool (no ahead-of-time kernel for this structure)"}
    ms, iters, _ = _time_runs(torch, s, stream, w.max_iters, reps)
    out["generic"] = {"kernel": s.kernel_name, "ms_per_step": ms, "frac_of_derived_peak": ALG_FLOP[d] * iters / (ms * 1e-3) / 1e12 / peak_tf}
    t0 = time.perf_counter()
    s.specialize()
    out["compile_s"] = time.perf_counter() - t0
    ms, iters, _ = _time_runs(torch, s, stream, w.max_iters, reps)
    out["specialized"] = {"kernel": s.kernel_name, "ms_per_step": ms, "frac_of_derived_peak": ALG_FLOP[d] * iters / (ms * 1e-3) / 1e12 / peak_tf}
    s.close()
    return out


def time_c3(lm, torch, wl, device, stream, peak_tf: float, reps: int = 10) -> dict:
    """BASELINE.json configs[2] at full size: 2048 x 300, the seeded 8-DoF chain (one prismatic joint), seeds N(0, 0.15),
    |r| < 1e-5 or 50 iterations -- and the same batch for exactly 50 iterations (tol = 0), which is the figure comparable
    with the headline's fraction (1762 FLOP per waypoint-iteration)."""
    ch = wl.random_chain_8dof(3)
    w = wl.config3(lm.device_fk(ch, device=str(device)))
    out = {"workload": f"C3: {w.B} x {w.n}, 8-DoF (1 prismatic), tol={w.tol:g}, max_iters={w.max_iters}"}
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=device)
    for key, tol in (("to_convergence", w.tol), ("fixed_50_iterations", 0.0)):
        prm = lm.lm_default_params(lambda0=w.lambda0, tol=tol)
        s = lm.Solver(ch, w.B, w.n, w.target_pos, w.target_quat, w.seeds, params=prm, device=str(device), stream=stream)
        ms, iters, conv = _time_runs(torch, s, stream, w.max_iters, reps, flush)
        name = s.kernel_name
        s.close()
        tf = ALG_FLOP[8] * iters / (ms * 1e-3) / 1e12
        out[key] = {"kernel": name, "ms_per_step": ms, "waypoint_iterations": iters, "waypoint_iterations_per_sec": iters / (ms * 1e-3),
                    "trajectories_per_sec": w.B / (ms * 1e-3), "converged_trajectories": conv,
                    "alg_flop_per_waypoint_iteration": ALG_FLOP[8], "achieved_tflops": tf, "frac_of_derived_peak": tf / peak_tf}
    return out


def time_sweep_c5(lm, torch, wl, fk, device, stream, reps: int = 5) -> dict:
    """BASELINE.json configs[4], compact: B in {1, 256, 4096, 16384} x n in {100, 300, 1000}, Panda, seeds N(0, 0.1), exactly
    20 iterations; median CUDA-event time of lm_reset + lm_run(20), L2 flushed before every launch."""
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=device)
    out = {"workload": "C5: Panda, smooth paths as configs[1], exactly 20 iterations", "points": []}
    for n in (100, 300, 1000):
        big = wl.config5(fk, B=16384, n=n)
        for B in (1, 256, 4096, 16384):
            w = big.subset(slice(0, B))
            prm = lm.lm_default_params(lambda0=w.lambda0, tol=w.tol)
            s = lm.Solver(w.chain, w.B, w.n, w.target_pos, w.target_quat, w.seeds, params=prm, device=str(device), stream=stream)
            ms, iters, _ = _time_runs(torch, s, stream, w.max_iters, reps, flush)
            s.close()
            out["points"].append({"B": B, "n": n, "ms": ms, "waypoint_iterations_per_sec": iters / (ms * 1e-3)})
    return out


def time_paper_shape(lm, torch, wl, fk, device, stream, reps: int = 7) -> dict:
    """The paper's own batch: K = 175 candidate plans x n = 300 poses of ONE target path (shared_targets),
    52 500 waypoints = 11 warps per SM, one wave -- the latency-bound regime.  Candidates = the
    path's joint-space truth + N(0, 0.1) per joint (as configs[4]).  Exactly 20 iterations with every block size / lane
    group the library offers, and to convergence (tol 1e-5) with the defaults; L2 flushed before every launch."""
    K, n = 175, 300
    w1 = wl.config5(fk, B=1, n=n)
    ch, d = w1.chain, int(w1.chain.dof)
    rng = np.random.default_rng(175)
    seeds = np.clip(w1.truth.reshape(1, n, d) + 0.1 * rng.normal(size=(K, n, d)), ch.q_lo, ch.q_hi).astype(np.float32).reshape(K * n, d)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=device)
    out = {"workload": f"{K} candidates x {n} waypoints of one path (shared targets), Panda", "exactly_20_iterations": []}
    for lanes in (1, 2, 4):
        for block in (32, 64, 128):
            s = lm.Solver(ch, K, n, w1.target_pos, w1.target_quat, seeds, params=lm.lm_default_params(lambda0=w1.lambda0, tol=0.0),
                          shared_targets=True, device=str(device), stream=stream)
            s.set_launch(block)
            try:
                if lanes > 1:
                    s.set_lanes_per_waypoint(lanes)
                ms, iters, _ = _time_runs(torch, s, stream, 20, reps, flush)
            except lm.LmError as e:
                out["exactly_20_iterations"].append({"lanes_per_waypoint": lanes, "block_threads": block, "error": str(e)})
                s.close()
                continue
            s.close()
            out["exactly_20_iterations"].append({"lanes_per_waypoint": lanes, "block_threads": block, "ms": ms, "us_per_iteration": 1e3 * ms / 20,
                                                 "waypoint_iterations_per_sec": iters / (ms * 1e-3)})
    s = lm.Solver(ch, K, n, w1.target_pos, w1.target_quat, seeds, params=lm.lm_default_params(lambda0=w1.lambda0, tol=1e-5),
                  shared_targets=True, device=str(device), stream=stream)
    ms, iters, conv = _time_runs(torch, s, stream, 50, reps, flush)
    s.close()
    out["to_convergence"] = {"tol": 1e-5, "ms": ms, "waypoint_iterations": int(iters), "converged_trajectories": int(conv),
                             "waypoint_iterations_per_sec": iters / (ms * 1e-3)}
    return out


def time_dual_variant(lm, torch, w, device, stream, peak_tf: float, reps: int = 10) -> dict:
    """The disclosed variant LM_SOLVER_DUAL (same LM step through the 6 x 6 system) on the same workload:
    median CUDA-event time of lm_reset + lm_run after 3 warm-ups."""
    d = int(w.chain.dof)
    prm = lm.lm_default_params(lambda0=w.lambda0, tol=w.tol, solver=lm.LM_SOLVER_DUAL)
    s = lm.Solver(w.chain, w.B, w.n, w.target_pos, w.target_quat, w.seeds, params=prm, device=str(device), stream=stream)
    ts = []
    with torch.cuda.stream(stream):
        for i in range(reps + 3):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            s.reset()
            a.record(stream)
            s.run(w.max_iters)
            b.record(stream)
            stream.synchronize()
            if i >= 3:
                ts.append(a.elapsed_time(b))
        iters, _ = s.fetch_totals()
    s.close()
    ms = float(np.median(ts))
    tf = ALG_FLOP_DUAL.get(d, 1055.0) * iters / (ms * 1e-3) / 1e12
    return {"solver": "LM_SOLVER_DUAL: delta = -J^T (J J^T + lambda I_6)^-1 r, no refinement", "ms_per_step": ms,
            "waypoint_iterations_per_sec": iters / (ms * 1e-3), "alg_flop_per_waypoint_iteration": ALG_FLOP_DUAL.get(d),
            "achieved_tflops": tf, "frac_of_derived_peak": tf / peak_tf}


def time_to_convergence(lm, torch, wl, fk, device, stream, reps: int = 20) -> dict:
    """Trajectories/s to convergence on configs[1] (512 x 300, Panda, |r| < 1e-5 or 50 iterations):
    median CUDA-event time of lm_reset + lm_run over `reps` launches after 3 warm-ups."""
    w = wl.config2(fk)
    prm = lm.lm_default_params(lambda0=w.lambda0, tol=w.tol)
    s = lm.Solver(w.chain, w.B, w.n, w.target_pos, w.target_quat, w.seeds, params=prm, device=str(device), stream=stream)
    ts = []
    with torch.cuda.stream(stream):
        for i in range(reps + 3):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            s.reset()
            a.record(stream)
            s.run(w.max_iters)
            b.record(stream)
            stream.synchronize()
            if i >= 3:
                ts.append(a.elapsed_time(b))
        iters, conv = s.fetch_totals()
    s.close()
    ms = float(np.median(ts))
    return {"workload": f"C2: {w.B} x {w.n}, tol={w.tol:g}, max_iters={w.max_iters}", "ms": ms,
            "trajectories_per_sec": w.B / (ms * 1e-3), "converged_trajectories": conv,
            "waypoint_iterations": iters, "waypoint_iterations_per_sec": iters / (ms * 1e-3),
            "mean_iterations_per_waypoint": iters / w.W}


def measure_e2e(lm, torch, chain, w, prm, device, steps: int, chunks: int = 0) -> dict:
    """The call a user with host data makes: pinned host inputs -> lm_init (H2D copies inside) ->
    lm_run -> lm_fetch into pinned host outputs (D2H inside), all inside the timed region."""
    d, W = int(chain.dof), w.W
    stream = torch.cuda.Stream(device=device)
    soa = lambda x: torch.from_numpy(np.ascontiguousarray(np.asarray(x, np.float32).T)).pin_memory()
    tp, tq, seeds = soa(w.target_pos), soa(w.target_quat), soa(w.seeds)
    nbytes = lm.lm_workspace_bytes(d, w.B, w.n, 0, lm.LM_MEM_HOST)
    ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=device)
    ws_ptr = (ws.data_ptr() + 255) // 256 * 256
    cchain, keep = lm.make_chain(chain)
    q_out = torch.empty((d, W), dtype=torch.float32).pin_memory()
    res = torch.empty(W, dtype=torch.float32).pin_memory()
    its = torch.empty(W, dtype=torch.int32).pin_memory()
    sts = torch.empty(W, dtype=torch.int32).pin_memory()
    h2d = 4 * W * (d + 3 + 4)
    d2h = 4 * W * (d + 3)
    times, units = [], 0

    msk = None
    pipe = None
    if chunks > 0:
        pipe = lm.lm_pipe_create(chunks)  # the handle (streams, events, pinned totals) outlives the calls, as in a serving loop
        nbytes = lm.lm_solve_host_workspace_bytes(d, w.B, w.n, chunks)
        ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=device)
        ws_ptr = (ws.data_ptr() + 255) // 256 * 256

    def once():
        pb = lm.LmProblem(w.B, w.n, tp.data_ptr(), tq.data_ptr(), 0, seeds.data_ptr(), lm.LM_MEM_HOST, ws_ptr, nbytes)
        st = lm.LmStats(res.data_ptr(), None, None, None, its.data_ptr(), None, sts.data_ptr(), None, None, 0, 0)
        if chunks > 0:  # one call: chunked, H2D / kernel / D2H pipelined over the library's streams
            lm.lm_pipe_solve(pipe, cchain, pb, prm, w.max_iters, chunks, q_out.data_ptr(), st, int(stream.cuda_stream))
            return int(st.total_waypoint_iters)
        ctx = lm.lm_init(cchain, pb, prm, int(stream.cuda_stream))
        lm.lm_run(ctx, w.max_iters)
        lm.lm_fetch(ctx, q_out.data_ptr(), st)  # synchronises the stream
        lm.lm_free(ctx)
        return int(st.total_waypoint_iters)

    once()
    once()
    dist_barrier()
    torch.cuda.synchronize(device)
    for _ in range(steps):
        t0 = time.perf_counter()
        units += once()
        times.append(time.perf_counter() - t0)
    dist_barrier()
    if pipe is not None:
        lm.lm_pipe_destroy(pipe)
    return {"ms_total": 1e3 * float(sum(times)), "units": float(units), "steps": steps, "h2d": h2d, "d2h": d2h}


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--workload", default="C4", choices=["C4", "C2", "C3", "C5"])
    ap.add_argument("--B", type=int, default=None, help="trajectories (default: the config's)")
    ap.add_argument("--n", type=int, default=None, help="waypoints per trajectory")
    ap.add_argument("--block", type=int, default=0, help="threads per block override")
    ap.add_argument("--ref-traj", type=int, default=0,
                    help="trajectories in the oracle's timed sample (default 256 for cpu_baseline, 16 per step for --impl reference)")
    ap.add_argument("--dist-selftest", action="store_true",
                    help="no GPU work: start the ranks, run the two cross-rank reductions of the bench over gloo and print their line")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
        return
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # `python bench.py --gpus N` without a launcher: start the N ranks ourselves (the torchrun path stays as it is)
        if not args.dist_selftest:
            import torch
            have = torch.cuda.device_count()
            if have < args.gpus:
                sys.exit(f"bench.py: {args.gpus} GPUs requested, {have} visible")
        sys.exit(spawn_ranks(args.gpus, sys.argv[1:]))
    if args.dist_selftest:
        run_dist_selftest(args)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()
