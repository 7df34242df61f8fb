#!/usr/bin/env python
"""bench.py — LSQR iterations/s of the hot path on synthetic paper-shaped systems (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference]

A *step* is one complete damped LSQR solve of the workload through the C ABI (libtomolsqr.so): the
init pass and every iteration (A v, A^T u, norms, scalar step, x/w update, stopping tests) of
BASELINE.json configs[C] with the solve parameters that config states (default C = 1: the paper-scale
array, atol = btol = 1e-6, at most 300 iterations).  `value` = iterations performed / device time with
the matrix, b and x resident in HBM; `e2e` = the same through tomo_lsqr_solve_host with pinned HOST
b and x (H2D of b and D2H of x inside the timed region).  The one-off create (validation + CSR->CSC
transpose) is reported separately (`create_ms`), as the metric is per iteration.

N > 1 (torchrun, one rank per GPU): the path has no exchange step on one GPU's problem, so ranks run
independent replicas of the workload; value = iterations of all
ranks / max-over-ranks device time, scaling "weak".

`--impl reference` times the CPU oracle (oracle/, plain fp64 mode, 1 core) on a bounded sample of the
same workload: the tier's reference arm.
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

METRIC = "lsqr_iterations_per_second"
UNIT = "iterations/s"


def algorithmic_bytes(m: int, n: int, nnz: int, vbytes: int = 8) -> dict:
    """Bytes the method must move per launch: matrix streams
    nnz*(vbytes+4) + pointers, the gathered vector once, the updated vector read + written."""
    k1 = (vbytes + 4) * nnz + 8 * (m + 1) + 8 * (2 * m + n)
    k2 = (vbytes + 4) * nnz + 8 * (n + 1) + 8 * (2 * n + m)
    k4 = 8 * 5 * n
    return dict(k1=k1, k2=k2, k4=k4, iteration=k1 + k2 + k4)


def measured_peak_gbs() -> tuple[float, str]:
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def ncu_traffic_bytes(config: int):
    """dram bytes per launch of the dominant kernel from the committed ncu --set full summary, or None."""
    p = os.path.join(ROOT, "profiles", "dram_traffic.csv")
    if not os.path.exists(p):
        return None
    try:
        for line in open(p):
            f = [t.strip() for t in line.split(",")]
            if len(f) >= 3 and f[0] == f"cfg{config}" and f[1] == "k_stream_mean_bytes_per_launch":
                return float(f[2])
    except Exception:
        return None
    return None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.lines, self.proc = index, [], None

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100",
                                          "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=lambda: [self.lines.append(l) for l in self.proc.stdout], daemon=True)
            self.t.start()
        except Exception:
            self.proc = None
        return self

    def __exit__(self, *a):
        if self.proc:
            time.sleep(0.15)
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except Exception:
                self.proc.kill()

    def summary(self) -> dict:
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for l in self.lines:
            f = [t.strip() for t in l.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for name, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unavailable"], "samples": 0}
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": max(mx), "reasons": sorted(reasons), "samples": len(sm)}


def load_system(config: int):
    import tomogen
    s = tomogen.System(config)
    rp, ci, va = s.csr()
    return s, rp, ci, va


def workload_name(s) -> str:
    d = s.dims
    return (f"configs[{s.config}]: {d.nx}x{d.ny}x{d.nz} grid, {d.m}x{d.n}, nnz {d.nnz}, damp {s.damp}, "
            f"atol=btol={s.solve['atol']:g}, max_iters {s.solve['max_iters']}")


def ref_iters_for(args) -> int:
    """Oracle iterations per timed sample: about 10-30 s of CPU work (config 2 is 19 x config 1)."""
    return args.ref_iters if args.config != 2 else max(1, args.ref_iters // 10)


def aggregate_over_ranks(dist, ms: float, its: int, launches: float, device: str = "cuda"):
    """Whole-job figures of N independent replicas: max over ranks of the device time, sums of the
    iterations and launches (the only communication of the N > 1 path; gloo on CPU in the tests)."""
    import torch
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    c = torch.tensor([float(its), launches], dtype=torch.float64, device=device)
    dist.all_reduce(c, op=dist.ReduceOp.SUM)
    return float(t[0]), int(c[0]), float(c[1])


# ---------------------------------------------------------------------------------------------------
def run_reference(args) -> dict:
    """The reference arm of this tier: the CPU oracle as it stands (plain fp64, single thread), each
    step a bounded sample (args.ref_iters iterations) of the same workload."""
    import oracle
    s, rp, ci, va = load_system(args.config)
    b = s.rhs(0)
    m, n = s.dims.m, s.dims.n
    iters = ref_iters_for(args)
    times = []
    for i in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        r = oracle.lsqr(m, n, rp, ci, va, b, damp=s.damp, atol=0.0, btol=0.0, max_iters=iters, mode=oracle.PLAIN)
        dt = time.perf_counter() - t0
        if i >= args.warmup:
            times.append(dt)
        assert r.itn == iters
    total = sum(times)
    value = iters * args.steps / total
    sample = f"{iters} iterations (plus the init pass) of the full configs[{args.config}] system per step"
    return {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(s), "l2": "per-iteration working set 4.7 GB >> L2"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }


def run_ours(args) -> dict | None:
    import numpy as np
    import torch
    import paper_2604_11920_b200 as tl
    tl.load()  # raises if libtomolsqr.so is missing: there is no fallback

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the hot path has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    import tomogen
    s = tomogen.System(args.config)
    m, n, nnz = s.dims.m, s.dims.n, s.dims.nnz
    damp, atol, btol, max_iters = s.damp, s.solve["atol"], s.solve["btol"], s.solve["max_iters"]
    b_host = torch.from_numpy(s.rhs(0)).pin_memory()
    x_host = torch.empty(n, dtype=torch.float64).pin_memory()
    rp_d, ci_d, va_d = s.csr_cuda()  # generated and uploaded block by block (config 2: 45 GB)
    vbytes = 8
    if args.vals == "f32":  # optional fp32 storage of the values (arithmetic stays fp64)
        va_d, vbytes = va_d.to(torch.float32), 4
    S = tl.TomoLsqr(m, n, rp_d, ci_d, va_d)
    S.set(accumulate=args.accumulate, check_every=args.check_every, graph=1, profile=0)
    if args.row_cost is not None:
        S.set(row_cost=args.row_cost)
    b = b_host.cuda()
    x = torch.empty(n, dtype=torch.float64, device="cuda")

    nrhs = s.dims.nrhs

    class _Its:  # a step's iteration count (all right-hand sides)
        def __init__(self, itn):
            self.itn = itn

    if nrhs > 1:  # configs[3]: the 8 right-hand sides (DESIGN.md a8: eight recurrences sharing every pass over A and A^T)
        B_host = torch.from_numpy(s.rhs_block()).pin_memory()
        X_host = torch.empty((n, nrhs), dtype=torch.float64).pin_memory()
        B = B_host.cuda()
        X = torch.empty((n, nrhs), dtype=torch.float64, device="cuda")

    def step_device():
        if nrhs > 1:
            return _Its(sum(r.itn for r in tl.tomo_lsqr_solve_multi(S.h, nrhs, B, damp, atol, btol, max_iters, X)))
        if args.solver == "lsmr":
            return tl.tomo_lsmr_solve(S.h, b, damp, atol, btol, max_iters, x)
        return tl.tomo_lsqr_solve(S.h, b, damp, atol, btol, max_iters, x)

    def step_host():
        if args.solver == "lsmr":  # no host-buffer entry for LSMR: copies around the device call
            b.copy_(b_host, non_blocking=True)
            r = tl.tomo_lsmr_solve(S.h, b, damp, atol, btol, max_iters, x)
            x_host.copy_(x)
            return r
        if nrhs > 1:  # no host-buffer entry for the block solve: copies around the device call
            B.copy_(B_host, non_blocking=True)
            r = _Its(sum(r.itn for r in tl.tomo_lsqr_solve_multi(S.h, nrhs, B, damp, atol, btol, max_iters, X)))
            X_host.copy_(X)
            return r
        return tl.tomo_lsqr_solve_host(S.h, b_host, damp, atol, btol, max_iters, x_host)

    def timed(step):
        for _ in range(args.warmup):
            step()
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        k0 = S.info("kernels_enqueued")
        e0.record()
        its = 0
        for _ in range(args.steps):
            its += step().itn
        e1.record()
        barrier()
        ms = e0.elapsed_time(e1)
        launches = S.info("kernels_enqueued") - k0
        if dist is not None:
            ms, its, launches = aggregate_over_ranks(dist, ms, its, launches, device="cuda")
        return ms, its, launches

    with ClockSampler(local) as clk:
        ms, its, launches = timed(step_device)
    clocks = clk.summary()
    ms_e2e, its_e2e, _ = timed(step_host)

    # per-kernel durations, live: the same solve launched kernel by kernel with CUDA events around each
    # launch on the launching stream (library option "profile")
    S.set(profile=1)
    for _ in range(2):
        if nrhs > 1:  # the block solve has no per-kernel read-out: time the single-side kernels on column 0
            tl.tomo_lsqr_solve(S.h, B[:, 0].contiguous(), damp, atol, btol, max_iters, x)
        else:
            step_device()
    nl = S.info("k_launches")
    k1_us, k2_us, k4_us = (1e3 * S.info(k) / nl for k in ("k1_ms", "k2_ms", "k4_ms"))
    S.set(profile=0)
    # fast-mode (plain fp64 FMA) numbers for context
    other = {}
    if args.both_modes:
        S.set(accumulate=1 - args.accumulate)
        ms_o, its_o, _ = timed(step_device)
        other = {"accumulate": 1 - args.accumulate, "value": its_o / (ms_o * 1e-3), "ms_per_step": ms_o / args.steps}
        S.set(accumulate=args.accumulate)

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return None

    ab = algorithmic_bytes(m, n, nnz, vbytes)
    peak, peak_src = measured_peak_gbs()
    spmv_bytes = ab["k1"] + ab["k2"]
    achieved = spmv_bytes / ((k1_us + k2_us) * 1e-6) / 1e9
    if nrhs > 1:  # shared pass: the matrix stream once per block iteration, the vector traffic nrhs times
        block_bytes = 2 * (vbytes + 4) * nnz + 8 * (m + n + 2) + nrhs * 8 * (3 * m + 3 * n + 5 * n)
        achieved = block_bytes * (its / nrhs / world) / (ms * 1e-3) / 1e9
    traffic = ncu_traffic_bytes(args.config)
    out = {
        "metric": METRIC, "value": its / (ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": workload_name(s), "iterations_per_step": its // max(1, args.steps * world),
                   "accumulate": "dd (double-double sums, rounded once)" if args.accumulate else "fast (fp64 FMA sums)",
                   "check_every": args.check_every, "solver": args.solver, "right_hand_sides": nrhs, "values": "fp64" if vbytes == 8 else "fp32 storage, fp64 arithmetic", "parallelism": "replicas" if world > 1 else "single GPU",
                   "l2": f"inputs larger than L2: {ab['iteration'] / 1e9:.2f} GB streamed per iteration vs 126 MB L2, no flush needed"},
        "effective_gbs": ab["iteration"] * its / world / (ms * 1e-3) / 1e9,
        "create_ms": S.info("create_ms"), "transpose_ms": S.info("transpose_ms"),
        "e2e": {"value": its_e2e / (ms_e2e * 1e-3), "unit": UNIT, "h2d_bytes_per_step": 8 * m * nrhs, "d2h_bytes_per_step": 8 * n * nrhs,
                "ms_per_step": ms_e2e / args.steps},
        "gpu_launches": int(launches),
        "clocks": clocks,
        "roofline": {"bound": "hbm", "kernel": "k_stream (K1: A v - alpha u + norm over CSR; K2: A^T u - beta v + norm over CSC), mean of the two launches of an iteration",
                     "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": traffic,
                     "algorithmic_bytes_per_launch": spmv_bytes / 2,
                     "peak_source": peak_src, "frac_of_8TBs": achieved / 8000.0,
                     "bytes_per_launch_pair": spmv_bytes, "k1_us": k1_us, "k2_us": k2_us, "k4_us": k4_us,
                     "k1_gbs": ab["k1"] / (k1_us * 1e-6) / 1e9, "k2_gbs": ab["k2"] / (k2_us * 1e-6) / 1e9},
    }
    if other:
        out["other_mode"] = other
    if world == 1 and not args.no_cpu:
        import oracle
        iters = ref_iters_for(args)
        rp, ci, va = s.csr()
        t0 = time.perf_counter()
        r = oracle.lsqr(m, n, rp, ci, va, s.rhs(0), damp=damp, atol=0.0, btol=0.0, max_iters=iters, mode=oracle.PLAIN)
        dt = time.perf_counter() - t0
        out["cpu_baseline"] = {"value": r.itn / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
                               "sample": f"{iters} iterations (plus the init pass) of the full configs[{args.config}] system, plain fp64 mode"}
    if dist is not None:
        dist.destroy_process_group()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=1)
    ap.add_argument("--accumulate", type=int, default=1, choices=[0, 1])
    ap.add_argument("--check-every", dest="check_every", type=int, default=10)
    ap.add_argument("--ref-iters", dest="ref_iters", type=int, default=20)
    ap.add_argument("--both-modes", dest="both_modes", action="store_true", default=True)
    ap.add_argument("--no-cpu", dest="no_cpu", action="store_true")
    ap.add_argument("--solver", default="lsqr", choices=["lsqr", "lsmr"], help="lsqr (BASELINE metric) or lsmr (the paper's solver)")
    ap.add_argument("--vals", default="f64", choices=["f64", "f32"], help="storage type of the matrix values")
    ap.add_argument("--row-cost", dest="row_cost", type=int, default=None, help="tuning: per-row weight of the element split")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        if int(os.environ.get("RANK", "0")) != 0:
            return
        print(json.dumps(run_reference(args)), flush=True)
        return
    out = run_ours(args)
    if out is not None:
        print(json.dumps(out), flush=True)


if __name__ == "__main__":
    main()
