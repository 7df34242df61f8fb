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


def ncu_traffic_bytes(config: int, nrhs: int = 1):
    """(dram bytes per launch of the dominant kernel, where the number comes from) read from the committed ncu
    --set full summary profiles/dram_traffic.csv: a figure captured ONCE per kernel generation under ncu, not in
    this run (a number taken under a profiler is never a bench value).  (None, reason) if there is no entry."""
    p = os.path.join(ROOT, "profiles", "dram_traffic.csv")
    key = "k_wstream_mean_bytes_per_launch" if nrhs == 1 else "k_spmm8_mean_bytes_per_launch"
    if not os.path.exists(p):
        return None, "profiles/dram_traffic.csv missing"
    try:
        src = ""
        for line in open(p):
            if line.startswith("#"):
                src = line.lstrip("# ").strip()
                continue
            f = [t.strip() for t in line.split(",")]
            if len(f) >= 3 and f[0] == f"cfg{config}" and f[1] == key:
                return float(f[2]), f"profiles/dram_traffic.csv ({src})"
    except Exception as e:  # noqa: BLE001
        return None, f"unreadable: {e}"
    return None, f"no {key} entry for cfg{config} in profiles/dram_traffic.csv"


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


def workload_config(s, args, iterations_per_step: int, world: int = 1) -> dict:
    """The `config` object of a bench line: names the workload and how the GPU arm is run on it.  Both arms print the
    SAME object for the same arguments (the reference arm times a bounded sample of this workload; its `cpu_baseline.sample`
    says which)."""
    m, n, nnz, nrhs = s.dims.m, s.dims.n, s.dims.nnz, s.dims.nrhs
    vbytes = 4 if args.vals == "f32" else 8
    ab = algorithmic_bytes(m, n, nnz, vbytes) if nrhs == 1 else block_bytes(m, n, nnz, nrhs, vbytes)
    return {"workload": workload_name(s), "iterations_per_step": iterations_per_step,
            "accumulate": ("dd (double-double sums, rounded once)" if args.accumulate else "fast (fp64 FMA sums)") +
                          (("; factored operator with exact entries W*g, depth contraction first (two_stage=2)" if args.accumulate else
                            "; depth contraction first (two_stage)") if getattr(args, "factored", 0) and
                           (getattr(args, "nodal", 0) or getattr(args, "two_stage", 1) == 2 or
                            (not args.accumulate and getattr(args, "two_stage", 1) >= 1)) else "") +
                          ("; kernel table per lateral node" if getattr(args, "factored", 0) and getattr(args, "nodal", 0) else ""),
            "check_every": args.check_every, "solver": args.solver, "right_hand_sides": nrhs,
            "values": "fp64" if vbytes == 8 else "fp32 storage, fp64 arithmetic",
            "index": ("none: factored operator (lateral footprint x depth kernel, tomo_lsqr_create_factored)" if getattr(args, "factored", 0)
                      else "run-compressed (compress=1)" if args.compress else "int32 per nonzero"),
            "parallelism": "replicas" if world > 1 else "single GPU",
            "l2": ("factored operator: tens of MB per product, L2-resident after the first pass; bound by fp64 arithmetic, no HBM stream to flush"
                   if getattr(args, "factored", 0) else
                   f"inputs larger than L2: {ab['iteration'] / 1e9:.2f} GB streamed per iteration vs 126 MB L2, no flush needed"
                   if ab["iteration"] > 2 * 126e6 else
                   f"working set {ab['iteration'] / 1e6:.1f} MB per iteration fits in L2: launch-latency-bound workload, no roofline claim")}


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
    sample = (f"{iters} iterations (plus the init pass) of the full configs[{args.config}] system per step, oracle in plain fp64 mode, "
              f"first right-hand side; the GPU arm runs the whole workload named in config")
    return {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(s, args, int(s.solve["max_iters"]) * int(s.dims.nrhs), max(1, args.gpus)),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }


def block_bytes(m: int, n: int, nnz: int, nrhs: int, vbytes: int = 8) -> dict:
    """Algorithmic bytes of one BLOCK iteration of the shared-pass multi-RHS solve (the matrix
    streams once for all sides, the vector traffic nrhs times): 24 nnz + 8 (32 m + 72 n) at nrhs = 8, fp64."""
    k1 = (vbytes + 4) * nnz + 8 * (m + 1) + nrhs * 8 * (2 * m + n)
    k2 = (vbytes + 4) * nnz + 8 * (n + 1) + nrhs * 8 * (2 * n + m)
    return dict(k1=k1, k2=k2, k4=nrhs * 40 * n, iteration=k1 + k2 + nrhs * 40 * n)


def measure(tl, torch, s, args, barrier, dist, world, steps, warmup, e2e=True, both_modes=True):
    """Times args.config-style steps on system `s` (already chosen); returns the raw numbers of one workload."""
    m, n, nnz = s.dims.m, s.dims.n, s.dims.nnz
    damp, atol, btol, max_iters = s.damp, s.solve["atol"], s.solve["btol"], s.solve["max_iters"]
    nrhs = s.dims.nrhs
    b_host = torch.from_numpy(s.rhs(0)).pin_memory()
    x_host = torch.empty(n, dtype=torch.float64).pin_memory()
    vbytes = 8
    factored = bool(getattr(args, "factored", 0))
    if factored:  # NEXT-2, factored form: lateral footprints + depth kernels + the smoothing block; nothing per nonzero
        f = s.factored()
        ft = {k: torch.from_numpy(v).cuda() for k, v in f.items() if hasattr(v, "dtype")}
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        S = tl.TomoLsqr.factored(f["npairs"], f["nper"], f["nnodes"], f["nz"], ft["lptr"], ft["lnode"], ft["lw"], ft["kj0"], ft["kern"],
                                 ft["sptr"], ft["sidx"], ft["svals"])
    else:
        rp_d, ci_d, va_d = s.csr_cuda()  # generated and uploaded block by block (config 2: 45 GB)
        if args.vals == "f32":  # optional fp32 storage of the values (arithmetic stays fp64)
            va_d, vbytes = va_d.to(torch.float32), 4
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        S = tl.TomoLsqr(m, n, rp_d, ci_d, va_d)
    torch.cuda.synchronize()
    create_wall_ms = 1e3 * (time.perf_counter() - t0)
    S.set(accumulate=args.accumulate, check_every=args.check_every, graph=1, profile=0, compress=0 if factored else args.compress)
    if factored:
        S.set(two_stage=getattr(args, "two_stage", 1))
        if getattr(args, "nodal", 0):
            # a kernel table per lateral node (the paper's Theta_k): here the shared table repeated for every node, so the
            # operator is the same and only the kernel path changes (the depth-contraction kernels in both modes)
            kj0n = ft["kj0"].repeat(f["nnodes"], 1).contiguous()
            kernn = ft["kern"].unsqueeze(0).repeat(f["nnodes"], 1, 1).contiguous()
            tl.tomo_lsqr_set_nodal_kernels(S.h, kj0n, kernn)
    if args.row_cost is not None:
        S.set(row_cost=args.row_cost)
    if args.pdl is not None:
        S.set(pdl=args.pdl)
    b = b_host.cuda()
    x = torch.empty(n, dtype=torch.float64, device="cuda")
    lsmr = args.solver == "lsmr"

    class _Its:  # a step's iteration count (all right-hand sides)
        def __init__(self, itn):
            self.itn = itn

    if nrhs > 1:  # configs[3]: 8 recurrences sharing every pass over A and A^T (DESIGN.md a8)
        B_host = torch.from_numpy(s.rhs_block()).pin_memory()
        X_host = torch.empty((n, nrhs), dtype=torch.float64).pin_memory()
        B = B_host.cuda()
        X = torch.empty((n, nrhs), dtype=torch.float64, device="cuda")
        multi = tl.tomo_lsmr_solve_multi if lsmr else tl.tomo_lsqr_solve_multi

    def step_device():
        if nrhs > 1:
            return _Its(sum(r.itn for r in multi(S.h, nrhs, B, damp, atol, btol, max_iters, X)))
        return (tl.tomo_lsmr_solve if lsmr else tl.tomo_lsqr_solve)(S.h, b, damp, atol, btol, max_iters, x)

    def step_host():
        if nrhs > 1:  # the block solve has no host-buffer entry: pinned copies around the device call, inside the timed region
            B.copy_(B_host, non_blocking=True)
            r = _Its(sum(r.itn for r in multi(S.h, nrhs, B, damp, atol, btol, max_iters, X)))
            X_host.copy_(X)
            return r
        return (tl.tomo_lsmr_solve_host if lsmr else tl.tomo_lsqr_solve_host)(S.h, b_host, damp, atol, btol, max_iters, x_host)

    def timed(step):
        for _ in range(warmup):
            step()
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        k0 = S.info("kernels_enqueued")
        e0.record()
        its = 0
        for _ in range(steps):
            its += step().itn
        e1.record()
        barrier()
        ms = e0.elapsed_time(e1)
        launches = S.info("kernels_enqueued") - k0
        if dist is not None:
            ms, its, launches = aggregate_over_ranks(dist, ms, its, launches, device="cuda")
        return ms, its, launches

    out = {"m": m, "n": n, "nnz": nnz, "nrhs": nrhs, "vbytes": vbytes, "create_wall_ms": create_wall_ms, "accumulate": args.accumulate,
           "create_ms": S.info("create_ms"), "transpose_ms": S.info("transpose_ms")}
    if factored:
        out["two_stage"] = getattr(args, "two_stage", 1)
        out["nodal"] = getattr(args, "nodal", 0)
        out["factored"] = {"lateral_entries": S.info("lateral_entries"), "operator_bytes": S.info("operator_bytes"),
                           "cut_nodes_pieces": S.info("cut_nodes_pieces")}
        if torch.cuda.mem_get_info()[0] > 14 * nnz + (2 << 30):
            # NEXT-4: on-device assembly of the CSR form from the same factored description (tomo_lsqr_assemble_csr): one
            # HBM-bound pass writing 12 bytes per nonzero + the row pointers
            rp_o = torch.empty(m + 1, dtype=torch.int64, device="cuda")
            ci_o = torch.empty(nnz, dtype=torch.int32, device="cuda")
            va_o = torch.empty(nnz, dtype=torch.float64, device="cuda")
            snnz = int(f["sidx"].shape[0])

            def asm():
                tl.tomo_lsqr_assemble_csr(f["npairs"], f["nper"], f["nnodes"], f["nz"], ft["lptr"], ft["lnode"], ft["lw"], f["klen"], ft["kj0"],
                                          ft["kern"], m - f["npairs"] * f["nper"], snnz, ft["sptr"], ft["sidx"], ft["svals"], nnz, rp_o, ci_o, va_o)
            for _ in range(2):
                asm()
            ea, eb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            ea.record()
            for _ in range(5):
                asm()
            eb.record()
            torch.cuda.synchronize()
            ams = ea.elapsed_time(eb) / 5
            out["factored"].update(assemble_csr_ms=ams, assemble_csr_gbs=(12.0 * nnz + 8.0 * (m + 1)) / (ams * 1e-3) / 1e9)
            del rp_o, ci_o, va_o
            torch.cuda.empty_cache()
    with ClockSampler(int(os.environ.get("LOCAL_RANK", "0"))) as clk:
        out["ms"], out["its"], out["launches"] = timed(step_device)
    out["clocks"] = clk.summary()
    if e2e:
        out["ms_e2e"], out["its_e2e"], _ = timed(step_host)
    # per-kernel durations, live: the same solve launched kernel by kernel with CUDA events around each launch on
    # the launching stream (library option "profile"); for the block solve these are the k_spmm8 / k_vec8 launches
    S.set(profile=1)
    for _ in range(2):
        step_device()
    nl = max(S.info("k_launches"), 1.0)
    out["k1_us"], out["k2_us"], out["k4_us"] = (1e3 * S.info(k) / nl for k in ("k1_ms", "k2_ms", "k4_ms"))
    S.set(profile=0)
    if both_modes:  # the other accumulation mode, for context
        S.set(accumulate=1 - args.accumulate)
        ms_o, its_o, _ = timed(step_device)
        out["other"] = {"accumulate": 1 - args.accumulate, "value": its_o / (ms_o * 1e-3), "ms_per_step": ms_o / steps}
        S.set(accumulate=args.accumulate)
    if args.compress and not factored:
        out["index_bytes"] = (S.info("compress_bytes_rows"), S.info("compress_bytes_cols"))
    S.close()
    return out


def run_sharded(args) -> dict | None:
    """`--shards P`: the configs[C] matrix cut into P nnz-balanced row blocks, solved by
    tomo_lsqr_solve_sharded.  One process: all P blocks on this GPU (the exchange is the identity; measures what the
    unrounded partials and the closing kernels cost).  Under torchrun with N ranks: P = N, rank r holds block r, the
    exchange is an NCCL all-gather; the total work is fixed (strong scaling)."""
    import numpy as np
    import torch
    import paper_2604_11920_b200 as tl
    import tomogen
    tl.load()
    world, rank, local = (int(os.environ.get(k, d)) for k, d in (("WORLD_SIZE", "1"), ("RANK", "0"), ("LOCAL_RANK", "0")))
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    s = tomogen.System(args.config)
    m, n, nnz = s.dims.m, s.dims.n, s.dims.nnz
    P = world if world > 1 else args.shards
    rp = s.rowptr()
    cuts = [0] + [int(np.searchsorted(rp, rp[-1] * q / P)) for q in range(1, P)] + [m]
    mine = [rank] if world > 1 else list(range(P))
    rp_d, ci_d, va_d = s.csr_cuda()
    b_all = torch.from_numpy(s.rhs(0)).cuda()
    blocks, bs = [], []
    for q in mine:
        a, c = cuts[q], cuts[q + 1]
        e0, e1 = int(rp[a]), int(rp[c])
        blocks.append(tl.TomoLsqr(c - a, n, (rp_d[a:c + 1] - e0).contiguous(), ci_d[e0:e1].clone(), va_d[e0:e1].clone()))
        bs.append(b_all[a:c].clone())
    del rp_d, ci_d, va_d
    blocks[0].set(accumulate=args.accumulate, check_every=args.check_every)
    cb = tl.make_allgather(dist, world) if world > 1 else None
    x = torch.empty(n, dtype=torch.float64, device="cuda")
    damp, atol, btol, max_iters = s.damp, s.solve["atol"], s.solve["btol"], s.solve["max_iters"]

    def step():
        return tl.tomo_lsqr_solve_sharded([B.h for B in blocks], bs, damp, atol, btol, max_iters, x, rank=rank, nranks=world, allgather=cb)

    for _ in range(args.warmup):
        step()
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(local) as clk:
        e0.record()
        its = sum(step().itn for _ in range(args.steps))
        e1.record()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    if dist is not None:
        t = torch.tensor([ms], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t[0])
        dist.destroy_process_group()
    if rank != 0:
        return None
    ab = algorithmic_bytes(m, n, nnz, 8)
    extra = P * 16 * n * 2 + P * 16 * n  # the unrounded column pairs: written by every block, read once by the closing kernel
    peak, peak_src = measured_peak_gbs()
    return {"metric": METRIC, "value": its / (ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": workload_name(s), "row_blocks": P, "blocks_per_gpu": len(mine),
                       "accumulate": "dd" if args.accumulate else "fast", "parallelism": f"row-sharded LSQR, {P} row blocks over {world} GPU(s)",
                       "exchange": "NCCL all-gather of (hi, lo) partials" if world > 1 else "none (all blocks on one GPU)",
                       "l2": "inputs larger than L2, no flush needed"},
            "effective_gbs": (ab["iteration"] + extra) * its / (ms * 1e-3) / 1e9, "clocks": clk.summary(),
            "roofline": {"bound": "hbm", "kernel": "k_wstream OP_K1S / OP_K2S over the row blocks + k_shard_combine (whole iteration, graph-less)",
                         "achieved": (ab["iteration"] + extra) * its / (ms * 1e-3) / 1e9, "peak": peak, "unit": "GB/s",
                         "frac": (ab["iteration"] + extra) * its / (ms * 1e-3) / 1e9 / peak, "traffic": None, "peak_source": peak_src},
            "gpu_launches": int(sum(B.info("kernels_enqueued") for B in blocks))}


def roofline_of(r: dict, peak: float, peak_src: str, compress: int) -> dict:
    """The roofline object of one measured workload: algorithmic bytes of the two sparse launches of an iteration
     over their live CUDA-event time."""
    m, n, nnz, nrhs, vb = r["m"], r["n"], r["nnz"], r["nrhs"], r["vbytes"]
    ab = algorithmic_bytes(m, n, nnz, vb) if nrhs == 1 else block_bytes(m, n, nnz, nrhs, vb)
    note = "general CSR byte count: (values + int32 index) per nonzero + pointers + vectors"
    if compress and "index_bytes" in r:  # NEXT-2: its own byte count, never mixed into the CSR roofline
        ab = dict(ab)
        ab["k1"] += int(r["index_bytes"][0]) - 4 * nnz
        ab["k2"] += int(r["index_bytes"][1]) - 4 * nnz
        note = "run-compressed index (option compress=1): values + measured compressed index bytes + pointers + vectors"
    if "factored" in r:
        # The factored operator is L2-resident (operator_bytes per product instead of 12 bytes per nonzero): bound by fp64
        # arithmetic.  Work per nonzero and product, in fp64 lane-instructions (an FMA counts once): dd 11 = the value
        # fl(W g) 1 + TwoProd 2 + TwoSum 6 + 2 error adds; fast 2 = the value + the FMA.  Peak as for the dd block solve.
        per = 11.0 if r.get("accumulate", 1) == 1 else 2.0
        two = r.get("two_stage", 1)
        contracted = r.get("nodal", 0) or ((two == 2) if r.get("accumulate", 1) == 1 else (two >= 1))
        sm_max = (r.get("clocks") or {}).get("sm_max_mhz") or 1965.0
        peak_t = 148 * 64 * sm_max * 1e6 / 1e12
        ach_t = per * nnz * 2 / ((r["k1_us"] + r["k2_us"]) * 1e-6) / 1e12
        if contracted:
            # two-stage contraction: the products per launch are entries x periods (+ the tiny depth stage), klen times fewer
            # than nonzeros; the kernels are bound by instruction issue and load latency around one (fast) or two (dd) products
            # per lane and step, so no pipe roofline is claimed: the line reports times only
            return {"bound": "alu", "kernel": "k_fac2_stage + k_fac2_rows (K1) / k_fac2_cols (K2): depth contraction per node, then W",
                    "achieved": None, "peak": None, "unit": "TFLOP/s", "frac": None, "traffic": None,
                    "note": "latency / issue bound: klen times fewer products than nonzeros; no roofline claim",
                    "operator_bytes_per_product": r["factored"]["operator_bytes"],
                    "k1_us": r["k1_us"], "k2_us": r["k2_us"], "k4_us": r["k4_us"]}
        return {"bound": "alu", "kernel": "k_fac_rows (K1) / k_fac_cols (K2): the two products of an iteration on the factored operator",
                "achieved": ach_t, "peak": peak_t, "unit": "TFLOP/s", "frac": ach_t / peak_t,
                "peak_source": "derived: 148 SMs x 64 fp64 lanes/clk x sm_max_mhz (fp64 lane-instructions/s, FMA counted once)",
                "work_per_launch": per * nnz, "traffic": None, "operator_bytes_per_product": r["factored"]["operator_bytes"],
                "k1_us": r["k1_us"], "k2_us": r["k2_us"], "k4_us": r["k4_us"]}
    spmv_bytes = ab["k1"] + ab["k2"]
    achieved = spmv_bytes / ((r["k1_us"] + r["k2_us"]) * 1e-6) / 1e9
    kern = ("k_wstream (K1: A v - alpha u + norm over CSR; K2: A^T u - beta v + norm over CSC), mean of the two launches of an iteration"
            if nrhs == 1 else
            "k_spmm8 (the same two products on len x 8 blocks, 8 right-hand sides per pass), mean of the two launches of a block iteration")
    if nrhs > 1 and r.get("accumulate", 1) == 1:
        # dd block solve: bound by the fp64 pipe, not by HBM.  Work = 10 fp64 instructions per (nonzero, side)
        # (TwoProd 2 + TwoSum 6 + 2 error adds; an FMA counts once); peak = 148 SMs x 64 fp64 lanes per clock x the SM's
        # maximum clock (B200: 40 TFLOP/s fp64 = 64 FMA lanes per SM and clock).
        sm_max = (r.get("clocks") or {}).get("sm_max_mhz") or 1965.0
        peak_t = 148 * 64 * sm_max * 1e6 / 1e12
        ach_t = 10.0 * nnz * nrhs * 2 / ((r["k1_us"] + r["k2_us"]) * 1e-6) / 1e12
        return {"bound": "alu", "kernel": kern, "achieved": ach_t, "peak": peak_t, "unit": "TFLOP/s", "frac": ach_t / peak_t,
                "peak_source": "derived: 148 SMs x 64 fp64 lanes/clk x sm_max_mhz (fp64 lane-instructions/s, FMA counted once)",
                "work_per_launch": 10.0 * nnz * nrhs, "traffic": None,
                "hbm_stream_gbs": achieved, "hbm_stream_frac_of_measured": achieved / peak, "bytes_per_launch_pair": spmv_bytes,
                "k1_us": r["k1_us"], "k2_us": r["k2_us"], "k4_us": r["k4_us"]}
    return {"bound": "hbm", "kernel": kern, "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
            "algorithmic_bytes_per_launch": spmv_bytes / 2, "byte_count": note, "peak_source": peak_src,
            "frac_of_8TBs": achieved / 8000.0, "bytes_per_launch_pair": spmv_bytes,
            "k1_us": r["k1_us"], "k2_us": r["k2_us"], "k4_us": r["k4_us"],
            "k1_gbs": ab["k1"] / (r["k1_us"] * 1e-6) / 1e9, "k2_gbs": ab["k2"] / (r["k2_us"] * 1e-6) / 1e9}


def run_ours(args) -> dict | None:
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
    r = measure(tl, torch, s, args, barrier, dist, world, args.steps, args.warmup, e2e=True, both_modes=args.both_modes)
    m, n, nnz, nrhs, vbytes = r["m"], r["n"], r["nnz"], r["nrhs"], r["vbytes"]
    ms, its = r["ms"], r["its"]

    also = {}
    if world == 1 and args.config == 1 and not args.no_also and torch.cuda.mem_get_info()[1] >= 150e9:
        # BASELINE.json north_star names configs[1] AND configs[2] for the >= 60 % target: the large system, 2 steps
        torch.cuda.empty_cache()
        s2 = tomogen.System(2)
        r2 = measure(tl, torch, s2, args, barrier, None, 1, 2, 3, e2e=False, both_modes=True)
        peak2, src2 = measured_peak_gbs()
        rf2 = roofline_of(r2, peak2, src2, args.compress)
        also["configs[2]"] = {"workload": workload_name(s2), "value": r2["its"] / (r2["ms"] * 1e-3), "unit": UNIT,
                              "accumulate": args.accumulate, "other_mode": r2.get("other"), "ms_per_step": r2["ms"] / 2, "steps": 2,
                              "warmup": 3, "k1_us": r2["k1_us"], "k2_us": r2["k2_us"], "k4_us": r2["k4_us"],
                              "achieved_gbs": rf2["achieved"] if rf2["bound"] == "hbm" else None, "frac": rf2["frac"], "frac_of_8TBs": rf2.get("frac_of_8TBs"),
                              "bound": rf2["bound"],
                              "create_ms": r2["create_ms"], "transpose_ms": r2["transpose_ms"], "clocks": r2["clocks"]}

    if world == 1 and args.config == 1 and not args.no_also and not args.factored and args.vals == "f64" and not args.compress:
        # the same system through the factored operator (NEXT-2, second form): its own line, never mixed into the CSR figures
        import copy
        fa = copy.copy(args)
        fa.factored = 1
        torch.cuda.empty_cache()
        rfac = measure(tl, torch, s, fa, barrier, None, 1, args.steps, args.warmup, e2e=False, both_modes=True)
        rff = roofline_of(rfac, *measured_peak_gbs(), 0)
        also["configs[1] factored"] = {"workload": workload_name(s), "operator": "factored (tomo_lsqr_create_factored): bitwise the CSR results in dd mode",
                                       "value": rfac["its"] / (rfac["ms"] * 1e-3), "unit": UNIT, "accumulate": args.accumulate,
                                       "other_mode": rfac.get("other"), "ms_per_step": rfac["ms"] / args.steps,
                                       "k1_us": rfac["k1_us"], "k2_us": rfac["k2_us"], "k4_us": rfac["k4_us"], "roofline": rff,
                                       "create_ms": rfac["create_ms"], "clocks": rfac["clocks"], **rfac["factored"]}
        # ... and with the depth contraction first in dd mode too (exact entries W*g, its own oracle: DESIGN.md F-fac3)
        fx = copy.copy(fa)
        fx.two_stage = 2
        rfx = measure(tl, torch, s, fx, barrier, None, 1, args.steps, args.warmup, e2e=False, both_modes=False)
        also["configs[1] factored, exact entries (two_stage=2)"] = {
            "workload": workload_name(s), "operator": "factored, entries W*g unrounded, depth contraction per node first; bitwise its own dd oracle",
            "value": rfx["its"] / (rfx["ms"] * 1e-3), "unit": UNIT, "accumulate": args.accumulate, "ms_per_step": rfx["ms"] / args.steps,
            "k1_us": rfx["k1_us"], "k2_us": rfx["k2_us"], "k4_us": rfx["k4_us"], "clocks": rfx["clocks"]}
        if "configs[2]" in also:
            # the large system through the factored operator (236 MB instead of 90 GB): rounded entries (the CSR bits) and exact entries
            s2f = tomogen.System(2)
            for key, two in (("configs[2] factored", 1), ("configs[2] factored, exact entries (two_stage=2)", 2)):
                f2 = copy.copy(fa)
                f2.two_stage = two
                r2f = measure(tl, torch, s2f, f2, barrier, None, 1, 2, 3, e2e=False, both_modes=(two == 1))
                also[key] = {"workload": workload_name(s2f), "value": r2f["its"] / (r2f["ms"] * 1e-3), "unit": UNIT, "accumulate": args.accumulate,
                             "other_mode": r2f.get("other"), "ms_per_step": r2f["ms"] / 2, "steps": 2, "warmup": 3,
                             "k1_us": r2f["k1_us"], "k2_us": r2f["k2_us"], "k4_us": r2f["k4_us"], "clocks": r2f["clocks"]}

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return None

    peak, peak_src = measured_peak_gbs()
    rf = roofline_of(r, peak, peak_src, args.compress)
    if rf["bound"] == "hbm":
        rf["traffic"], rf["traffic_source"] = ncu_traffic_bytes(args.config, nrhs)
    ab = algorithmic_bytes(m, n, nnz, vbytes) if nrhs == 1 else block_bytes(m, n, nnz, nrhs, vbytes)
    # bytes moved per second by the whole step: single side per iteration, block solve per BLOCK iteration (its / nrhs)
    eff = ab["iteration"] * (its / nrhs) / world / (ms * 1e-3) / 1e9
    out = {
        "metric": METRIC, "value": its / (ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": workload_config(s, args, its // max(1, args.steps * world), world),
        "effective_gbs": None if args.factored else eff,  # the factored operator does not move the CSR bytes
        "create_ms": r["create_ms"], "transpose_ms": r["transpose_ms"], "create_wall_ms": r["create_wall_ms"],
        "create_note": "create_ms / transpose_ms: CUDA events inside tomo_lsqr_create (kernels + its cudaMalloc calls); create_wall_ms: host clock around the call",
        "e2e": {"value": r["its_e2e"] / (r["ms_e2e"] * 1e-3), "unit": UNIT, "h2d_bytes_per_step": 8 * m * nrhs,
                "d2h_bytes_per_step": 8 * n * nrhs, "ms_per_step": r["ms_e2e"] / args.steps},
        "gpu_launches": int(r["launches"]),
        "clocks": r["clocks"],
        "roofline": rf,
    }
    if "factored" in r:
        out["factored"] = r["factored"]
    if "other" in r:
        out["other_mode"] = r["other"]
    if also:
        out["also"] = also
    if world == 1 and not args.no_cpu:
        import oracle
        iters = ref_iters_for(args)
        rp, ci, va = s.csr()
        t0 = time.perf_counter()
        ro = oracle.lsqr(m, n, rp, ci, va, s.rhs(0), damp=s.damp, atol=0.0, btol=0.0, max_iters=iters, mode=oracle.PLAIN)
        dt = time.perf_counter() - t0
        out["cpu_baseline"] = {"value": ro.itn / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
                               "sample": f"{iters} iterations (plus the init pass) of the full configs[{args.config}] system, plain fp64 mode"}
    if dist is not None:
        dist.destroy_process_group()
    return out


def relaunch_under_torchrun(args) -> int:
    """`python bench.py --gpus N` with N > 1 and no torchrun around it: start the N ranks here (one process per
    GPU, NCCL for the timing reduction) and pass their output through."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "INFO")  # communicator lines stay visible (rank count evidence)
    return subprocess.call(cmd, env=env)


def run_stub(args) -> dict | None:
    """TEST-ONLY (tests/test_bench_ranks.py, `--stub-step`): the rank plumbing of the N > 1 path — environment,
    process group (gloo, CPU), barrier, max / sum aggregation, rank 0 prints — with a step that does NO work and
    touches neither the GPU nor the library.  Its line says "stub": true and carries no value."""
    import torch
    import torch.distributed as dist
    world, rank = int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("RANK", "0"))
    if world > 1:
        dist.init_process_group("gloo")
        dist.barrier()
    ms, its, launches = 10.0 * (rank + 1), 7 * args.steps, 21.0 * args.steps
    if world > 1:
        ms, its, launches = aggregate_over_ranks(dist, ms, its, launches, device="cpu")
        dist.barrier()
        dist.destroy_process_group()
    if rank != 0:
        return None
    return {"stub": True, "metric": METRIC, "value": None, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "scaling": "weak", "stub_iterations": its, "stub_launches": launches}


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
    ap.add_argument("--one-mode", dest="both_modes", action="store_false", default=True, help="skip the other accumulation mode")
    ap.add_argument("--no-cpu", dest="no_cpu", action="store_true")
    ap.add_argument("--no-also", dest="no_also", action="store_true", help="skip the configs[2] lines attached to a configs[1] run")
    ap.add_argument("--solver", default="lsqr", choices=["lsqr", "lsmr"], help="lsqr (BASELINE metric) or lsmr (the paper's solver)")
    ap.add_argument("--vals", default="f64", choices=["f64", "f32"], help="storage type of the matrix values")
    ap.add_argument("--compress", type=int, default=0, choices=[0, 1], help="1: run-compressed index (NEXT-2), reported with its own byte count")
    ap.add_argument("--factored", type=int, default=0, choices=[0, 1], help="1: the factored operator (NEXT-2, second form), reported against the fp64 pipe")
    ap.add_argument("--two-stage", dest="two_stage", type=int, default=1, choices=[0, 1, 2],
                    help="factored operator: 0 per-entry products in both modes, 1 (default) depth contraction first in fast mode, "
                         "2 also in dd mode (exact entries W*g, DESIGN.md F-fac3)")
    ap.add_argument("--nodal", type=int, default=0, choices=[0, 1], help="factored operator: install a kernel table per lateral node (tomo_lsqr_set_nodal_kernels)")
    ap.add_argument("--row-cost", dest="row_cost", type=int, default=None, help="tuning: per-row weight of the element split")
    ap.add_argument("--pdl", type=int, default=None, choices=[0, 1], help="tuning: programmatic dependent launch between the kernels of an iteration")
    ap.add_argument("--shards", type=int, default=0, help="NEXT-3: P row blocks solved by tomo_lsqr_solve_sharded (one GPU: all blocks local; torchrun: one block per rank)")
    ap.add_argument("--stub-step", dest="stub", action="store_true", help="TEST-ONLY: rank plumbing with a step that does no work (no GPU)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        if int(os.environ.get("RANK", "0")) != 0:
            return
        print(json.dumps(run_reference(args)), flush=True)
        return
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        sys.exit(relaunch_under_torchrun(args))
    out = run_stub(args) if args.stub else (run_sharded(args) if args.shards > 0 else run_ours(args))
    if out is not None:
        print(json.dumps(out), flush=True)


if __name__ == "__main__":
    main()
