"""Background runs of the CPU oracle for the GPU parity tests (test infrastructure).

The dd-mode oracle needs ~1 s per iteration on a config-1-sized system, so the full-size expected
values are computed in worker processes that start when the first GPU test asks for one and run
while the other GPU tests execute.  Workers call only ``tomogen`` (inputs) and ``oracle`` (expected
values); nothing here ever sees a CUDA result.
"""
from __future__ import annotations

import multiprocessing as mp
import os
from concurrent.futures import Future, ProcessPoolExecutor

import numpy as np

_pool: ProcessPoolExecutor | None = None
_jobs: dict[tuple, Future] = {}


def _available_ram() -> float:
    try:
        import psutil
        return float(psutil.virtual_memory().available)
    except Exception:
        for line in open("/proc/meminfo"):
            if line.startswith("MemAvailable:"):
                return 1024.0 * float(line.split()[1])
    return 0.0


def _run(cfg: int, rhs: int, mode: int, damp: float, atol: float, btol: float, max_iters: int, snapshots: tuple,
         f32_values: bool = False, solver: str = "lsqr", exact_entries: bool = False):
    import oracle
    import tomogen
    s = tomogen.System(cfg)
    if exact_entries:  # the factored operator with exact entries W*g as two-word values (oracle/factored.py expand_exact)
        from oracle import factored as ofac
        f = s.factored()
        rp, ci, va, lo = ofac.expand_exact(f["npairs"], f["nper"], f["nnodes"], f["nz"], f["lptr"], f["lnode"], f["lw"], f["kj0"], f["kern"],
                                           f["sptr"], f["sidx"], f["svals"])
        r = oracle.lsqr(s.dims.m, s.dims.n, rp, ci, va, s.rhs(rhs), damp=damp, atol=atol, btol=btol, max_iters=max_iters, mode=mode,
                        snapshots=snapshots, vals_lo=lo)
        return dict(x=r.x, itn=r.itn, istop=r.istop, r2hist=r.r2norm_hist, snapshots=r.snapshots)
    need = 13.0 * s.dims.nnz + 64.0 * (s.dims.m + s.dims.n)  # CSR (12 B/nnz) + vectors + slack
    if cfg == 2 and _available_ram() < need + 8e9:
        return dict(skipped=f"host RAM: {_available_ram() / 1e9:.0f} GB available, the config-2 CSR needs {need / 1e9:.0f} GB")
    rp, ci, va = s.csr()
    if f32_values:  # the fp32-storage path: the oracle sees the same rounded values, widened to fp64
        va = va.astype(np.float32).astype(np.float64)
    if solver == "lsmr":
        r = oracle.lsmr(s.dims.m, s.dims.n, rp, ci, va, s.rhs(rhs), damp=damp, atol=atol, btol=btol, max_iters=max_iters,
                        mode=mode, snapshots=snapshots)
        return dict(x=r.x, itn=r.itn, istop=r.istop, snapshots=r.snapshots)
    b = s.rhs(rhs)
    r = oracle.lsqr(s.dims.m, s.dims.n, rp, ci, va, b, damp=damp, atol=atol, btol=btol, max_iters=max_iters,
                    mode=mode, snapshots=snapshots)
    return dict(x=r.x, itn=r.itn, istop=r.istop, r1norm=r.r1norm, r2norm=r.r2norm, arnorm=r.arnorm, anorm=r.anorm,
                acond=r.acond, xnorm=r.xnorm, r2hist=r.r2norm_hist, arhist=r.arnorm_hist, snapshots=r.snapshots)


# every full-size oracle run the GPU suite needs; all are submitted together so that they overlap
def _all_jobs():
    import oracle
    import tomogen
    d1, d4 = tomogen.System(1).damp, tomogen.System(4).damp
    return {
        # config 1: tolerance run (BASELINE configs[1]); the same run yields x_50 as a snapshot
        ("cfg1_dd_tol",): (1, 0, oracle.DD, d1, 1e-6, 1e-6, 300, (10, 50)),
        ("cfg1_plain_50",): (1, 0, oracle.PLAIN, d1, 0.0, 0.0, 50, (10,)),
        # config 1 with fp32-rounded values (DESIGN.md R-f32 (i))
        ("cfg1_dd_f32_50",): (1, 0, oracle.DD, d1, 0.0, 0.0, 50, (), True),
        # config 1 by LSMR (NEXT-1)
        ("cfg1_lsmr_dd_50",): (1, 0, oracle.DD, d1, 0.0, 0.0, 50, (), False, "lsmr"),
        # config 1 through the factored operator with exact entries (two-stage dd mode, DESIGN.md F-fac3)
        ("cfg1_ddx_50",): (1, 0, oracle.DD, d1, 0.0, 0.0, 50, (10,), False, "lsqr", True),
        # config 4: skewed system, 100 iterations with x_50 as a snapshot
        ("cfg4_dd_100",): (4, 0, oracle.DD, d4, 0.0, 0.0, 100, (50,)),
        # config 2 (3.7e9 nnz): x_5 of the dd oracle at full size (~45 GB of host RAM, ~25 s per iteration)
        ("cfg2_dd_5",): (2, 0, oracle.DD, tomogen.System(2).damp, 0.0, 0.0, 5, (1, 2)),
        # config 3: every one of the 8 right-hand sides, 100 iterations as BASELINE.json states (x_50 as a snapshot)
        **{(f"cfg3_dd_rhs{r}",): (3, r, oracle.DD, d1, 0.0, 0.0, 100, (50,)) for r in range(8)},
        # config 1 by LSMR on the block path (columns 0 and 5 of config 3's right-hand sides)
        ("cfg3_lsmr_dd_rhs0",): (3, 0, oracle.DD, d1, 0.0, 0.0, 50, (), False, "lsmr"),
        ("cfg3_lsmr_dd_rhs5",): (3, 5, oracle.DD, d1, 0.0, 0.0, 50, (), False, "lsmr"),
    }


def start():
    global _pool
    if _pool is not None:
        return
    jobs = _all_jobs()
    # one worker per job if the host has the cores and the memory (a config-1-sized job holds ~3 GB, the
    # config-2 job ~50 GB); the long jobs are submitted first
    by_ram = int(max(1.0, (_available_ram() - 60e9) / 4e9))
    workers = max(1, min(len(jobs), (os.cpu_count() or 2) - 1, by_ram))
    _pool = ProcessPoolExecutor(max_workers=workers, mp_context=mp.get_context("spawn"))
    order = sorted(jobs.items(), key=lambda kv: -(kv[1][6] * (20 if kv[1][0] == 2 else 1)))
    for key, args in order:
        _jobs[key] = _pool.submit(_run, *args)


def get(name: str) -> dict:
    start()
    return _jobs[(name,)].result()


def shutdown():
    global _pool
    if _pool is not None:
        _pool.shutdown(wait=False, cancel_futures=True)
        _pool = None
