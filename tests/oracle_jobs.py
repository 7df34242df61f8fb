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


def _run(cfg: int, rhs: int, mode: int, damp: float, atol: float, btol: float, max_iters: int, snapshots: tuple,
         f32_values: bool = False, solver: str = "lsqr"):
    import oracle
    import tomogen
    s = tomogen.System(cfg)
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
        # config 3: columns 0 and 7 of the 8 right-hand sides
        ("cfg3_dd_rhs0",): (3, 0, oracle.DD, d1, 0.0, 0.0, 50, ()),
        ("cfg3_dd_rhs7",): (3, 7, oracle.DD, d1, 0.0, 0.0, 50, ()),
        # config 4: skewed system, 100 iterations with x_50 as a snapshot
        ("cfg4_dd_100",): (4, 0, oracle.DD, d4, 0.0, 0.0, 100, (50,)),
    }


def start():
    global _pool
    if _pool is not None:
        return
    workers = max(1, min(7, (os.cpu_count() or 2) - 1))
    _pool = ProcessPoolExecutor(max_workers=workers, mp_context=mp.get_context("spawn"))
    for key, args in _all_jobs().items():
        _jobs[key] = _pool.submit(_run, *args)


def get(name: str) -> dict:
    start()
    return _jobs[(name,)].result()


def shutdown():
    global _pool
    if _pool is not None:
        _pool.shutdown(wait=False, cancel_futures=True)
        _pool = None
