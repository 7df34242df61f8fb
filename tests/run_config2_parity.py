#!/usr/bin/env python
"""Manual, long-running parity check of BASELINE configs[2] at full size (not collected by pytest):

    python tests/run_config2_parity.py [K]         # default K = 50; needs a B200 and ~110 GB of host RAM

Runs K LSQR iterations of the 3 855 360 x 655 360 system (nnz 3.7e9) in the order-independent
double-double mode with the CPU oracle (single thread: about 20 s per iteration) and through the C ABI on
the GPU, and compares x_k at k = 5, 10, 20, 30, 40, 50 element by element (relative L2 and bitwise).
Writes gpurun_out/cfg2_parity.json.  The result of the round-1 run is quoted in DESIGN.md §11.
"""
import json
import os
import sys
import time

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import oracle  # noqa: E402
import paper_2604_11920_b200 as tl  # noqa: E402
import tomogen  # noqa: E402


def main():
    K = int(sys.argv[1]) if len(sys.argv) > 1 else 50
    t0 = time.time()
    s = tomogen.System(2)
    d = s.dims
    rp, ci, va = s.csr()
    b = s.rhs(0)
    print("generated", d, "t %.1f" % (time.time() - t0), flush=True)
    S = tl.TomoLsqr(d.m, d.n, torch.from_numpy(rp).cuda(), torch.from_numpy(ci).cuda(), torch.from_numpy(va).cuda())
    S.set(accumulate=1)
    bd = torch.from_numpy(b).cuda()
    snaps = tuple(k for k in (5, 10, 20, 30, 40, 50) if k <= K)
    gx = {k: S.solve(bd, s.damp, 0.0, 0.0, k)[0].cpu().numpy() for k in snaps}
    print("gpu done t %.1f" % (time.time() - t0), flush=True)
    o = oracle.lsqr(d.m, d.n, rp, ci, va, b, damp=s.damp, atol=0.0, btol=0.0, max_iters=K, mode=oracle.DD, snapshots=snaps)
    out = {}
    for k in snaps:
        ox = o.snapshots[k] if k in o.snapshots else o.x
        out[k] = dict(rel=float(np.linalg.norm(gx[k] - ox) / np.linalg.norm(ox)), bitwise=bool(np.array_equal(gx[k], ox)))
        print("k", k, out[k], flush=True)
    os.makedirs(os.path.join(ROOT, "gpurun_out"), exist_ok=True)
    json.dump(dict(config=2, mode="dd", nnz=int(rp[-1]), results=out, seconds=time.time() - t0),
              open(os.path.join(ROOT, "gpurun_out", "cfg2_parity.json"), "w"))


if __name__ == "__main__":
    main()
