"""The N > 1 host logic of the row-sharded solve (tomo_lsqr_solve_sharded) on CPU: the exchange callback
the binding builds on torch.distributed (make_allgather) is called the way the library calls it — raw addresses, byte
counts — by two gloo ranks, and must deliver every rank's block at offset rank * bytes, for both message sizes of an
iteration (the 16-byte norm pair per block and the 16 n bytes of column pairs per block)."""
import os
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_allgather_callback_two_gloo_ranks(tmp_path):
    script = tmp_path / "ranks.py"
    script.write_text(textwrap.dedent(f"""
        import ctypes, json, sys
        sys.path.insert(0, {ROOT!r})
        import numpy as np, torch, torch.distributed as dist
        import paper_2604_11920_b200 as tl
        dist.init_process_group("gloo")
        rank, world = dist.get_rank(), dist.get_world_size()
        cb = tl.make_allgather(dist, world, device="cpu")
        ok = True
        n, nlocal = 1000, 2
        for pairs in (nlocal, nlocal * n):            # norm pairs, column pairs (double2 = 16 bytes each)
            send = np.arange(2 * pairs, dtype=np.float64) + 1e6 * rank
            recv = np.full(2 * pairs * world, np.nan)
            rc = cb(None, send.ctypes.data, recv.ctypes.data, 16 * pairs, None)
            want = np.concatenate([np.arange(2 * pairs, dtype=np.float64) + 1e6 * r for r in range(world)])
            ok = ok and rc == 0 and np.array_equal(recv, want)
        # a failing exchange is reported as a status, never raised through the C frame
        bad = tl.make_allgather(None, world, device="cpu")
        ok = ok and bad(None, send.ctypes.data, recv.ctypes.data, 16, None) == 1
        t = torch.tensor([1.0 if ok else 0.0])
        dist.all_reduce(t, op=dist.ReduceOp.MIN)
        if rank == 0:
            print(json.dumps(dict(ok=bool(t[0] == 1.0), world=world)))
        dist.destroy_process_group()
    """))
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
                          "127.0.0.1", "--master-port", "29741", str(script)], capture_output=True, text=True, env=env, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    import json
    d = json.loads([l for l in out.stdout.splitlines() if l.startswith("{")][-1])
    assert d == dict(ok=True, world=2)
