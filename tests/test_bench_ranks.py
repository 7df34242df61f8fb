"""The N > 1 path of bench.py on CPU: two gloo ranks run the rank-aggregation logic (max of the times,
sum of the units) that the NCCL path uses on GPUs (replicas only, no data-path collective)."""
import os
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_two_gloo_ranks_aggregate_like_the_bench(tmp_path):
    script = tmp_path / "ranks.py"
    script.write_text(textwrap.dedent(f"""
        import os, sys, json
        sys.path.insert(0, {ROOT!r})
        import torch, torch.distributed as dist
        import bench
        dist.init_process_group("gloo")
        rank = dist.get_rank()
        # rank r "measured" (ms, iterations, launches); the aggregate must be max / sum / sum
        ms, its, launches = bench.aggregate_over_ranks(dist, 100.0 + 50.0 * rank, 300 + rank, 903.0, device="cpu")
        if rank == 0:
            print(json.dumps(dict(ms=ms, its=its, launches=launches, world=dist.get_world_size())))
        dist.destroy_process_group()
    """))
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
                          "127.0.0.1", "--master-port", "29731", str(script)], capture_output=True, text=True, env=env, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    import json
    line = [l for l in out.stdout.splitlines() if l.startswith("{")][-1]
    d = json.loads(line)
    assert d == dict(ms=150.0, its=601, launches=1806.0, world=2)
