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


def test_bench_gpus_2_self_launches_its_ranks():
    """`python bench.py --gpus 2` as the driver invokes it (no torchrun around it) must start its own two ranks;
    here with the test-only stub step (no GPU): one JSON line, n_gpus = 2, max-over-ranks time, summed units."""
    import json
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "3", "--warmup", "3", "--stub-step"],
                         capture_output=True, text=True, env=env, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["stub"] is True and d["n_gpus"] == 2 and d["value"] is None
    assert d["ms_per_step"] == 20.0 / 3 and d["stub_iterations"] == 42 and d["stub_launches"] == 126.0
