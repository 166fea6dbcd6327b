"""The N > 1 path on CPU: world_size 2, gloo, 127.0.0.1 (replicas only -- the process
group carries the barrier and the max-over-ranks of the step time, never field data)."""
import json
import os
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _torchrun(args, port):
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", OMP_NUM_THREADS="2")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr", "127.0.0.1",
           "--master-port", str(port)] + args
    return subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=600)


def test_dist_helper_max_over_ranks_and_replica_value(tmp_path):
    script = tmp_path / "probe.py"
    script.write_text(textwrap.dedent(f"""
        import json, os, sys
        sys.path.insert(0, {ROOT!r})
        import bench
        rank, world, local, barrier, vmax = bench._dist(backend="gloo")
        barrier()
        ms = vmax(10.0 * (rank + 1))          # rank 1 is the slow replica
        barrier()
        if rank == 0:
            print(json.dumps({{"world": world, "ms": ms, "value": bench.replica_value(world, 1000, 5, ms)}}))
        import torch.distributed as dist
        dist.destroy_process_group()
    """))
    r = _torchrun([str(script)], 29611)
    assert r.returncode == 0, r.stderr[-2000:]
    line = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(line) == 1, r.stdout  # rank 0 alone prints
    d = json.loads(line[0])
    assert d["world"] == 2 and d["ms"] == 20.0
    assert d["value"] == 2 * 1000 * 5 / 20e-3


def test_reference_arm_under_torchrun_rank0_only():
    r = _torchrun(["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0", "--workload", "c3",
                   "--ref-sites", "2000"], 29612)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, r.stdout
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
    assert d["metric"] == "smear-step site-updates/s" and d["higher_is_better"] is True
