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


# ------------------------------------------------------------------------------------------------
# NEXT-4: decomposition along t (paper_1105_2279_b200/tsplit.py).  The plumbing -- who sends which slice to whom,
# which slices a launch covers, the all-reduce of the plaquette -- on two gloo ranks with the CPU oracle doing the
# arithmetic on each rank's local lattice: the ranks' own slabs, concatenated, must equal the oracle's step of the
# whole lattice BIT FOR BIT (every own site reads the same operand values in the same order), over several steps.
# ------------------------------------------------------------------------------------------------
def test_tsplit_two_gloo_ranks_equal_the_single_lattice_oracle(tmp_path):
    script = tmp_path / "tsplit_probe.py"
    script.write_text(textwrap.dedent(f"""
        import json, os, sys
        sys.path.insert(0, {ROOT!r}); sys.path.insert(0, os.path.join({ROOT!r}, "tests"))
        import numpy as np, torch
        import torch.distributed as dist
        import lattice_inputs as li, oracle as orc
        from paper_1105_2279_b200 import tsplit
        import tsplit_helpers as th
        dist.init_process_group("gloo")
        rank, world = dist.get_rank(), dist.get_world_size()
        gdims = (4, 4, 2, 8)                      # V3 = 32, four own slices per rank
        u = [t.numpy() for t in li.gauge_field(3, gdims, "f64", "near_unit")]
        comm = tsplit.DistComm()
        ts = tsplit.TSplit(th.OracleBackend(tsplit.local_dims(gdims, world), "n64"), comm, gdims)
        cur = [torch.from_numpy(th.scatter_no_halo(f, gdims, rank, world)) for f in u]   # halos poisoned with NaN
        nxt = [torch.full_like(f, float("nan")) for f in cur]
        want = u
        ok, plaq_err = True, 0.0
        for step in range(3):
            ts.smear_step(nxt, cur, 0.5, overlap=(step != 1))
            cur, nxt = nxt, cur
            want = orc.smear_step(gdims, want, 0.5, "n64")
            p = ts.plaquette_sum(cur) / (18.0 * np.prod(gdims))
            plaq_err = max(plaq_err, abs(p - orc.plaquette_avg(gdims, want, "n64")))
            for mu in range(4):
                own = cur[mu].numpy()[ts.be.v3:-ts.be.v3]
                ref = th.scatter(want[mu], gdims, rank, world)[ts.be.v3:-ts.be.v3]
                ok = ok and np.array_equal(own, ref)
        flags = [None] * world
        dist.all_gather_object(flags, (bool(ok), float(plaq_err)))
        if rank == 0:
            print(json.dumps({{"ok": [f[0] for f in flags], "plaq_err": max(f[1] for f in flags), "lt": ts.lt}}))
        dist.destroy_process_group()
    """))
    r = _torchrun([str(script)], 29613)
    assert r.returncode == 0, r.stderr[-3000:]
    d = json.loads([l for l in r.stdout.splitlines() if l.startswith("{")][0])
    assert d["ok"] == [True, True] and d["lt"] == 4
    assert d["plaq_err"] < 1e-13
