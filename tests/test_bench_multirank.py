"""N > 1 path of bench.py on CPU: two ranks under torchrun with the gloo-free reference arm (rank 0 alone works and
prints, the other rank exits 0), and the max-over-ranks / sum-over-ranks aggregation the GPU arm uses, run with gloo
at world_size 2.  The hot path does not shard ("replicas only"): there is no data-path collective."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _torchrun(args, port):
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", OMP_NUM_THREADS="2")
    return subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                           "--master-addr", "127.0.0.1", "--master-port", str(port)] + args, cwd=ROOT, env=env,
                          capture_output=True, text=True, timeout=600)


def test_reference_arm_two_ranks_prints_one_line():
    r = _torchrun(["bench.py", "--impl", "reference", "--gpus", "2", "--config", "1", "--steps", "3", "--warmup", "1"],
                  29611)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["value"] > 0 and d["e2e"]["h2d_bytes_per_step"] == 0 and d["config"]["workload"] == "config1"


def test_rank_aggregation_with_gloo(tmp_path):
    script = tmp_path / "agg.py"
    script.write_text(
        "import os, sys, json\n"
        f"sys.path.insert(0, {ROOT!r})\n"
        "import torch, torch.distributed as dist\n"
        "import bench\n"
        "dist.init_process_group('gloo')\n"
        "r = dist.get_rank()\n"
        "tmax, temax, ntot = bench.aggregate(dist, torch.device('cpu'), ms=10.0 + 5 * r, ms_e2e=30.0 - 7 * r, n=1000 * (r + 1))\n"
        "if r == 0: print(json.dumps([tmax, temax, ntot]))\n"
        "dist.destroy_process_group()\n")
    r = _torchrun([str(script)], 29613)
    assert r.returncode == 0, r.stderr[-2000:]
    out = [l for l in r.stdout.splitlines() if l.startswith("[")]
    assert json.loads(out[0]) == [15.0, 30.0, 3000.0]   # max time over ranks, particles summed over ranks
