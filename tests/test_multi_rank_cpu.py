"""CPU-only, world_size 2 over gloo: the N > 1 path of bench.py.

The hot path does not shard (BASELINE north_star: one GPU, no collectives), so `bench.py --gpus N`
runs N independent replicas; the only multi-rank logic is the max-over-ranks step time and the
whole-job throughput.  Rank 0 of the reference arm alone prints, the other ranks exit without work.
"""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
import bench
dist.init_process_group("gloo", rank=int(os.environ["RANK"]), world_size=int(os.environ["WORLD_SIZE"]))
rank = dist.get_rank()
ms = 2.0 if rank == 0 else 5.0                       # rank 1 is the slow replica
step = bench.max_over_ranks(ms, dist, torch.device("cpu"))
val = bench.whole_job_value(128.0, dist.get_world_size(), step)
dist.barrier()
print(json.dumps({{"rank": rank, "step_ms": step, "value": val}}), flush=True)
dist.destroy_process_group()
"""


def run_two_ranks(code, port):
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, "-c", code], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True, cwd=ROOT))
    outs = []
    for p in procs:
        out, err = p.communicate(timeout=180)
        assert p.returncode == 0, err[-2000:]
        outs.append(out)
    return outs


def test_replicas_only_max_over_ranks_and_whole_job_value():
    outs = run_two_ranks(WORKER.format(root=ROOT), 29631)
    recs = [json.loads(o.strip().splitlines()[-1]) for o in outs]
    for r in recs:
        assert r["step_ms"] == 5.0                       # the slowest rank sets the job's step time
        assert r["value"] == pytest.approx(2 * 128.0 / 5e-3)   # both replicas' tokens over that time


def test_reference_arm_prints_on_rank0_only():
    """`bench.py --impl reference` under a 2-rank launch: rank 0 runs the CPU oracle and prints the one
    JSON line, rank 1 exits 0 without work (tiny fp32 workload so that this stays a CPU-suite test)."""
    outs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT="29632")
        p = subprocess.run([sys.executable, "bench.py", "--impl", "reference", "--gpus", "2", "--workload", "cfg1",
                            "--steps", "3", "--warmup", "3"], env=env, capture_output=True, text=True, cwd=ROOT,
                           timeout=300)
        assert p.returncode == 0, p.stderr[-2000:]
        outs.append(p.stdout.strip())
    line = json.loads(outs[0].splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle" and line["n_gpus"] == 2
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["value"] > 0
    assert outs[1] == ""
