"""N > 1 plumbing of bench.py on CPU: world_size 2, gloo backend, 127.0.0.1 rendezvous.

The path does not shard ("replicas only"): every rank runs an independent replica of the
workload and the only exchange is the aggregation of the timing outside the timed region.  Checked here:
ranks draw different replicas of the same recipe, the aggregate is (max time, sum of pushes), and the
reference arm prints its line on rank 0 only."""
import json
import os
import socket
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = textwrap.dedent("""
    import json, os, sys
    sys.path.insert(0, %r)
    import numpy as np
    import torch
    import torch.distributed as dist
    import bench
    from paper_2603_24508_b200 import workloads
    rank, local_rank, world = bench.env_rank()
    dist.init_process_group("gloo")
    inp = workloads.make(1, nc=64, ppc=8, replica=rank)
    x = inp["species"][0]["x"]
    seconds, pushes = 1.0 + rank, float(len(x)) * 3
    t, p = bench.aggregate_over_ranks(dist, seconds, pushes, torch.device("cpu"))
    sums = [None] * world
    dist.all_gather_object(sums, float(np.sum(x)))
    print(json.dumps({"rank": rank, "world": world, "t": t, "p": p, "n": len(x), "sums": sums}), flush=True)
    dist.destroy_process_group()
""") % ROOT


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _spawn(code_or_args, world=2, script=True):
    port = _free_port()
    procs = []
    for rank in range(world):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), CUDA_VISIBLE_DEVICES="")
        cmd = [sys.executable, "-c", code_or_args] if script else [sys.executable] + code_or_args
        procs.append(subprocess.Popen(cmd, env=env, cwd=ROOT, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        out, err = p.communicate(timeout=300)
        assert p.returncode == 0, err[-2000:]
        outs.append(out)
    return outs


def test_replica_aggregation_world2_gloo():
    outs = _spawn(WORKER)
    recs = sorted((json.loads(o.strip().splitlines()[-1]) for o in outs), key=lambda r: r["rank"])
    assert [r["rank"] for r in recs] == [0, 1] and all(r["world"] == 2 for r in recs)
    n = recs[0]["n"]
    for r in recs:
        assert r["t"] == 2.0              # max over ranks of (1.0, 2.0)
        assert r["p"] == 2 * 3.0 * n      # sum over ranks
    assert recs[0]["sums"][0] != recs[0]["sums"][1], "ranks must draw independent replicas"


def test_reference_arm_prints_on_rank0_only():
    outs = _spawn([os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "2", "--warmup", "1",
                   "--config", "1"], script=False)
    lines = [o.strip() for o in outs]
    assert lines[1] == ""
    rec = json.loads(lines[0].splitlines()[-1])
    assert rec["impl"] == "reference" and rec["cpu_baseline"]["kind"].startswith("oracle") and rec["value"] > 0
    assert rec["e2e"]["h2d_bytes_per_step"] == 0 and rec["n_gpus"] == 2
    assert rec["cpu_baseline"]["cores"] >= 1 and rec["cpu_baseline"]["same_config"] is True and rec["steps"] == 2
