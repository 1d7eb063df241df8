"""Host logic of the N > 1 bench path on CPU (gloo, world_size 2): the path does not shard (DESIGN.md Sec. 9,
"replicas only"), so what there is to cover is the aggregation (all ranks' units / max-over-ranks time) and the
reference arm's "rank 0 alone runs and prints" rule."""
import json
import os
import re
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
# rank r processed (r + 1) * 1000 units in (r + 1) * 0.5 s of device time
value, tmax = bench.aggregate_replicas((rank + 1) * 1000.0, (rank + 1) * 0.5, world, torch.device("cpu"))
print(json.dumps(dict(rank=rank, value=value, tmax=tmax)), flush=True)
dist.destroy_process_group()
"""


def torchrun(args, env_extra=None, timeout=300):
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    env.update(env_extra or {})
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", "29731", *args]
    return subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=timeout)


def test_replica_aggregation_gloo_world2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    res = torchrun([str(script)])
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [json.loads(m) for m in re.findall(r"\{[^{}]*\}", res.stdout)]      # (two ranks may share a line)
    assert sorted(l["rank"] for l in lines) == [0, 1]
    for l in lines:                       # (1000 + 2000) units / max(0.5, 1.0) s on every rank
        assert l["tmax"] == 1.0 and l["value"] == 3000.0


def test_reference_arm_rank0_only_world2():
    res = torchrun(["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0",
                    "--config", "1", "--cpu-sample-n", "16"])
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [json.loads(l) for l in res.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1                # rank 0 alone prints; rank 1 exits 0 without work
    d = lines[0]
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
